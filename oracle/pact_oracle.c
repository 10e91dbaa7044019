/*
 * oracle/pact_oracle.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, fp64 CPU implementation of the discrete forward operator H and its exact
 * transpose H^T of arXiv 1709.02733 (Mitsuhashi et al.), written step by step from the paper.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
 * call it.  It shares no code with the CUDA path (paper_1709_02733_b200/csrc) and neither
 * includes the other.
 *
 * What it computes (citations are PAPER.md line + equation):
 *   forward  H  = M' T'_{M-1} ... T'_1 T'_0            PAPER.md:644-645, Eq. 58
 *   adjoint  H^T= T'_0^T T'_1^T ... T'_{M-1}^T M'^T    PAPER.md:649-650, Eq. 59
 *   one step W' = Eq. 46a-d:  phi <- B phi + E sigma ; u <- J u + Phi sigma +
 *                 Gamma phi ; psi <- B~ psi + E~ u ; sigma <- sigma + Psi u + Delta psi
 *   derivative   = 4th-order staggered difference, Eq. 8
 *   J, Phi, Psi  = Eq. 7a-c
 *   C-PML a, b   = Eq. 38 with kappa = 1
 *   tau, Theta   = Eq. 21 / Eq. 23: sigma^ii = -p0/3,
 *                  p^_m = -R (sigma11+sigma22+sigma33)_m, R = trilinear interpolation rows
 *   adjoint recursion = Eq. 27 / 60, taken with Eq. 27b's indexing
 *
 * Readings of passages where the paper is silent or garbled are those of SURVEY.md 8(c)
 * (G1..G19) and are listed again in DESIGN.md:
 *   - sample positions: standard Virieux/Moczo cell (Fig. 1 is unreadable): normal stresses,
 *     lambda, mu, p0 at nodes (x,y,z); u1 at (x+1/2,y,z); u2 at (x,y+1/2,z); u3 at (x,y,z+1/2);
 *     s12 at (x+1/2,y+1/2,z); s13 at (x+1/2,y,z+1/2); s23 at (x,y+1/2,z+1/2);
 *   - samples outside the index range are zero (zero padding) for every field;
 *   - rho, alpha at velocity points: 2-point arithmetic mean, clamped at the last
 *     index; mu at shear points: 4-point harmonic mean, 0 if any of the four is 0;
 *   - PML profile: d = d0 xi^2, d0 = -3 c_ref ln(R) / (2 P h), beta = beta_max (1 - xi),
 *     xi = depth/P; a := 0 where d = 0.  PARITY UNPINNED by the paper (it gives no profile);
 *     the constants are parameters shared with the CUDA path as values, not code.
 *
 * Every floating-point operation is fp64.  Loops are plain; the only concession to run time is
 * `#pragma omp parallel for` over independent grid lines/points and storing the C-PML memory
 * variables only in the boundary slabs where their coefficient a is non-zero (elsewhere they
 * are identically zero by Eq. 37 with a = 0 and zero initial value).
 *
 * Build:  gcc -O2 -fopenmp -shared -fPIC -o liboracle.so pact_oracle.c -lm
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int nx, ny, nz;
    double h, dt;
    int nt, npml;
    double pml_R, pml_cref, pml_beta_max;
} oracle_params;

/* field ids for oracle_field() */
enum { F_U1 = 0, F_U2, F_U3, F_S11, F_S22, F_S33, F_S23, F_S13, F_S12, F_COUNT };

typedef struct oracle_state {
    oracle_params p;
    long N;
    int L;
    const float *lam, *mu, *rho, *alpha; /* borrowed, [nz][ny][nx]; alpha may be NULL */
    double *f[F_COUNT];                  /* u1,u2,u3,s11,s22,s33,s23,s13,s12 */
    /* C-PML 1-D tables per axis (0=x,1=y,2=z): "int" at s=i, "half" at s=i+1/2 */
    double *a_int[3], *b_int[3], *a_half[3], *b_half[3];
    /* memory variables, slab-confined along their derivative axis.
       phi[a][b]: memory of d_b sigma^{ab}, stored at u^a's position   (Eq. 41a, reading G5)
       psi[a][b]: memory of d_b u^a,        stored at sigma^{ab}'s pos (Eq. 41b, reading G5) */
    double *phi[3][3], *psi[3][3];
    int slabw;                           /* 2*npml+1 (0 if npml == 0) */
    /* receivers: 8 node indices and weights each (trilinear) */
    long *rnode;
    double *rw;
    double *tmp[3];                      /* scratch fields for the adjoint */
} oracle_state;

static const double C1 = 9.0 / 8.0, C2 = -1.0 / 24.0; /* Eq. 8 */

/* ------------------------------------------------------------------ indexing helpers */

static inline long IDX(const oracle_state *s, int x, int y, int z)
{
    return (long)x + (long)s->p.nx * ((long)y + (long)s->p.ny * (long)z);
}

/* zero padding outside the grid (reading G9) */
static inline double at(const oracle_state *s, const double *f, int x, int y, int z)
{
    if (x < 0 || y < 0 || z < 0 || x >= s->p.nx || y >= s->p.ny || z >= s->p.nz) return 0.0;
    return f[IDX(s, x, y, z)];
}

static inline int axis_len(const oracle_state *s, int b)
{
    return b == 0 ? s->p.nx : (b == 1 ? s->p.ny : s->p.nz);
}

/* position of index i inside the boundary slab of an axis of length n, or -1 */
static inline int slab_pos(int i, int n, int P)
{
    if (P <= 0) return -1;
    if (i < P) return i;
    if (i >= n - 1 - P) return i - (n - 1 - P) + P;
    return -1;
}

/* linear index of a memory variable of derivative axis b at grid point (x,y,z), or -1 */
static inline long mv_index(const oracle_state *s, int b, int x, int y, int z)
{
    const int P = s->p.npml, W = s->slabw;
    if (P <= 0) return -1;
    if (b == 0) {
        int q = slab_pos(x, s->p.nx, P);
        return q < 0 ? -1 : (long)q + (long)W * ((long)y + (long)s->p.ny * (long)z);
    } else if (b == 1) {
        int q = slab_pos(y, s->p.ny, P);
        return q < 0 ? -1 : (long)x + (long)s->p.nx * ((long)q + (long)W * (long)z);
    } else {
        int q = slab_pos(z, s->p.nz, P);
        return q < 0 ? -1 : (long)x + (long)s->p.nx * ((long)y + (long)s->p.ny * (long)q);
    }
}

static inline long mv_size(const oracle_state *s, int b)
{
    const long W = s->slabw;
    if (b == 0) return W * s->p.ny * (long)s->p.nz;
    if (b == 1) return (long)s->p.nx * W * s->p.nz;
    return (long)s->p.nx * s->p.ny * W;
}

/* ------------------------------------------------------------------ Eq. 8 differences */

/* D+ along axis b: integer -> half positions; result belongs to i+1/2 */
static inline double Dp(const oracle_state *s, const double *f, int b, int x, int y, int z)
{
    const int dx = (b == 0), dy = (b == 1), dz = (b == 2);
    return (C1 * (at(s, f, x + dx, y + dy, z + dz) - at(s, f, x, y, z)) +
            C2 * (at(s, f, x + 2 * dx, y + 2 * dy, z + 2 * dz) - at(s, f, x - dx, y - dy, z - dz))) /
           s->p.h;
}

/* D- along axis b: half -> integer positions; result belongs to i */
static inline double Dm(const oracle_state *s, const double *f, int b, int x, int y, int z)
{
    const int dx = (b == 0), dy = (b == 1), dz = (b == 2);
    return (C1 * (at(s, f, x, y, z) - at(s, f, x - dx, y - dy, z - dz)) +
            C2 * (at(s, f, x + dx, y + dy, z + dz) - at(s, f, x - 2 * dx, y - 2 * dy, z - 2 * dz))) /
           s->p.h;
}

/* ------------------------------------------------------------------ staggered material (Eq. 5) */

static inline int clampi(int i, int n) { return i < 0 ? 0 : (i >= n ? n - 1 : i); }

static inline double node(const oracle_state *s, const float *v, int x, int y, int z)
{
    return (double)v[IDX(s, clampi(x, s->p.nx), clampi(y, s->p.ny), clampi(z, s->p.nz))];
}

/* arithmetic 2-point mean at the velocity point displaced by +1/2 along axis b */
static inline double avg2(const oracle_state *s, const float *v, int b, int x, int y, int z)
{
    if (!v) return 0.0;
    return 0.5 * (node(s, v, x, y, z) + node(s, v, x + (b == 0), y + (b == 1), z + (b == 2)));
}

/* harmonic 4-point mean of mu at the shear point displaced by +1/2 along axes b and c */
static inline double mu_shear(const oracle_state *s, int b, int c, int x, int y, int z)
{
    const int bx = (b == 0), by = (b == 1), bz = (b == 2);
    const int cx = (c == 0), cy = (c == 1), cz = (c == 2);
    const double m0 = node(s, s->mu, x, y, z);
    const double m1 = node(s, s->mu, x + bx, y + by, z + bz);
    const double m2 = node(s, s->mu, x + cx, y + cy, z + cz);
    const double m3 = node(s, s->mu, x + bx + cx, y + by + cy, z + bz + cz);
    if (m0 == 0.0 || m1 == 0.0 || m2 == 0.0 || m3 == 0.0) return 0.0;
    return 4.0 / (1.0 / m0 + 1.0 / m1 + 1.0 / m2 + 1.0 / m3);
}

/* ------------------------------------------------------------------ C-PML tables (Eq. 38) */

static void pml_tables(const oracle_params *p, int n, double *a_int, double *b_int, double *a_half,
                       double *b_half)
{
    const int P = p->npml;
    for (int i = 0; i < n; ++i) {
        for (int half = 0; half < 2; ++half) {
            double a = 0.0, b = 1.0;
            if (P > 0) {
                const double sc = (double)i + (half ? 0.5 : 0.0);
                double depth = 0.0;
                if ((double)P - sc > depth) depth = (double)P - sc;
                if (sc - (double)(n - 1 - P) > depth) depth = sc - (double)(n - 1 - P);
                if (depth > 0.0) {
                    const double xi = depth / (double)P;
                    const double d0 = -3.0 * p->pml_cref * log(p->pml_R) / (2.0 * (double)P * p->h);
                    const double d = d0 * xi * xi;
                    const double beta = p->pml_beta_max * (1.0 - xi);
                    b = exp(-(d + beta) * p->dt);            /* Eq. 38a, kappa = 1 */
                    a = d > 0.0 ? d / (d + beta) * (b - 1.0) : 0.0; /* Eq. 38b */
                }
            }
            if (half) { a_half[i] = a; b_half[i] = b; } else { a_int[i] = a; b_int[i] = b; }
        }
    }
}

/* ------------------------------------------------------------------ life cycle */

void oracle_destroy(oracle_state *s)
{
    if (!s) return;
    for (int i = 0; i < F_COUNT; ++i) free(s->f[i]);
    for (int b = 0; b < 3; ++b) {
        free(s->a_int[b]); free(s->b_int[b]); free(s->a_half[b]); free(s->b_half[b]);
        for (int a = 0; a < 3; ++a) { free(s->phi[a][b]); free(s->psi[a][b]); }
        free(s->tmp[b]);
    }
    free(s->rnode); free(s->rw);
    free(s);
}

static void zero_state(oracle_state *s)
{
    for (int i = 0; i < F_COUNT; ++i) memset(s->f[i], 0, sizeof(double) * (size_t)s->N);
    if (s->slabw)
        for (int a = 0; a < 3; ++a)
            for (int b = 0; b < 3; ++b) {
                memset(s->phi[a][b], 0, sizeof(double) * (size_t)mv_size(s, b));
                memset(s->psi[a][b], 0, sizeof(double) * (size_t)mv_size(s, b));
            }
}

/* rcv: L x 3 doubles (x,y,z metres; node (0,0,0) at the origin).  Returns NULL on bad input. */
oracle_state *oracle_create(const oracle_params *prm, const float *lam, const float *mu,
                            const float *rho, const float *alpha, const double *rcv, int L)
{
    if (!prm || !lam || !mu || !rho || L < 0 || (L > 0 && !rcv)) return NULL;
    if (prm->nx < 2 || prm->ny < 2 || prm->nz < 2 || prm->nt < 1 || prm->npml < 0) return NULL;
    if (!(prm->h > 0.0) || !(prm->dt > 0.0)) return NULL;
    if (prm->npml > 0) {
        int nmin = prm->nx < prm->ny ? prm->nx : prm->ny;
        if (prm->nz < nmin) nmin = prm->nz;
        if (2 * prm->npml + 1 > nmin) return NULL; /* the two slabs must not overlap */
    }
    oracle_state *s = (oracle_state *)calloc(1, sizeof(*s));
    if (!s) return NULL;
    s->p = *prm;
    s->N = (long)prm->nx * prm->ny * prm->nz;
    s->L = L;
    s->lam = lam; s->mu = mu; s->rho = rho; s->alpha = alpha;
    s->slabw = prm->npml > 0 ? 2 * prm->npml + 1 : 0;
    for (int i = 0; i < F_COUNT; ++i) {
        s->f[i] = (double *)calloc((size_t)s->N, sizeof(double));
        if (!s->f[i]) { oracle_destroy(s); return NULL; }
    }
    for (int b = 0; b < 3; ++b) {
        const int n = axis_len(s, b);
        s->a_int[b] = (double *)calloc((size_t)n, sizeof(double));
        s->b_int[b] = (double *)calloc((size_t)n, sizeof(double));
        s->a_half[b] = (double *)calloc((size_t)n, sizeof(double));
        s->b_half[b] = (double *)calloc((size_t)n, sizeof(double));
        pml_tables(prm, n, s->a_int[b], s->b_int[b], s->a_half[b], s->b_half[b]);
        if (s->slabw)
            for (int a = 0; a < 3; ++a) {
                s->phi[a][b] = (double *)calloc((size_t)mv_size(s, b), sizeof(double));
                s->psi[a][b] = (double *)calloc((size_t)mv_size(s, b), sizeof(double));
                if (!s->phi[a][b] || !s->psi[a][b]) { oracle_destroy(s); return NULL; }
            }
    }
    /* trilinear rows R_l: i0 = floor(r/h) clamped to [0, n-2], t = r/h - i0 */
    s->rnode = (long *)calloc((size_t)(8 * (L > 0 ? L : 1)), sizeof(long));
    s->rw = (double *)calloc((size_t)(8 * (L > 0 ? L : 1)), sizeof(double));
    for (int l = 0; l < L; ++l) {
        int i0[3];
        double t[3];
        for (int b = 0; b < 3; ++b) {
            const int n = axis_len(s, b);
            double fpos = rcv[3 * l + b] / prm->h;
            /* outside [0,(n-1)h] is an error; 1e-9 cells of slack absorbs the rounding of r/h */
            if (!(fpos >= -1e-9) || !(fpos <= (double)(n - 1) + 1e-9)) { oracle_destroy(s); return NULL; }
            if (fpos < 0.0) fpos = 0.0;
            if (fpos > (double)(n - 1)) fpos = (double)(n - 1);
            int i = (int)floor(fpos);
            if (i > n - 2) i = n - 2;
            if (i < 0) i = 0;
            i0[b] = i;
            t[b] = fpos - (double)i;
        }
        for (int c = 0; c < 8; ++c) {
            const int cx = c & 1, cy = (c >> 1) & 1, cz = (c >> 2) & 1;
            s->rnode[8 * l + c] = IDX(s, i0[0] + cx, i0[1] + cy, i0[2] + cz);
            s->rw[8 * l + c] = (cx ? t[0] : 1.0 - t[0]) * (cy ? t[1] : 1.0 - t[1]) *
                               (cz ? t[2] : 1.0 - t[2]);
        }
    }
    return s;
}

double *oracle_field(oracle_state *s, int id) { return (id >= 0 && id < F_COUNT) ? s->f[id] : NULL; }
int oracle_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------ forward pieces */

/* tau, Eq. 21 (reading G1): sigma11 = sigma22 = sigma33 = -p0/3, all else 0
   (memory variables zero initially: PAPER.md:623) */
void oracle_set_p0(oracle_state *s, const double *p0)
{
    zero_state(s);
    for (long i = 0; i < s->N; ++i) {
        const double v = -p0[i] / 3.0;
        s->f[F_S11][i] = v; s->f[F_S22][i] = v; s->f[F_S33][i] = v;
    }
}

/* Theta, Eq. 23/56: p^_l = -R_l (s11 + s22 + s33) */
void oracle_sample(const oracle_state *s, double *out)
{
    for (int l = 0; l < s->L; ++l) {
        double acc = 0.0;
        for (int c = 0; c < 8; ++c) {
            const long n = s->rnode[8 * l + c];
            acc += s->rw[8 * l + c] * (s->f[F_S11][n] + s->f[F_S22][n] + s->f[F_S33][n]);
        }
        out[l] = -acc;
    }
}

/* Eq. 37 + Eq. 36 (kappa = 1): mem <- b mem + a d ; return d + mem.  Outside the slab a = 0 and
   mem = 0, so the return value is d. */
static inline double cpml_fwd(double *mem, long mi, double a, double b, double d)
{
    if (mi < 0) return d;
    mem[mi] = b * mem[mi] + a * d;
    return d + mem[mi];
}

/* Eq. 46a + 46b: phi update, then u <- J u + Phi sigma + Gamma phi */
static void velocity_update(oracle_state *s)
{
    const int nx = s->p.nx, ny = s->p.ny, nz = s->p.nz;
    const double dt = s->p.dt;
    double *u1 = s->f[F_U1], *u2 = s->f[F_U2], *u3 = s->f[F_U3];
    const double *s11 = s->f[F_S11], *s22 = s->f[F_S22], *s33 = s->f[F_S33];
    const double *s23 = s->f[F_S23], *s13 = s->f[F_S13], *s12 = s->f[F_S12];
#pragma omp parallel for collapse(2) schedule(static)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                const long i = IDX(s, x, y, z);
                const long mx = mv_index(s, 0, x, y, z), my = mv_index(s, 1, x, y, z),
                           mz = mv_index(s, 2, x, y, z);
                double t;
                /* u1 at (x+1/2, y, z): d1 s11 (half_x), d2 s12 (int_y), d3 s13 (int_z) */
                t = cpml_fwd(s->phi[0][0], mx, s->a_half[0][x], s->b_half[0][x], Dp(s, s11, 0, x, y, z)) +
                    cpml_fwd(s->phi[0][1], my, s->a_int[1][y], s->b_int[1][y], Dm(s, s12, 1, x, y, z)) +
                    cpml_fwd(s->phi[0][2], mz, s->a_int[2][z], s->b_int[2][z], Dm(s, s13, 2, x, y, z));
                u1[i] = (1.0 - dt * avg2(s, s->alpha, 0, x, y, z)) * u1[i] +
                        dt / avg2(s, s->rho, 0, x, y, z) * t;
                /* u2 at (x, y+1/2, z): d1 s12 (int_x), d2 s22 (half_y), d3 s23 (int_z) */
                t = cpml_fwd(s->phi[1][0], mx, s->a_int[0][x], s->b_int[0][x], Dm(s, s12, 0, x, y, z)) +
                    cpml_fwd(s->phi[1][1], my, s->a_half[1][y], s->b_half[1][y], Dp(s, s22, 1, x, y, z)) +
                    cpml_fwd(s->phi[1][2], mz, s->a_int[2][z], s->b_int[2][z], Dm(s, s23, 2, x, y, z));
                u2[i] = (1.0 - dt * avg2(s, s->alpha, 1, x, y, z)) * u2[i] +
                        dt / avg2(s, s->rho, 1, x, y, z) * t;
                /* u3 at (x, y, z+1/2): d1 s13 (int_x), d2 s23 (int_y), d3 s33 (half_z) */
                t = cpml_fwd(s->phi[2][0], mx, s->a_int[0][x], s->b_int[0][x], Dm(s, s13, 0, x, y, z)) +
                    cpml_fwd(s->phi[2][1], my, s->a_int[1][y], s->b_int[1][y], Dm(s, s23, 1, x, y, z)) +
                    cpml_fwd(s->phi[2][2], mz, s->a_half[2][z], s->b_half[2][z], Dp(s, s33, 2, x, y, z));
                u3[i] = (1.0 - dt * avg2(s, s->alpha, 2, x, y, z)) * u3[i] +
                        dt / avg2(s, s->rho, 2, x, y, z) * t;
            }
}

/* Eq. 46c + 46d: psi update, then sigma <- sigma + Psi u + Delta psi (Psi: Eq. 7c) */
static void stress_update(oracle_state *s)
{
    const int nx = s->p.nx, ny = s->p.ny, nz = s->p.nz;
    const double dt = s->p.dt;
    const double *u1 = s->f[F_U1], *u2 = s->f[F_U2], *u3 = s->f[F_U3];
    double *s11 = s->f[F_S11], *s22 = s->f[F_S22], *s33 = s->f[F_S33];
    double *s23 = s->f[F_S23], *s13 = s->f[F_S13], *s12 = s->f[F_S12];
#pragma omp parallel for collapse(2) schedule(static)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                const long i = IDX(s, x, y, z);
                const long mx = mv_index(s, 0, x, y, z), my = mv_index(s, 1, x, y, z),
                           mz = mv_index(s, 2, x, y, z);
                /* normal stresses at the node: d_k u^k with "int" tables */
                const double e11 = cpml_fwd(s->psi[0][0], mx, s->a_int[0][x], s->b_int[0][x], Dm(s, u1, 0, x, y, z));
                const double e22 = cpml_fwd(s->psi[1][1], my, s->a_int[1][y], s->b_int[1][y], Dm(s, u2, 1, x, y, z));
                const double e33 = cpml_fwd(s->psi[2][2], mz, s->a_int[2][z], s->b_int[2][z], Dm(s, u3, 2, x, y, z));
                const double lam = (double)s->lam[i], mu = (double)s->mu[i];
                const double div = e11 + e22 + e33;
                s11[i] += dt * (lam * div + 2.0 * mu * e11);
                s22[i] += dt * (lam * div + 2.0 * mu * e22);
                s33[i] += dt * (lam * div + 2.0 * mu * e33);
                /* s12 at (x+1/2, y+1/2, z): d2 u1 (half_y) + d1 u2 (half_x) */
                double g;
                g = cpml_fwd(s->psi[0][1], my, s->a_half[1][y], s->b_half[1][y], Dp(s, u1, 1, x, y, z)) +
                    cpml_fwd(s->psi[1][0], mx, s->a_half[0][x], s->b_half[0][x], Dp(s, u2, 0, x, y, z));
                s12[i] += dt * mu_shear(s, 0, 1, x, y, z) * g;
                /* s13 at (x+1/2, y, z+1/2): d3 u1 (half_z) + d1 u3 (half_x) */
                g = cpml_fwd(s->psi[0][2], mz, s->a_half[2][z], s->b_half[2][z], Dp(s, u1, 2, x, y, z)) +
                    cpml_fwd(s->psi[2][0], mx, s->a_half[0][x], s->b_half[0][x], Dp(s, u3, 0, x, y, z));
                s13[i] += dt * mu_shear(s, 0, 2, x, y, z) * g;
                /* s23 at (x, y+1/2, z+1/2): d3 u2 (half_z) + d2 u3 (half_y) */
                g = cpml_fwd(s->psi[1][2], mz, s->a_half[2][z], s->b_half[2][z], Dp(s, u2, 2, x, y, z)) +
                    cpml_fwd(s->psi[2][1], my, s->a_half[1][y], s->b_half[1][y], Dp(s, u3, 1, x, y, z));
                s23[i] += dt * mu_shear(s, 1, 2, x, y, z) * g;
            }
}

/* one application of W' (Eq. 49 = Eq. 46a-d in sequence) */
void oracle_step(oracle_state *s)
{
    velocity_update(s);
    stress_update(s);
}

/* H p0 (Eq. 58).  p0: N doubles; data: nt x L doubles, time-major (Eq. 12). */
int oracle_forward(oracle_state *s, const double *p0, double *data)
{
    if (!s || !p0 || (!data && s->L > 0)) return -1;
    oracle_set_p0(s, p0);
    for (int m = 0; m < s->p.nt; ++m) {
        oracle_sample(s, data + (size_t)m * (size_t)s->L);
        if (m == s->p.nt - 1) break;
        oracle_step(s);
    }
    return 0;
}

/* ------------------------------------------------------------------ adjoint pieces */

/* Literal transposes of the 1-D difference matrices of Eq. 8 under zero padding: for every
   row i of D (the stencil that produces out[i] from in[..]) scatter d[i] times the row's
   entries into the positions the row reads.  Lines along the axis are independent. */
static void add_DT(const oracle_state *s, double *out, const double *d, int b, int plus)
{
    const int nx = s->p.nx, ny = s->p.ny, nz = s->p.nz;
    const int n = axis_len(s, b);
    const int n1 = b == 0 ? ny : nx, n2 = b == 2 ? ny : nz; /* the two other axes */
    const long stride = b == 0 ? 1 : (b == 1 ? nx : (long)nx * ny);
    const double ih = 1.0 / s->p.h;
#pragma omp parallel for collapse(2) schedule(static)
    for (int q2 = 0; q2 < n2; ++q2)
        for (int q1 = 0; q1 < n1; ++q1) {
            long base;
            if (b == 0) base = IDX(s, 0, q1, q2);
            else if (b == 1) base = IDX(s, q1, 0, q2);
            else base = IDX(s, q1, q2, 0);
            for (int i = 0; i < n; ++i) {
                const double v = d[base + i * stride];
                if (v == 0.0) continue;
                /* row i of D+: +C1 at i+1, -C1 at i, +C2 at i+2, -C2 at i-1
                   row i of D-: +C1 at i,   -C1 at i-1, +C2 at i+1, -C2 at i-2 */
                const int o = plus ? 0 : -1;
                const int jp1 = i + 1 + o, jm1 = i + o, jp2 = i + 2 + o, jm2 = i - 1 + o;
                if (jp1 >= 0 && jp1 < n) out[base + jp1 * stride] += C1 * ih * v;
                if (jm1 >= 0 && jm1 < n) out[base + jm1 * stride] -= C1 * ih * v;
                if (jp2 >= 0 && jp2 < n) out[base + jp2 * stride] += C2 * ih * v;
                if (jm2 >= 0 && jm2 < n) out[base + jm2 * stride] -= C2 * ih * v;
            }
        }
}

/* transpose of cpml_fwd as a map (mem, d) -> (mem', out = d + mem'):
     mem' = b mem + a d ; out = d + mem'
   adjoint, given incoming bar_out (g) and bar_mem:
     t = bar_mem + g ; bar_d = g + a t ; bar_mem = b t */
static inline double cpml_adj(double *mem, long mi, double a, double b, double g)
{
    if (mi < 0) return g;
    const double t = mem[mi] + g;
    mem[mi] = b * t;
    return g + a * t;
}

/* Theta'^T p^_m added to the adjoint state: sigma_bar^ii[node] += -w p^_m[l] */
void oracle_adj_source(oracle_state *s, const double *pm)
{
    for (int l = 0; l < s->L; ++l)
        for (int c = 0; c < 8; ++c) {
            const long n = s->rnode[8 * l + c];
            const double v = -s->rw[8 * l + c] * pm[l];
            s->f[F_S11][n] += v; s->f[F_S22][n] += v; s->f[F_S33][n] += v;
        }
}

/* W'^T = S1^T S2^T S3^T S4^T with W' = S4 S3 S2 S1 (S1: 46a, S2: 46b, S3: 46c, S4: 46d);
   equals Eq. 61a-g.  The state arrays hold the adjoint variables. */
void oracle_adj_step(oracle_state *s)
{
    const int nx = s->p.nx, ny = s->p.ny, nz = s->p.nz;
    const double dt = s->p.dt;
    double *u1 = s->f[F_U1], *u2 = s->f[F_U2], *u3 = s->f[F_U3];
    double *s11 = s->f[F_S11], *s22 = s->f[F_S22], *s33 = s->f[F_S33];
    double *s23 = s->f[F_S23], *s13 = s->f[F_S13], *s12 = s->f[F_S12];
    double *t0 = s->tmp[0], *t1 = s->tmp[1], *t2 = s->tmp[2];

    /* ---- S4^T, S3^T: normal stresses -> d_bar of e11, e22, e33 at nodes */
#pragma omp parallel for collapse(2) schedule(static)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                const long i = IDX(s, x, y, z);
                const double lam = (double)s->lam[i], mu = (double)s->mu[i];
                const double tr = s11[i] + s22[i] + s33[i];
                const double e11 = dt * (lam * tr + 2.0 * mu * s11[i]);
                const double e22 = dt * (lam * tr + 2.0 * mu * s22[i]);
                const double e33 = dt * (lam * tr + 2.0 * mu * s33[i]);
                t0[i] = cpml_adj(s->psi[0][0], mv_index(s, 0, x, y, z), s->a_int[0][x], s->b_int[0][x], e11);
                t1[i] = cpml_adj(s->psi[1][1], mv_index(s, 1, x, y, z), s->a_int[1][y], s->b_int[1][y], e22);
                t2[i] = cpml_adj(s->psi[2][2], mv_index(s, 2, x, y, z), s->a_int[2][z], s->b_int[2][z], e33);
            }
    add_DT(s, u1, t0, 0, 0); /* e11 = D-x u1 */
    add_DT(s, u2, t1, 1, 0); /* e22 = D-y u2 */
    add_DT(s, u3, t2, 2, 0); /* e33 = D-z u3 */

    /* ---- shear stresses.  s12: g = D+y u1 (psi12, half_y) + D+x u2 (psi21, half_x) */
#pragma omp parallel for collapse(2) schedule(static)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                const long i = IDX(s, x, y, z);
                const double g = dt * mu_shear(s, 0, 1, x, y, z) * s12[i];
                t0[i] = cpml_adj(s->psi[0][1], mv_index(s, 1, x, y, z), s->a_half[1][y], s->b_half[1][y], g);
                t1[i] = cpml_adj(s->psi[1][0], mv_index(s, 0, x, y, z), s->a_half[0][x], s->b_half[0][x], g);
            }
    add_DT(s, u1, t0, 1, 1);
    add_DT(s, u2, t1, 0, 1);
    /* s13: g = D+z u1 (psi13, half_z) + D+x u3 (psi31, half_x) */
#pragma omp parallel for collapse(2) schedule(static)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                const long i = IDX(s, x, y, z);
                const double g = dt * mu_shear(s, 0, 2, x, y, z) * s13[i];
                t0[i] = cpml_adj(s->psi[0][2], mv_index(s, 2, x, y, z), s->a_half[2][z], s->b_half[2][z], g);
                t1[i] = cpml_adj(s->psi[2][0], mv_index(s, 0, x, y, z), s->a_half[0][x], s->b_half[0][x], g);
            }
    add_DT(s, u1, t0, 2, 1);
    add_DT(s, u3, t1, 0, 1);
    /* s23: g = D+z u2 (psi23, half_z) + D+y u3 (psi32, half_y) */
#pragma omp parallel for collapse(2) schedule(static)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                const long i = IDX(s, x, y, z);
                const double g = dt * mu_shear(s, 1, 2, x, y, z) * s23[i];
                t0[i] = cpml_adj(s->psi[1][2], mv_index(s, 2, x, y, z), s->a_half[2][z], s->b_half[2][z], g);
                t1[i] = cpml_adj(s->psi[2][1], mv_index(s, 1, x, y, z), s->a_half[1][y], s->b_half[1][y], g);
            }
    add_DT(s, u2, t0, 2, 1);
    add_DT(s, u3, t1, 1, 1);

    /* ---- S2^T, S1^T.  u1: t = (D+x s11 | phi11 half_x) + (D-y s12 | phi12 int_y) + (D-z s13 | phi13 int_z) */
#pragma omp parallel for collapse(2) schedule(static)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                const long i = IDX(s, x, y, z);
                const double ut = u1[i];
                const double g = dt / avg2(s, s->rho, 0, x, y, z) * ut;
                u1[i] = (1.0 - dt * avg2(s, s->alpha, 0, x, y, z)) * ut;
                t0[i] = cpml_adj(s->phi[0][0], mv_index(s, 0, x, y, z), s->a_half[0][x], s->b_half[0][x], g);
                t1[i] = cpml_adj(s->phi[0][1], mv_index(s, 1, x, y, z), s->a_int[1][y], s->b_int[1][y], g);
                t2[i] = cpml_adj(s->phi[0][2], mv_index(s, 2, x, y, z), s->a_int[2][z], s->b_int[2][z], g);
            }
    add_DT(s, s11, t0, 0, 1);
    add_DT(s, s12, t1, 1, 0);
    add_DT(s, s13, t2, 2, 0);
    /* u2: (D-x s12 | int_x) + (D+y s22 | half_y) + (D-z s23 | int_z) */
#pragma omp parallel for collapse(2) schedule(static)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                const long i = IDX(s, x, y, z);
                const double ut = u2[i];
                const double g = dt / avg2(s, s->rho, 1, x, y, z) * ut;
                u2[i] = (1.0 - dt * avg2(s, s->alpha, 1, x, y, z)) * ut;
                t0[i] = cpml_adj(s->phi[1][0], mv_index(s, 0, x, y, z), s->a_int[0][x], s->b_int[0][x], g);
                t1[i] = cpml_adj(s->phi[1][1], mv_index(s, 1, x, y, z), s->a_half[1][y], s->b_half[1][y], g);
                t2[i] = cpml_adj(s->phi[1][2], mv_index(s, 2, x, y, z), s->a_int[2][z], s->b_int[2][z], g);
            }
    add_DT(s, s12, t0, 0, 0);
    add_DT(s, s22, t1, 1, 1);
    add_DT(s, s23, t2, 2, 0);
    /* u3: (D-x s13 | int_x) + (D-y s23 | int_y) + (D+z s33 | half_z) */
#pragma omp parallel for collapse(2) schedule(static)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                const long i = IDX(s, x, y, z);
                const double ut = u3[i];
                const double g = dt / avg2(s, s->rho, 2, x, y, z) * ut;
                u3[i] = (1.0 - dt * avg2(s, s->alpha, 2, x, y, z)) * ut;
                t0[i] = cpml_adj(s->phi[2][0], mv_index(s, 0, x, y, z), s->a_int[0][x], s->b_int[0][x], g);
                t1[i] = cpml_adj(s->phi[2][1], mv_index(s, 1, x, y, z), s->a_int[1][y], s->b_int[1][y], g);
                t2[i] = cpml_adj(s->phi[2][2], mv_index(s, 2, x, y, z), s->a_half[2][z], s->b_half[2][z], g);
            }
    add_DT(s, s13, t0, 0, 0);
    add_DT(s, s23, t1, 1, 0);
    add_DT(s, s33, t2, 2, 1);
}

/* tau^T (Eq. 27c / 60c with tau of Eq. 21): image = -(s11+s22+s33)/3 */
void oracle_adj_image(const oracle_state *s, double *image)
{
    for (long i = 0; i < s->N; ++i)
        image[i] = -(s->f[F_S11][i] + s->f[F_S22][i] + s->f[F_S33][i]) / 3.0;
}

static int ensure_tmp(oracle_state *s)
{
    for (int k = 0; k < 3; ++k)
        if (!s->tmp[k]) {
            s->tmp[k] = (double *)calloc((size_t)s->N, sizeof(double));
            if (!s->tmp[k]) return -1;
        }
    return 0;
}

void oracle_adj_begin(oracle_state *s) { zero_state(s); ensure_tmp(s); }

/* H^T p^ (Eq. 59 / Eq. 27 with 27b's indexing, reading G4):
   v = 0 ; for m = M-1 .. 0: [if m < M-1: v <- W'^T v] ; v += Theta'^T p^_m ; image = tau^T v */
int oracle_adjoint(oracle_state *s, const double *data, double *image)
{
    if (!s || !image || (!data && s->L > 0)) return -1;
    zero_state(s);
    if (ensure_tmp(s)) return -2;
    for (int m = s->p.nt - 1; m >= 0; --m) {
        if (m < s->p.nt - 1) oracle_adj_step(s);
        oracle_adj_source(s, data + (size_t)m * (size_t)s->L);
    }
    oracle_adj_image(s, image);
    return 0;
}

/* ------------------------------------------------------------------ introspection for tests */

/* staggered coefficients as the oracle uses them: kind 0 rho_b, 1 alpha_b (b = axis),
   2 mu at the shear point of axes (b, c) */
double oracle_coef(const oracle_state *s, int kind, int b, int c, int x, int y, int z)
{
    if (kind == 0) return avg2(s, s->rho, b, x, y, z);
    if (kind == 1) return avg2(s, s->alpha, b, x, y, z);
    return mu_shear(s, b, c, x, y, z);
}

/* copy the PML tables of axis b: out = [a_int | b_int | a_half | b_half], each of length n_b */
void oracle_pml_tables(const oracle_state *s, int b, double *out)
{
    const int n = axis_len(s, b);
    memcpy(out, s->a_int[b], sizeof(double) * (size_t)n);
    memcpy(out + n, s->b_int[b], sizeof(double) * (size_t)n);
    memcpy(out + 2 * n, s->a_half[b], sizeof(double) * (size_t)n);
    memcpy(out + 3 * n, s->b_half[b], sizeof(double) * (size_t)n);
}

/* sum of squares of all memory variables (phi if which == 0, psi otherwise) */
double oracle_memvar_energy(const oracle_state *s, int which)
{
    double acc = 0.0;
    if (!s->slabw) return 0.0;
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) {
            const double *m = which == 0 ? s->phi[a][b] : s->psi[a][b];
            const long n = mv_size(s, b);
            for (long i = 0; i < n; ++i) acc += m[i] * m[i];
        }
    return acc;
}

/* trilinear row l: 8 node indices and weights */
void oracle_receiver_row(const oracle_state *s, int l, long *nodes, double *w)
{
    memcpy(nodes, s->rnode + 8 * l, 8 * sizeof(long));
    memcpy(w, s->rw + 8 * l, 8 * sizeof(double));
}
