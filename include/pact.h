/*
 * pact.h — C ABI of the B200-native forward/adjoint operator pair of arXiv 1709.02733
 * (Mitsuhashi et al., "A forward-adjoint operator pair based on the elastic wave equation for use
 * in transcranial photoacoustic computed tomography").  Citations are PAPER.md line + equation.
 *
 *   H   : p0 volume  -> receiver time series    H  = M' T'_{M-1} ... T'_1 T'_0   (Eq. 58)
 *   H^T : time series -> image                  H^T = T'_0^T ... T'_{M-1}^T M'^T (Eq. 59)
 *
 * One time step T'_m applies W' (Eq. 49), i.e. Eq. 46a-d in sequence
 * (PAPER.md:550-560): C-PML memory variables phi, particle velocity u, memory variables psi,
 * stress sigma, on a 4th-order staggered grid (Eq. 8).  T'_0 = tau' sets
 * sigma11 = sigma22 = sigma33 = -p0/3 (Eq. 21); M' samples
 * p^_m = -R (sigma11+sigma22+sigma33) by trilinear interpolation (Eq. 23/56, PAPER.md:216-219,
 * 634-637).  Readings of silent/garbled passages are listed in DESIGN.md.
 *
 * The library is fp32, single GPU (sm_100a), no CPU fallback.  All work is enqueued on the
 * CUDA stream given to pact_create; calls return without synchronising unless stated.  A
 * context is not thread-safe.  No exception or abort crosses this boundary: every entry point
 * returns an int (0 = PACT_OK, negative = error) except pact_destroy and pact_strerror.
 */
#ifndef PACT_H
#define PACT_H

#ifdef __cplusplus
extern "C" {
#endif

#define PACT_OK          0
#define PACT_EINVAL     -1  /* NULL pointer, non-positive size/h/dt/nt, n < 8 or 2*npml+8 > min(nx,ny,nz), bad PML constants */
#define PACT_ECFL       -2  /* dt * c_max > 6 h / (7 sqrt 3), c_max^2 = max over nodes of (lambda+2mu)/rho: the scheme is
                               unstable (reading G11).  A NECESSARY condition only: next to a much lighter
                               neighbour the staggered density is below the node's, so stay a few per cent under it
                               (the paper's and BASELINE's media run at <= 0.57 of the limit) */
#define PACT_ERCV       -3  /* a receiver lies outside [0,(n-1)h] on some axis */
#define PACT_EMATERIAL  -4  /* rho <= 0, mu < 0, lambda + 2 mu <= 0, alpha < 0 or a non-finite value */
#define PACT_ENOMEM     -5  /* device or host allocation failed */
#define PACT_ECUDA      -6  /* a CUDA call failed; pact_last_cuda_error() has the text */
#define PACT_ENUMERIC   -7  /* option "check_finite": the result holds a NaN or an Inf (the output buffer is still written) */

typedef struct pact_ctx pact_ctx;   /* opaque; owns every internal device buffer */

typedef struct {
    int    nx, ny, nz;     /* grid nodes; x fastest: idx = x + nx*(y + ny*z); x,y,z = paper directions 1,2,3 */
    double h;              /* grid pitch [m], isotropic */
    double dt;             /* time step [s] */
    int    nt;             /* = M: recorded samples p^_0 .. p^_{M-1}; M-1 applications of W' (Eq. 17) */
    int    npml;           /* C-PML thickness in cells on all six faces, inside the grid; 0 = none */
    double pml_R;          /* theoretical reflection coefficient of the profile, in (0,1); 0 = default 1e-4 */
    double pml_cref;       /* reference speed of the profile [m/s]; 0 = default: max c_l of the medium */
    double pml_beta_max;   /* CFS frequency shift beta at the PML entrance [rad/s] (Eq. 32) */
} pact_params;

/*
 * pact_create — build a context for one medium and receiver set (Eq. 5; Eq. 38
 * PAPER.md:416-420; trilinear rows R_l PAPER.md:219).
 *   out        [out] receives the context (NULL on error).
 *   prm        [in]  HOST pointer.
 *   lambda, mu, rho  [in] DEVICE pointers, float[nz][ny][nx], Lame parameters [Pa] and density
 *              [kg/m^3] at the grid nodes.
 *   alpha      [in]  DEVICE pointer, float[nz][ny][nx], diffusive absorption [1/s] (Eq. 3a,
 *              PAPER.md:52-53), or NULL for a lossless medium.
 *   rcv_xyz    [in]  HOST pointer, double[L][3], receiver positions [m]; node (0,0,0) at the origin.
 *   L          number of receivers (>= 0).
 *   cuda_stream  a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream), 0 = default stream.
 * The volumes and the receiver list are read once; only derived copies are kept, so the caller may
 * free them as soon as pact_create returns (it synchronises the stream before returning).
 * Errors: PACT_EINVAL, PACT_ECFL, PACT_ERCV, PACT_EMATERIAL, PACT_ENOMEM, PACT_ECUDA.
 */
int pact_create(pact_ctx** out, const pact_params* prm, const float* lambda, const float* mu,
                const float* rho, const float* alpha, const double* rcv_xyz, int L, void* cuda_stream);

/*
 * pact_forward — data = H p0 (Eq. 58).
 *   p0    [in]  DEVICE float[nz][ny][nx].
 *   data  [out] DEVICE float[nt][L], time-major (Eq. 12); overwritten.
 * Internal state is reset first, so calls are independent and repeatable bit for bit.
 * Asynchronous on the context's stream.  Errors: PACT_EINVAL, PACT_ECUDA.
 */
int pact_forward(pact_ctx* ctx, const float* p0, float* data);

/*
 * pact_adjoint — image = H^T data (Eq. 59-61; recursion of Eq. 27,
 * PAPER.md:240-249).
 *   data   [in]  DEVICE float[nt][L].
 *   image  [out] DEVICE float[nz][ny][nx]; overwritten.
 * The result is the exact transpose of pact_forward up to fp32 rounding; receivers that share
 * grid nodes are accumulated in a fixed order (no atomics), so results are deterministic.
 */
int pact_adjoint(pact_ctx* ctx, const float* data, float* image);

/*
 * Host-buffer variants: same operators with HOST pointers (pinned memory overlaps best, pageable
 * works).  The host<->device copies are enqueued on the context's stream around the operator and
 * the call returns after the result has landed in host memory (it synchronises the stream).
 */
int pact_forward_host(pact_ctx* ctx, const float* p0_host, float* data_host);
int pact_adjoint_host(pact_ctx* ctx, const float* data_host, float* image_host);

/*
 * pact_pgd — projected-gradient reconstruction with the pair, the use the paper builds it for (
 * BASELINE config 5):  p_{k+1} = P(p_k - step * H^T (H p_k - data)),  k = 0 .. iters-1,  P = max(0, .) if nonneg
 * else the identity.  Each iteration is one pact_forward, a fused residual kernel, one pact_adjoint and a fused
 * update-and-clamp kernel; nothing leaves the device inside the loop.
 *   p          [in/out] DEVICE float[nz][ny][nx]: p_0 on entry, p_iters on return.
 *   data       [in]  DEVICE float[nt][L].
 *   step       > 0; 1 / ||H||^2 (pact_power_iteration) makes the iteration non-expansive.
 *   resid_l2   [out] HOST double[iters] or NULL: ||H p_k - data||_2 of every iteration (fp64 accumulation,
 *              bit-reproducible).
 *   update_l2  [out] HOST double[iters] or NULL: ||p_{k+1} - p_k||_2.
 * Synchronises the stream once, at the end.  Errors: PACT_EINVAL, PACT_ENOMEM, PACT_ECUDA, PACT_ENUMERIC (option).
 */
int pact_pgd(pact_ctx* ctx, float* p, const float* data, double step, int iters, int nonneg,
             double* resid_l2, double* update_l2);

/*
 * pact_power_iteration — largest eigenvalue of H^T H, i.e. ||H||^2, by `iters` power iterations.
 *   v       [in/out] DEVICE float[nz][ny][nx]: non-zero start vector (the caller's seeded random numbers); on
 *           return the normalised iterate (approximate dominant right singular vector of H).
 *   sigma2  [out] HOST: ||H^T H v|| for the last normalised v.
 * Synchronises the stream.  Errors: PACT_EINVAL, PACT_ENOMEM, PACT_ECUDA, PACT_ENUMERIC (the result is not finite).
 */
int pact_power_iteration(pact_ctx* ctx, float* v, int iters, double* sigma2);

/* pact_destroy — free the context and everything it owns; NULL is allowed. */
void pact_destroy(pact_ctx* ctx);

/* pact_strerror — static text for an error code. */
const char* pact_strerror(int code);

/* pact_last_cuda_error — text of the last CUDA failure seen by this thread ("" if none). */
const char* pact_last_cuda_error(void);

/*
 * Options (all optional).  Unknown keys give PACT_EINVAL.
 *   "profile"  1: record CUDA events on the context's stream around the time loop and around
 *              sampled kernel launches of the next pact_forward/pact_adjoint; read them with
 *              pact_get_timing.  0 (default): no events.
 *   "variant"  step-kernel implementation: 0 = automatic (fused when the grid has at least one
 *              32 x 32 x 32 brick per SM, else plain), 1 = plain two-kernel in-place path, 2 = fused
 *              single-pass path (TMA-staged z-marching kernel, two state buffers).  A medium with
 *              3 lambda + 2 mu <= 0 somewhere always takes the plain path.
 *   "graph"    1: replay the time loop from a captured CUDA graph (default for small grids);
 *              0: launch directly; -1: automatic.
 *   "zchunk"   planes of z each CTA of the fused kernel marches over (0 = automatic).  Any value
 *              gives the same operator; it only changes how the grid is cut into CTAs.
 *   "chunk_long", "chunk_short"  tuning knobs of the automatic cut (0 = built-in 128 / 40): longest chunk of the
 *              first five sixths of a tile column, and of its last sixth (listed last, so that a launch ends on
 *              short bricks).  Any value gives the same operator.
 *   "split_launch"  1 (default): a fused time step runs its C-PML (slab) bricks and then its C-PML-free
 *              (interior) bricks as two launches on the context's stream, each timed on its own
 *              (PACT_K_*_SLAB / PACT_K_*_INTERIOR); 0: one persistent launch over the whole work list
 *              (PACT_K_*_FUSED).  Same bricks, same operator, same bits (measured within 2 % of each other).
 *   "acoustic"  -1 (default): a medium with mu = 0 everywhere (the paper's H^dagger_{mu=0}) takes
 *              the fused path's fluid-only kernels (one stress field + three velocities, 44 B per cell-step instead
 *              of 88); 0: always the elastic kernels.  Same results to rounding (1-2 ulp).
 *   "material_elision"  1 (default): the fused path fetches (tile, plane) material boxes that are one constant
 *              4-tuple (water around a skull) from an L2-resident palette plane instead of HBM; 0: always the
 *              real plane.  Bit-identical results.
 *   "check_finite"  1: pact_forward / pact_adjoint (and their _host forms) finish with a reduction over
 *              the output, synchronise the stream and return PACT_ENUMERIC if it holds a NaN or an Inf
 *              (a blow-up of the time stepping).  0 (default): no check, fully asynchronous.
 */
int pact_set_option(pact_ctx* ctx, const char* key, long long value);

/*
 * pact_get_timing — timings of the LAST pact_forward (op = 0) or pact_adjoint (op = 1) call made
 * with "profile" = 1.  Synchronises the context's stream.
 *   loop_ms      [out] device time of the whole time loop (IC / read-out excluded).
 *   kernel_ms    [out] double[PACT_K_COUNT]: mean device time of one launch of kernel kind k (CUDA events on
 *                      the context's stream around launches sampled evenly over the loop), 0 if
 *                      that kind did not run.  Kinds: PACT_K_*.
 *   launches     [out] long long[PACT_K_COUNT]: number of launches of kind k in that call.
 * Any output pointer may be NULL.  Errors: PACT_EINVAL (no profiled call of that op yet), PACT_ECUDA.
 */
#define PACT_K_FWD_VEL   0   /* Eq. 46a,b */
#define PACT_K_FWD_STR   1   /* Eq. 46c,d */
#define PACT_K_FWD_FUSED 2   /* Eq. 46a-d in one pass: the persistent launch of one fused time step */
#define PACT_K_ADJ_A     3   /* Eq. 61a,b,f : sigma_bar -> u_bar, psi_bar */
#define PACT_K_ADJ_B     4   /* Eq. 61c,d,e,g : u_bar -> sigma_bar, phi_bar */
#define PACT_K_ADJ_FUSED 5
#define PACT_K_RECV      6   /* Theta gather / Theta^T scatter, Eq. 56, 60 */
#define PACT_K_OTHER     7   /* tau^T read-out */
#define PACT_K_FWD_SLAB      8   /* option "split_launch": the C-PML bricks of a fused forward step */
#define PACT_K_FWD_INTERIOR  9   /*                        the C-PML-free bricks */
#define PACT_K_ADJ_SLAB     10
#define PACT_K_ADJ_INTERIOR 11
#define PACT_K_COUNT        12
int pact_get_timing(pact_ctx* ctx, int op, double* loop_ms, double* kernel_ms, long long* launches);

/* Bytes of device memory owned by the context. */
long long pact_device_bytes(const pact_ctx* ctx);

/*
 * pact_get_info — read-only facts about a context.  Keys:
 *   "elided_material_planes"  fraction of the fused path's (32 x 32 tile, z plane) material boxes that are
 *                             homogeneous and served from a palette plane (builds the fused path's tables)
 *   "num_sms"                 multiprocessors of the context's device
 *   "fluid"                   1 if mu = 0 everywhere in the medium
 *   "acoustic_path"           1 if the next operator call runs the fluid-only kernels
 * Errors: PACT_EINVAL (NULL or unknown key), PACT_ENOMEM, PACT_ECUDA.
 */
int pact_get_info(pact_ctx* ctx, const char* key, double* value);

#ifdef __cplusplus
}
#endif
#endif /* PACT_H */
