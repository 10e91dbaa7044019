// pact.cu — host side of libpact: the C ABI of include/pact.h.
//
// Everything numerical happens in the kernels of kernels_*.cuh; this file validates arguments,
// derives the tables that depend only on the parameters (C-PML profiles, trilinear rows), owns the
// device buffers and enqueues the time loops of Eq. 58 (forward) and Eq. 59/27 (adjoint).
// There is no CPU fallback: every entry point either enqueues CUDA work or returns an error.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include <cuda_runtime.h>

#include "../../include/pact.h"
#include "common.cuh"
#include "kernels_io.cuh"
#include "kernels_plain.cuh"
#include "kernels_fused.cuh"
#include "kernels_pgd.cuh"
#include "kernels_acoustic.cuh"


// ------------------------------------------------------------------------------------------------
static thread_local char g_cuda_err[512] = "";

static int cuda_fail(cudaError_t e, const char* what, int line)
{
    snprintf(g_cuda_err, sizeof(g_cuda_err), "%s (pact.cu:%d): %s", what, line, cudaGetErrorString(e));
    return e == cudaErrorMemoryAllocation ? PACT_ENOMEM : PACT_ECUDA;
}
#define CK(call)                                                          \
    do {                                                                  \
        cudaError_t e_ = (call);                                          \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call, __LINE__);     \
    } while (0)

#define MAX_SAMPLES 48

struct EvPair { cudaEvent_t a, b; };

struct pact_ctx {
    pact_params prm;
    cudaStream_t stream;
    cudaStream_t cap_stream;   // private stream for graph capture (the legacy default stream cannot capture)
    long long N;             // nx ny nz
    int L;
    int pitch, py, pz;       // padded box extents
    long long box;           // elements of one padded field
    long long mbox;          // elements of one padded material field: PACT_NPAL palette planes follow its pz planes
    unsigned char* d_mflag;  // [tiles][nzp] material-plane flags of the fused path (kernels_fused.cuh)
    int nzp;
    double elided;           // fraction of (tile, plane) material boxes the fused path fetches from a palette plane
    int elide;               // option "material_elision"
    DevGrid g;
    RcvTables rcv;
    IoArgs* d_io;
    std::vector<void*> allocs;
    long long bytes;
    // zeroed at the start of every operator call: state fields + memory variables (contiguous)
    float* state_base;
    long long state_bytes;
    float* scratch_base;     // adjoint scratch of the plain variant, allocated on first use
    // fused variant (kernels_fused.cuh): second state buffer, ping-pong memory variables, TMA maps
    bool fluid;              // mu = 0 everywhere: the fused path runs its acoustic specialisation (option "acoustic")
    int acoustic;            // option: -1 automatic (acoustic kernels when the medium is a fluid), 0 never
    bool bulk_positive;      // 3 lambda + 2 mu > 0 everywhere (the fused adjoint carries C sigma_bar and divides by it)
    bool fused_ready;
    DevGrid g2;              // view of state buffer B for the I/O kernels
    float* stateB_base;
    long long stateB_bytes;
    CUtensorMap tmS40[2], tmS36[2], tmS32[2], tmM37, tmM36, tmL;
    FusedArgs fa;
    int zchunk;              // planes per CTA along z (0 = auto)
    int chunk_long, chunk_short;   // automatic chunking: longest long / short chunk (options "chunk_long", "chunk_short")
    // work list of the fused launch, heaviest first: [0, nslab) bricks that touch a C-PML slab (they run the C-PML
    // code), [nslab, nwork) bricks whose every tap (those of the adjoint included) stays clear of the slabs
    int4* d_work;
    int nwork, nslab;
    int work_zc;             // zchunk value the list was built for (-1 = not built)
    long long work_cap;
    unsigned int* d_queue;   // [2] ticket counter + exit counter of the persistent launch
    int split_launch;        // diagnostic option: slab bricks and interior bricks as two launches, timed apart
    float* mvbuf[2][18];     // fused memory variables, two sets (read / written alternate every step)
    float* mgbuf[2][6];      // the same storage as the elastic kernels see it: six groups of three interleaved components
    // host-buffer variants and pact_pgd / pact_power_iteration (gradient and residual)
    float* d_vol;            // [N]
    float* d_dat;            // [nt][L]
    double* d_partial;       // [PGD_MAXBLOCKS] block partial sums of the fp64 norms
    double* d_norms;         // [PGD_MAXNORMS] norms left on the device by a pact_pgd / pact_power_iteration call
    // options
    int variant;             // 0 auto, 1 plain, 2 tiled
    int use_graph;           // -1 auto, 0 off, 1 on
    int profile;
    int check_finite;        // option: reduce the output of every operator call to a NaN/Inf flag (synchronises)
    unsigned int* d_flag;    // that flag
    int num_sms;             // cudaDevAttrMultiProcessorCount of the context's device
    cudaGraphExec_t gexec[2];     // forward / adjoint loop
    int gexec_variant[2];
    // timing of the last profiled call
    // timing of the last profiled forward ([0]) / adjoint ([1]) call
    cudaEvent_t ev_loop[2][2];
    std::vector<EvPair> samples[2][PACT_K_COUNT];
    size_t used[2][PACT_K_COUNT];
    long long launches[2][PACT_K_COUNT];
    bool have_timing[2];
};

static int dev_alloc(pact_ctx* c, void** p, size_t bytes)
{
    if (bytes == 0) bytes = 16;
    cudaError_t e = cudaMalloc(p, bytes);
    if (e != cudaSuccess) { *p = nullptr; return cuda_fail(e, "cudaMalloc", __LINE__); }
    c->allocs.push_back(*p);
    c->bytes += (long long)bytes;
    return PACT_OK;
}

template <typename T>
static int upload(pact_ctx* c, T** dst, const std::vector<T>& v)
{
    int rc = dev_alloc(c, (void**)dst, v.size() * sizeof(T));
    if (rc) return rc;
    if (!v.empty()) CK(cudaMemcpyAsync(*dst, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice, c->stream));
    CK(cudaStreamSynchronize(c->stream));   // v may be a temporary
    return PACT_OK;
}

// ---- C-PML profiles, Eq. 38 with kappa = 1; profile shape: DESIGN.md reading G8
//   depth = max(P - s, s - (n-1-P), 0) cells, xi = depth/P, d = d0 xi^2, d0 = -3 c_ref ln R/(2 P h),
//   beta = beta_max (1 - xi);  b = exp(-(d + beta) dt),  a = d/(d + beta) (b - 1), a = 0 where d = 0.
static void cpml_profile(const pact_params& p, int n, bool half, std::vector<float>& a, std::vector<float>& b)
{
    a.assign(n, 0.0f);
    b.assign(n, 1.0f);
    const int P = p.npml;
    if (P <= 0) return;
    const double d0 = -3.0 * p.pml_cref * std::log(p.pml_R) / (2.0 * P * p.h);
    for (int i = 0; i < n; ++i) {
        const double s = i + (half ? 0.5 : 0.0);
        const double depth = std::max(std::max((double)P - s, s - (double)(n - 1 - P)), 0.0);
        if (depth <= 0.0) continue;
        const double xi = depth / P;
        const double d = d0 * xi * xi, beta = p.pml_beta_max * (1.0 - xi);
        const double bb = std::exp(-(d + beta) * p.dt);
        b[i] = (float)bb;
        a[i] = d > 0.0 ? (float)(d / (d + beta) * (bb - 1.0)) : 0.0f;
    }
}

static void free_graphs(pact_ctx* c)
{
    for (int k = 0; k < 2; ++k)
        if (c->gexec[k]) { cudaGraphExecDestroy(c->gexec[k]); c->gexec[k] = nullptr; }
}

extern "C" void pact_destroy(pact_ctx* c)
{
    if (!c) return;
    cudaStreamSynchronize(c->stream);
    free_graphs(c);
    if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
    for (int op = 0; op < 2; ++op) {
        for (int k = 0; k < PACT_K_COUNT; ++k)
            for (auto& s : c->samples[op][k]) { cudaEventDestroy(s.a); cudaEventDestroy(s.b); }
        for (int k = 0; k < 2; ++k) if (c->ev_loop[op][k]) cudaEventDestroy(c->ev_loop[op][k]);
    }
    for (void* p : c->allocs) cudaFree(p);
    delete c;
}

extern "C" const char* pact_strerror(int code)
{
    switch (code) {
    case PACT_OK: return "ok";
    case PACT_EINVAL: return "invalid argument";
    case PACT_ECFL: return "time step exceeds the stability limit dt*c_max <= 6h/(7 sqrt 3)";
    case PACT_ERCV: return "receiver outside the grid";
    case PACT_EMATERIAL: return "invalid material value";
    case PACT_ENOMEM: return "out of memory";
    case PACT_ECUDA: return "CUDA error";
    case PACT_ENUMERIC: return "the result holds a NaN or an Inf";
    default: return "unknown error";
    }
}

extern "C" const char* pact_last_cuda_error(void) { return g_cuda_err; }

extern "C" long long pact_device_bytes(const pact_ctx* c) { return c ? c->bytes : 0; }

static int ensure_fused(pact_ctx* c);
static int resolve_variant(const pact_ctx* c);
static bool use_acoustic(const pact_ctx* c);

extern "C" int pact_get_info(pact_ctx* c, const char* key, double* value)
{
    if (!c || !key || !value) return PACT_EINVAL;
    if (!strcmp(key, "elided_material_planes")) {
        int rc = ensure_fused(c);
        if (rc) return rc;
        *value = c->elided;
        return PACT_OK;
    }
    if (!strcmp(key, "num_sms")) { *value = c->num_sms; return PACT_OK; }
    if (!strcmp(key, "fluid")) { *value = c->fluid ? 1.0 : 0.0; return PACT_OK; }
    if (!strcmp(key, "acoustic_path")) { *value = (use_acoustic(c) && resolve_variant(c) == 2) ? 1.0 : 0.0; return PACT_OK; }
    return PACT_EINVAL;
}

// ------------------------------------------------------------------------------------------------
// pact_create
static int create_impl(pact_ctx* c, const pact_params* prm, const float* lam, const float* mu,
                       const float* rho, const float* alpha, const double* rcv_xyz, int L)
{
    const int nx = prm->nx, ny = prm->ny, nz = prm->nz, P = prm->npml;
    c->N = (long long)nx * ny * nz;
    c->L = L;
    c->pitch = ((nx + PACT_HALO_X + 4 + 31) / 32) * 32;
    c->py = ny + 2 * PACT_HALO_Y;
    c->pz = nz + 2 * PACT_HALO_Z;
    c->box = (long long)c->pitch * c->py * c->pz;
    DevGrid& g = c->g;
    g.nx = nx; g.ny = ny; g.nz = nz; g.P = P; g.W = P > 0 ? 2 * P + 1 : 0;
    g.sy = c->pitch; g.sz = (long long)c->pitch * c->py;
    const long long org = (long long)PACT_HALO_Z * g.sz + (long long)PACT_HALO_Y * g.sy + PACT_HALO_X;

    // ---- 1. scan the caller's volumes: validity and c_max (stability bound, reading G11)
    unsigned int* d_scan = nullptr;
    int rc = dev_alloc(c, (void**)&d_scan, 2 * sizeof(unsigned int));
    if (rc) return rc;
    CK(cudaMemsetAsync(d_scan, 0, 2 * sizeof(unsigned int), c->stream));
    {
        int dev = 0;
        CK(cudaGetDevice(&dev));
        CK(cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, dev));
        if (c->num_sms <= 0) c->num_sms = 148;
    }
    k_scan_materials<<<c->num_sms * 8, 256, 0, c->stream>>>(lam, mu, rho, alpha, c->N, d_scan, d_scan + 1);
    CK(cudaGetLastError());
    unsigned int h_scan[2];
    CK(cudaMemcpyAsync(h_scan, d_scan, sizeof(h_scan), cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    if (h_scan[0] & 31u) return PACT_EMATERIAL;
    c->bulk_positive = !(h_scan[0] & 32u);
    c->fluid = !(h_scan[0] & 64u);
    float c2;
    memcpy(&c2, &h_scan[1], sizeof(float));
    const double cmax = std::sqrt((double)c2);
    if (prm->npml > 0) {   // documented defaults of include/pact.h
        if (c->prm.pml_R == 0.0) c->prm.pml_R = 1e-4;
        if (c->prm.pml_cref == 0.0) c->prm.pml_cref = cmax;
    }
    const double limit = 6.0 * prm->h / (7.0 * std::sqrt(3.0));   // DESIGN.md reading G11
    if (prm->dt * cmax > limit * (1.0 + 1e-6)) return PACT_ECFL;

    // ---- 2. receivers: trilinear rows R_l and their node-sorted transpose
    std::vector<long long> node8((size_t)8 * L);
    std::vector<float> w8((size_t)8 * L);
    {
        const int n[3] = {nx, ny, nz};
        for (int l = 0; l < L; ++l) {
            int i0[3];
            double t[3];
            for (int b = 0; b < 3; ++b) {
                double f = rcv_xyz[3 * l + b] / prm->h;
                if (!(f >= -1e-9) || !(f <= (double)(n[b] - 1) + 1e-9)) return PACT_ERCV;
                f = std::min(std::max(f, 0.0), (double)(n[b] - 1));
                int i = (int)std::floor(f);
                i = std::min(std::max(i, 0), n[b] - 2);
                i0[b] = i;
                t[b] = f - i;
            }
            for (int k = 0; k < 8; ++k) {
                const int cx = k & 1, cy = (k >> 1) & 1, cz = (k >> 2) & 1;
                node8[8 * l + k] = (long long)(i0[2] + cz) * g.sz + (long long)(i0[1] + cy) * g.sy + (i0[0] + cx);
                w8[8 * l + k] = (float)((cx ? t[0] : 1.0 - t[0]) * (cy ? t[1] : 1.0 - t[1]) * (cz ? t[2] : 1.0 - t[2]));
            }
        }
    }
    std::vector<long long> tnode;
    std::vector<int> row_ptr(1, 0), trcv;
    std::vector<float> tw;
    {
        std::vector<std::pair<long long, int>> e((size_t)8 * L);   // (node, entry id) ; entry id = 8 l + k
        for (int q = 0; q < 8 * L; ++q) e[q] = {node8[q], q};
        std::sort(e.begin(), e.end());   // by node, then by receiver (ascending): fixed summation order
        for (size_t q = 0; q < e.size(); ++q) {
            if (q == 0 || e[q].first != e[q - 1].first) {
                if (q) row_ptr.push_back((int)q);
                tnode.push_back(e[q].first);
            }
            trcv.push_back(e[q].second / 8);
            tw.push_back(w8[e[q].second]);
        }
        if (!e.empty()) row_ptr.push_back((int)e.size());
    }
    c->rcv.L = L;
    c->rcv.nnodes = (int)tnode.size();
    long long* d_ll; float* d_f; int* d_i;
    if ((rc = upload(c, &d_ll, node8))) return rc; c->rcv.node8 = d_ll;
    if ((rc = upload(c, &d_f, w8))) return rc;     c->rcv.w8 = d_f;
    if ((rc = upload(c, &d_ll, tnode))) return rc; c->rcv.tnode = d_ll;
    if ((rc = upload(c, &d_i, row_ptr))) return rc; c->rcv.row_ptr = d_i;
    if ((rc = upload(c, &d_i, trcv))) return rc;   c->rcv.trcv = d_i;
    if ((rc = upload(c, &d_f, tw))) return rc;     c->rcv.tw = d_f;

    // ---- 3. C-PML tables
    for (int b = 0; b < 3; ++b) {
        const int n = b == 0 ? nx : (b == 1 ? ny : nz);
        std::vector<float> ai, bi, ah, bh;
        cpml_profile(c->prm, n, false, ai, bi);
        cpml_profile(c->prm, n, true, ah, bh);
        float* d;
        if ((rc = upload(c, &d, ai))) return rc; g.tab[b][T_A_INT] = d;
        if ((rc = upload(c, &d, bi))) return rc; g.tab[b][T_B_INT] = d;
        if ((rc = upload(c, &d, ah))) return rc; g.tab[b][T_A_HALF] = d;
        if ((rc = upload(c, &d, bh))) return rc; g.tab[b][T_B_HALF] = d;
    }

    // ---- 4. scaled, padded material volumes
    float* mat = nullptr;
    c->mbox = (long long)c->pitch * c->py * (c->pz + PACT_NPAL);
    if ((rc = dev_alloc(c, (void**)&mat, (size_t)c->mbox * 4 * sizeof(float)))) return rc;
    float* Ll = mat + org; float* Mi = Ll + c->mbox; float* Rr = Mi + c->mbox; float* Aa = Rr + c->mbox;
    {
        dim3 blk(128), grd((c->pitch + 127) / 128, c->py, c->pz);
        k_scale_materials<<<grd, blk, 0, c->stream>>>(lam, mu, rho, alpha, nx, ny, nz, g.sy, g.sz, c->pitch,
                                                      Ll, Mi, Rr, Aa, prm->dt / prm->h, prm->dt);
        CK(cudaGetLastError());
    }
    g.Ll = Ll; g.Mi = Mi; g.Rr = Rr; g.Aa = Aa;

    // ---- 5. state fields + memory variables, one contiguous block (zeroed per call)
    long long mv[3] = {0, 0, 0};
    if (P > 0) {
        mv[0] = (long long)g.W * ny * nz;
        mv[1] = (long long)nx * g.W * nz;
        mv[2] = (long long)nx * ny * g.W;
    }
    auto r32 = [](long long v) { return (v + 31) / 32 * 32; };
    long long total = c->box * NFIELD;
    for (int b = 0; b < 3; ++b) total += 6 * r32(mv[b]);
    c->state_bytes = total * (long long)sizeof(float);
    if ((rc = dev_alloc(c, (void**)&c->state_base, (size_t)c->state_bytes))) return rc;
    for (int k = 0; k < NFIELD; ++k) g.f[k] = c->state_base + (long long)k * c->box + org;
    {
        float* p = c->state_base + c->box * NFIELD;
        for (int a = 0; a < 3; ++a)
            for (int b = 0; b < 3; ++b) { g.phi[3 * a + b] = p; p += r32(mv[b]); }
        for (int a = 0; a < 3; ++a)
            for (int b = 0; b < 3; ++b) { g.psi[3 * a + b] = p; p += r32(mv[b]); }
    }
    for (int k = 0; k < 9; ++k) g.scr[k] = nullptr;

    if ((rc = dev_alloc(c, (void**)&c->d_flag, sizeof(unsigned int)))) return rc;
    if ((rc = dev_alloc(c, (void**)&c->d_io, sizeof(IoArgs)))) return rc;
    CK(cudaMemsetAsync(c->d_io, 0, sizeof(IoArgs), c->stream));
    for (int op = 0; op < 2; ++op)
        for (int k = 0; k < 2; ++k) CK(cudaEventCreate(&c->ev_loop[op][k]));
    CK(cudaStreamSynchronize(c->stream));   // the caller may free its volumes now
    CK(cudaGetLastError());
    return PACT_OK;
}

extern "C" int pact_create(pact_ctx** out, const pact_params* prm, const float* lam, const float* mu,
                           const float* rho, const float* alpha, const double* rcv_xyz, int L, void* cuda_stream)
{
    if (out) *out = nullptr;
    if (!out || !prm || !lam || !mu || !rho || L < 0 || (L > 0 && !rcv_xyz)) return PACT_EINVAL;
    if (prm->nx < 8 || prm->ny < 8 || prm->nz < 8 || prm->nt < 1 || prm->npml < 0) return PACT_EINVAL;
    if (!(prm->h > 0.0) || !(prm->dt > 0.0) || !std::isfinite(prm->h) || !std::isfinite(prm->dt)) return PACT_EINVAL;
    if (2 * prm->npml + 8 > std::min(prm->nx, std::min(prm->ny, prm->nz))) return PACT_EINVAL;
    if (prm->npml > 0 && (!(prm->pml_R >= 0.0 && prm->pml_R < 1.0) || !(prm->pml_cref >= 0.0) || !std::isfinite(prm->pml_cref) ||
                          !(prm->pml_beta_max >= 0.0) || !std::isfinite(prm->pml_beta_max)))
        return PACT_EINVAL;   // pml_R = 0 / pml_cref = 0 select the defaults (1e-4, max c_l)
    if ((double)prm->nx * prm->ny * prm->nz > 2.0e9) return PACT_EINVAL;   // 32-bit cell counts inside kernels
    pact_ctx* c = new (std::nothrow) pact_ctx();
    if (!c) return PACT_ENOMEM;
    c->prm = *prm;
    c->stream = (cudaStream_t)cuda_stream;
    c->variant = 0;
    c->use_graph = -1;
    c->split_launch = 1;
    c->elide = 1;
    c->acoustic = -1;
    int rc = create_impl(c, prm, lam, mu, rho, alpha, rcv_xyz, L);
    if (rc != PACT_OK) { pact_destroy(c); return rc; }
    *out = c;
    return PACT_OK;
}

// ------------------------------------------------------------------------------------------------
// time loops
__global__ void k_set_io(IoArgs* io, IoArgs v) { *io = v; }

struct Launcher {
    pact_ctx* c;
    int op;          // 0 forward, 1 adjoint
    bool sample;     // record events around the launches of this step
    int err;
    template <typename F>
    void run(int kind, F&& launch)
    {
        if (err) return;
        EvPair* ev = nullptr;
        if (sample && c->used[op][kind] < MAX_SAMPLES) {
            if (c->used[op][kind] == c->samples[op][kind].size()) {
                EvPair p;
                if (cudaEventCreate(&p.a) != cudaSuccess || cudaEventCreate(&p.b) != cudaSuccess) {
                    err = cuda_fail(cudaGetLastError(), "cudaEventCreate", __LINE__);
                    return;
                }
                c->samples[op][kind].push_back(p);
            }
            ev = &c->samples[op][kind][c->used[op][kind]++];
            cudaError_t e = cudaEventRecord(ev->a, c->stream);
            if (e != cudaSuccess) { err = cuda_fail(e, "cudaEventRecord", __LINE__); return; }
        }
        launch();
        cudaError_t e = cudaGetLastError();
        if (e == cudaSuccess && ev) e = cudaEventRecord(ev->b, c->stream);
        c->launches[op][kind]++;
        if (e != cudaSuccess) err = cuda_fail(e, "kernel launch", __LINE__);
    }
};

// 1 = plain two-kernel path, 2 = fused single-pass path.  Automatic: the fused kernel runs one CTA per SM over
// 32 x 32 x (>= 32) bricks, so it needs a grid with at least one brick per SM; smaller grids (which fit in L2 and
// are launch/latency bound anyway) take the one-thread-per-cell kernels.
static int resolve_variant(const pact_ctx* c)
{
    if (!c->bulk_positive) return 1;
    if (c->variant != 0) return c->variant;
    const long long bricks = (long long)((c->prm.nx + FT_TX - 1) / FT_TX) * ((c->prm.ny + FT_TY - 1) / FT_TY) * ((c->prm.nz + 31) / 32);
    return bricks >= c->num_sms ? 2 : 1;
}

static int ensure_scratch(pact_ctx* c)
{
    if (c->scratch_base) return PACT_OK;
    int rc = dev_alloc(c, (void**)&c->scratch_base, (size_t)c->box * 9 * sizeof(float));
    if (rc) return rc;
    CK(cudaMemsetAsync(c->scratch_base, 0, (size_t)c->box * 9 * sizeof(float), c->stream));   // halo stays 0
    const long long org = (long long)PACT_HALO_Z * c->g.sz + (long long)PACT_HALO_Y * c->g.sy + PACT_HALO_X;
    for (int k = 0; k < 9; ++k) c->g.scr[k] = c->scratch_base + (long long)k * c->box + org;
    return PACT_OK;
}

static void forward_step(pact_ctx* c, Launcher& ln, int variant)
{
    const DevGrid& g = c->g;
    cudaStream_t st = c->stream;
    dim3 blk(PLAIN_BX, PLAIN_BY, PLAIN_BZ);
    dim3 grd((g.nx + PLAIN_BX - 1) / PLAIN_BX, (g.ny + PLAIN_BY - 1) / PLAIN_BY, (g.nz + PLAIN_BZ - 1) / PLAIN_BZ);
    ln.run(PACT_K_FWD_VEL, [&] { k_fwd_vel<<<grd, blk, 0, st>>>(g); });
    ln.run(PACT_K_FWD_STR, [&] { k_fwd_str<<<grd, blk, 0, st>>>(g); });
}

static void adjoint_step(pact_ctx* c, Launcher& ln, int variant)
{
    const DevGrid& g = c->g;
    cudaStream_t st = c->stream;
    dim3 blk(PLAIN_BX, PLAIN_BY, PLAIN_BZ);
    dim3 grd((g.nx + PLAIN_BX - 1) / PLAIN_BX, (g.ny + PLAIN_BY - 1) / PLAIN_BY, (g.nz + PLAIN_BZ - 1) / PLAIN_BZ);
    ln.run(PACT_K_ADJ_A, [&] { k_adj_a1<<<grd, blk, 0, st>>>(g); });
    ln.run(PACT_K_ADJ_A, [&] { k_adj_a2<<<grd, blk, 0, st>>>(g); });
    ln.run(PACT_K_ADJ_B, [&] { k_adj_b1<<<grd, blk, 0, st>>>(g); });
    ln.run(PACT_K_ADJ_B, [&] { k_adj_b2<<<grd, blk, 0, st>>>(g); });
}


// ---- fused variant: buffers, TMA descriptors, launch ---------------------------------------------
typedef CUresult (*encode_tiled_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                    const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// 4-D map [field][z][y][x] over `nf` padded fields starting at `base` (start of the padded box), box {bw, bh, 1, 1}
static int make_map(pact_ctx* c, encode_tiled_fn enc, CUtensorMap* tm, const float* base, int nf, int bw, int bh,
                    int planes = 0, long long field_stride = 0)
{
    if (planes == 0) { planes = c->pz; field_stride = c->box; }
    const cuuint64_t dims[4] = {(cuuint64_t)c->pitch, (cuuint64_t)c->py, (cuuint64_t)planes, (cuuint64_t)nf};
    const cuuint64_t strides[3] = {(cuuint64_t)c->pitch * 4, (cuuint64_t)c->pitch * c->py * 4, (cuuint64_t)field_stride * 4};
    const cuuint32_t boxd[4] = {(cuuint32_t)bw, (cuuint32_t)bh, 1, 1};
    const cuuint32_t es[4] = {1, 1, 1, 1};
    // L2 promotion 64 B: box rows are 160 B starting 112 B into a 128-B line; with 128-B promotion every row pulls
    // three whole lines (measured: 12.0 GB of DRAM reads per 512^3 step against 9.5 GB with 64 B, 7.0 GB algorithmic)
    CUresult r = enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, (void*)base, dims, strides, boxd, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                     CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_64B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
        return PACT_ECUDA;
    }
    return PACT_OK;
}

// Homogeneous material planes: flag every (tile, plane) whose material box is one 4-tuple, give the
// PACT_NPAL most frequent tuples a palette plane each behind the material volumes, and let the fused kernel fetch
// flagged planes from there.  Same bytes arrive in shared memory, so the result does not change by a bit; what
// changes is that the palette planes live in L2 while the flagged planes are never read from HBM.
static int scan_material_planes(pact_ctx* c)
{
    const DevGrid& g = c->g;
    const int ntx = (g.nx + FT_TX - 1) / FT_TX, nty = (g.ny + FT_TY - 1) / FT_TY, tiles = ntx * nty;
    c->nzp = c->pz + 8;
    const long long nrec = (long long)tiles * c->nzp;
    const long long org = (long long)PACT_HALO_Z * g.sz + (long long)PACT_HALO_Y * g.sy + PACT_HALO_X;
    float* mat0 = const_cast<float*>(g.Ll) - org;
    MatPlaneRec* d_rec = nullptr;
    CK(cudaMalloc((void**)&d_rec, (size_t)nrec * sizeof(MatPlaneRec)));
    k_scan_material_planes<<<dim3(tiles, c->nzp), 128, 0, c->stream>>>(mat0, c->mbox, c->pitch, c->py, c->pz, ntx, c->nzp, d_rec);
    std::vector<MatPlaneRec> rec((size_t)nrec);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaMemcpyAsync(rec.data(), d_rec, (size_t)nrec * sizeof(MatPlaneRec), cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    cudaFree(d_rec);
    if (e != cudaSuccess) return cuda_fail(e, "k_scan_material_planes", __LINE__);
    // palette = the most frequent homogeneous tuples
    struct Entry { unsigned int v[4]; long long n; };
    std::vector<Entry> ent;
    for (const MatPlaneRec& r : rec) {
        if (!r.homog) continue;
        size_t k = 0;
        for (; k < ent.size(); ++k)
            if (!memcmp(ent[k].v, r.v, sizeof(r.v))) break;
        if (k == ent.size()) {
            if (ent.size() >= 4096) continue;     // a medium with that many distinct homogeneous planes gains nothing here
            Entry en; memcpy(en.v, r.v, sizeof(r.v)); en.n = 0;
            ent.push_back(en);
        }
        ent[k].n++;
    }
    std::sort(ent.begin(), ent.end(), [](const Entry& a, const Entry& b) { return a.n > b.n; });
    if (ent.size() > PACT_NPAL) ent.resize(PACT_NPAL);
    std::vector<unsigned char> flag((size_t)nrec, 0);
    long long hit = 0, planes = 0;
    for (long long i = 0; i < nrec; ++i) {
        if (i % c->nzp < c->pz) planes++;
        if (!rec[(size_t)i].homog) continue;
        for (size_t k = 0; k < ent.size(); ++k)
            if (!memcmp(ent[k].v, rec[(size_t)i].v, sizeof(ent[k].v))) { flag[(size_t)i] = (unsigned char)(k + 1); hit++; break; }
    }
    c->elided = planes ? (double)hit / (double)planes : 0.0;
    const long long plane = (long long)c->pitch * c->py;
    for (size_t k = 0; k < ent.size(); ++k)
        for (int f = 0; f < 4; ++f) {
            k_fill<<<64, 256, 0, c->stream>>>(mat0 + (long long)f * c->mbox + (long long)(c->pz + (int)k) * plane, ent[k].v[f], plane);
            CK(cudaGetLastError());
        }
    int rc = dev_alloc(c, (void**)&c->d_mflag, (size_t)nrec);
    if (rc) return rc;
    CK(cudaMemcpyAsync(c->d_mflag, flag.data(), (size_t)nrec, cudaMemcpyHostToDevice, c->stream));
    CK(cudaStreamSynchronize(c->stream));   // the vector is a temporary
    c->fa.mflag = c->d_mflag;
    c->fa.ntx = ntx; c->fa.nzp = c->nzp; c->fa.mpal = c->pz;
    return PACT_OK;
}

static int ensure_fused(pact_ctx* c)
{
    if (c->fused_ready) return PACT_OK;
    const DevGrid& g = c->g;
    const int P = g.P;
    FusedArgs& fa = c->fa;
    memset(&fa, 0, sizeof(fa));
    fa.nx = g.nx; fa.ny = g.ny; fa.nz = g.nz;
    fa.sy = g.sy; fa.sz = g.sz; fa.box = c->box;
    fa.P = P;
    fa.nxq = (g.nx + 3) / 4 * 4;
    fa.wyz = P > 0 ? 2 * P + 1 : 0;
    if (P > 0) {
        fa.xl = (P + 3) / 4 * 4;
        fa.xr = (g.nx - 1 - P) / 4 * 4;
        if (fa.xl >= fa.xr) { fa.xl = fa.nxq; fa.xr = fa.nxq; }
        fa.wx = fa.xl + (fa.nxq - fa.xr);
    }
    for (int b = 0; b < 3; ++b)
        for (int t = 0; t < 4; ++t) fa.tab[b][t] = g.tab[b][t];
    // state buffer B + ping-pong memory variables in one block (zeroed at the start of every call)
    long long mv[3] = {0, 0, 0};
    if (P > 0) {
        mv[0] = (long long)fa.wx * g.ny * g.nz;
        mv[1] = (long long)fa.nxq * fa.wyz * g.nz;
        mv[2] = (long long)fa.nxq * g.ny * fa.wyz;
    }
    auto r32 = [](long long v) { return (v + 31) / 32 * 32; };
    for (int b = 0; b < 3; ++b)     // the kernels index a group with 32-bit float offsets
        if (3 * r32(mv[b]) + 64 > 0x7fffffffLL) {
            snprintf(g_cuda_err, sizeof(g_cuda_err), "C-PML slab of axis %d too large for the fused kernels' 32-bit offsets", b);
            return PACT_EINVAL;
        }
    long long total = c->box * NFIELD;
    for (int b = 0; b < 3; ++b) total += 2 * 6 * r32(mv[b]);
    c->stateB_bytes = total * (long long)sizeof(float);
    int rc = dev_alloc(c, (void**)&c->stateB_base, (size_t)c->stateB_bytes);
    if (rc) return rc;
    const long long org = (long long)PACT_HALO_Z * g.sz + (long long)PACT_HALO_Y * g.sy + PACT_HALO_X;
    c->g2 = c->g;
    for (int k = 0; k < NFIELD; ++k) c->g2.f[k] = c->stateB_base + (long long)k * c->box + org;
    {
        float* p = c->stateB_base + c->box * NFIELD;
        for (int set = 0; set < 2; ++set)            // [0]: read at even steps, [1]: read at odd steps
        {
            float* q = p;       // elastic view (FusedArgs::mgi): group g = 3 * kind + axis, 3 * r32(mv[axis]) floats each
            for (int gk = 0; gk < 6; ++gk) { c->mgbuf[set][gk] = q; q += 3 * r32(mv[gk % 3]); }
            for (int k = 0; k < 18; ++k) { c->mvbuf[set][k] = p; p += r32(mv[k % 3]); }
        }
    }
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    CK(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
    if (!fn || qres != cudaDriverEntryPointSuccess) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "cuTensorMapEncodeTiled is not available from the driver");
        return PACT_ECUDA;
    }
    encode_tiled_fn enc = (encode_tiled_fn)fn;
    const float* baseA = c->state_base;
    const float* baseB = c->stateB_base;
    const float* baseM = g.Ll - org;
    if ((rc = make_map(c, enc, &c->tmS40[0], baseA, NFIELD, FT_BW, FT_BH))) return rc;
    if ((rc = make_map(c, enc, &c->tmS36[0], baseA, NFIELD, FT_BW, FT_UH))) return rc;
    if ((rc = make_map(c, enc, &c->tmS40[1], baseB, NFIELD, FT_BW, FT_BH))) return rc;
    if ((rc = make_map(c, enc, &c->tmS32[0], baseA, NFIELD, FT_TX, FT_TY))) return rc;
    if ((rc = make_map(c, enc, &c->tmS32[1], baseB, NFIELD, FT_TX, FT_TY))) return rc;
    if ((rc = make_map(c, enc, &c->tmS36[1], baseB, NFIELD, FT_BW, FT_UH))) return rc;
    if ((rc = make_map(c, enc, &c->tmM37, baseM, 4, FT_BW, FT_RH, c->pz + PACT_NPAL, c->mbox))) return rc;
    if ((rc = make_map(c, enc, &c->tmL, baseM, 4, FT_TX, FT_TY, c->pz + PACT_NPAL, c->mbox))) return rc;
    if ((rc = make_map(c, enc, &c->tmM36, baseM, 4, FT_MW, FT_MH, c->pz + PACT_NPAL, c->mbox))) return rc;
    if ((rc = scan_material_planes(c))) return rc;
    CK(cudaFuncSetAttribute(k_step<FM_PLAIN>, cudaFuncAttributeMaxDynamicSharedMemorySize, FT_SMEM_BYTES));
    CK(cudaFuncSetAttribute(k_step<FM_FWD>, cudaFuncAttributeMaxDynamicSharedMemorySize, FT_SMEM_BYTES));
    CK(cudaFuncSetAttribute(k_step<FM_ADJ>, cudaFuncAttributeMaxDynamicSharedMemorySize, FT_SMEM_BYTES));
    CK(cudaFuncSetAttribute(k_step_acoustic<FM_PLAIN>, cudaFuncAttributeMaxDynamicSharedMemorySize, FT_SMEM_BYTES));
    CK(cudaFuncSetAttribute(k_step_acoustic<FM_FWD>, cudaFuncAttributeMaxDynamicSharedMemorySize, FT_SMEM_BYTES));
    CK(cudaFuncSetAttribute(k_step_acoustic<FM_ADJ>, cudaFuncAttributeMaxDynamicSharedMemorySize, FT_SMEM_BYTES));
    c->work_zc = -1;
    c->work_cap = (long long)((g.nx + FT_TX - 1) / FT_TX) * ((g.ny + FT_TY - 1) / FT_TY) * (2 * g.nz + 2);   // worst case: one-plane chunks
    if ((rc = dev_alloc(c, (void**)&c->d_work, (size_t)c->work_cap * sizeof(int4)))) return rc;
    if ((rc = dev_alloc(c, (void**)&c->d_queue, 2 * sizeof(unsigned int)))) return rc;
    CK(cudaMemsetAsync(c->d_queue, 0, 2 * sizeof(unsigned int), c->stream));
    fa.queue = c->d_queue;
    c->fused_ready = true;
    return PACT_OK;
}

// z chunks of the plane range [z0, z1).  zc > 0: `zc` planes each (tests).  Automatic: the
// persistent launch hands bricks out dynamically, so what matters is (a) few start-up planes (4 per brick, plus the
// pipeline prologue) and (b) a short tail: about five sixths of the range in long chunks (<= FT_CHUNK_LONG planes),
// the rest in short ones (<= FT_CHUNK_SHORT) that the host lists last.
#define FT_CHUNK_LONG 128
#define FT_CHUNK_SHORT 40
static void cut_chunks(int z0, int z1, int zc, int len_long, int len_short, std::vector<std::pair<int, int>>& longs,
                       std::vector<std::pair<int, int>>& shorts)
{
    const int n = z1 - z0;
    if (n <= 0) return;
    auto equal_parts = [](int a, int b, int maxlen, std::vector<std::pair<int, int>>& out) {
        const int m = b - a;
        if (m <= 0) return;
        const int k = (m + maxlen - 1) / maxlen;
        for (int i = 0; i < k; ++i) out.push_back({a + (int)((long long)m * i / k), a + (int)((long long)m * (i + 1) / k)});
    };
    if (zc > 0) { equal_parts(z0, z1, zc, longs); return; }
    if (n <= len_short + 8) { shorts.push_back({z0, z1}); return; }
    const int tail = std::max(n / 6, 24);
    equal_parts(z0, z1 - tail, len_long, longs);
    equal_parts(z1 - tail, z1, len_short, shorts);
}

// Work list: a brick is "interior" when its u region with the +-2 taps of the transposed
// C-PML recursion (x0-4 .. x0+35, likewise y, planes zb-4 .. ze+2) misses every slab; such bricks run the brick
// routine without C-PML code.  Everything else (boundary tiles over all z; the z slabs of interior tiles) carries
// the FT_WORK_SLAB flag.  Order = the order the persistent launch hands them out: slab bricks first (they cost
// about twice as much per plane), long before short, and chunk-major inside a class so that neighbouring tiles
// march the same planes together (their shared box rows then meet in L2).
static int build_work(pact_ctx* c)
{
    if (c->work_zc == c->zchunk) return PACT_OK;
    const DevGrid& g = c->g;
    const int LL = c->chunk_long > 0 ? c->chunk_long : FT_CHUNK_LONG, LS = c->chunk_short > 0 ? c->chunk_short : FT_CHUNK_SHORT;
    const int P = g.P, ntx = (g.nx + FT_TX - 1) / FT_TX, nty = (g.ny + FT_TY - 1) / FT_TY;
    auto interior_1d = [&](int t0, int n) { return P == 0 || (t0 - 4 >= P && t0 + 36 <= n - 1 - P); };
    int zlo = 0, zhi = g.nz;
    if (P > 0) { zlo = P + 4; zhi = g.nz - 5 - P; }
    std::vector<std::pair<int, int>> tin, tbd;
    for (int ty = 0; ty < nty; ++ty)
        for (int tx = 0; tx < ntx; ++tx)
            ((interior_1d(tx * FT_TX, g.nx) && interior_1d(ty * FT_TY, g.ny) && zhi - zlo >= 8) ? tin : tbd).push_back({tx, ty});
    std::vector<int4> wl;
    auto add = [&](const std::vector<std::pair<int, int>>& tiles, const std::vector<std::pair<int, int>>& chunks, int flag) {
        for (auto& ch : chunks)
            for (auto& t : tiles) {
                // nothing the brick touches sticks out of the grid: its instance without lane masks (FT_WORK_NOEDGE)
                const int x0 = t.first * FT_TX, y0 = t.second * FT_TY;
                const bool clear = x0 >= 4 && x0 + FT_TX + 4 <= g.nx && y0 >= 4 && y0 + FT_TY + 4 <= g.ny && ch.first >= 4 && ch.second + 4 <= g.nz;
                wl.push_back(make_int4(t.first | flag | (clear && !flag ? FT_WORK_NOEDGE : 0), t.second, ch.first, ch.second));
            }
    };
    std::vector<std::pair<int, int>> bl, bs, il, is, zl, zs;
    // C-PML bricks: the long / short chunk lengths that give the shortest makespan when the launch hands the bricks out
    // in list order to num_sms CTAs (greedy list scheduling, 7 start-up iterations per brick, corner tiles 1.6 x, other
    // boundary tiles 1.3 x the cost of a z-slab brick of an interior tile per plane: the adjoint's ratios).  On large
    // grids this reproduces 128 / 40 ; on small ones (256^3: 28 boundary columns for 148 SMs) one long brick would
    // otherwise be the whole launch.
    int LLs = LL, LSs = LS;
    if (P > 0 && c->zchunk == 0 && c->chunk_long == 0 && c->chunk_short == 0 && !tbd.empty()) {
        auto weight = [&](const std::pair<int, int>& t) {
            return (!interior_1d(t.first * FT_TX, g.nx) && !interior_1d(t.second * FT_TY, g.ny)) ? 1.6 : 1.3;
        };
        double best = 1e300;
        const int cl[] = {24, 32, 48, 64, 96, 128}, cs[] = {16, 24, 40};
        for (int a = 0; a < 6; ++a)
            for (int b = 0; b < 3; ++b) {
                if (cs[b] > cl[a]) continue;
                std::vector<std::pair<int, int>> l1, s1, l2, s2;
                cut_chunks(0, g.nz, 0, cl[a], cs[b], l1, s1);
                if (!tin.empty()) { cut_chunks(0, zlo, 0, cl[a], cs[b], l2, s2); cut_chunks(zhi, g.nz, 0, cl[a], cs[b], l2, s2); }
                std::vector<double> costs;
                for (auto& ch : l1) for (auto& t : tbd) costs.push_back(weight(t) * (ch.second - ch.first + 7));
                for (auto& ch : s1) for (auto& t : tbd) costs.push_back(weight(t) * (ch.second - ch.first + 7));
                for (auto& ch : l2) for (size_t t = 0; t < tin.size(); ++t) costs.push_back(1.0 * (ch.second - ch.first + 7));
                for (auto& ch : s2) for (size_t t = 0; t < tin.size(); ++t) costs.push_back(1.0 * (ch.second - ch.first + 7));
                std::vector<double> sm(c->num_sms, 0.0);        // min-heap of the CTAs' finish times
                auto gt = [](double x, double y) { return x > y; };
                for (double w : costs) {
                    std::pop_heap(sm.begin(), sm.end(), gt);
                    sm.back() += w;
                    std::push_heap(sm.begin(), sm.end(), gt);
                }
                const double mk = *std::max_element(sm.begin(), sm.end());
                if (mk < best * 0.995) { best = mk; LLs = cl[a]; LSs = cs[b]; }      // (a later candidate must be clearly better)
            }
    }
    if (!tbd.empty()) cut_chunks(0, g.nz, c->zchunk, LLs, LSs, bl, bs);
    if (!tin.empty()) {
        // Interior bricks all cost the same per plane, so equal chunks in a whole number of waves beat the long / short mix:
        // k chunks per column minimising waves x (planes per chunk + 7 start-up iterations).  (512^3, npml 16: 196 columns
        // of 472 planes -> k = 3, 588 bricks = 3.97 waves of 148 ; measured 1.557 -> 1.538 ms against 6 chunks per column.)
        if (c->zchunk > 0) cut_chunks(zlo, zhi, c->zchunk, LL + LL / 4, LS, il, is);
        else {
            const int n = zhi - zlo, nt = (int)tin.size();
            int best_k = 1; double best = 1e30;
            for (int k = 1; k <= 16 && n / k >= 24; ++k) {
                const int waves = (nt * k + c->num_sms - 1) / c->num_sms;
                const double cost = (double)waves * ((n + k - 1) / k + 7);
                if (cost < best) { best = cost; best_k = k; }
            }
            cut_chunks(zlo, zhi, (n + best_k - 1) / best_k, 0, 0, il, is);
        }
        if (P > 0) {   // the z slabs of interior tiles: thin bricks
            cut_chunks(0, zlo, c->zchunk, LLs, LSs, zl, zs);
            cut_chunks(zhi, g.nz, c->zchunk, LLs, LSs, zl, zs);
        }
    }
    const int slab = P > 0 ? FT_WORK_SLAB : 0;
    add(tbd, bl, slab); add(tbd, bs, slab); add(tin, zl, slab); add(tin, zs, slab);
    c->nslab = P > 0 ? (int)wl.size() : 0;
    add(tin, il, 0); add(tin, is, 0);
    if ((long long)wl.size() > c->work_cap) return PACT_EINVAL;
    c->nwork = (int)wl.size();
    if (!wl.empty()) CK(cudaMemcpyAsync(c->d_work, wl.data(), wl.size() * sizeof(int4), cudaMemcpyHostToDevice, c->stream));
    CK(cudaStreamSynchronize(c->stream));   // the vector is a temporary
    c->work_zc = c->zchunk;
    return PACT_OK;
}

static bool use_acoustic(const pact_ctx* c) { return c->fluid && c->acoustic != 0; }

// one time step cur -> 1-cur ; sgn = +1: W' ; sgn = -1: W'^T on the scaled adjoint variables.  One persistent
// launch (option "split_launch": the slab bricks and the interior bricks as two launches, each with its own events)
static void fused_step(pact_ctx* c, Launcher& ln, int cur, float sgn, int kind)
{
    FusedArgs fa = c->fa;
    const DevGrid& gi = cur ? c->g2 : c->g;
    const DevGrid& go = cur ? c->g : c->g2;
    fa.in = gi.f[0]; fa.out = go.f[0];
    fa.sgn = sgn;
    fa.work = c->d_work;
    fa.mflag = c->elide ? c->d_mflag : nullptr;
    for (int k = 0; k < 18; ++k) { fa.mvi[k] = c->mvbuf[cur][k]; fa.mvo[k] = c->mvbuf[1 - cur][k]; }
    for (int k = 0; k < 6; ++k) { fa.mgi[k] = c->mgbuf[cur][k]; fa.mgo[k] = c->mgbuf[1 - cur][k]; }
    cudaStream_t st = c->stream;
    // plain: the range holds no C-PML brick, so the kernel without C-PML code (and its register budget) serves it
    auto launch = [&](int b0, int b1, bool plain) {
        if (b1 <= b0) return;
        fa.work_begin = b0; fa.work_end = b1;
        const int grid = std::min(c->num_sms, b1 - b0);
        if (use_acoustic(c)) {      // mu = 0 everywhere: one stress field, 44 B per cell-step (kernels_acoustic.cuh)
            if (fa.P == 0 || plain) k_step_acoustic<FM_PLAIN><<<grid, FT_NT, FT_SMEM_BYTES, st>>>(c->tmS40[cur], c->tmS36[cur], c->tmM37, c->tmL, c->tmS32[cur], fa);
            else if (sgn > 0.0f) k_step_acoustic<FM_FWD><<<grid, FT_NT, FT_SMEM_BYTES, st>>>(c->tmS40[cur], c->tmS36[cur], c->tmM37, c->tmL, c->tmS32[cur], fa);
            else k_step_acoustic<FM_ADJ><<<grid, FT_NT, FT_SMEM_BYTES, st>>>(c->tmS40[cur], c->tmS36[cur], c->tmM37, c->tmL, c->tmS32[cur], fa);
        }
        else if (fa.P == 0 || plain) k_step<FM_PLAIN><<<grid, FT_NT, FT_SMEM_BYTES, st>>>(c->tmS40[cur], c->tmS36[cur], c->tmM37, c->tmM36, c->tmL, c->tmS32[cur], fa);
        else if (sgn > 0.0f) k_step<FM_FWD><<<grid, FT_NT, FT_SMEM_BYTES, st>>>(c->tmS40[cur], c->tmS36[cur], c->tmM37, c->tmM36, c->tmL, c->tmS32[cur], fa);
        else k_step<FM_ADJ><<<grid, FT_NT, FT_SMEM_BYTES, st>>>(c->tmS40[cur], c->tmS36[cur], c->tmM37, c->tmM36, c->tmL, c->tmS32[cur], fa);
    };
    if (!c->split_launch || c->nslab == 0 || c->nslab == c->nwork) {
        ln.run(kind, [&] { launch(0, c->nwork, c->nslab == 0); });
        return;
    }
    const int k_slab = sgn > 0.0f ? PACT_K_FWD_SLAB : PACT_K_ADJ_SLAB, k_int = sgn > 0.0f ? PACT_K_FWD_INTERIOR : PACT_K_ADJ_INTERIOR;
    ln.run(k_slab, [&] { launch(0, c->nslab, false); });
    ln.run(k_int, [&] { launch(c->nslab, c->nwork, true); });
}

// Eq. 58 right to left: tau, then for m = 0..M-1 { Theta ; W' unless m = M-1 }
static int enqueue_forward_loop(pact_ctx* c, bool profile, int variant)
{
    const DevGrid& g = c->g;
    cudaStream_t st = c->stream;
    const int nt = c->prm.nt;
    Launcher ln{c, 0, false, 0};
    const int every = std::max(1, (nt - 1) / MAX_SAMPLES);
    const dim3 rblk(128), rgrd((c->L + 127) / 128);
    int cur = 0;   // fused variant: which state buffer holds v'_m
    for (int m = 0; m < nt; ++m) {
        ln.sample = profile && (m % every == every / 2);
        const DevGrid& gc = cur ? c->g2 : g;
        const int fl = variant == 2 && use_acoustic(c);
        if (c->L > 0) ln.run(PACT_K_RECV, [&] { k_gather<<<rgrd, rblk, 0, st>>>(gc, c->rcv, c->d_io, m, fl); });
        if (m < nt - 1) {
            if (variant == 2) { fused_step(c, ln, cur, 1.0f, PACT_K_FWD_FUSED); cur ^= 1; }
            else forward_step(c, ln, variant);
        }
    }
    return ln.err;
}

// Eq. 27 / 60 with 27b's indexing (reading G4):
//   v = 0 ; for m = M-1..0 { v <- W'^T v unless m = M-1 ; v += Theta'^T p^_m } ; image = tau^T v
static int enqueue_adjoint_loop(pact_ctx* c, bool profile, int variant)
{
    const DevGrid& g = c->g;
    cudaStream_t st = c->stream;
    const int nt = c->prm.nt;
    Launcher ln{c, 1, false, 0};
    const int every = std::max(1, (nt - 1) / MAX_SAMPLES);
    const dim3 rblk(128), rgrd((c->rcv.nnodes + 127) / 128);
    int cur = 0;
    for (int m = nt - 1; m >= 0; --m) {
        ln.sample = profile && (m % every == every / 2);
        if (m < nt - 1) {
            if (variant == 2) { fused_step(c, ln, cur, -1.0f, PACT_K_ADJ_FUSED); cur ^= 1; }
            else adjoint_step(c, ln, variant);
        }
        const DevGrid& gc = cur ? c->g2 : g;
        if (c->L > 0) {
            if (variant == 2) ln.run(PACT_K_RECV, [&] { k_scatter_scaled<<<rgrd, rblk, 0, st>>>(gc, c->rcv, c->d_io, m, (int)use_acoustic(c)); });
            else ln.run(PACT_K_RECV, [&] { k_scatter<<<rgrd, rblk, 0, st>>>(gc, c->rcv, c->d_io, m); });
        }
    }
    ln.sample = false;
    {   // tau^T (Eq. 27c / 60c)
        const DevGrid& gc = cur ? c->g2 : g;
        dim3 blk(64, 4), grd((g.nx + 63) / 64, (g.ny + 3) / 4, g.nz);
        if (variant == 2) ln.run(PACT_K_OTHER, [&] { k_image_scaled<<<grd, blk, 0, st>>>(gc, c->d_io, (int)use_acoustic(c)); });
        else ln.run(PACT_K_OTHER, [&] { k_image<<<grd, blk, 0, st>>>(gc, c->d_io); });
    }
    return ln.err;
}

static bool want_graph(const pact_ctx* c)
{
    if (c->profile) return false;
    if (c->use_graph >= 0) return c->use_graph != 0;
    // auto: small grids are launch-bound (a 64^3 step is a few microseconds); big ones are not
    return c->N <= (1ll << 22) && c->prm.nt <= 4096;
}

static int run_loop(pact_ctx* c, int which /*0 fwd, 1 adj*/)
{
    const int variant = resolve_variant(c);
    if (which == 1 && variant == 1) { int rc = ensure_scratch(c); if (rc) return rc; }
    if (variant == 2) {
        int rc = ensure_fused(c);
        if (rc) return rc;
        if ((rc = build_work(c))) return rc;
        CK(cudaMemsetAsync(c->stateB_base, 0, (size_t)c->stateB_bytes, c->stream));
    }
    for (int k = 0; k < PACT_K_COUNT; ++k) { c->used[which][k] = 0; c->launches[which][k] = 0; }
    c->have_timing[which] = c->profile != 0;
    if (want_graph(c)) {
        if (c->gexec[which] && c->gexec_variant[which] != variant) {
            cudaGraphExecDestroy(c->gexec[which]);
            c->gexec[which] = nullptr;
        }
        if (!c->gexec[which]) {
            cudaGraph_t graph = nullptr;
            if (!c->cap_stream) CK(cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking));
            cudaStream_t user = c->stream;
            CK(cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeThreadLocal));
            c->stream = c->cap_stream;
            int rc = which == 0 ? enqueue_forward_loop(c, false, variant) : enqueue_adjoint_loop(c, false, variant);
            c->stream = user;
            cudaError_t e = cudaStreamEndCapture(c->cap_stream, &graph);
            if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
            if (e != cudaSuccess) return cuda_fail(e, "cudaStreamEndCapture", __LINE__);
            e = cudaGraphInstantiate(&c->gexec[which], graph, 0);
            cudaGraphDestroy(graph);
            if (e != cudaSuccess) { c->gexec[which] = nullptr; return cuda_fail(e, "cudaGraphInstantiate", __LINE__); }
            c->gexec_variant[which] = variant;
        }
        CK(cudaGraphLaunch(c->gexec[which], c->stream));
        return PACT_OK;
    }
    if (c->profile) CK(cudaEventRecord(c->ev_loop[which][0], c->stream));
    int rc = which == 0 ? enqueue_forward_loop(c, c->profile != 0, variant) : enqueue_adjoint_loop(c, c->profile != 0, variant);
    if (rc) return rc;
    if (c->profile) CK(cudaEventRecord(c->ev_loop[which][1], c->stream));
    return PACT_OK;
}

// option "check_finite" (failure detection): NaN / Inf anywhere in the result -> PACT_ENUMERIC
static int finite_check(pact_ctx* c, const float* out, long long n)
{
    if (!c->check_finite || n <= 0) return PACT_OK;
    CK(cudaMemsetAsync(c->d_flag, 0, sizeof(unsigned int), c->stream));
    k_check_finite<<<c->num_sms * 4, 256, 0, c->stream>>>(out, n, c->d_flag);
    CK(cudaGetLastError());
    unsigned int h = 0;
    CK(cudaMemcpyAsync(&h, c->d_flag, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    return h ? PACT_ENUMERIC : PACT_OK;
}

extern "C" int pact_forward(pact_ctx* c, const float* p0, float* data)
{
    if (!c || !p0 || (!data && c->L > 0)) return PACT_EINVAL;
    cudaStream_t st = c->stream;
    IoArgs io{p0, data, nullptr, nullptr};
    k_set_io<<<1, 1, 0, st>>>(c->d_io, io);
    CK(cudaGetLastError());
    CK(cudaMemsetAsync(c->state_base, 0, (size_t)c->state_bytes, st));
    dim3 blk(64, 4), grd((c->g.nx + 63) / 64, (c->g.ny + 3) / 4, c->g.nz);
    k_inject<<<grd, blk, 0, st>>>(c->g, c->d_io);
    CK(cudaGetLastError());
    int rc = run_loop(c, 0);
    if (rc) return rc;
    return finite_check(c, data, (long long)c->prm.nt * c->L);
}

extern "C" int pact_adjoint(pact_ctx* c, const float* data, float* image)
{
    if (!c || !image || (!data && c->L > 0)) return PACT_EINVAL;
    cudaStream_t st = c->stream;
    IoArgs io{nullptr, nullptr, data, image};
    k_set_io<<<1, 1, 0, st>>>(c->d_io, io);
    CK(cudaGetLastError());
    CK(cudaMemsetAsync(c->state_base, 0, (size_t)c->state_bytes, st));
    int rc = run_loop(c, 1);
    if (rc) return rc;
    return finite_check(c, image, c->N);
}

// ---- host-buffer variants -----------------------------------------------------------------------
static int ensure_host_staging(pact_ctx* c)
{
    if (!c->d_vol) { int rc = dev_alloc(c, (void**)&c->d_vol, (size_t)c->N * sizeof(float)); if (rc) return rc; }
    if (!c->d_dat) { int rc = dev_alloc(c, (void**)&c->d_dat, (size_t)c->prm.nt * (size_t)std::max(c->L, 1) * sizeof(float)); if (rc) return rc; }
    return PACT_OK;
}

extern "C" int pact_forward_host(pact_ctx* c, const float* p0_host, float* data_host)
{
    if (!c || !p0_host || (!data_host && c->L > 0)) return PACT_EINVAL;
    int rc = ensure_host_staging(c);
    if (rc) return rc;
    CK(cudaMemcpyAsync(c->d_vol, p0_host, (size_t)c->N * sizeof(float), cudaMemcpyHostToDevice, c->stream));
    rc = pact_forward(c, c->d_vol, c->d_dat);
    if (rc && rc != PACT_ENUMERIC) return rc;
    if (c->L > 0)
        CK(cudaMemcpyAsync(data_host, c->d_dat, (size_t)c->prm.nt * c->L * sizeof(float), cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    return rc;
}

extern "C" int pact_adjoint_host(pact_ctx* c, const float* data_host, float* image_host)
{
    if (!c || !image_host || (!data_host && c->L > 0)) return PACT_EINVAL;
    int rc = ensure_host_staging(c);
    if (rc) return rc;
    if (c->L > 0)
        CK(cudaMemcpyAsync(c->d_dat, data_host, (size_t)c->prm.nt * c->L * sizeof(float), cudaMemcpyHostToDevice, c->stream));
    rc = pact_adjoint(c, c->d_dat, c->d_vol);
    if (rc && rc != PACT_ENUMERIC) return rc;
    CK(cudaMemcpyAsync(image_host, c->d_vol, (size_t)c->N * sizeof(float), cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    return rc;
}

// ---- projected-gradient reconstruction ------------------------------
#define PGD_MAXNORMS 4096
static int ensure_pgd(pact_ctx* c)
{
    int rc = ensure_host_staging(c);
    if (rc) return rc;
    if (!c->d_partial && (rc = dev_alloc(c, (void**)&c->d_partial, PGD_MAXBLOCKS * sizeof(double)))) return rc;
    if (!c->d_norms && (rc = dev_alloc(c, (void**)&c->d_norms, PGD_MAXNORMS * sizeof(double)))) return rc;
    return PACT_OK;
}

static int pgd_blocks(const pact_ctx* c, long long n)
{
    const long long want = (n + PGD_BLOCK - 1) / PGD_BLOCK;
    return (int)std::max(1ll, std::min(want, (long long)std::min(c->num_sms * 8, PGD_MAXBLOCKS)));
}

// p_{k+1} = P_+(p_k - s H^T (H p_k - d)), k = 0 .. iters-1.  Everything stays on the device; the two norms per
// iteration are copied out once at the end (one synchronisation per call).
extern "C" int pact_pgd(pact_ctx* c, float* p, const float* data, double step, int iters, int nonneg,
                        double* resid_l2, double* update_l2)
{
    if (!c || !p || (!data && c->L > 0) || !(step > 0.0) || !std::isfinite(step) || iters < 0 || 2 * iters > PGD_MAXNORMS)
        return PACT_EINVAL;
    int rc = ensure_pgd(c);
    if (rc) return rc;
    const long long nd = (long long)c->prm.nt * c->L;
    const int bd = pgd_blocks(c, nd), bn = pgd_blocks(c, c->N);
    const int check = c->check_finite;
    c->check_finite = 0;              // checked once, on the final iterate
    for (int k = 0; k < iters && !rc; ++k) {
        if ((rc = pact_forward(c, p, c->d_dat))) break;                       // H p_k
        k_pgd_residual<<<bd, PGD_BLOCK, 0, c->stream>>>(c->d_dat, data, nd, c->d_partial);     // r = H p_k - d
        k_pgd_finish<<<1, 32, 0, c->stream>>>(c->d_partial, bd, c->d_norms, 2 * k);
        if ((rc = pact_adjoint(c, c->d_dat, c->d_vol))) break;                // g = H^T r
        k_pgd_update<<<bn, PGD_BLOCK, 0, c->stream>>>(p, c->d_vol, (float)step, nonneg, c->N, c->d_partial);
        k_pgd_finish<<<1, 32, 0, c->stream>>>(c->d_partial, bn, c->d_norms, 2 * k + 1);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) rc = cuda_fail(e, "pact_pgd kernels", __LINE__);
    }
    c->check_finite = check;
    if (rc) return rc;
    if (iters > 0 && (resid_l2 || update_l2)) {
        std::vector<double> h((size_t)2 * iters);
        CK(cudaMemcpyAsync(h.data(), c->d_norms, h.size() * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        CK(cudaStreamSynchronize(c->stream));
        for (int k = 0; k < iters; ++k) {
            if (resid_l2) resid_l2[k] = h[(size_t)2 * k];
            if (update_l2) update_l2[k] = h[(size_t)2 * k + 1];
        }
    }
    return finite_check(c, p, c->N);
}

// ||H||^2 by power iteration on H^T H:  v <- H^T H v / ||H^T H v|| ; with ||v|| = 1 the norm before scaling tends to
// the largest eigenvalue.  v is normalised first, so any non-zero start works (the caller supplies the seeded one).
extern "C" int pact_power_iteration(pact_ctx* c, float* v, int iters, double* sigma2)
{
    if (!c || !v || iters < 1 || iters + 1 > PGD_MAXNORMS || !sigma2) return PACT_EINVAL;
    int rc = ensure_pgd(c);
    if (rc) return rc;
    const int bn = pgd_blocks(c, c->N);
    const int check = c->check_finite;
    c->check_finite = 0;
    for (int k = 0; k <= iters && !rc; ++k) {
        k_pgd_norm2<<<bn, PGD_BLOCK, 0, c->stream>>>(v, c->N, c->d_partial);
        k_pgd_finish<<<1, 32, 0, c->stream>>>(c->d_partial, bn, c->d_norms, k);          // k >= 1: ||H^T H v_{k-1}||
        k_pgd_scale_by_inverse<<<bn, PGD_BLOCK, 0, c->stream>>>(v, c->N, c->d_norms, k);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) { rc = cuda_fail(e, "pact_power_iteration kernels", __LINE__); break; }
        if (k == iters) break;
        if ((rc = pact_forward(c, v, c->d_dat))) break;
        if ((rc = pact_adjoint(c, c->d_dat, v))) break;
    }
    c->check_finite = check;
    if (rc) return rc;
    double h = 0.0;
    CK(cudaMemcpyAsync(&h, c->d_norms + iters, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    *sigma2 = h;
    if (!std::isfinite(h)) return PACT_ENUMERIC;
    return PACT_OK;
}

// ---- options and timing -------------------------------------------------------------------------
extern "C" int pact_set_option(pact_ctx* c, const char* key, long long value)
{
    if (!c || !key) return PACT_EINVAL;
    if (!strcmp(key, "profile")) { c->profile = value != 0; return PACT_OK; }
    if (!strcmp(key, "check_finite")) { c->check_finite = value != 0; return PACT_OK; }
    if (!strcmp(key, "variant")) {
        if (value < 0 || value > 2) return PACT_EINVAL;
        c->variant = (int)value;
        return PACT_OK;
    }
    if (!strcmp(key, "chunk_long") || !strcmp(key, "chunk_short")) {
        if (value < 0 || value > 65535) return PACT_EINVAL;
        (key[6] == 'l' ? c->chunk_long : c->chunk_short) = (int)value;
        c->work_zc = -1; free_graphs(c);
        return PACT_OK;
    }
    if (!strcmp(key, "zchunk")) { if (value < 0) return PACT_EINVAL; c->zchunk = (int)value; free_graphs(c); return PACT_OK; }
    if (!strcmp(key, "graph")) { c->use_graph = value < 0 ? -1 : (value != 0); return PACT_OK; }
    if (!strcmp(key, "acoustic")) { c->acoustic = value < 0 ? -1 : (value != 0 ? -1 : 0); free_graphs(c); return PACT_OK; }
    if (!strcmp(key, "material_elision")) { c->elide = value != 0; free_graphs(c); return PACT_OK; }
    if (!strcmp(key, "split_launch")) { c->split_launch = value != 0; free_graphs(c); return PACT_OK; }
    return PACT_EINVAL;
}

extern "C" int pact_get_timing(pact_ctx* c, int op, double* loop_ms, double* kernel_ms, long long* launches)
{
    if (!c || op < 0 || op > 1 || !c->have_timing[op]) return PACT_EINVAL;
    CK(cudaStreamSynchronize(c->stream));
    if (loop_ms) {
        float ms = 0.0f;
        CK(cudaEventElapsedTime(&ms, c->ev_loop[op][0], c->ev_loop[op][1]));
        *loop_ms = ms;
    }
    for (int k = 0; k < PACT_K_COUNT; ++k) {
        if (kernel_ms) {
            double acc = 0.0;
            for (size_t s = 0; s < c->used[op][k]; ++s) {
                float ms = 0.0f;
                CK(cudaEventElapsedTime(&ms, c->samples[op][k][s].a, c->samples[op][k][s].b));
                acc += ms;
            }
            kernel_ms[k] = c->used[op][k] ? acc / (double)c->used[op][k] : 0.0;
        }
        if (launches) launches[k] = c->launches[op][k];
    }
    return PACT_OK;
}
