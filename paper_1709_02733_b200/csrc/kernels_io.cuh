// kernels_io.cuh — set-up, initial condition, receiver sampling and read-out kernels of libpact.
//
//   k_scan_materials  : validity flags and max c_l^2 of the caller's volumes (pact_create)
//   k_scale_materials : caller's [nz][ny][nx] volumes -> scaled, padded, edge-replicated volumes
//   k_inject          : tau,   Eq. 21: sigma11 = sigma22 = sigma33 = -p0/3
//   k_gather          : Theta, Eq. 23/56: p^_l = -R_l (s11+s22+s33)
//   k_scatter         : Theta^T (Eq. 60a,b PAPER.md:654-658) via the node-sorted transpose table
//   k_image           : tau^T, Eq. 27c/60c: image = -(s11+s22+s33)/3
#pragma once
#include "common.cuh"

// ---- pact_create: scan the caller's volumes -----------------------------------------------------
// flags bit 0: non-finite value ; bit 1: rho <= 0 ; bit 2: mu < 0 ; bit 3: lambda + 2 mu <= 0 ;
// bit 4: alpha < 0 ; bit 5: 3 lambda + 2 mu <= 0 (legal, but the fused adjoint divides by it) ; bit 6: mu > 0 somewhere
// (clear = a fluid everywhere: the acoustic specialisation applies).  cmax2 = max (lambda + 2 mu)/rho as float bits (positive floats order as ints).
__global__ void k_scan_materials(const float* __restrict__ lam, const float* __restrict__ mu,
                                 const float* __restrict__ rho, const float* __restrict__ alpha,
                                 long long N, unsigned int* flags, unsigned int* cmax2_bits)
{
    unsigned int f = 0;
    float c2 = 0.0f;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < N;
         i += (long long)gridDim.x * blockDim.x) {
        const float l = lam[i], m = mu[i], r = rho[i], a = alpha ? alpha[i] : 0.0f;
        if (!isfinite(l) || !isfinite(m) || !isfinite(r) || !isfinite(a)) f |= 1u;
        if (!(r > 0.0f)) f |= 2u;
        if (m < 0.0f) f |= 4u;
        if (!(l + 2.0f * m > 0.0f)) f |= 8u;
        if (a < 0.0f) f |= 16u;
        if (!(3.0f * l + 2.0f * m > 0.0f)) f |= 32u;   // not an error: only rules out the scaled adjoint variables of the fused path
        if (m > 0.0f) f |= 64u;
        if (r > 0.0f) c2 = fmaxf(c2, (l + 2.0f * m) / r);
    }
    for (int o = 16; o > 0; o >>= 1) {
        f |= __shfl_xor_sync(0xffffffffu, f, o);
        c2 = fmaxf(c2, __shfl_xor_sync(0xffffffffu, c2, o));
    }
    if ((threadIdx.x & 31) == 0) {
        if (f) atomicOr(flags, f);
        if (c2 > 0.0f && isfinite(c2)) atomicMax(cmax2_bits, __float_as_uint(c2));
    }
}

// ---- pact_create: scaled padded material volumes ------------------------------------------------
// Covers the whole padded box; indices are clamped into the grid (edge replication implements the
// "missing neighbour = own value" rule of reading G10).  Scale factors are applied in fp64 and
// rounded once:  Ll = lambda dt/h ; Mi = h/(mu dt) (+inf where mu = 0) ; Rr = rho h/dt ; Aa = alpha dt.
__global__ void k_scale_materials(const float* __restrict__ lam, const float* __restrict__ mu,
                                  const float* __restrict__ rho, const float* __restrict__ alpha,
                                  int nx, int ny, int nz, long long sy, long long sz, int pitch,
                                  float* Ll, float* Mi, float* Rr, float* Aa, double dt_over_h, double dt)
{
    // thread (px, py, pz) over the padded box; px = 0 corresponds to x = -PACT_HALO_X
    const int px = blockIdx.x * blockDim.x + threadIdx.x;
    const int py = blockIdx.y;
    const int pz = blockIdx.z;
    if (px >= pitch) return;
    const int x = px - PACT_HALO_X, y = py - PACT_HALO_Y, z = pz - PACT_HALO_Z;
    const int cx = min(max(x, 0), nx - 1), cy = min(max(y, 0), ny - 1), cz = min(max(z, 0), nz - 1);
    const long long src = (long long)cx + (long long)nx * ((long long)cy + (long long)ny * cz);
    const long long dst = (long long)z * sz + (long long)y * sy + x;   // relative to node (0,0,0)
    const double m = (double)mu[src];
    Ll[dst] = (float)((double)lam[src] * dt_over_h);
    Mi[dst] = m > 0.0 ? (float)(1.0 / (m * dt_over_h)) : __int_as_float(0x7f800000);
    Rr[dst] = (float)((double)rho[src] / dt_over_h);
    Aa[dst] = alpha ? (float)((double)alpha[src] * dt) : 0.0f;
}

// ---- pact_create: homogeneous material planes -------------------------
// One block per (tile, padded plane): are the four scaled materials each one bit pattern over the tile's whole box
// (x0-4 .. x0+35, y0-4 .. y0+35, clipped to the padded array) on that plane?  rec[(tile * nzp + zp)] = {homogeneous,
// bits of Ll, Mi, Rr, Aa}.  The host turns the most frequent tuples into palette planes and per-plane flags.
struct MatPlaneRec { unsigned int homog, v[4]; };
__global__ void k_scan_material_planes(const float* __restrict__ mat /* start of the padded box of field 0 */, long long mbox,
                                       int pitch, int py, int pz, int ntx, int nzp, MatPlaneRec* rec)
{
    const int tile = blockIdx.x, zp = blockIdx.y;
    const int tx = tile % ntx, ty = tile / ntx;
    MatPlaneRec r;
    r.homog = 0; r.v[0] = r.v[1] = r.v[2] = r.v[3] = 0;
    if (zp < pz) {
        const int xa = tx * 32 - 4 + PACT_HALO_X, ya = ty * 32 - 4 + PACT_HALO_Y;
        const int x0 = max(xa, 0), x1 = min(xa + 40, pitch), y0 = max(ya, 0), y1 = min(ya + 40, py);
        const int w = x1 - x0, n = w * (y1 - y0);
        bool same = true;
        for (int k = 0; k < 4; ++k) {
            const unsigned int* f = reinterpret_cast<const unsigned int*>(mat + (long long)k * mbox + (long long)zp * pitch * py);
            const unsigned int first = f[(long long)y0 * pitch + x0];
            r.v[k] = first;
            for (int i = threadIdx.x; i < n; i += blockDim.x) same &= f[(long long)(y0 + i / w) * pitch + x0 + i % w] == first;
        }
        r.homog = __syncthreads_and(same) ? 1u : 0u;
    }
    if (threadIdx.x == 0) rec[(long long)tile * nzp + zp] = r;
}

__global__ void k_fill(float* p, unsigned int bits, long long n)
{
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        p[i] = __uint_as_float(bits);
}

// ---- option "check_finite": flag <- 1 if any of the n values is a NaN or an Inf ------------------------
__global__ void k_check_finite(const float* __restrict__ v, long long n, unsigned int* flag)
{
    bool bad = false;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        bad |= !isfinite(v[i]);
    if (__any_sync(0xffffffffu, bad) && (threadIdx.x & 31) == 0) atomicOr(flag, 1u);
}

// ---- device-resident call arguments (so that captured graphs survive new user pointers) ---------
struct IoArgs {
    const float* p0;     // pact_forward input
    float* data_out;     // pact_forward output  [nt][L]
    const float* data_in;// pact_adjoint input   [nt][L]
    float* image;        // pact_adjoint output
};

// ---- tau (Eq. 21): interior of the three normal stresses; everything else was zeroed by memset --
__global__ void k_inject(const DevGrid g, const IoArgs* __restrict__ io)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= g.nx || y >= g.ny) return;
    const float v = io->p0[(long long)x + (long long)g.nx * ((long long)y + (long long)g.ny * z)] * (-1.0f / 3.0f);
    const long long i = (long long)z * g.sz + (long long)y * g.sy + x;
    g.f[S11][i] = v; g.f[S22][i] = v; g.f[S33][i] = v;
}

// ---- tau^T -------------------------------------------------------------------------------------
__global__ void k_image(const DevGrid g, const IoArgs* __restrict__ io)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= g.nx || y >= g.ny) return;
    const long long i = (long long)z * g.sz + (long long)y * g.sy + x;
    io->image[(long long)x + (long long)g.nx * ((long long)y + (long long)g.ny * z)] =
        (g.f[S11][i] + g.f[S22][i] + g.f[S33][i]) * (-1.0f / 3.0f);
}

// ---- receivers ---------------------------------------------------------------------------------
struct RcvTables {
    int L;                       // receivers
    int nnodes;                  // distinct grid nodes touched by any receiver
    const long long* node8;      // [L][8] padded-layout offsets of the 8 corners
    const float* w8;             // [L][8] trilinear weights
    // transpose (node-sorted) table: node k owns entries row_ptr[k] .. row_ptr[k+1]-1
    const long long* tnode;      // [nnodes] padded-layout offset
    const int* row_ptr;          // [nnodes + 1]
    const int* trcv;             // [8L] receiver index
    const float* tw;             // [8L] weight
};

// Theta: one thread per receiver, fixed summation order c = 0..7
// (fluid = 1: the acoustic path keeps the common normal stress in the S11 field only)
__global__ void k_gather(const DevGrid g, const RcvTables r, const IoArgs* __restrict__ io, int m, int fluid = 0)
{
    const int l = blockIdx.x * blockDim.x + threadIdx.x;
    if (l >= r.L) return;
    const float* __restrict__ s11 = g.f[S11];
    const float* __restrict__ s22 = g.f[S22];
    const float* __restrict__ s33 = g.f[S33];
    float acc = 0.0f;
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        const long long n = r.node8[8 * l + c];
        const float s = s11[n];
        acc = fmaf(r.w8[8 * l + c], fluid ? s + s + s : s + s22[n] + s33[n], acc);
    }
    io->data_out[(long long)m * r.L + l] = -acc;
}

// Theta^T: one thread per touched node, receivers of that node in ascending order (deterministic)
__global__ void k_scatter(const DevGrid g, const RcvTables r, const IoArgs* __restrict__ io, int m)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= r.nnodes) return;
    const float* __restrict__ d = io->data_in + (long long)m * r.L;
    float acc = 0.0f;
    for (int e = r.row_ptr[k]; e < r.row_ptr[k + 1]; ++e) acc = fmaf(r.tw[e], d[r.trcv[e]], acc);
    const long long n = r.tnode[k];
    g.f[S11][n] -= acc; g.f[S22][n] -= acc; g.f[S33][n] -= acc;
}

// ---- scaled adjoint variables of the fused variant --------------------
// The fused adjoint carries s = C sigma_bar (C = the dt/h-scaled isotropic stiffness of Eq. 7c).  For a
// source that adds the same value v to the three normal components, C (v,v,v) = (3 Ll + 2 Ml) (v,v,v).
__device__ __forceinline__ float bulk3(const DevGrid& g, long long n) { return 3.0f * g.Ll[n] + 2.0f / g.Mi[n]; }

__global__ void k_scatter_scaled(const DevGrid g, const RcvTables r, const IoArgs* __restrict__ io, int m, int fluid = 0)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= r.nnodes) return;
    const float* __restrict__ d = io->data_in + (long long)m * r.L;
    float acc = 0.0f;
    for (int e = r.row_ptr[k]; e < r.row_ptr[k + 1]; ++e) acc = fmaf(r.tw[e], d[r.trcv[e]], acc);
    const long long n = r.tnode[k];
    acc *= bulk3(g, n);
    g.f[S11][n] -= acc;
    if (!fluid) { g.f[S22][n] -= acc; g.f[S33][n] -= acc; }
}

// tau^T on the scaled variables: sigma_bar11+22+33 = (s11+s22+s33) / (3 Ll + 2 Ml)
__global__ void k_image_scaled(const DevGrid g, const IoArgs* __restrict__ io, int fluid = 0)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= g.nx || y >= g.ny) return;
    const long long i = (long long)z * g.sz + (long long)y * g.sy + x;
    const float s = g.f[S11][i];
    io->image[(long long)x + (long long)g.nx * ((long long)y + (long long)g.ny * z)] =
        (fluid ? s + s + s : s + g.f[S22][i] + g.f[S33][i]) / bulk3(g, i) * (-1.0f / 3.0f);
}
