// kernels_fused.cuh — variant 2: one fused, TMA-staged, z-marching kernel per time step.
//
// One launch applies the whole propagator W' (Eq. 46a-d) — or, with sgn = -1 and
// the scaled adjoint variables of DESIGN.md "Adjoint step", the whole W'^T (Eq. 61) —
// reading state buffer A and writing state buffer B, so that every state field crosses HBM once
// in each direction per time step (88 B per cell).
//
// Tiling (2.5-D): a CTA owns a 32 x 32 (x,y) tile and marches along z
// over a chunk of planes.  A thread owns one float4 (4 consecutive x) of one row.
//   stage 1 (Eq. 46a,b): u(kk) on the tile + 2 cells of ring, from sigma on the tile + 4 cells;
//   stage 2 (Eq. 46c,d): sigma(kk-2) on the tile, from u(kk-4 .. kk) kept in a shared-memory ring.
// Fields whose x/y neighbours are needed (s11,s22,s12,s13,s23, rho, alpha, mu) and s33 arrive in
// shared memory by TMA (cp.async.bulk.tensor, mbarrier complete_tx), one plane ahead of use; the
// z neighbours of s13,s23,s33 live in per-thread register windows; u_old, lambda and the old
// s11,s22,s12 are own-column values fetched with 128-bit loads one stage ahead of use.
// The ring of 2 (4) cells around the tile is recomputed by the neighbouring CTAs; nothing is
// exchanged between CTAs, hence the two state buffers.
#pragma once
#include <cuda.h>
#include "common.cuh"

#define FT_TX 32
#define FT_TY 32
#define FT_BW 40                      // box width: tile + 4 on each side (floats)
#define FT_BH 40                      // box rows of the sigma / rho / alpha planes
#define FT_UH 36                      // rows of the u region: tile + 2 on each side
#define FT_NT 384                     // threads: 360 quads of the u region, 12 warps
#define FT_BOX (FT_BW * FT_BH)        // floats per 40x40 plane
#define FT_UPL (FT_BW * FT_UH)        // floats per 40x36 plane
#define FT_MW 36                      // mu box: tile + 1 (rounded up to a quad) in x
#define FT_MH 33                      //         tile + 1 in y
#define FT_MPL 1216                   // floats per mu plane buffer (36*33 = 1188, padded to 128 B)
#define FT_RING 5                     // u planes kept for stage 2: ks-2 .. ks+2

// shared memory map (floats)
#define FT_OFF_S11 0
#define FT_OFF_S22 (FT_OFF_S11 + 2 * FT_BOX)
#define FT_OFF_S12 (FT_OFF_S22 + 2 * FT_BOX)
#define FT_OFF_S13 (FT_OFF_S12 + 2 * FT_BOX)
#define FT_OFF_S23 (FT_OFF_S13 + 3 * FT_BOX)
#define FT_OFF_RHO (FT_OFF_S23 + 3 * FT_BOX)
#define FT_OFF_ALP (FT_OFF_RHO + 3 * FT_BOX)
#define FT_OFF_S33 (FT_OFF_ALP + 3 * FT_BOX)
#define FT_OFF_MU (FT_OFF_S33 + 2 * FT_UPL)
#define FT_OFF_UR (FT_OFF_MU + 3 * FT_MPL)
#define FT_OFF_END (FT_OFF_UR + 3 * FT_RING * FT_UPL)
#define FT_SMEM_BYTES (FT_OFF_END * 4 + 64)   // + 8 mbarriers

struct FusedArgs {
    int nx, ny, nz;
    int ntx, nty;          // tiles along x, y
    int zc;                // planes per z chunk
    int nzc;               // chunks
    long long sy, sz, box; // strides (elements) of the padded box; elements per field
    const float* in;       // state read  (field k at in + k*box; pointer to node (0,0,0))
    float* out;            // state written
    const float* mat;      // scaled materials Ll, Mi, Rr, Aa at mat + k*box (node (0,0,0))
    float sgn;             // +1: W' on (u, sigma) ; -1: W'^T on the scaled adjoint variables
    // C-PML (PML variant only)
    int P;
    const float* tab[3][4];
    int xl, xr, wx;        // x slab: columns [0,xl) and [xr, nxq) ; wx = xl + nxq - xr ; quad aligned
    int nxq;               // nx rounded up to a multiple of 4
    int wyz;               // slab width along y and z: 2P+1
    const float* mvi[18];  // memory variables read:  phi[3a+b] = [0..9), psi[3a+b] = [9..18)
    float* mvo[18];        // memory variables written
};

// ---- PTX wrappers: mbarrier + TMA (SASS: SYNCS.*, UTMALDG) --------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t"
        "}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// one plane of one field: box {w, h, 1, 1} at (c0, c1, c2, c3) of a 4-D map [field][z][y][x]
__device__ __forceinline__ void tma_plane(const CUtensorMap* tm, float* dst, uint64_t* bar, int c0, int c1, int c2, int c3)
{
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
        ::"r"(smem_u32(dst)), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar))
        : "memory");
}

// ---- float4 helpers -----------------------------------------------------------------------------
__device__ __forceinline__ float4 ld4s(const float* p, int quad) { return *reinterpret_cast<const float4*>(p + 4 * quad); }
__device__ __forceinline__ float2 ld2s(const float* p, int off) { return *reinterpret_cast<const float2*>(p + off); }
__device__ __forceinline__ float4 f4(float v) { return make_float4(v, v, v, v); }
__device__ __forceinline__ float4 operator+(float4 a, float4 b) { return make_float4(a.x + b.x, a.y + b.y, a.z + b.z, a.w + b.w); }
__device__ __forceinline__ float4 operator*(float4 a, float4 b) { return make_float4(a.x * b.x, a.y * b.y, a.z * b.z, a.w * b.w); }
__device__ __forceinline__ float4 operator*(float a, float4 b) { return make_float4(a * b.x, a * b.y, a * b.z, a * b.w); }
__device__ __forceinline__ float4 fma4(float4 a, float4 b, float4 c)
{
    return make_float4(fmaf(a.x, b.x, c.x), fmaf(a.y, b.y, c.y), fmaf(a.z, b.z, c.z), fmaf(a.w, b.w, c.w));
}
// the value one x to the right of each lane of `c`, `r0` being the element after c.w
__device__ __forceinline__ float4 shl1(float4 c, float r0) { return make_float4(c.y, c.z, c.w, r0); }
__device__ __forceinline__ float4 rcp4(float4 a) { return make_float4(__frcp_rn(a.x), __frcp_rn(a.y), __frcp_rn(a.z), __frcp_rn(a.w)); }

// Eq. 8 without 1/h, along y or z: taps t0..t3 at consecutive samples;
//   D+ at i uses (i-1, i, i+1, i+2) ; D- at i uses (i-2, i-1, i, i+1)
__device__ __forceinline__ float4 d4(float4 t0, float4 t1, float4 t2, float4 t3)
{
    return make_float4(fmaf(PACT_C1, t2.x - t1.x, PACT_C2 * (t3.x - t0.x)), fmaf(PACT_C1, t2.y - t1.y, PACT_C2 * (t3.y - t0.y)),
                       fmaf(PACT_C1, t2.z - t1.z, PACT_C2 * (t3.z - t0.z)), fmaf(PACT_C1, t2.w - t1.w, PACT_C2 * (t3.w - t0.w)));
}
// along x on a quad c = f[0..3]: l = (f[-2], f[-1]), r = (f[4], f[5])
__device__ __forceinline__ float4 dpx(float2 l, float4 c, float2 r)   // D+ : result at i + 1/2
{
    return make_float4(fmaf(PACT_C1, c.y - c.x, PACT_C2 * (c.z - l.y)), fmaf(PACT_C1, c.z - c.y, PACT_C2 * (c.w - c.x)),
                       fmaf(PACT_C1, c.w - c.z, PACT_C2 * (r.x - c.y)), fmaf(PACT_C1, r.x - c.w, PACT_C2 * (r.y - c.z)));
}
__device__ __forceinline__ float4 dmx(float2 l, float4 c, float2 r)   // D- : result at i
{
    return make_float4(fmaf(PACT_C1, c.x - l.y, PACT_C2 * (c.y - l.x)), fmaf(PACT_C1, c.y - c.x, PACT_C2 * (c.z - l.y)),
                       fmaf(PACT_C1, c.z - c.y, PACT_C2 * (c.w - c.x)), fmaf(PACT_C1, c.w - c.z, PACT_C2 * (r.x - c.y)));
}

__device__ __forceinline__ float4 ldg4(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }
__device__ __forceinline__ void stg4(float* p, float4 v) { *reinterpret_cast<float4*>(p) = v; }

// store the in-grid lanes of a quad starting at column x
__device__ __forceinline__ void store_quad(float* p, float4 v, int x, int nx)
{
    if (x + 3 < nx) { stg4(p, v); return; }
    if (x < nx) p[0] = v.x;
    if (x + 1 < nx) p[1] = v.y;
    if (x + 2 < nx) p[2] = v.z;
}

// ---- C-PML pieces (PML variant) -------------------------------------------------------------------
struct PmlCtx {
    bool bx, by;           // this CTA's box touches the x / y slabs
};

// slab column of grid column x (multiple of 4), or -1 ; x slab = [0,xl) U [xr,nxq)
__device__ __forceinline__ int xslab_col(const FusedArgs& a, int x)
{
    if (x < 0 || x >= a.nxq) return -1;
    if (x < a.xl) return x;
    if (x >= a.xr) return a.xl + (x - a.xr);
    return -1;
}
__device__ __forceinline__ int yzslab_row(int i, int n, int P)
{
    if (i < 0 || i >= n) return -1;
    if (i < P) return i;
    if (i >= n - 1 - P) return i - (n - 1 - P) + P;
    return -1;
}
__device__ __forceinline__ float4 tab4(const float* t, int x, int n)
{
    // table values at x..x+3 ; outside [0,n): identity (a = 0 / b = 1 are chosen by the caller)
    float4 v;
    v.x = (unsigned)x < (unsigned)n ? __ldg(t + x) : 0.0f;
    v.y = (unsigned)(x + 1) < (unsigned)n ? __ldg(t + x + 1) : 0.0f;
    v.z = (unsigned)(x + 2) < (unsigned)n ? __ldg(t + x + 2) : 0.0f;
    v.w = (unsigned)(x + 3) < (unsigned)n ? __ldg(t + x + 3) : 0.0f;
    return v;
}

// =================================================================================================
// The fused step.  PML: the CTA applies the C-PML recursions (all CTAs of a launch share the
// template; interior CTAs are launched with PML = false).  See DESIGN.md for the index algebra.
template <bool PML>
__global__ void __launch_bounds__(FT_NT, 1)
k_fused(const __grid_constant__ CUtensorMap tmS40, const __grid_constant__ CUtensorMap tmS36,
        const __grid_constant__ CUtensorMap tmM40, const __grid_constant__ CUtensorMap tmM36, const FusedArgs a)
{
    extern __shared__ __align__(1024) float sm[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(sm + FT_OFF_END);
    uint64_t* barL = bars;        // [2]  s11, s22, s12 of plane j          -> slot j & 1
    uint64_t* barE = bars + 2;    // [3]  s13, s23, rho, alpha of plane j ; s33 of plane j + 1 -> slot j % 3
    uint64_t* barM = bars + 5;    // [3]  mu of plane j                     -> slot j % 3

    const int tid = threadIdx.x;
    int b = blockIdx.x;
    const int tx = b % a.ntx; b /= a.ntx;
    const int ty = b % a.nty; b /= a.nty;
    const int zb = b * a.zc, ze = min(zb + a.zc, a.nz);
    const int x0 = tx * FT_TX, y0 = ty * FT_TY;
    const int itn = ze - zb + 4;            // iterations: u planes kk = zb-2 .. ze+1

    // thread -> quad of the u region (10 quads x 36 rows)
    const bool act1 = tid < 360;
    const int qx = tid % 10, r = tid / 10;
    const int x = x0 - 4 + 4 * qx, y = y0 - 2 + r;
    const bool inner = act1 && qx >= 1 && qx <= 8 && r >= 2 && r < 34 && x < a.nx && y < a.ny;
    const int q = tid + 20;                 // quad index in a 40x40 plane (two rows further down)
    const int uq = tid;                     // quad index in a 40x36 plane
    const int mq = (r - 2) * 9 + (qx - 1);  // quad index in a mu plane (inner threads)
    // own-column global loads are legal where the padded box has storage
    const bool ld_ok = act1 && (y + PACT_HALO_Y < a.ny + 2 * PACT_HALO_Y) && (x + 3 + PACT_HALO_X < (int)a.sy);
    const long long gxy = (long long)y * a.sy + x;
    // lanes of the quad that are grid points (u outside the grid is zero: reading G9)
    const bool yin = (unsigned)y < (unsigned)a.ny;
    const bool m0 = yin && (unsigned)x < (unsigned)a.nx, m1 = yin && (unsigned)(x + 1) < (unsigned)a.nx;
    const bool m2 = yin && (unsigned)(x + 2) < (unsigned)a.nx, m3 = yin && (unsigned)(x + 3) < (unsigned)a.nx;

    const float* in = a.in;
    const long long box = a.box;

    if (tid == 0) {
        for (int k = 0; k < 8; ++k) mbar_init(&bars[k], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();

    const int cx40 = x0 - 4 + PACT_HALO_X, cy40 = y0 - 4 + PACT_HALO_Y, cy36 = y0 - 2 + PACT_HALO_Y;
    const int cxm = x0 + PACT_HALO_X, cym = y0 + PACT_HALO_Y;
    const int cz0 = zb - 2 + PACT_HALO_Z;   // padded z of relative plane j = 0

    auto issueL = [&](int j) {
        uint64_t* bar = &barL[j & 1];
        mbar_expect_tx(bar, 3 * FT_BOX * 4);
        tma_plane(&tmS40, sm + FT_OFF_S11 + (j & 1) * FT_BOX, bar, cx40, cy40, cz0 + j, S11);
        tma_plane(&tmS40, sm + FT_OFF_S22 + (j & 1) * FT_BOX, bar, cx40, cy40, cz0 + j, S22);
        tma_plane(&tmS40, sm + FT_OFF_S12 + (j & 1) * FT_BOX, bar, cx40, cy40, cz0 + j, S12);
    };
    auto issueE = [&](int j) {
        const int s = j % 3;
        uint64_t* bar = &barE[s];
        mbar_expect_tx(bar, (4 * FT_BOX + FT_UPL) * 4);
        tma_plane(&tmS40, sm + FT_OFF_S13 + s * FT_BOX, bar, cx40, cy40, cz0 + j, S13);
        tma_plane(&tmS40, sm + FT_OFF_S23 + s * FT_BOX, bar, cx40, cy40, cz0 + j, S23);
        tma_plane(&tmM40, sm + FT_OFF_RHO + s * FT_BOX, bar, cx40, cy40, cz0 + j, 2);
        tma_plane(&tmM40, sm + FT_OFF_ALP + s * FT_BOX, bar, cx40, cy40, cz0 + j, 3);
        tma_plane(&tmS36, sm + FT_OFF_S33 + ((j + 1) & 1) * FT_UPL, bar, cx40, cy36, cz0 + j + 1, S33);
    };
    auto issueM = [&](int j) {
        uint64_t* bar = &barM[j % 3];
        mbar_expect_tx(bar, FT_MW * FT_MH * 4);
        tma_plane(&tmM36, sm + FT_OFF_MU + (j % 3) * FT_MPL, bar, cxm, cym, cz0 + j, 1);
    };

    if (tid == 0) { issueL(0); issueE(0); issueE(1); }

    // register windows along z (own column), relative plane j <-> z = zb - 2 + j
    float4 w13a, w13b, w13c;          // s13 at kk-2, kk-1, kk
    float4 w23a, w23b, w23c;          // s23
    float4 w33a, w33b, w33c, w33d;    // s33 at kk-2, kk-1, kk, kk+1
    float4 uo1, uo2, uo3;             // u_old(kk)
    float4 lam, so11, so22, so12;     // lambda, old s11, s22, s12 at ks = kk - 2
    const float4 z4 = f4(0.0f);
    {
        const long long g = (long long)(zb - 2) * a.sz + gxy;
        w13a = ld_ok ? ldg4(in + S13 * box + g - 2 * a.sz) : z4;
        w13b = ld_ok ? ldg4(in + S13 * box + g - a.sz) : z4;
        w13c = ld_ok ? ldg4(in + S13 * box + g) : z4;
        w23a = ld_ok ? ldg4(in + S23 * box + g - 2 * a.sz) : z4;
        w23b = ld_ok ? ldg4(in + S23 * box + g - a.sz) : z4;
        w23c = ld_ok ? ldg4(in + S23 * box + g) : z4;
        w33a = ld_ok ? ldg4(in + S33 * box + g - 2 * a.sz) : z4;
        w33b = ld_ok ? ldg4(in + S33 * box + g - a.sz) : z4;
        w33c = ld_ok ? ldg4(in + S33 * box + g) : z4;
        w33d = ld_ok ? ldg4(in + S33 * box + g + a.sz) : z4;
        uo1 = ld_ok ? ldg4(in + U1 * box + g) : z4;
        uo2 = ld_ok ? ldg4(in + U2 * box + g) : z4;
        uo3 = ld_ok ? ldg4(in + U3 * box + g) : z4;
        lam = so11 = so22 = so12 = z4;
    }
    mbar_wait(&barE[0], 0);

    const float sgn = a.sgn;
    const float* Rbase = sm + FT_OFF_RHO;
    const float* Abase = sm + FT_OFF_ALP;

    for (int it = 0; it < itn; ++it) {
        const int kk = zb - 2 + it;
        if (tid == 0) {
            if (it + 1 < itn) issueL(it + 1);
            if (it + 2 <= itn) issueE(it + 2);
            if (it <= itn - 2) issueM(it);
        }
        mbar_wait(&barL[it & 1], (it >> 1) & 1);
        mbar_wait(&barE[(it + 1) % 3], ((it + 1) / 3) & 1);
        if (it >= 1) mbar_wait(&barM[(it - 1) % 3], ((it - 1) / 3) & 1);

        const int s3 = it % 3, s3n = (it + 1) % 3;
        float4 f13 = z4, f23 = z4, f33 = z4;     // fresh window entries: s13, s23 at kk+1, s33 at kk+2
        // ------------------------------------------------------------------ stage 1: u(kk)
        if (act1) {
            const float* P11 = sm + FT_OFF_S11 + (it & 1) * FT_BOX;
            const float* P22 = sm + FT_OFF_S22 + (it & 1) * FT_BOX;
            const float* P12 = sm + FT_OFF_S12 + (it & 1) * FT_BOX;
            const float* P13 = sm + FT_OFF_S13 + s3 * FT_BOX;
            const float* P23 = sm + FT_OFF_S23 + s3 * FT_BOX;
            const float* PR = Rbase + s3 * FT_BOX;
            const float* PA = Abase + s3 * FT_BOX;
            f13 = ld4s(sm + FT_OFF_S13 + s3n * FT_BOX, q);
            f23 = ld4s(sm + FT_OFF_S23 + s3n * FT_BOX, q);
            f33 = ld4s(sm + FT_OFF_S33 + (it & 1) * FT_UPL, uq);   // plane kk+2 = relative it+2 -> slot (it+2)&1

            // staggered coefficients (reading G10): J = 1 - dt alpha_b, B = dt/(h rho_b)
            const float4 r0 = ld4s(PR, q), a0 = ld4s(PA, q);
            const float4 rxp = shl1(r0, PR[4 * q + 4]), axp = shl1(a0, PA[4 * q + 4]);
            const float4 ryp = ld4s(PR, q + 10), ayp = ld4s(PA, q + 10);
            const float4 rzp = ld4s(Rbase + s3n * FT_BOX, q), azp = ld4s(Abase + s3n * FT_BOX, q);
            const float4 one = f4(1.0f), mh = f4(-0.5f);
            const float4 J1 = fma4(mh, a0 + axp, one), J2 = fma4(mh, a0 + ayp, one), J3 = fma4(mh, a0 + azp, one);
            const float4 B1 = (2.0f * sgn) * rcp4(r0 + rxp), B2 = (2.0f * sgn) * rcp4(r0 + ryp), B3 = (2.0f * sgn) * rcp4(r0 + rzp);

            // nine derivatives of sigma (Eq. 46b)
            const float4 c11 = ld4s(P11, q), c12 = ld4s(P12, q), c22 = ld4s(P22, q);
            float4 d1 = dpx(ld2s(P11, 4 * q - 2), c11, ld2s(P11, 4 * q + 4));                       // D+x s11
            d1 = d1 + d4(ld4s(P12, q - 20), ld4s(P12, q - 10), c12, ld4s(P12, q + 10));             // D-y s12
            d1 = d1 + d4(w13a, w13b, w13c, f13);                                                    // D-z s13
            float4 d2 = dmx(ld2s(P12, 4 * q - 2), c12, ld2s(P12, 4 * q + 4));                       // D-x s12
            d2 = d2 + d4(ld4s(P22, q - 10), c22, ld4s(P22, q + 10), ld4s(P22, q + 20));             // D+y s22
            d2 = d2 + d4(w23a, w23b, w23c, f23);                                                    // D-z s23
            float4 d3 = dmx(ld2s(P13, 4 * q - 2), w13c, ld2s(P13, 4 * q + 4));                      // D-x s13
            d3 = d3 + d4(ld4s(P23, q - 20), ld4s(P23, q - 10), w23c, ld4s(P23, q + 10));            // D-y s23
            d3 = d3 + d4(w33b, w33c, w33d, f33);                                                    // D+z s33

            float4 n1 = fma4(J1, uo1, B1 * d1), n2 = fma4(J2, uo2, B2 * d2), n3 = fma4(J3, uo3, B3 * d3);
            const bool zin = (unsigned)kk < (unsigned)a.nz;
            if (!(zin && m0)) { n1.x = 0.0f; n2.x = 0.0f; n3.x = 0.0f; }
            if (!(zin && m1)) { n1.y = 0.0f; n2.y = 0.0f; n3.y = 0.0f; }
            if (!(zin && m2)) { n1.z = 0.0f; n2.z = 0.0f; n3.z = 0.0f; }
            if (!(zin && m3)) { n1.w = 0.0f; n2.w = 0.0f; n3.w = 0.0f; }
            const int sl = it % FT_RING;
            *reinterpret_cast<float4*>(sm + FT_OFF_UR + (0 * FT_RING + sl) * FT_UPL + 4 * uq) = n1;
            *reinterpret_cast<float4*>(sm + FT_OFF_UR + (1 * FT_RING + sl) * FT_UPL + 4 * uq) = n2;
            *reinterpret_cast<float4*>(sm + FT_OFF_UR + (2 * FT_RING + sl) * FT_UPL + 4 * uq) = n3;
            const long long g = (long long)kk * a.sz + gxy;
            if (inner && kk >= zb && kk < ze) {
                store_quad(a.out + U1 * box + g, n1, x, a.nx);
                store_quad(a.out + U2 * box + g, n2, x, a.nx);
                store_quad(a.out + U3 * box + g, n3, x, a.nx);
            }
            // u_old of the next plane (in flight during stage 2 and the next waits)
            if (ld_ok && it + 1 < itn) {
                uo1 = ldg4(in + U1 * box + g + a.sz);
                uo2 = ldg4(in + U2 * box + g + a.sz);
                uo3 = ldg4(in + U3 * box + g + a.sz);
            }
        }
        __syncthreads();
        // ------------------------------------------------------------------ stage 2: sigma(ks), ks = kk - 2
        const int ks = kk - 2;
        if (inner && it >= 4) {
            const int j = it - 2;             // relative plane of ks
            const float* U1p = sm + FT_OFF_UR + 0 * FT_RING * FT_UPL;
            const float* U2p = sm + FT_OFF_UR + 1 * FT_RING * FT_UPL;
            const float* U3p = sm + FT_OFF_UR + 2 * FT_RING * FT_UPL;
            const int p0 = (j % FT_RING) * FT_UPL, pm1 = ((j + 4) % FT_RING) * FT_UPL, pm2 = ((j + 3) % FT_RING) * FT_UPL;
            const int pp1 = ((j + 1) % FT_RING) * FT_UPL, pp2 = ((j + 2) % FT_RING) * FT_UPL;
            const float4 c1 = ld4s(U1p + p0, uq), c2 = ld4s(U2p + p0, uq), c3 = ld4s(U3p + p0, uq);
            float4 e11 = dmx(ld2s(U1p + p0, 4 * uq - 2), c1, ld2s(U1p + p0, 4 * uq + 4));                        // D-x u1
            float4 g12 = d4(ld4s(U1p + p0, uq - 10), c1, ld4s(U1p + p0, uq + 10), ld4s(U1p + p0, uq + 20));     // D+y u1
            float4 g13 = d4(ld4s(U1p + pm1, uq), c1, ld4s(U1p + pp1, uq), ld4s(U1p + pp2, uq));                 // D+z u1
            float4 g21 = dpx(ld2s(U2p + p0, 4 * uq - 2), c2, ld2s(U2p + p0, 4 * uq + 4));                        // D+x u2
            float4 e22 = d4(ld4s(U2p + p0, uq - 20), ld4s(U2p + p0, uq - 10), c2, ld4s(U2p + p0, uq + 10));     // D-y u2
            float4 g23 = d4(ld4s(U2p + pm1, uq), c2, ld4s(U2p + pp1, uq), ld4s(U2p + pp2, uq));                 // D+z u2
            float4 g31 = dpx(ld2s(U3p + p0, 4 * uq - 2), c3, ld2s(U3p + p0, 4 * uq + 4));                        // D+x u3
            float4 g32 = d4(ld4s(U3p + p0, uq - 10), c3, ld4s(U3p + p0, uq + 10), ld4s(U3p + p0, uq + 20));     // D+y u3
            float4 e33 = d4(ld4s(U3p + pm2, uq), ld4s(U3p + pm1, uq), c3, ld4s(U3p + pp1, uq));                 // D-z u3

            // Lame coefficients: lambda, 2 mu at the node; 4-point harmonic mu at shear points (reading G10)
            const float* M0 = sm + FT_OFF_MU + (j % 3) * FT_MPL;
            const float* M1 = sm + FT_OFF_MU + ((j + 1) % 3) * FT_MPL;
            const float4 i0 = ld4s(M0, mq), iy = ld4s(M0, mq + 9), iz = ld4s(M1, mq), iyz = ld4s(M1, mq + 9);
            const float4 ix = shl1(i0, M0[4 * mq + 4]), ixy = shl1(iy, M0[4 * mq + 40]), ixz = shl1(iz, M1[4 * mq + 4]);
            const float4 mn2 = (2.0f * sgn) * rcp4(i0);
            const float4 mxy = (4.0f * sgn) * rcp4((i0 + ix) + (iy + ixy));
            const float4 mxz = (4.0f * sgn) * rcp4((i0 + ix) + (iz + ixz));
            const float4 myz = (4.0f * sgn) * rcp4((i0 + iy) + (iz + iyz));
            const float4 ldiv = (sgn * lam) * (e11 + e22 + e33);
            const float4 n11 = so11 + fma4(mn2, e11, ldiv);
            const float4 n22 = so22 + fma4(mn2, e22, ldiv);
            const float4 n33 = w33a + fma4(mn2, e33, ldiv);
            const float4 n12 = fma4(mxy, g12 + g21, so12);
            const float4 n13 = fma4(mxz, g13 + g31, w13a);
            const float4 n23 = fma4(myz, g23 + g32, w23a);
            const long long g = (long long)ks * a.sz + gxy;
            store_quad(a.out + S11 * box + g, n11, x, a.nx);
            store_quad(a.out + S22 * box + g, n22, x, a.nx);
            store_quad(a.out + S33 * box + g, n33, x, a.nx);
            store_quad(a.out + S12 * box + g, n12, x, a.nx);
            store_quad(a.out + S13 * box + g, n13, x, a.nx);
            store_quad(a.out + S23 * box + g, n23, x, a.nx);
        }
        if (inner && it >= 3 && it + 1 < itn) {   // own-column inputs of the next stage 2 (plane ks + 1)
            const long long g = (long long)(ks + 1) * a.sz + gxy;
            lam = ldg4(a.mat + g);
            so11 = ldg4(in + S11 * box + g);
            so22 = ldg4(in + S22 * box + g);
            so12 = ldg4(in + S12 * box + g);
        }
        // slide the z windows
        w13a = w13b; w13b = w13c; w13c = f13;
        w23a = w23b; w23b = w23c; w23c = f23;
        w33a = w33b; w33b = w33c; w33c = w33d; w33d = f33;
        __syncthreads();
    }
}
