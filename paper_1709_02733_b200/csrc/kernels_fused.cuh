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
// Fields whose x/y neighbours are needed (s11,s22,s12,s13,s23, rho, alpha, mu), s33 and lambda arrive in
// shared memory by TMA (cp.async.bulk.tensor, mbarrier complete_tx), one or two planes ahead of use;
// u_old(kk) lands by TMA in the very ring slot that u_new(kk) then overwrites in place; the z neighbours
// of s13,s23,s33 (and the oldest u3 tap) live in per-thread registers; the old s11,s22,s12 of stage 2 are
// own-column 128-bit loads issued one stage ahead of use (L2 hits: TMA fetched those planes two
// iterations earlier).  Global loads through the LSU that miss L2 are what this kernel cannot afford.
// The ring of 2 (4) cells around the tile is recomputed by the neighbouring CTAs; nothing is
// exchanged between CTAs, hence the two state buffers.
//
// Synchronisation: ONE __syncthreads per plane (between the stages).  The z taps of stage 2 are
// own-column reads of the u ring, so the only cross-thread reads of a ring slot happen while it is
// the centre plane; TMA refills are issued by thread 0 right after the barrier into slots whose
// last readers finished before it (slot algebra in DESIGN.md "Fused kernel").
//
// C-PML (Eq. 46a,c / 61): memory variables are slab-confined, read from one set and written to the
// other (the tile ring recomputes them without writing).  Forward: the recursion follows the
// difference (own quad only).  Adjoint: the recursion precedes the difference, so the taps of the
// difference along the slab axis are re-derived from the neighbours' old memory variables.
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
#define FT_RH 37                      // rows of the rho / alpha planes: u region + 1
#define FT_RPL 1504                   // floats per rho / alpha plane buffer (40*37 = 1480, padded to 128 B)
#define FT_LPL (FT_TX * FT_TY)        // floats per lambda plane (the tile itself)
// The thread that issues every TMA of the loop.  Warp 11 holds only 8 quads of the u region's last ring row (no stage 2
// work), so its spare lane 12 runs the ~250 instructions of the issue block off the critical path of the other warps.
#ifndef FT_PROD
#define FT_PROD 364
#endif
// Where stage 2 finds the old s11, s22, s12 of its plane (own quad): 0 = s11, s22 as 32 x 32 tile planes by TMA and s12 by
// an own-column load (u ring of 4) ; 1 = three own-column loads ; 2 = parked in tensor memory by stage 1 of the same
// thread two iterations earlier.  1 and 2 free the tile planes for a fifth ring slot: u_old is then requested a whole
// iteration earlier.
// The mode is a property of the kernel (template parameter SOM of the brick routine, FusedMap below).
#define FT_RING 4                     // mode 0: u planes in the ring: ks .. ks+2 and the slot u_old(kk+1) is landing in
// C-PML memory variables stream from HBM and are used right after they are requested: each thread asks for the record
// it will load FT_PFMV planes later to be brought into L2 (measured at 512^3: 2 planes ahead -2 % forward, -5 % adjoint
// slab launch; 1, 3, 4 planes ahead and L1 prefetches did not pay)
#ifndef FT_PFMV
#define FT_PFMV 2
#endif
// Windows in tensor memory (WT): the z windows of s13, s23, s33 (10 quads per thread) live in tensor memory instead of
// registers; every warp then executes stage 1 convergently (the 24 spare lanes of warp 11 compute on in-range
// shared-memory garbage and store nothing), because tcgen05.ld / st are warp-wide instructions.
// Measured at 512^3: C-PML kernels -14 % (adjoint) / -3 % (forward) and room for SO mode 2 there (-7 % / -2 % more) ; the
// C-PML-free kernel +3.5 % (it has no register shortage to relieve), so only the C-PML kernels use it.
#ifndef FT_WT_PML
#define FT_WT_PML 1
#endif
#ifndef FT_WT_PLAIN
#define FT_WT_PLAIN 0
#endif
#define FT_WT(MODE) ((MODE) == FM_PLAIN ? FT_WT_PLAIN : FT_WT_PML)
// Adjoint, z slabs (FT_ZX 1, needs WT): the filtered increment X = a T of a plane is computed once, when the plane enters
// the z window as its newest tap (one load of the old T, requested at the top of the iteration), and kept in a TMEM ring
// of four planes per term ; the other three taps of the transposed recursion come from that ring instead of three more
// loads per term and plane whose latency sat in front of every use.  Stage 1 terms (sigma13, sigma23, sigma33).
#ifndef FT_ZX
#define FT_ZX 1
#endif
// columns per warp with WT: parked old s11, s22, s12, s33 3 x 16 | s13 ring 16 | s23 ring 16 | s33 ring 16 | X rings of
// stage 1 3 x 12 | X rings of stage 2 3 x 12  (3 warps per lane quarter: 504 of 512 columns)
#define FT_TM_WARP 168
#define FT_TMEM_COLS_X 512
#define FT_TMEM_COLS 128              // tensor-memory columns allocated per CTA (mode 2): 3 warps per lane quarter x 36

// shared memory map (floats).  Planes are only as tall as their readers need: s11, s13 (x neighbours only) and
// s33 (own column) cover the u region (36 rows), rho / alpha one row more, s22, s12, s23 the full 40.
#define FT_OFF_S22 0
#define FT_OFF_S12 (FT_OFF_S22 + 2 * FT_BOX)
#define FT_OFF_S11 (FT_OFF_S12 + 2 * FT_BOX)
#define FT_OFF_S13 (FT_OFF_S11 + 2 * FT_UPL)
#define FT_OFF_S23 (FT_OFF_S13 + 3 * FT_UPL)
#define FT_OFF_RHO (FT_OFF_S23 + 3 * FT_BOX)
#define FT_OFF_ALP (FT_OFF_RHO + 3 * FT_RPL)
#define FT_OFF_S33 (FT_OFF_ALP + 3 * FT_RPL)
#define FT_OFF_MU (FT_OFF_S33 + 2 * FT_UPL)
#define FT_OFF_LAM (FT_OFF_MU + 3 * FT_MPL)
#define FT_OFF_SO (FT_OFF_LAM + 2 * FT_LPL)       // old s11, s22 of plane ks (tile only): [slot][field]
#define FT_OFF_UR (FT_OFF_SO + 4 * FT_LPL)
#define FT_OFF_END (FT_OFF_UR + 3 * FT_RING * FT_UPL)
#define FT_TABW 48                     // x / y C-PML table window: tile - 8 .. tile + 39
#define FT_ZRING 16                   // z C-PML table ring (planes)
#define FT_OFF_XT (FT_OFF_END + 16)   // after 8 mbarriers (64 B)
#define FT_OFF_YT (FT_OFF_XT + 4 * FT_TABW)
#define FT_OFF_ZT (FT_OFF_YT + 4 * FT_TABW)
// the tail of the map for a given SO mode: modes 1, 2 trade the four old-stress tile planes for a fifth ring slot
template <int SOM>
struct FusedMap {
    static constexpr int RING = SOM == 0 ? 4 : 5;      // ... and the slots of u_old(kk+1) (landed), u_old(kk+2) (landing)
    static constexpr int ULEAD = RING - 3;             // u_old(c) is requested after the block barrier of iteration c - ULEAD
    static constexpr int OFF_UR = FT_OFF_SO + (SOM == 0 ? 4 : 0) * FT_LPL;
    static constexpr int OFF_END = OFF_UR + 3 * RING * FT_UPL;
    static constexpr int OFF_XT = OFF_END + 16;
    static constexpr int OFF_YT = OFF_XT + 4 * FT_TABW;
    static constexpr int OFF_ZT = OFF_YT + 4 * FT_TABW;
    static constexpr int OFF_TICKET = OFF_ZT + 4 * FT_ZRING;   // the work-queue ticket, then the tensor-memory base address
    static constexpr int BYTES = (OFF_TICKET + 4) * 4;
};
#define FT_SMEM_BYTES (FusedMap<2>::BYTES > FusedMap<0>::BYTES ? FusedMap<2>::BYTES : FusedMap<0>::BYTES)
static_assert(FT_SMEM_BYTES <= 232448, "shared-memory map exceeds 227 KB");
// SO mode of the kernel that carries C-PML mode MODE (the C-PML kernels need WT for mode 2: registers)
#ifndef FT_SOM_PML
#define FT_SOM_PML 2
#endif
#ifndef FT_SOM_PLAIN
#define FT_SOM_PLAIN 2
#endif
#define FT_SOM(MODE) ((MODE) == FM_PLAIN ? FT_SOM_PLAIN : FT_SOM_PML)

// kernel modes: which C-PML code a launch carries (CTAs away from the slabs skip it at run time)
#define FM_PLAIN 0     // no C-PML (npml = 0)
#define FM_FWD 1       // W'   : Eq. 46a-d, memory variables updated after differencing
#define FM_ADJ 2       // W'^T : Eq. 61, memory variables (tilde form) applied before differencing

#define FT_WORK_SLAB 0x10000           // flag in work[b].x: the brick touches a C-PML slab (runs the launch's C-PML code)
#define FT_WORK_NOEDGE 0x20000         // flag in work[b].x: u region, taps and planes zb-2 .. ze+1 lie inside the grid (no lane masks)

struct FusedArgs {
    int nx, ny, nz;
    const int4* work;      // brick b: tile (work[b].x & 0xffff, work[b].y), planes [work[b].z, work[b].w) ; FT_WORK_SLAB flag in .x
    int work_begin, work_end;   // the launch processes bricks [work_begin, work_end) of the list, in list order
    unsigned int* queue;   // [2]: next brick (relative to work_begin), CTAs that left ; both reset by the last CTA to leave
    long long sy, sz, box; // strides (elements) of the padded box; elements per field
    const float* in;       // state read  (field k at in + k*box; pointer to node (0,0,0))
    float* out;            // state written
    // Material elision: mflag[(tile y * ntx + tile x) * nzp + z + HALO_Z] is
    // 0, or 1 + p when all four scaled materials are constant over the tile's whole box on plane z and equal palette
    // entry p; such planes are fetched from palette plane p (padded z index mpal + p: the same bytes, always in L2)
    // instead of their own plane in HBM.  NULL = no elision.
    const unsigned char* mflag;
    int ntx, nzp, mpal;
    float sgn;             // +1: W' on (u, sigma) ; -1: W'^T on the scaled adjoint variables
    // C-PML
    int P;
    const float* tab[3][4];
    int xl, xr, wx;        // x slab: columns [0,xl) and [xr, nxq) ; wx = xl + nxq - xr ; quad aligned
    int nxq;               // nx rounded up to a multiple of 4
    int wyz;               // slab width along y and z: 2P+1
    const float* mvi[18];  // memory variables read:  phi[3a+b] = [0..9), psi[3a+b] = [9..18)   (fluid-only kernels)
    float* mvo[18];        // memory variables written
    // The elastic kernels see the same storage as six groups g = 3 * kind + b (kind 0: phi, 1: psi ; b = slab axis), the
    // three components a of a quad interleaved: float offset 3 * o + 4 * a, o = the quad's offset in the layout above.
    // One address per axis and stage then serves three loads and three stores (immediate offsets 0, 16, 32 bytes).
    const float* mgi[6];
    float* mgo[6];
};

// ---- PTX wrappers: mbarrier + TMA (SASS: SYNCS.*, UTMALDG) --------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_inval(uint64_t* bar)
{
    asm volatile("mbarrier.inval.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
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

// ---- tensor memory as per-thread scratch (SASS: STTM / LDTM): 32x32b = lane <-> thread, 4 consecutive 32-bit columns
__device__ __forceinline__ void tmem_st4(uint32_t taddr, float4 v)
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};"
                 ::"r"(taddr), "r"(__float_as_uint(v.x)), "r"(__float_as_uint(v.y)), "r"(__float_as_uint(v.z)), "r"(__float_as_uint(v.w)) : "memory");
}
__device__ __forceinline__ float4 tmem_ld4(uint32_t taddr)
{
    uint32_t x, y, z, w;
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(x), "=r"(y), "=r"(z), "=r"(w) : "r"(taddr) : "memory");
    return make_float4(__uint_as_float(x), __uint_as_float(y), __uint_as_float(z), __uint_as_float(w));
}
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// ---- float4 helpers -----------------------------------------------------------------------------
__device__ __forceinline__ float4 ld4s(const float* p, int quad) { return *reinterpret_cast<const float4*>(p + 4 * quad); }
__device__ __forceinline__ float2 ld2s(const float* p, int off) { return *reinterpret_cast<const float2*>(p + off); }
__device__ __forceinline__ float4 f4(float v) { return make_float4(v, v, v, v); }
// Packed fp32 arithmetic of sm_100 (PTX add/sub/mul/fma .f32x2 -> SASS FADD2 / FMUL2 / FFMA2): one instruction works on
// an aligned register pair, i.e. on half a quad, with the rounding of the scalar instruction.  The step kernels are
// bound by issue slots and latency, not by the FMA pipe, so halving the lane-parallel arithmetic instructions pays.
// The (x,y) and (z,w) halves of a float4 that came from a 128-bit load are aligned pairs already (no moves).
#define FT_X2_OP(name, op)                                                                                          \
    __device__ __forceinline__ void name(float& d0, float& d1, float a0, float a1, float b0, float b1)              \
    {                                                                                                               \
        asm("{\n\t.reg .b64 ra, rb, rd;\n\tmov.b64 ra, {%2, %3};\n\tmov.b64 rb, {%4, %5};\n\t" op                    \
            " rd, ra, rb;\n\tmov.b64 {%0, %1}, rd;\n\t}"                                                            \
            : "=f"(d0), "=f"(d1) : "f"(a0), "f"(a1), "f"(b0), "f"(b1));                                             \
    }
FT_X2_OP(add2, "add.rn.f32x2")
FT_X2_OP(sub2, "sub.rn.f32x2")
FT_X2_OP(mul2, "mul.rn.f32x2")
__device__ __forceinline__ void fma2(float& d0, float& d1, float a0, float a1, float b0, float b1, float c0, float c1)
{
    asm("{\n\t.reg .b64 ra, rb, rc, rd;\n\tmov.b64 ra, {%2, %3};\n\tmov.b64 rb, {%4, %5};\n\tmov.b64 rc, {%6, %7};\n\t"
        "fma.rn.f32x2 rd, ra, rb, rc;\n\tmov.b64 {%0, %1}, rd;\n\t}"
        : "=f"(d0), "=f"(d1) : "f"(a0), "f"(a1), "f"(b0), "f"(b1), "f"(c0), "f"(c1));
}
__device__ __forceinline__ float4 operator+(float4 a, float4 b) { float4 d; add2(d.x, d.y, a.x, a.y, b.x, b.y); add2(d.z, d.w, a.z, a.w, b.z, b.w); return d; }
__device__ __forceinline__ float4 operator-(float4 a, float4 b) { float4 d; sub2(d.x, d.y, a.x, a.y, b.x, b.y); sub2(d.z, d.w, a.z, a.w, b.z, b.w); return d; }
__device__ __forceinline__ float4 operator*(float4 a, float4 b) { float4 d; mul2(d.x, d.y, a.x, a.y, b.x, b.y); mul2(d.z, d.w, a.z, a.w, b.z, b.w); return d; }
__device__ __forceinline__ float4 operator*(float a, float4 b) { float4 d; mul2(d.x, d.y, a, a, b.x, b.y); mul2(d.z, d.w, a, a, b.z, b.w); return d; }
__device__ __forceinline__ float4 fma4(float4 a, float4 b, float4 c)
{
    float4 d; fma2(d.x, d.y, a.x, a.y, b.x, b.y, c.x, c.y); fma2(d.z, d.w, a.z, a.w, b.z, b.w, c.z, c.w); return d;
}
__device__ __forceinline__ float4 fma4(float a, float4 b, float4 c)
{
    float4 d; fma2(d.x, d.y, a, a, b.x, b.y, c.x, c.y); fma2(d.z, d.w, a, a, b.z, b.w, c.z, c.w); return d;
}
// lane-wise sum where one operand is not pair aligned (a quad shifted by one lane): scalar adds, no register moves
__device__ __forceinline__ float4 adds(float4 a, float4 b) { return make_float4(a.x + b.x, a.y + b.y, a.z + b.z, a.w + b.w); }
// the value one x to the right of each lane of `c`, `r0` being the element after c.w
__device__ __forceinline__ float4 shl1(float4 c, float r0) { return make_float4(c.y, c.z, c.w, r0); }
// 1/x by the special-function unit (MUFU.RCP, <= 1 ulp): 1/inf = 0 (fluid: mu = 0), 1/0 = inf
__device__ __forceinline__ float rcpa(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float4 rcp4(float4 a) { return make_float4(rcpa(a.x), rcpa(a.y), rcpa(a.z), rcpa(a.w)); }

// Eq. 8 without 1/h and divided by c2 = -1/24 (both folded into the scaled
// coefficients):  (9/8 (t2 - t1) - 1/24 (t3 - t0)) / c2 = (t3 - t0) - 27 (t2 - t1).
// Taps t0..t3 at consecutive samples: D+ at i uses (i-1, i, i+1, i+2) ; D- at i uses (i-2, i-1, i, i+1).
#define FT_K 27.0f
__device__ __forceinline__ float d1(float t0, float t1, float t2, float t3) { return fmaf(-FT_K, t2 - t1, t3 - t0); }
__device__ __forceinline__ float4 d4(float4 t0, float4 t1, float4 t2, float4 t3) { return fma4(-FT_K, t2 - t1, t3 - t0); }
// along x on a quad c = f[0..3]: l = (f[-2], f[-1]), r = (f[4], f[5])
__device__ __forceinline__ float4 dpx(float2 l, float4 c, float2 r)   // D+ : result at i + 1/2
{
    return make_float4(d1(l.y, c.x, c.y, c.z), d1(c.x, c.y, c.z, c.w), d1(c.y, c.z, c.w, r.x), d1(c.z, c.w, r.x, r.y));
}
__device__ __forceinline__ float4 dmx(float2 l, float4 c, float2 r)   // D- : result at i
{
    return make_float4(d1(l.x, l.y, c.x, c.y), d1(l.y, c.x, c.y, c.z), d1(c.x, c.y, c.z, c.w), d1(c.y, c.z, c.w, r.x));
}

__device__ __forceinline__ float4 ldg4(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }
// Predicated 128-bit load INTO the registers of v (no copy of the loaded value, so that the scoreboard
// wait lands on the first real use, a stage later, and not on a loop-carried register move).
__device__ __forceinline__ void ldg4_into(float4& v, const float* p, bool pred)
{
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %5, 0;\n\t"
        "@p ld.global.nc.v4.f32 {%0, %1, %2, %3}, [%4];\n\t"
        "}"
        : "+f"(v.x), "+f"(v.y), "+f"(v.z), "+f"(v.w)
        : "l"(p), "r"((int)pred));
}
// request the line at p into L2 (no register, no scoreboard)
__device__ __forceinline__ void prefetch_l2(const float* p, bool pred)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %1, 0;\n\t@p prefetch.global.L2 [%0];\n\t}" ::"l"(p), "r"((int)pred) : "memory");
}
// 128-bit store that does not allocate in L1 (st.global.cg): the step kernels leave ~20 KB of L1 beside their shared
// memory, and the default write-allocating stores of the nine output fields kept evicting what little of it the loads
// use (interior launch -4 % at 512^3 ; .cs and .wt measured within 1 % of it)
__device__ __forceinline__ void stg4(float* p, float4 v)
{
    asm volatile("st.global.cg.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}

// store the in-grid lanes of a quad starting at column x (EDGE = false: the whole quad is in the grid)
template <bool EDGE = true>
__device__ __forceinline__ void store_quad(float* p, float4 v, int x, int nx)
{
    if (!EDGE || x + 3 < nx) { stg4(p, v); return; }
    if (x < nx) p[0] = v.x;
    if (x + 1 < nx) p[1] = v.y;
    if (x + 2 < nx) p[2] = v.z;
}

// ---- C-PML pieces ---------------------------------------------------------------------------------
// Memory variables are stored slab-compressed, quad aligned in x (FusedArgs):
//   axis x: [nz][ny][wx]   columns [0,xl) U [xr,nxq)      axis y: [nz][wyz][nxq]      axis z: [wyz][ny][nxq]
// slab column of the quad starting at grid column x (multiple of 4), or -1
__device__ __forceinline__ int xslab_col(const FusedArgs& a, int x)
{
    if (x < 0 || x >= a.nxq) return -1;
    if (x < a.xl) return x;
    if (x >= a.xr) return a.xl + (x - a.xr);
    return -1;
}
// slab row of index i on an axis of length n (y or z), or -1
__device__ __forceinline__ int yzslab_row(int i, int n, int P)
{
    if (i < 0 || i >= n) return -1;
    if (i < P) return i;
    if (i >= n - 1 - P) return i - (n - 1 - P) + P;
    return -1;
}
__device__ __forceinline__ long long idx_x(const FusedArgs& a, int col, int y, int z) { return ((long long)z * a.ny + y) * a.wx + col; }
__device__ __forceinline__ long long idx_y(const FusedArgs& a, int x, int row, int z) { return ((long long)z * a.wyz + row) * a.nxq + x; }
__device__ __forceinline__ long long idx_z(const FusedArgs& a, int x, int y, int row) { return ((long long)row * a.ny + y) * a.nxq + x; }

// The C-PML tables (Eq. 38) of the CTA's x / y window and a ring of z planes are staged in shared
// memory (zeros outside the grid: a = 0 means no C-PML term ; b = 0 only ever multiplies zeros).
// Helpers take pointers pre-offset so that t[i] is the value at grid index i (z: t[i & 15]).
__device__ __forceinline__ float4 tab4(const float* t, int x) { return *reinterpret_cast<const float4*>(t + x); }

// Forward recursion on the thread's own quad (Eq. 46a / 46c with Eq. 38): m <- b m + a t ; returns t + m
__device__ __forceinline__ float4 pml_fwd(const float* mi, float* mo, long long idx, float4 a4, float4 b4, float4 t, bool wr)
{
    const float4 m = fma4(b4, ldg4(mi + idx), a4 * t);
    if (wr) stg4(mo + idx, m);
    return t + m;
}
__device__ __forceinline__ float4 pml_fwd(const float* mi, float* mo, long long idx, float a1, float b1, float4 t, bool wr)
{
    const float4 m = fma4(b1, ldg4(mi + idx), a1 * t);
    if (wr) stg4(mo + idx, m);
    return t + m;
}

// same with the old value already in registers (loaded a barrier earlier)
__device__ __forceinline__ float4 pml_fwd_m(float4 m_old, float* mo, long long idx, float4 a4, float4 b4, float4 t, bool wr)
{
    const float4 m = fma4(b4, m_old, a4 * t);
    if (wr) stg4(mo + idx, m);
    return t + m;
}
__device__ __forceinline__ float4 pml_fwd_m(float4 m_old, float* mo, long long idx, float a1, float b1, float4 t, bool wr)
{
    const float4 m = fma4(b1, m_old, a1 * t);
    if (wr) stg4(mo + idx, m);
    return t + m;
}

// Transposed recursion in tilde form (Eq. 61b / 61d-g): T <- b T + s at the
// sample, and the differenced quantity is s + a T.  The a T part ("X") is needed at every tap of
// the difference along the slab axis, so it is re-derived from the neighbours' old T.
// X along y: rows r0..r0+3 of plane z at the thread's quad ; tap `own` is the thread's own row.  Returns d4 of X.
// The four loads are predicated, not branched around, so that they issue back to back.
__device__ __forceinline__ float4 adj_y(const FusedArgs& a, const float* __restrict__ Ti, float* __restrict__ To,
                                        const float* __restrict__ ta, const float* __restrict__ tb,
                                        int x, int r0, int z, int own, float4 s0, float4 s1, float4 s2, float4 s3, bool wr)
{
    const float4 s[4] = {s0, s1, s2, s3};
    float4 T[4];
    long long i[4];
    bool in[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int p = yzslab_row(r0 + k, a.ny, a.P);
        in[k] = p >= 0;
        i[k] = in[k] ? idx_y(a, x, p, z) : 0;
        T[k] = f4(0.0f);
        ldg4_into(T[k], Ti + i[k], in[k]);
    }
    float4 X[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const float bk = in[k] ? tb[r0 + k] : 0.0f, ak = in[k] ? ta[r0 + k] : 0.0f;
        const float4 Tn = fma4(bk, T[k], s[k]);
        if (wr && k == own && in[k]) stg4(To + i[k], Tn);
        X[k] = ak * Tn;
    }
    return d4(X[0], X[1], X[2], X[3]);
}
// X along z: planes z0..z0+3 at the thread's quad of row y
__device__ __forceinline__ float4 adj_z(const FusedArgs& a, const float* __restrict__ Ti, float* __restrict__ To,
                                        const float* __restrict__ ta, const float* __restrict__ tb,
                                        int x, int y, int z0, int own, float4 s0, float4 s1, float4 s2, float4 s3, bool wr)
{
    const float4 s[4] = {s0, s1, s2, s3};
    float4 T[4];
    long long i[4];
    bool in[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int p = yzslab_row(z0 + k, a.nz, a.P);
        in[k] = p >= 0;
        i[k] = in[k] ? idx_z(a, x, y, p) : 0;
        T[k] = f4(0.0f);
        ldg4_into(T[k], Ti + i[k], in[k]);
    }
    float4 X[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const float bk = tb[(z0 + k) & (FT_ZRING - 1)], ak = in[k] ? ta[(z0 + k) & (FT_ZRING - 1)] : 0.0f;
        const float4 Tn = fma4(bk, T[k], s[k]);
        if (wr && k == own && in[k]) stg4(To + i[k], Tn);
        X[k] = ak * Tn;
    }
    return d4(X[0], X[1], X[2], X[3]);
}
// the same with the old T already in registers (loaded ahead of a barrier)
__device__ __forceinline__ float4 adj_own_x(float4 Told, float* To, long long i, bool in_slab, float4 a4, float4 b4, float4 s, bool wr)
{
    if (!in_slab) return f4(0.0f);
    const float4 Tn = fma4(b4, Told, s);
    if (wr) stg4(To + i, Tn);
    return a4 * Tn;
}
// ---- the same pieces on the interleaved layout (FusedArgs::mgi / mgo) with 32-bit float offsets --------------------
// Forward recursion, branch-free: outside the slab a = 0 and the old value is 0, so m = 0 and t is returned unchanged.
// `mo` points at the quad's record (component offset included).
__device__ __forceinline__ float4 pml_fwd_p(float4 m_old, float* mo, float4 a4, float4 b4, float4 t, bool wr)
{
    const float4 m = fma4(b4, m_old, a4 * t);
    if (wr) stg4(mo, m);
    return t + m;
}
__device__ __forceinline__ float4 pml_fwd_p(float4 m_old, float* mo, float a1, float b1, float4 t, bool wr)
{
    const float4 m = fma4(b1, m_old, a1 * t);
    if (wr) stg4(mo, m);
    return t + m;
}
// X along y: rows r0..r0+3 ; obase = float offset of (row 0 of the y slab, own x) on the plane ; rs = floats per slab row
__device__ __forceinline__ float4 adj_y3(const FusedArgs& a, const float* __restrict__ Ti, float* __restrict__ To,
                                         const float* __restrict__ ta, const float* __restrict__ tb,
                                         int obase, int rs, int r0, int own, float4 s0, float4 s1, float4 s2, float4 s3, bool wr)
{
    const float4 s[4] = {s0, s1, s2, s3};
    float4 T[4];
    int i[4];
    bool in[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int p = yzslab_row(r0 + k, a.ny, a.P);
        in[k] = p >= 0;
        i[k] = in[k] ? obase + p * rs : 0;
        T[k] = f4(0.0f);
        ldg4_into(T[k], Ti + i[k], in[k]);
    }
    float4 X[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const float bk = in[k] ? tb[r0 + k] : 0.0f, ak = in[k] ? ta[r0 + k] : 0.0f;
        const float4 Tn = fma4(bk, T[k], s[k]);
        if (wr && k == own && in[k]) stg4(To + i[k], Tn);
        X[k] = ak * Tn;
    }
    return d4(X[0], X[1], X[2], X[3]);
}
// X along z: planes z0..z0+3 ; oq = float offset of the own quad on slab row 0 ; rs = floats per slab row (plane)
__device__ __forceinline__ float4 adj_z3(const FusedArgs& a, const float* __restrict__ Ti, float* __restrict__ To,
                                         const float* __restrict__ ta, const float* __restrict__ tb,
                                         int oq, int rs, int z0, int own, float4 s0, float4 s1, float4 s2, float4 s3, bool wr)
{
    const float4 s[4] = {s0, s1, s2, s3};
    float4 T[4];
    int i[4];
    bool in[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int p = yzslab_row(z0 + k, a.nz, a.P);
        in[k] = p >= 0;
        i[k] = in[k] ? oq + p * rs : 0;
        T[k] = f4(0.0f);
        ldg4_into(T[k], Ti + i[k], in[k]);
    }
    float4 X[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const float bk = tb[(z0 + k) & (FT_ZRING - 1)], ak = in[k] ? ta[(z0 + k) & (FT_ZRING - 1)] : 0.0f;
        const float4 Tn = fma4(bk, T[k], s[k]);
        if (wr && k == own && in[k]) stg4(To + i[k], Tn);
        X[k] = ak * Tn;
    }
    return d4(X[0], X[1], X[2], X[3]);
}
// own quad, old T already in registers ; `To` points at the quad's record
__device__ __forceinline__ float4 adj_own_p(float4 Told, float* To, bool in_slab, float4 a4, float4 b4, float4 s, bool wr)
{
    if (!in_slab) return f4(0.0f);
    const float4 Tn = fma4(b4, Told, s);
    if (wr) stg4(To, Tn);
    return a4 * Tn;
}
// =================================================================================================
// The fused step.  MODE selects the C-PML code carried by the launch (FM_*); see DESIGN.md for the
// index algebra.  Relative plane j <-> z = zb - 2 + j ; iteration `it` computes u(kk = zb - 2 + it)
// and sigma(ks = kk - 2).
// EDGE = false: the host vouches (FT_WORK_NOEDGE) that nothing this brick touches sticks out of the grid, so the lane
// masks, the in-grid tests of the stores and the z range tests are compiled out.
template <int MODE, bool EDGE, int SOM, bool WT>
__device__ __forceinline__ void fused_brick(float* __restrict__ sm, const CUtensorMap& tmS40, const CUtensorMap& tmS36,
                                            const CUtensorMap& tmM37, const CUtensorMap& tmM36, const CUtensorMap& tmL,
                                            const CUtensorMap& tmS32, const FusedArgs& a, const int4 wk, const bool first,
                                            const uint32_t tmem_base)
{
    constexpr int RING = FusedMap<SOM>::RING, ULEAD = FusedMap<SOM>::ULEAD, OFF_UR = FusedMap<SOM>::OFF_UR;
    constexpr int OFF_END = FusedMap<SOM>::OFF_END, OFF_XT = FusedMap<SOM>::OFF_XT, OFF_YT = FusedMap<SOM>::OFF_YT, OFF_ZT = FusedMap<SOM>::OFF_ZT;
    uint64_t* bars = reinterpret_cast<uint64_t*>(sm + OFF_END);
    uint64_t* barG = bars;        // [2]  everything first read by stage 1 of iteration c -> slot c & 1
    uint64_t* barM = bars + 2;    // [3]  mu of plane j -> slot j % 3
    uint64_t* barU = bars + 5;    // [2]  u_old of plane c, landed in ring slot c % RING -> barrier c & 1

    const int tid = threadIdx.x;
    const int zb = wk.z, ze = wk.w;
    const int x0 = (wk.x & 0xffff) * FT_TX, y0 = wk.y * FT_TY;
    const int itn = ze - zb + 4;            // iterations: u planes kk = zb-2 .. ze+1

    // thread -> quad of the u region (10 quads x 36 rows)
    const bool act1 = tid < 360;
    const int qx = tid % 10, r = tid / 10;
    const int x = x0 - 4 + 4 * qx, y = y0 - 2 + r;
    const bool inner = act1 && qx >= 1 && qx <= 8 && r >= 2 && r < 34 && (!EDGE || (x < a.nx && y < a.ny));
    const int q = tid + 20;                 // quad index in a 40x40 plane (two rows further down)
    const int uq = tid;                     // quad index in a 40x36 plane
    // SOM 2: the thread's tensor-memory scratch (lane = its lane in the warp's lane quarter ; 36 columns per warp:
    // [plane % 3][s11, s22, s12][4]).  Warp 11 holds no tile quad and takes no part (its u-region lanes diverge).
    const bool tmw = SOM == 2 && (WT || tid < 352);
    const uint32_t tm0 = tmem_base + ((uint32_t)((tid >> 5) & 3) << 21) + (uint32_t)(tid >> 7) * (WT ? FT_TM_WARP : 36u);
    const uint32_t tW13 = tm0 + 48u, tW23 = tm0 + 64u, tW33 = tm0 + 80u;      // WT: ring slots of 4 columns, plane j -> j & 3
    constexpr uint32_t SOS = WT ? 16u : 12u;      // columns per parking slot (WT: the old s33 is parked as well)
    constexpr bool ZX = FT_ZX != 0 && WT && MODE == FM_ADJ;
    const uint32_t tXZ = tm0 + 96u;       // ZX: X rings of sigma13, sigma23, sigma33 (12 columns each), plane j -> j mod 3
    const int mq = (r - 2) * 9 + (qx - 1);  // quad index in a mu plane (inner threads)
    // own-column global loads are legal where the padded box has storage
    const bool ld_ok = act1 && (!EDGE || ((y + PACT_HALO_Y < a.ny + 2 * PACT_HALO_Y) && (x + 3 + PACT_HALO_X < (int)a.sy)));
    const long long gxy = (long long)y * a.sy + x;
    // lanes of the quad that are grid points (u outside the grid is zero: reading G9)
    const bool yin = (unsigned)y < (unsigned)a.ny;
    const bool m0 = yin && (unsigned)x < (unsigned)a.nx, m1 = yin && (unsigned)(x + 1) < (unsigned)a.nx;
    const bool m2 = yin && (unsigned)(x + 2) < (unsigned)a.nx, m3 = yin && (unsigned)(x + 3) < (unsigned)a.nx;
    // the CTA's u region sticks out of the grid in x or y (then lanes are masked every plane)
    const bool edge_xy = EDGE && (x0 == 0 || y0 == 0 || x0 + FT_TX + 4 > a.nx || y0 + FT_TY + 2 > a.ny);

    // C-PML: does the CTA's region (plus the taps of the adjoint) touch the x / y slabs; own-quad slab positions
    const bool pml = MODE != FM_PLAIN && a.P > 0;
    const bool bx = pml && (x0 - 8 < a.xl || x0 + FT_TX + 8 > a.xr);
    const bool by = pml && (y0 - 4 < a.P || y0 + FT_TY + 4 > a.ny - 1 - a.P);
    const bool pok = pml && act1 && x >= 0 && x < a.nxq && yin;     // quad has memory-variable storage (given z in range)
    const int colq = pok ? xslab_col(a, x) : -1;
    const int prow = pok ? yzslab_row(y, a.ny, a.P) : -1;
    // adjoint: does any tap of this thread's differences along y fall into a slab (x taps always go through the
    // shared-memory exchange: a CTA that touches the x slabs takes x as its exchange axis)
    const bool neary = pok && (y - 2 < a.P || y + 2 >= a.ny - 1 - a.P);

    // adjoint: slab axis whose filtered taps this CTA exchanges through shared memory (x if it touches the x slabs,
    // else y), -1 = none.  CTA-uniform: it adds block barriers.
    const int exa = (MODE == FM_ADJ) ? (bx ? 0 : (by ? 1 : -1)) : -1;
    // Memory variables (interleaved layout): running float offsets of the own quad's record at plane kk in the x and y
    // slabs, of row 0 of the y slab (adjoint taps), and the plane-independent part in the z slabs.  32 bits suffice
    // (pact_create checks) and one add per plane replaces the 64-bit index products.
    const bool hx = pok && colq >= 0, hy = pok && prow >= 0;
    const int sxp = 3 * a.ny * a.wx, syp = 3 * a.wyz * a.nxq, szp = 3 * a.ny * a.nxq, rsy = 3 * a.nxq;
    int ox = hx ? 3 * (((zb - 2) * a.ny + y) * a.wx + colq) : 0;
    int oy = hy ? 3 * (((zb - 2) * a.wyz + prow) * a.nxq + x) : 0;
    int oyb = pok ? 3 * ((zb - 2) * a.wyz * a.nxq + x) : 0;
    const int ozq = pok ? 3 * (y * a.nxq + x) : 0;

    const float* in = a.in;
    const long long box = a.box;

    if (pml) {   // stage the C-PML tables: x / y windows and the first planes of the z ring (zeros outside the grid)
        for (int i = tid; i < 4 * FT_TABW; i += FT_NT) {
            const int t = i / FT_TABW, o = i % FT_TABW - 8;
            sm[OFF_XT + i] = (unsigned)(x0 + o) < (unsigned)a.nx ? __ldg(a.tab[0][t] + x0 + o) : 0.0f;
            sm[OFF_YT + i] = (unsigned)(y0 + o) < (unsigned)a.ny ? __ldg(a.tab[1][t] + y0 + o) : 0.0f;
        }
        if (tid < 4 * 12) {     // planes zb - 10 .. zb + 1 ; the loop adds plane kk + 3 = zb + 1 + it every iteration
            const int t = tid / 12, z = zb - 10 + tid % 12;
            sm[OFF_ZT + t * FT_ZRING + (z & (FT_ZRING - 1))] = (unsigned)z < (unsigned)a.nz ? __ldg(a.tab[2][t] + z) : 0.0f;
        }
    }
    if (tid == 0) {   // fresh barriers per brick (every transaction of the previous brick was waited for)
        for (int k = 0; k < 8; ++k) {
            if (!first) mbar_inval(&bars[k]);
            mbar_init(&bars[k], 1);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();

    const int cx40 = x0 - 4 + PACT_HALO_X, cy40 = y0 - 4 + PACT_HALO_Y, cy36 = y0 - 2 + PACT_HALO_Y;
    const int cxm = x0 + PACT_HALO_X, cym = y0 + PACT_HALO_Y;
    const int cz0 = zb - 2 + PACT_HALO_Z;   // padded z of relative plane j = 0
    // material-plane flags of this tile, relative plane j at mfl[j] (thread 0 only reads them)
    const unsigned char* mfl = a.mflag ? a.mflag + ((size_t)wk.y * a.ntx + (wk.x & 0xffff)) * a.nzp + cz0 : nullptr;
    auto mflag_at = [&](int j) -> unsigned { return mfl ? (unsigned)__ldg(mfl + j) : 0u; };
    // padded z of the material plane to fetch for relative plane j, given its flag
    auto mz = [&](int j, unsigned f) { return f ? a.mpal + (int)f - 1 : cz0 + j; };
    // flags of the planes the next issues need, newest in the low byte: after the update in iteration `it`
    // byte 0 = plane it + 3, ..., byte 3 = plane it, byte 4 = plane it - 1
    unsigned long long fh = 0;

    // E(j): s13, s23, rho, alpha of plane j -> slot j % 3 ; f = material flag of plane j ; keep = the slot already
    // holds this plane's rho and alpha (the plane three below came from the same palette plane): nothing to fetch
    auto issueE = [&](int j, uint64_t* bar, unsigned f, bool keep) {
        const int s = j % 3;
        tma_plane(&tmS36, sm + FT_OFF_S13 + s * FT_UPL, bar, cx40, cy36, cz0 + j, S13);
        tma_plane(&tmS40, sm + FT_OFF_S23 + s * FT_BOX, bar, cx40, cy40, cz0 + j, S23);
        if (!keep) {
            tma_plane(&tmM37, sm + FT_OFF_RHO + s * FT_RPL, bar, cx40, cy36, mz(j, f), 2);
            tma_plane(&tmM37, sm + FT_OFF_ALP + s * FT_RPL, bar, cx40, cy36, mz(j, f), 3);
        }
    };
    // group c = what stage 1 of iteration c reads for the first time:
    //   s11, s22, s12 of plane c -> slot c & 1 ; E(c + 1) ; s33 of plane c + 2 -> slot c & 1 ; (c = 0: E(0) too)
    auto issueG = [&](int c, unsigned fE1, unsigned fE0, bool keep) {     // flags of planes c + 1 and (c = 0 only) 0
        uint64_t* bar = &barG[c & 1];
        const uint32_t mBytes = 2 * FT_BW * FT_RH * 4;                        // rho, alpha
        const uint32_t eBytes = (FT_UPL + FT_BOX) * 4 + mBytes;               // s13, s23, rho, alpha
        mbar_expect_tx(bar, (2 * FT_UPL + 2 * FT_BOX) * 4 + eBytes - (keep ? mBytes : 0) + (c == 0 ? eBytes : 0));
        tma_plane(&tmS36, sm + FT_OFF_S11 + (c & 1) * FT_UPL, bar, cx40, cy36, cz0 + c, S11);
        tma_plane(&tmS40, sm + FT_OFF_S22 + (c & 1) * FT_BOX, bar, cx40, cy40, cz0 + c, S22);
        tma_plane(&tmS40, sm + FT_OFF_S12 + (c & 1) * FT_BOX, bar, cx40, cy40, cz0 + c, S12);
        issueE(c + 1, bar, fE1, keep);
        tma_plane(&tmS36, sm + FT_OFF_S33 + (c & 1) * FT_UPL, bar, cx40, cy36, cz0 + c + 2, S33);
        if (c == 0) issueE(0, bar, fE0, false);
    };
    // flags of planes j (mu) and j - 1 (lambda) ; keep*: the slot holds the same palette plane already
    auto issueM = [&](int j, unsigned fmu, unsigned flam, bool keep_mu, bool keep_lam) {
        uint64_t* bar = &barM[j % 3];
        mbar_expect_tx(bar, ((keep_mu ? 0 : FT_MW * FT_MH) + ((keep_lam ? 0 : 1) + (SOM == 0 ? 2 : 0)) * FT_LPL) * 4);
        if (!keep_mu) tma_plane(&tmM36, sm + FT_OFF_MU + (j % 3) * FT_MPL, bar, cxm, cym, mz(j, fmu), 1);
        // lambda of plane j - 1 (read by stage 2 of iteration j + 1, which waits on this barrier) -> slot (j - 1) & 1
        if (!keep_lam) tma_plane(&tmL, sm + FT_OFF_LAM + ((j + 1) & 1) * FT_LPL, bar, cxm, cym, mz(j - 1, flam), 0);
        // and the old s11, s22 of that plane (the tile itself): they are the sigma(ks) that stage 2 adds to
        if (SOM == 0) {
            tma_plane(&tmS32, sm + FT_OFF_SO + (2 * ((j + 1) & 1) + 0) * FT_LPL, bar, cxm, cym, cz0 + j - 1, S11);
            tma_plane(&tmS32, sm + FT_OFF_SO + (2 * ((j + 1) & 1) + 1) * FT_LPL, bar, cxm, cym, cz0 + j - 1, S22);
        }
    };

    // u_old(c) lands in the ring slot that u_new(c) will overwrite in place (own quads only)
    auto issueU = [&](int c) {
        uint64_t* bar = &barU[c & 1];
        mbar_expect_tx(bar, 3 * FT_UPL * 4);
        tma_plane(&tmS36, sm + OFF_UR + (0 * RING + c % RING) * FT_UPL, bar, cx40, cy36, cz0 + c, U1);
        tma_plane(&tmS36, sm + OFF_UR + (1 * RING + c % RING) * FT_UPL, bar, cx40, cy36, cz0 + c, U2);
        tma_plane(&tmS36, sm + OFF_UR + (2 * RING + c % RING) * FT_UPL, bar, cx40, cy36, cz0 + c, U3);
    };

    if (tid == FT_PROD) {
        const unsigned f0 = mflag_at(0), f1 = mflag_at(1), f2 = mflag_at(2);
        fh = (unsigned long long)f2 | ((unsigned long long)f1 << 8) | ((unsigned long long)f0 << 16) | ((unsigned long long)mflag_at(-1) << 24);
        issueG(0, f1, f0, false); issueG(1, f2, 0u, false); issueU(0);
        if (ULEAD > 1) issueU(1);
    }

    // register windows along z (own column)
    float4 w13a, w13b, w13c;          // s13 at kk-2, kk-1, kk
    float4 w23a, w23b, w23c;          // s23
    float4 w33a, w33b, w33c, w33d;    // s33 at kk-2, kk-1, kk, kk+1
    // own-quad z taps of stage 2 that are older than the ring: u(ks-1) and u3(ks-2) (their slots are being refilled)
    float4 u1m1 = f4(0.0f), u2m1 = f4(0.0f), u3m1 = f4(0.0f), u3m2 = f4(0.0f);
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
        if (WT) {      // planes -2, -1, 0 (s33: and 1) of the rings
            tmem_st4(tW13 + 8u, w13a); tmem_st4(tW13 + 12u, w13b); tmem_st4(tW13, w13c);
            tmem_st4(tW23 + 8u, w23a); tmem_st4(tW23 + 12u, w23b); tmem_st4(tW23, w23c);
            tmem_st4(tW33 + 12u, w33b); tmem_st4(tW33, w33c); tmem_st4(tW33 + 4u, w33d);      // (the oldest entry is parked, not ringed)
            if (ZX && pml) {     // X of the three planes below the newest taps of iteration 0: planes -2 .. 0 (sigma33: -1 .. 1), not owned
                const float4 sv[3][3] = {{w13a, w13b, w13c}, {w23a, w23b, w23c}, {w33b, w33c, w33d}};
#pragma unroll
                for (int cc = 0; cc < 3; ++cc)
#pragma unroll
                    for (int k = 0; k < 3; ++k) {
                        const int j = k - 2 + (cc == 2 ? 1 : 0), z = zb - 2 + j;
                        const int p = yzslab_row(z, a.nz, a.P);
                        const bool in = pok && p >= 0;
                        float4 T = f4(0.0f);
                        ldg4_into(T, a.mgi[5] + 4 * cc + (in ? ozq + p * szp : 0), in);
                        const float* ztp = sm + OFF_ZT;
                        const float bk = ztp[(cc == 2 ? T_B_INT : T_B_HALF) * FT_ZRING + (z & (FT_ZRING - 1))];
                        const float ak = in ? ztp[(cc == 2 ? T_A_INT : T_A_HALF) * FT_ZRING + (z & (FT_ZRING - 1))] : 0.0f;
                        tmem_st4(tXZ + 12u * cc + 4u * ((j + 3) % 3), ak * fma4(bk, T, sv[cc][k]));
                    }
            }
            tmem_wait_st();
        }
    }

    // coefficient scales: sign of the step and the 1/c2 of the unnormalised differences (d1)
    const float kB = 2.0f * a.sgn * PACT_C2, kM = 4.0f * a.sgn * PACT_C2, kL = a.sgn * PACT_C2;
    const float* Rbase = sm + FT_OFF_RHO;
    const float* Abase = sm + FT_OFF_ALP;
    // C-PML tables in shared memory, pre-offset: XT(t)[x], YT(t)[y], ZT(t)[z & 15] (t = T_A_INT ..)
    const float* xt0 = sm + OFF_XT + 8 - x0;
    const float* yt0 = sm + OFF_YT + 8 - y0;
    const float* zt0 = sm + OFF_ZT;
#define XT(t) (xt0 + (t) * FT_TABW)
#define YT(t) (yt0 + (t) * FT_TABW)
#define ZT(t) (zt0 + (t) * FT_ZRING)

    for (int it = 0; it < itn; ++it) {
        const int kk = zb - 2 + it;
        unsigned fnew = 0;      // thread 0: material flag of plane it + 3, fetched half an iteration before its use
        if (tid == FT_PROD) fnew = mflag_at(it + 3);
        // forward C-PML: the nine phi of this thread's quad at plane kk, issued together ahead of the wait
        // (one exposed latency per stage instead of nine serialised ones)
        float4 pm[9];
        if (MODE == FM_FWD) {
#pragma unroll
            for (int k = 0; k < 9; ++k) pm[k] = f4(0.0f);
            if (bx || by || (pml && (kk - 2 < a.P || kk + 2 >= a.nz - 1 - a.P))) {
                const bool zok = (unsigned)kk < (unsigned)a.nz;
                const int pzk = zok ? yzslab_row(kk, a.nz, a.P) : -1;          // CTA-uniform
                const bool ex = hx && zok, ey = hy && zok, ez = pok && pzk >= 0;
                const float* gx = a.mgi[0] + ox;
                const float* gy = a.mgi[1] + oy;
                const float* gz = a.mgi[2] + (ez ? ozq + pzk * szp : 0);
                if (bx) { ldg4_into(pm[0], gx, ex); ldg4_into(pm[3], gx + 4, ex); ldg4_into(pm[6], gx + 8, ex); }
                if (by) { ldg4_into(pm[1], gy, ey); ldg4_into(pm[4], gy + 4, ey); ldg4_into(pm[7], gy + 8, ey); }
                if (pzk >= 0) { ldg4_into(pm[2], gz, ez); ldg4_into(pm[5], gz + 4, ez); ldg4_into(pm[8], gz + 8, ez); }
#if FT_PFMV > 0
                const bool zpf = kk + FT_PFMV < a.nz;
                if (bx) prefetch_l2(gx + FT_PFMV * sxp, ex && zpf);
                if (by) prefetch_l2(gy + FT_PFMV * syp, ey && zpf);
                const int pzf = yzslab_row(kk + FT_PFMV, a.nz, a.P);
                if (pzf >= 0) prefetch_l2(a.mgi[2] + (ozq + pzf * szp), pok);
#endif
            }
        }
        // adjoint exchange CTAs: the three old T of the own quad (plane kk) for the pre-block of stage 1, issued ahead
        float4 e1[3];
        int oe1 = 0;
        bool se1 = false;
        if (MODE == FM_ADJ) {
#if FT_PFMV > 0
            if (pml) {      // z slabs: the newest planes the transposed recursions of stage 1 / stage 2 will tap, FT_PFMV iterations on
                const int p1 = yzslab_row(kk + 2 + FT_PFMV, a.nz, a.P), p2 = yzslab_row(kk + FT_PFMV, a.nz, a.P);
                if (p1 >= 0) prefetch_l2(a.mgi[5] + (ozq + p1 * szp), pok);
                if (p2 >= 0) prefetch_l2(a.mgi[2] + (ozq + p2 * szp), pok);
            }
#endif
            e1[0] = e1[1] = e1[2] = f4(0.0f);
            if (exa >= 0) {
                const bool ok = pok && (unsigned)kk < (unsigned)a.nz;
                se1 = ok && (exa == 0 ? colq >= 0 : prow >= 0);
                oe1 = se1 ? (exa == 0 ? ox : oy) : 0;
                const float* ge = a.mgi[3 + exa] + oe1;
                ldg4_into(e1[0], ge, se1); ldg4_into(e1[1], ge + 4, se1); ldg4_into(e1[2], ge + 8, se1);
#if FT_PFMV > 0
                prefetch_l2(ge + FT_PFMV * (exa == 0 ? sxp : syp), se1 && kk + FT_PFMV < a.nz);
#endif
            }
        }
        // ZX: old T of the planes that enter the z windows in this iteration (sigma13, sigma23: kk + 1 ; sigma33: kk + 2)
        float4 zT[3];
        bool zin_[2] = {false, false};
        int zo[2] = {0, 0};
        const bool bzm = ZX && pml && (kk - 3 < a.P || kk + 5 >= a.nz - 1 - a.P);     // a tap of this or a later plane may lie in a z slab
        if (ZX) {
            zT[0] = zT[1] = zT[2] = f4(0.0f);
            if (bzm) {
                const int p1 = yzslab_row(kk + 1, a.nz, a.P), p2 = yzslab_row(kk + 2, a.nz, a.P);
                zin_[0] = pok && p1 >= 0; zin_[1] = pok && p2 >= 0;
                zo[0] = zin_[0] ? ozq + p1 * szp : 0; zo[1] = zin_[1] ? ozq + p2 * szp : 0;
                ldg4_into(zT[0], a.mgi[5] + zo[0], zin_[0]); ldg4_into(zT[1], a.mgi[5] + 4 + zo[0], zin_[0]);
                ldg4_into(zT[2], a.mgi[5] + 8 + zo[1], zin_[1]);
            }
        }
        mbar_wait(&barG[it & 1], (it >> 1) & 1);

        const int s3 = it % 3, s3n = (it + 1) % 3;
        float4 f13 = z4, f23 = z4, f33 = z4;     // fresh window entries: s13, s23 at kk+1, s33 at kk+2
        const bool zin = !EDGE || (unsigned)kk < (unsigned)a.nz;
        // ------------------------------------------------------------------ stage 1: u(kk)
        // Adjoint slab CTAs: X = a T of the own quad for the three terms of the exchange axis, T <- b T + s, into the ring
        // slot that u_old(kk+1) will land in after the barrier (free: the closing barrier of the previous iteration's
        // stage 2 was passed by every thread).
        float* const SC1 = sm + OFF_UR + ((it + ULEAD) % RING) * FT_UPL;     // + f * RING * FT_UPL
        if (exa >= 0) {
            if (WT) {
                if (exa == 0) w13c = tmem_ld4(tW13 + 4u * (it & 3)); else w23c = tmem_ld4(tW23 + 4u * (it & 3));
                tmem_wait_ld();
            }
            if (WT || act1) {
                float4 X0 = z4, X1 = z4, X2 = z4;
                if (pok && zin) {
                    const bool wr = inner && kk >= zb && kk < ze;
                    const float4 o12 = ld4s(sm + FT_OFF_S12 + (it & 1) * FT_BOX, q);
                    if (exa == 0) {
                        const float4 o11 = ld4s(sm + FT_OFF_S11 + (it & 1) * FT_UPL, uq);
                        const float4 ai = tab4(XT(T_A_INT), x), bi = tab4(XT(T_B_INT), x), ah = tab4(XT(T_A_HALF), x), bh = tab4(XT(T_B_HALF), x);
                        X0 = adj_own_p(e1[0], a.mgo[3] + oe1, se1, ai, bi, o11, wr);
                        X1 = adj_own_p(e1[1], a.mgo[3] + oe1 + 4, se1, ah, bh, o12, wr);
                        X2 = adj_own_p(e1[2], a.mgo[3] + oe1 + 8, se1, ah, bh, w13c, wr);
                    } else {
                        const float4 o22 = ld4s(sm + FT_OFF_S22 + (it & 1) * FT_BOX, q);
                        const float4 ai = f4(YT(T_A_INT)[y]), bi = f4(YT(T_B_INT)[y]), ah = f4(YT(T_A_HALF)[y]), bh = f4(YT(T_B_HALF)[y]);
                        X0 = adj_own_p(e1[0], a.mgo[4] + oe1, se1, ah, bh, o12, wr);
                        X1 = adj_own_p(e1[1], a.mgo[4] + oe1 + 4, se1, ai, bi, o22, wr);
                        X2 = adj_own_p(e1[2], a.mgo[4] + oe1 + 8, se1, ah, bh, w23c, wr);
                    }
                }
                if (!WT || act1) {
                    *reinterpret_cast<float4*>(SC1 + 0 * RING * FT_UPL + 4 * uq) = X0;
                    *reinterpret_cast<float4*>(SC1 + 1 * RING * FT_UPL + 4 * uq) = X1;
                    *reinterpret_cast<float4*>(SC1 + 2 * RING * FT_UPL + 4 * uq) = X2;
                }
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // TMA overwrites these planes later
            }
            __syncthreads();
        }
        const bool yex = exa == 1 && r >= 2 && r < 34;      // all four y taps of this thread lie in the exchanged region
        if (WT || act1) {
            const float* P11 = sm + FT_OFF_S11 + (it & 1) * FT_UPL;
            const float* P22 = sm + FT_OFF_S22 + (it & 1) * FT_BOX;
            const float* P12 = sm + FT_OFF_S12 + (it & 1) * FT_BOX;
            const float* P13 = sm + FT_OFF_S13 + s3 * FT_UPL;
            const float* P23 = sm + FT_OFF_S23 + s3 * FT_BOX;
            const float* PR = Rbase + s3 * FT_RPL;
            const float* PA = Abase + s3 * FT_RPL;
            f13 = ld4s(sm + FT_OFF_S13 + s3n * FT_UPL, uq);
            f23 = ld4s(sm + FT_OFF_S23 + s3n * FT_BOX, q);
            f33 = ld4s(sm + FT_OFF_S33 + (it & 1) * FT_UPL, uq);   // plane kk+2
            if (WT) {
                tmem_st4(tW13 + 4u * ((it + 1) & 3), f13); tmem_st4(tW23 + 4u * ((it + 1) & 3), f23); tmem_st4(tW33 + 4u * ((it + 2) & 3), f33);
            }
            // ZX: T <- b T + s and X = a T of the entering planes ; T is stored by the brick that owns the plane
            float4 zX[3];
            if (ZX) {
                zX[0] = zX[1] = zX[2] = f4(0.0f);
                if (bzm) {
                    const int z1 = kk + 1, z2 = kk + 2;
                    const bool w1 = inner && zin_[0] && z1 >= zb && z1 < ze, w2 = inner && zin_[1] && z2 >= zb && z2 < ze;
                    const float b1h = ZT(T_B_HALF)[z1 & (FT_ZRING - 1)], a1h = zin_[0] ? ZT(T_A_HALF)[z1 & (FT_ZRING - 1)] : 0.0f;
                    const float b2i = ZT(T_B_INT)[z2 & (FT_ZRING - 1)], a2i = zin_[1] ? ZT(T_A_INT)[z2 & (FT_ZRING - 1)] : 0.0f;
                    const float4 Ta = fma4(b1h, zT[0], f13), Tb = fma4(b1h, zT[1], f23), Tc = fma4(b2i, zT[2], f33);
                    if (w1) { stg4(a.mgo[5] + zo[0], Ta); stg4(a.mgo[5] + 4 + zo[0], Tb); }
                    if (w2) stg4(a.mgo[5] + 8 + zo[1], Tc);
                    zX[0] = a1h * Ta; zX[1] = a1h * Tb; zX[2] = a2i * Tc;
                }
            }
            // ZX: the z differences of X (taps kk - 2 .. kk + 1 ; sigma33: kk - 1 .. kk + 2), three taps from the rings.  Warp-wide
            // tensor-memory loads: under the CTA-uniform test only.
            float4 zD[3];
            if (ZX) {
                zD[0] = zD[1] = zD[2] = f4(0.0f);
                const uint32_t q0 = 4u * (uint32_t)s3, q1 = 4u * (uint32_t)s3n, q2 = 4u * (uint32_t)((it + 2) % 3);    // planes it, it + 1 (= it - 2), it + 2 (= it - 1)
                if (pml && (kk - 2 < a.P || kk + 2 >= a.nz - 1 - a.P)) {
                    const float4 xa0 = tmem_ld4(tXZ + q1), xb0 = tmem_ld4(tXZ + q2), xc0 = tmem_ld4(tXZ + q0);
                    const float4 xa1 = tmem_ld4(tXZ + 12u + q1), xb1 = tmem_ld4(tXZ + 12u + q2), xc1 = tmem_ld4(tXZ + 12u + q0);
                    const float4 xa2 = tmem_ld4(tXZ + 24u + q2), xb2 = tmem_ld4(tXZ + 24u + q0), xc2 = tmem_ld4(tXZ + 24u + q1);
                    tmem_wait_ld();
                    zD[0] = d4(xa0, xb0, xc0, zX[0]); zD[1] = d4(xa1, xb1, xc1, zX[1]); zD[2] = d4(xa2, xb2, xc2, zX[2]);
                }
                if (bzm) {      // the entering planes take the slots of the planes that just left the windows (read above)
                    tmem_st4(tXZ + q1, zX[0]); tmem_st4(tXZ + 12u + q1, zX[1]); tmem_st4(tXZ + 24u + q2, zX[2]);
                }
            }

            const bool wr1 = inner && kk >= zb && kk < ze;          // this CTA owns u(x..x+3, y, kk)
            // C-PML at this plane: z slab position of kk ; is any tap of the thread inside a slab
            const int pz = (pml && zin) ? yzslab_row(kk, a.nz, a.P) : -1;
            const bool bz = pml && (kk - 2 < a.P || kk + 2 >= a.nz - 1 - a.P);
            const bool slab1 = bx || by || bz;                       // CTA-uniform
            const bool pml1 = slab1 && pok && zin;
            const int oz1 = ozq + (pz >= 0 ? pz : 0) * szp;          // z-slab record of the own quad at plane kk

            // staggered coefficients (reading G10): J = 1 - dt alpha_b, B = dt/(h rho_b)
            const float4 r0 = ld4s(PR, uq), a0 = ld4s(PA, uq);
            const float4 one = f4(1.0f), mh = f4(-0.5f);
            const float4 c12 = ld4s(P12, q);
            const uint32_t tms = tm0 + (uint32_t)(it % 3) * SOS;      // SOM 2: this plane's parking columns
            float4 n1, n2, n3;
            const int sl = it % RING;
            float* const R1 = sm + OFF_UR + (0 * RING + sl) * FT_UPL + 4 * uq;
            float* const R2 = sm + OFF_UR + (1 * RING + sl) * FT_UPL + 4 * uq;
            float* const R3 = sm + OFF_UR + (2 * RING + sl) * FT_UPL + 4 * uq;
            {   // ---- u1 at (x+1/2, y, z): D+x s11, D-y s12, D-z s13
                const float4 c11 = ld4s(P11, uq);
                const float2 l = ld2s(P11, 4 * uq - 2), rr = ld2s(P11, 4 * uq + 4);
                const float4 ya = ld4s(P12, q - 20), yb = ld4s(P12, q - 10), yd = ld4s(P12, q + 10);
                if (WT) {
                    w13a = tmem_ld4(tW13 + 4u * ((it + 2) & 3)); w13b = tmem_ld4(tW13 + 4u * ((it + 3) & 3)); w13c = tmem_ld4(tW13 + 4u * (it & 3));
                    tmem_wait_ld();
                }
                float4 t1 = dpx(l, c11, rr), t2 = d4(ya, yb, c12, yd), t3 = d4(w13a, w13b, w13c, f13);
                if (tmw) { tmem_st4(tms, c11); tmem_st4(tms + 8u, c12); }      // parked after their first use: no wait for the LDS here
                if (MODE == FM_FWD && slab1) {
                    if (bx) t1 = pml_fwd_p(pm[0], a.mgo[0] + ox, tab4(XT(T_A_HALF), x), tab4(XT(T_B_HALF), x), t1, wr1 && hx);
                    if (by) t2 = pml_fwd_p(pm[1], a.mgo[1] + oy, YT(T_A_INT)[y], YT(T_B_INT)[y], t2, wr1 && hy);
                    if (pz >= 0) t3 = pml_fwd_p(pm[2], a.mgo[2] + oz1, ZT(T_A_INT)[kk & (FT_ZRING - 1)], ZT(T_B_INT)[kk & (FT_ZRING - 1)], t3, wr1);
                }
                if (MODE == FM_ADJ && pml1) {
                    const float* S = SC1 + 0 * RING * FT_UPL;
                    if (exa == 0) t1 = t1 + dpx(ld2s(S, 4 * uq - 2), ld4s(S, uq), ld2s(S, 4 * uq + 4));
                    if (yex) t2 = t2 + d4(ld4s(S, uq - 20), ld4s(S, uq - 10), ld4s(S, uq), ld4s(S, uq + 10));
                    else if (neary) t2 = t2 + adj_y3(a, a.mgi[4], a.mgo[4], YT(T_A_HALF), YT(T_B_HALF), oyb, rsy, y - 2, 2, ya, yb, c12, yd, wr1 && exa != 1);
                    if (bz) t3 = t3 + (ZX ? zD[0] : adj_z3(a, a.mgi[5], a.mgo[5], ZT(T_A_HALF), ZT(T_B_HALF), ozq, szp, kk - 2, 2, w13a, w13b, w13c, f13, wr1));
                }
                const float4 rxp = shl1(r0, PR[4 * uq + 4]), axp = shl1(a0, PA[4 * uq + 4]);
                mbar_wait(&barU[it & 1], (it >> 1) & 1);      // u_old(kk) has landed in the ring slot
                n1 = fma4(fma4(mh, adds(a0, axp), one), *reinterpret_cast<const float4*>(R1), (kB * rcp4(adds(r0, rxp))) * (t1 + t2 + t3));
            }
            {   // ---- u2 at (x, y+1/2, z): D-x s12, D+y s22, D-z s23
                const float2 l = ld2s(P12, 4 * q - 2), rr = ld2s(P12, 4 * q + 4);
                const float4 yb = ld4s(P22, q - 10), c22 = ld4s(P22, q), yc = ld4s(P22, q + 10), yd = ld4s(P22, q + 20);
                if (WT) {
                    w23a = tmem_ld4(tW23 + 4u * ((it + 2) & 3)); w23b = tmem_ld4(tW23 + 4u * ((it + 3) & 3)); w23c = tmem_ld4(tW23 + 4u * (it & 3));
                    tmem_wait_ld();
                }
                float4 t1 = dmx(l, c12, rr), t2 = d4(yb, c22, yc, yd), t3 = d4(w23a, w23b, w23c, f23);
                if (tmw) tmem_st4(tms + 4u, c22);
                if (MODE == FM_FWD && slab1) {
                    if (bx) t1 = pml_fwd_p(pm[3], a.mgo[0] + ox + 4, tab4(XT(T_A_INT), x), tab4(XT(T_B_INT), x), t1, wr1 && hx);
                    if (by) t2 = pml_fwd_p(pm[4], a.mgo[1] + oy + 4, YT(T_A_HALF)[y], YT(T_B_HALF)[y], t2, wr1 && hy);
                    if (pz >= 0) t3 = pml_fwd_p(pm[5], a.mgo[2] + oz1 + 4, ZT(T_A_INT)[kk & (FT_ZRING - 1)], ZT(T_B_INT)[kk & (FT_ZRING - 1)], t3, wr1);
                }
                if (MODE == FM_ADJ && pml1) {
                    const float* S = SC1 + 1 * RING * FT_UPL;
                    if (exa == 0) t1 = t1 + dmx(ld2s(S, 4 * uq - 2), ld4s(S, uq), ld2s(S, 4 * uq + 4));
                    if (yex) t2 = t2 + d4(ld4s(S, uq - 10), ld4s(S, uq), ld4s(S, uq + 10), ld4s(S, uq + 20));
                    else if (neary) t2 = t2 + adj_y3(a, a.mgi[4] + 4, a.mgo[4] + 4, YT(T_A_INT), YT(T_B_INT), oyb, rsy, y - 1, 1, yb, c22, yc, yd, wr1 && exa != 1);
                    if (bz) t3 = t3 + (ZX ? zD[1] : adj_z3(a, a.mgi[5] + 4, a.mgo[5] + 4, ZT(T_A_HALF), ZT(T_B_HALF), ozq, szp, kk - 2, 2, w23a, w23b, w23c, f23, wr1));
                }
                const float4 ryp = ld4s(PR, uq + 10), ayp = ld4s(PA, uq + 10);
                n2 = fma4(fma4(mh, a0 + ayp, one), *reinterpret_cast<const float4*>(R2), (kB * rcp4(r0 + ryp)) * (t1 + t2 + t3));
            }
            {   // ---- u3 at (x, y, z+1/2): D-x s13, D-y s23, D+z s33
                const float2 l = ld2s(P13, 4 * uq - 2), rr = ld2s(P13, 4 * uq + 4);
                const float4 ya = ld4s(P23, q - 20), yb = ld4s(P23, q - 10), yd = ld4s(P23, q + 10);
                if (WT) {
                    w33b = tmem_ld4(tW33 + 4u * ((it + 3) & 3)); w33c = tmem_ld4(tW33 + 4u * (it & 3)); w33d = tmem_ld4(tW33 + 4u * ((it + 1) & 3));
                    tmem_wait_ld();
                    tmem_st4(tms + 12u, w33c);      // s33 of plane kk: the old value stage 2 adds to two iterations on
                }
                float4 t1 = dmx(l, w13c, rr), t2 = d4(ya, yb, w23c, yd), t3 = d4(w33b, w33c, w33d, f33);
                if (MODE == FM_FWD && slab1) {
                    if (bx) t1 = pml_fwd_p(pm[6], a.mgo[0] + ox + 8, tab4(XT(T_A_INT), x), tab4(XT(T_B_INT), x), t1, wr1 && hx);
                    if (by) t2 = pml_fwd_p(pm[7], a.mgo[1] + oy + 8, YT(T_A_INT)[y], YT(T_B_INT)[y], t2, wr1 && hy);
                    if (pz >= 0) t3 = pml_fwd_p(pm[8], a.mgo[2] + oz1 + 8, ZT(T_A_HALF)[kk & (FT_ZRING - 1)], ZT(T_B_HALF)[kk & (FT_ZRING - 1)], t3, wr1);
                }
                if (MODE == FM_ADJ && pml1) {
                    const float* S = SC1 + 2 * RING * FT_UPL;
                    if (exa == 0) t1 = t1 + dmx(ld2s(S, 4 * uq - 2), ld4s(S, uq), ld2s(S, 4 * uq + 4));
                    if (yex) t2 = t2 + d4(ld4s(S, uq - 20), ld4s(S, uq - 10), ld4s(S, uq), ld4s(S, uq + 10));
                    else if (neary) t2 = t2 + adj_y3(a, a.mgi[4] + 8, a.mgo[4] + 8, YT(T_A_HALF), YT(T_B_HALF), oyb, rsy, y - 2, 2, ya, yb, w23c, yd, wr1 && exa != 1);
                    if (bz) t3 = t3 + (ZX ? zD[2] : adj_z3(a, a.mgi[5] + 8, a.mgo[5] + 8, ZT(T_A_INT), ZT(T_B_INT), ozq, szp, kk - 1, 1, w33b, w33c, w33d, f33, wr1));
                }
                const float4 rzp = ld4s(Rbase + s3n * FT_RPL, uq), azp = ld4s(Abase + s3n * FT_RPL, uq);
                n3 = fma4(fma4(mh, a0 + azp, one), *reinterpret_cast<const float4*>(R3), (kB * rcp4(r0 + rzp)) * (t1 + t2 + t3));
            }
            if (EDGE && (edge_xy || !zin)) {
                if (!(zin && m0)) { n1.x = 0.0f; n2.x = 0.0f; n3.x = 0.0f; }
                if (!(zin && m1)) { n1.y = 0.0f; n2.y = 0.0f; n3.y = 0.0f; }
                if (!(zin && m2)) { n1.z = 0.0f; n2.z = 0.0f; n3.z = 0.0f; }
                if (!(zin && m3)) { n1.w = 0.0f; n2.w = 0.0f; n3.w = 0.0f; }
            }
            if (!WT || act1) {
                *reinterpret_cast<float4*>(R1) = n1;
                *reinterpret_cast<float4*>(R2) = n2;
                *reinterpret_cast<float4*>(R3) = n3;
            }
            // generic-proxy writes to a slot that issueU refills through the async proxy four iterations later
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            const long long g = (long long)kk * a.sz + gxy;
            if (wr1) {
                store_quad<EDGE>(a.out + U1 * box + g, n1, x, a.nx);
                store_quad<EDGE>(a.out + U2 * box + g, n2, x, a.nx);
                store_quad<EDGE>(a.out + U3 * box + g, n3, x, a.nx);
            }
        }
        // forward C-PML: the nine psi of the quad at plane ks = kk - 2, issued ahead of the barrier
        float4 qm[9];
        if (MODE == FM_FWD) {
#pragma unroll
            for (int k = 0; k < 9; ++k) qm[k] = f4(0.0f);
            if (bx || by || (pml && (kk - 4 < a.P || kk >= a.nz - 1 - a.P))) {
                const bool ok = inner && it >= 4;
                const int pzk = it >= 4 ? yzslab_row(kk - 2, a.nz, a.P) : -1;      // CTA-uniform
                const bool ex = ok && colq >= 0, ey = ok && prow >= 0, ez = ok && pzk >= 0;
                const float* gx = a.mgi[3] + (ox - 2 * sxp);
                const float* gy = a.mgi[4] + (oy - 2 * syp);
                const float* gz = a.mgi[5] + (ez ? ozq + pzk * szp : 0);
                if (bx) { ldg4_into(qm[0], gx, ex); ldg4_into(qm[3], gx + 4, ex); ldg4_into(qm[6], gx + 8, ex); }
                if (by) { ldg4_into(qm[1], gy, ey); ldg4_into(qm[4], gy + 4, ey); ldg4_into(qm[7], gy + 8, ey); }
                if (pzk >= 0) { ldg4_into(qm[2], gz, ez); ldg4_into(qm[5], gz + 4, ez); ldg4_into(qm[8], gz + 8, ez); }
#if FT_PFMV > 0
                const bool zpf = kk - 2 + FT_PFMV < a.nz;
                if (bx) prefetch_l2(gx + FT_PFMV * sxp, ex && zpf);
                if (by) prefetch_l2(gy + FT_PFMV * syp, ey && zpf);
                const int pzf = yzslab_row(kk - 2 + FT_PFMV, a.nz, a.P);
                if (pzf >= 0) prefetch_l2(a.mgi[5] + (ozq + pzf * szp), ok);
#endif
            }
        }
        // adjoint exchange CTAs: the three old T' of the own quad (plane ks = kk - 2) for the pre-block of stage 2
        float4 e2[3];
        int oe2 = 0;
        bool se2 = false;
        if (MODE == FM_ADJ) {
            e2[0] = e2[1] = e2[2] = f4(0.0f);
            if (exa >= 0 && it >= 4) {
                const bool ok = pok && (unsigned)(kk - 2) < (unsigned)a.nz;
                se2 = ok && (exa == 0 ? colq >= 0 : prow >= 0);
                oe2 = se2 ? (exa == 0 ? ox - 2 * sxp : oy - 2 * syp) : 0;
                const float* ge = a.mgi[exa] + oe2;
                ldg4_into(e2[0], ge, se2); ldg4_into(e2[1], ge + 4, se2); ldg4_into(e2[2], ge + 8, se2);
#if FT_PFMV > 0
                prefetch_l2(ge + FT_PFMV * (exa == 0 ? sxp : syp), se2 && kk - 2 + FT_PFMV < a.nz);
#endif
            }
        }
        // SOM 2: the old s11, s22, s12 of plane ks = kk - 2, parked by this thread in stage 1 two iterations ago ; WT: the
        // oldest window entries.  Warp-wide instructions, hence outside the divergent block of stage 2 ; requested here, ahead
        // of the block barrier, and waited for at the top of stage 2.
        float4 so11 = z4, so22 = z4, so12 = z4;
        // ZX, stage 2: old T' of the u planes that enter the z taps of the stress update (u1, u2: plane kk ; u3: plane kk - 1)
        float4 yT[3];
        bool yin_[2] = {false, false};
        int yo[2] = {0, 0};
        const bool bzm2 = ZX && pml && it >= 1 && (kk - 4 < a.P || kk + 5 >= a.nz - 1 - a.P);
        if (ZX) {
            yT[0] = yT[1] = yT[2] = f4(0.0f);
            if (bzm2) {
                const int p1 = yzslab_row(kk, a.nz, a.P), p2 = yzslab_row(kk - 1, a.nz, a.P);
                yin_[0] = inner && p1 >= 0; yin_[1] = inner && p2 >= 0;
                yo[0] = yin_[0] ? ozq + p1 * szp : 0; yo[1] = yin_[1] ? ozq + p2 * szp : 0;
                ldg4_into(yT[0], a.mgi[2] + yo[0], yin_[0]); ldg4_into(yT[1], a.mgi[2] + 4 + yo[0], yin_[0]);
                ldg4_into(yT[2], a.mgi[2] + 8 + yo[1], yin_[1]);
            }
        }
        if ((WT || tmw) && it >= 4) {
            if (tmw) {
                const uint32_t tml = tm0 + (uint32_t)((it + 1) % 3) * SOS;     // plane it - 2
                so11 = tmem_ld4(tml); so22 = tmem_ld4(tml + 4u); so12 = tmem_ld4(tml + 8u);
            }
            if (WT) {   // old s13, s23, s33 of plane ks = the oldest window entries
                w13a = tmem_ld4(tW13 + 4u * ((it + 2) & 3)); w23a = tmem_ld4(tW23 + 4u * ((it + 2) & 3)); w33a = tmem_ld4(tm0 + (uint32_t)((it + 1) % 3) * SOS + 12u);
            }
        }
        if (WT || tmw) tmem_wait_st();
        if (pml && tid >= 360 && tid < 364) {   // z table ring: plane kk + 3 (first read after the barrier)
            const int t = tid - 360, z = kk + 3;
            sm[OFF_ZT + t * FT_ZRING + (z & (FT_ZRING - 1))] = (unsigned)z < (unsigned)a.nz ? __ldg(a.tab[2][t] + z) : 0.0f;
        }
        __syncthreads();
        // every thread is past stage 1 of `it` and stage 2 of `it - 1`: refill the slots they freed
        // thread 0: flags of planes it + 3 (E), it (mu), it - 1 (lambda) and of the planes that filled their slots last
        unsigned fE = 0, fMu = 0, fLam = 0;
        bool kE = false, kMu = false, kLam = false;
        if (tid == FT_PROD) {
            fh = (fh << 8) | fnew;
            fE = (unsigned)fh & 0xffu; fMu = (unsigned)(fh >> 24) & 0xffu; fLam = (unsigned)(fh >> 32) & 0xffu;
            const unsigned fM3 = (unsigned)(fh >> 48) & 0xffu;             // plane it - 3: previous tenant of the mu and lambda slots
            kE = fE != 0 && fE == fMu;                                     // rho, alpha slot (it + 3) % 3 holds plane it (>= 0)
            kMu = it >= 3 && fMu != 0 && fMu == fM3;
            kLam = it >= 2 && fLam != 0 && fLam == fM3;
            // needed first ; ring of 4: slot of plane it - 3, whose last cross-thread reads were in stage 2 of it - 1 (ring of 5:
            // plane it + 2 into the slot of plane it - 3 likewise)
            if (it + ULEAD < itn) issueU(it + ULEAD);
            if (it + 2 <= itn) issueM(it, fMu, fLam, kMu, kLam);
            if (exa < 0 && it + 2 < itn) issueG(it + 2, fE, 0u, kE);   // exchange CTAs: after stage 2 (its slots are their scratch)
        }
        if (it >= 1) mbar_wait(&barM[(it - 1) % 3], ((it - 1) / 3) & 1);
        // ------------------------------------------------------------------ stage 2: sigma(ks), ks = kk - 2
        const int ks = kk - 2;
        // centre-plane values of the own quad: they become the (ks-1) taps of the next iteration (from it = 2 on, so
        // that the first stage 2, at it = 4, finds u(ks-1) and u3(ks-2) in registers)
        float4 cc1 = z4, cc2 = z4, cc3 = z4;
        if (inner && it >= 2) {
            const int pc = ((it + RING - 2) % RING) * FT_UPL;      // slot of plane it - 2
            cc1 = ld4s(sm + OFF_UR + 0 * RING * FT_UPL + pc, uq);
            cc2 = ld4s(sm + OFF_UR + 1 * RING * FT_UPL + pc, uq);
            cc3 = ld4s(sm + OFF_UR + 2 * RING * FT_UPL + pc, uq);
        }
        // Adjoint slab CTAs: Y = a T' of the own quad (T' = b T'_old + u_bar(ks), not stored here: stage 1 of plane ks did)
        // for the three terms of the exchange axis, into the s22 / s12 / s11 planes that stage 1 has finished with.
        float* const SC2a = sm + FT_OFF_S22 + (it & 1) * FT_BOX;
        float* const SC2b = sm + FT_OFF_S12 + (it & 1) * FT_BOX;
        float* const SC2c = sm + FT_OFF_S11 + (it & 1) * FT_UPL;
        if (exa >= 0) {
            if (act1 && it >= 4) {
                float4 Y0 = z4, Y1 = z4, Y2 = z4;
                if (pok && (unsigned)ks < (unsigned)a.nz) {
                    const int pc = ((it + RING - 2) % RING) * FT_UPL;      // slot of the centre plane it - 2
                    const float4 v1 = ld4s(sm + OFF_UR + 0 * RING * FT_UPL + pc, uq);
                    const float4 v2 = ld4s(sm + OFF_UR + 1 * RING * FT_UPL + pc, uq);
                    const float4 v3 = ld4s(sm + OFF_UR + 2 * RING * FT_UPL + pc, uq);
                    if (exa == 0) {
                        const float4 ai = tab4(XT(T_A_INT), x), bi = tab4(XT(T_B_INT), x);
                        Y0 = adj_own_p(e2[0], a.mgo[0] + oe2, se2, tab4(XT(T_A_HALF), x), tab4(XT(T_B_HALF), x), v1, inner);
                        Y1 = adj_own_p(e2[1], a.mgo[0] + oe2 + 4, se2, ai, bi, v2, inner);
                        Y2 = adj_own_p(e2[2], a.mgo[0] + oe2 + 8, se2, ai, bi, v3, inner);
                    } else {
                        const float4 ai = f4(YT(T_A_INT)[y]), bi = f4(YT(T_B_INT)[y]);
                        Y0 = adj_own_p(e2[0], a.mgo[1] + oe2, se2, ai, bi, v1, inner);
                        Y1 = adj_own_p(e2[1], a.mgo[1] + oe2 + 4, se2, f4(YT(T_A_HALF)[y]), f4(YT(T_B_HALF)[y]), v2, inner);
                        Y2 = adj_own_p(e2[2], a.mgo[1] + oe2 + 8, se2, ai, bi, v3, inner);
                    }
                }
                *reinterpret_cast<float4*>(SC2a + 4 * uq) = Y0;
                *reinterpret_cast<float4*>(SC2b + 4 * uq) = Y1;
                *reinterpret_cast<float4*>(SC2c + 4 * uq) = Y2;
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            }
            __syncthreads();
        }
        if ((WT || tmw) && it >= 4) tmem_wait_ld();      // (requested ahead of the block barrier)
        // ZX, stage 2: T' <- b T' + u and Y = a T' of the entering planes (stored by the brick that owns the plane), the z
        // differences of Y from the rings (taps ks - 1 .. ks + 2 ; u3: ks - 2 .. ks + 1), then the entering planes take the
        // slots of the planes that left.  CTA-uniform tests around the warp-wide tensor-memory instructions.
        float4 yD[3];
        if (ZX) {
            yD[0] = yD[1] = yD[2] = f4(0.0f);
            float4 yX[3];
            yX[0] = yX[1] = yX[2] = f4(0.0f);
            const uint32_t tYZ = tm0 + 132u;
            const uint32_t q0 = 4u * (uint32_t)(it % 3), q1 = 4u * (uint32_t)((it + 1) % 3), q2 = 4u * (uint32_t)((it + 2) % 3);
            if (bzm2) {
                const int z1 = kk, z2 = kk - 1;
                const float4 v1 = ld4s(sm + OFF_UR + (0 * RING + it % RING) * FT_UPL, uq), v2 = ld4s(sm + OFF_UR + (1 * RING + it % RING) * FT_UPL, uq);
                const float4 v3 = ld4s(sm + OFF_UR + (2 * RING + (it + RING - 1) % RING) * FT_UPL, uq);
                const bool w1 = yin_[0] && z1 >= zb && z1 < ze, w2 = yin_[1] && z2 >= zb && z2 < ze;
                const float b1i = ZT(T_B_INT)[z1 & (FT_ZRING - 1)], a1i = yin_[0] ? ZT(T_A_INT)[z1 & (FT_ZRING - 1)] : 0.0f;
                const float b2h = ZT(T_B_HALF)[z2 & (FT_ZRING - 1)], a2h = yin_[1] ? ZT(T_A_HALF)[z2 & (FT_ZRING - 1)] : 0.0f;
                const float4 Ta = fma4(b1i, yT[0], v1), Tb = fma4(b1i, yT[1], v2), Tc = fma4(b2h, yT[2], v3);
                if (w1) { stg4(a.mgo[2] + yo[0], Ta); stg4(a.mgo[2] + 4 + yo[0], Tb); }
                if (w2) stg4(a.mgo[2] + 8 + yo[1], Tc);
                yX[0] = a1i * Ta; yX[1] = a1i * Tb; yX[2] = a2h * Tc;
            }
            if (it >= 4 && pml && (kk - 4 < a.P || kk >= a.nz - 1 - a.P)) {      // bz of stage 2 (ks = kk - 2)
                const float4 xa0 = tmem_ld4(tYZ + q0), xb0 = tmem_ld4(tYZ + q1), xc0 = tmem_ld4(tYZ + q2);                      // planes it - 3, it - 2, it - 1
                const float4 xa1 = tmem_ld4(tYZ + 12u + q0), xb1 = tmem_ld4(tYZ + 12u + q1), xc1 = tmem_ld4(tYZ + 12u + q2);
                const float4 xa2 = tmem_ld4(tYZ + 24u + q2), xb2 = tmem_ld4(tYZ + 24u + q0), xc2 = tmem_ld4(tYZ + 24u + q1);    // planes it - 4, it - 3, it - 2
                tmem_wait_ld();
                yD[0] = d4(xa0, xb0, xc0, yX[0]); yD[1] = d4(xa1, xb1, xc1, yX[1]); yD[2] = d4(xa2, xb2, xc2, yX[2]);
            }
            if (bzm2) { tmem_st4(tYZ + q0, yX[0]); tmem_st4(tYZ + 12u + q0, yX[1]); tmem_st4(tYZ + 24u + q2, yX[2]); }
        }
        if (inner && it >= 4) {
            const int j = it - 2;             // relative plane of ks
            // SOM 0, 1: old s12(ks) (and s11, s22) by own-column loads (L2 hits: group ks fetched the planes two
            // iterations ago).  Issued here and consumed at the end of the stage: a load in flight across the loop
            // back-edge makes ptxas wait for it at the loop head, every iteration.
            if (SOM != 2) so12 = ldg4(in + S12 * box + (long long)ks * a.sz + gxy);
            if (SOM == 1) {
                so11 = ldg4(in + S11 * box + (long long)ks * a.sz + gxy);
                so22 = ldg4(in + S22 * box + (long long)ks * a.sz + gxy);
            }
            const float* U1p = sm + OFF_UR + 0 * RING * FT_UPL;
            const float* U2p = sm + OFF_UR + 1 * RING * FT_UPL;
            const float* U3p = sm + OFF_UR + 2 * RING * FT_UPL;
            const int p0 = (j % RING) * FT_UPL;
            const int pp1 = ((j + 1) % RING) * FT_UPL, pp2 = ((j + 2) % RING) * FT_UPL;
            const int pz = pml ? yzslab_row(ks, a.nz, a.P) : -1;
            const bool bz = pml && (ks - 2 < a.P || ks + 2 >= a.nz - 1 - a.P);
            const bool pml2 = bx || by || bz;       // inner threads have storage: 0 <= x < nx, 0 <= y < ny, zb <= ks < ze
            const int ox2 = ox - 2 * sxp, oy2 = oy - 2 * syp, oyb2 = oyb - 2 * syp;      // plane ks
            const int oz2 = ozq + (pz >= 0 ? pz : 0) * szp;
            float4 e11, e22, e33, g12, g21, g13, g31, g23, g32;
            {   // ---- derivatives of u1: D-x (e11), D+y (g12), D+z (g13)
                const float4 c = cc1;
                const float2 l = ld2s(U1p + p0, 4 * uq - 2), rr = ld2s(U1p + p0, 4 * uq + 4);
                const float4 ya = ld4s(U1p + p0, uq - 10), yc = ld4s(U1p + p0, uq + 10), yd = ld4s(U1p + p0, uq + 20);
                const float4 za = u1m1, zc = ld4s(U1p + pp1, uq), zd = ld4s(U1p + pp2, uq);
                e11 = dmx(l, c, rr); g12 = d4(ya, c, yc, yd); g13 = d4(za, c, zc, zd);
                if (MODE == FM_FWD && pml2) {
                    if (bx) e11 = pml_fwd_p(qm[0], a.mgo[3] + ox2, tab4(XT(T_A_INT), x), tab4(XT(T_B_INT), x), e11, colq >= 0);
                    if (by) g12 = pml_fwd_p(qm[1], a.mgo[4] + oy2, YT(T_A_HALF)[y], YT(T_B_HALF)[y], g12, prow >= 0);
                    if (pz >= 0) g13 = pml_fwd_p(qm[2], a.mgo[5] + oz2, ZT(T_A_HALF)[ks & (FT_ZRING - 1)], ZT(T_B_HALF)[ks & (FT_ZRING - 1)], g13, true);
                }
                if (MODE == FM_ADJ && pml2) {
                    if (exa == 0) e11 = e11 + dmx(ld2s(SC2a, 4 * uq - 2), ld4s(SC2a, uq), ld2s(SC2a, 4 * uq + 4));
                    if (exa == 1) g12 = g12 + d4(ld4s(SC2a, uq - 10), ld4s(SC2a, uq), ld4s(SC2a, uq + 10), ld4s(SC2a, uq + 20));
                    else if (neary) g12 = g12 + adj_y3(a, a.mgi[1], a.mgo[1], YT(T_A_INT), YT(T_B_INT), oyb2, rsy, y - 1, 1, ya, c, yc, yd, true);
                    if (bz) g13 = g13 + (ZX ? yD[0] : adj_z3(a, a.mgi[2], a.mgo[2], ZT(T_A_INT), ZT(T_B_INT), ozq, szp, ks - 1, 1, za, c, zc, zd, true));
                }
            }
            {   // ---- derivatives of u2: D+x (g21), D-y (e22), D+z (g23)
                const float4 c = cc2;
                const float2 l = ld2s(U2p + p0, 4 * uq - 2), rr = ld2s(U2p + p0, 4 * uq + 4);
                const float4 ya = ld4s(U2p + p0, uq - 20), yb = ld4s(U2p + p0, uq - 10), yd = ld4s(U2p + p0, uq + 10);
                const float4 za = u2m1, zc = ld4s(U2p + pp1, uq), zd = ld4s(U2p + pp2, uq);
                g21 = dpx(l, c, rr); e22 = d4(ya, yb, c, yd); g23 = d4(za, c, zc, zd);
                if (MODE == FM_FWD && pml2) {
                    if (bx) g21 = pml_fwd_p(qm[3], a.mgo[3] + ox2 + 4, tab4(XT(T_A_HALF), x), tab4(XT(T_B_HALF), x), g21, colq >= 0);
                    if (by) e22 = pml_fwd_p(qm[4], a.mgo[4] + oy2 + 4, YT(T_A_INT)[y], YT(T_B_INT)[y], e22, prow >= 0);
                    if (pz >= 0) g23 = pml_fwd_p(qm[5], a.mgo[5] + oz2 + 4, ZT(T_A_HALF)[ks & (FT_ZRING - 1)], ZT(T_B_HALF)[ks & (FT_ZRING - 1)], g23, true);
                }
                if (MODE == FM_ADJ && pml2) {
                    if (exa == 0) g21 = g21 + dpx(ld2s(SC2b, 4 * uq - 2), ld4s(SC2b, uq), ld2s(SC2b, 4 * uq + 4));
                    if (exa == 1) e22 = e22 + d4(ld4s(SC2b, uq - 20), ld4s(SC2b, uq - 10), ld4s(SC2b, uq), ld4s(SC2b, uq + 10));
                    else if (neary) e22 = e22 + adj_y3(a, a.mgi[1] + 4, a.mgo[1] + 4, YT(T_A_HALF), YT(T_B_HALF), oyb2, rsy, y - 2, 2, ya, yb, c, yd, true);
                    if (bz) g23 = g23 + (ZX ? yD[1] : adj_z3(a, a.mgi[2] + 4, a.mgo[2] + 4, ZT(T_A_INT), ZT(T_B_INT), ozq, szp, ks - 1, 1, za, c, zc, zd, true));
                }
            }
            {   // ---- derivatives of u3: D+x (g31), D+y (g32), D-z (e33)
                const float4 c = cc3;
                const float2 l = ld2s(U3p + p0, 4 * uq - 2), rr = ld2s(U3p + p0, 4 * uq + 4);
                const float4 ya = ld4s(U3p + p0, uq - 10), yc = ld4s(U3p + p0, uq + 10), yd = ld4s(U3p + p0, uq + 20);
                const float4 za = u3m2, zb_ = u3m1, zd = ld4s(U3p + pp1, uq);
                g31 = dpx(l, c, rr); g32 = d4(ya, c, yc, yd); e33 = d4(za, zb_, c, zd);
                if (MODE == FM_FWD && pml2) {
                    if (bx) g31 = pml_fwd_p(qm[6], a.mgo[3] + ox2 + 8, tab4(XT(T_A_HALF), x), tab4(XT(T_B_HALF), x), g31, colq >= 0);
                    if (by) g32 = pml_fwd_p(qm[7], a.mgo[4] + oy2 + 8, YT(T_A_HALF)[y], YT(T_B_HALF)[y], g32, prow >= 0);
                    if (pz >= 0) e33 = pml_fwd_p(qm[8], a.mgo[5] + oz2 + 8, ZT(T_A_INT)[ks & (FT_ZRING - 1)], ZT(T_B_INT)[ks & (FT_ZRING - 1)], e33, true);
                }
                if (MODE == FM_ADJ && pml2) {
                    if (exa == 0) g31 = g31 + dpx(ld2s(SC2c, 4 * uq - 2), ld4s(SC2c, uq), ld2s(SC2c, 4 * uq + 4));
                    if (exa == 1) g32 = g32 + d4(ld4s(SC2c, uq - 10), ld4s(SC2c, uq), ld4s(SC2c, uq + 10), ld4s(SC2c, uq + 20));
                    else if (neary) g32 = g32 + adj_y3(a, a.mgi[1] + 8, a.mgo[1] + 8, YT(T_A_INT), YT(T_B_INT), oyb2, rsy, y - 1, 1, ya, c, yc, yd, true);
                    if (bz) e33 = e33 + (ZX ? yD[2] : adj_z3(a, a.mgi[2] + 8, a.mgo[2] + 8, ZT(T_A_HALF), ZT(T_B_HALF), ozq, szp, ks - 2, 2, za, zb_, c, zd, true));
                }
            }

            // Lame coefficients: lambda, 2 mu at the node; 4-point harmonic mu at shear points (reading G10)
            const float* M0 = sm + FT_OFF_MU + (j % 3) * FT_MPL;
            const float* M1 = sm + FT_OFF_MU + ((j + 1) % 3) * FT_MPL;
            const float4 i0 = ld4s(M0, mq), iy = ld4s(M0, mq + 9), iz = ld4s(M1, mq), iyz = ld4s(M1, mq + 9);
            const float4 ix = shl1(i0, M0[4 * mq + 4]), ixy = shl1(iy, M0[4 * mq + 40]), ixz = shl1(iz, M1[4 * mq + 4]);
            const float4 mn2 = kB * rcp4(i0);
            const float4 i0x = adds(i0, ix);
            const float4 mxy = kM * rcp4(i0x + adds(iy, ixy));
            const float4 mxz = kM * rcp4(i0x + adds(iz, ixz));
            const float4 myz = kM * rcp4((i0 + iy) + (iz + iyz));
            const float4 lam = ld4s(sm + FT_OFF_LAM + (it & 1) * FT_LPL, (r - 2) * 8 + (qx - 1));   // lambda(ks), by TMA
            const float4 ldiv = (kL * lam) * (e11 + e22 + e33);
            const int lq = (r - 2) * 8 + (qx - 1);
            if (SOM == 0) {
                so11 = ld4s(sm + FT_OFF_SO + (2 * (it & 1) + 0) * FT_LPL, lq);
                so22 = ld4s(sm + FT_OFF_SO + (2 * (it & 1) + 1) * FT_LPL, lq);
            }
            const float4 n11 = so11 + fma4(mn2, e11, ldiv);
            const float4 n22 = so22 + fma4(mn2, e22, ldiv);
            const float4 n33 = w33a + fma4(mn2, e33, ldiv);
            const float4 n12 = fma4(mxy, g12 + g21, so12);
            const float4 n13 = fma4(mxz, g13 + g31, w13a);
            const float4 n23 = fma4(myz, g23 + g32, w23a);
            const long long g = (long long)ks * a.sz + gxy;
            store_quad<EDGE>(a.out + S11 * box + g, n11, x, a.nx);
            store_quad<EDGE>(a.out + S22 * box + g, n22, x, a.nx);
            store_quad<EDGE>(a.out + S33 * box + g, n33, x, a.nx);
            store_quad<EDGE>(a.out + S12 * box + g, n12, x, a.nx);
            store_quad<EDGE>(a.out + S13 * box + g, n13, x, a.nx);
            store_quad<EDGE>(a.out + S23 * box + g, n23, x, a.nx);
        }
        if (exa >= 0) {   // every thread is done with the exchange planes: now the group that refills them may go
            __syncthreads();
            if (tid == FT_PROD && it + 2 < itn) issueG(it + 2, fE, 0u, kE);
        }
        u3m2 = u3m1; u1m1 = cc1; u2m1 = cc2; u3m1 = cc3;
        if (MODE != FM_PLAIN) { ox += sxp; oy += syp; oyb += syp; }
        // slide the z windows
        if (!WT) {
            w13a = w13b; w13b = w13c; w13c = f13;
            w23a = w23b; w23b = w23c; w23c = f23;
            w33a = w33b; w33b = w33c; w33c = w33d; w33d = f33;
        }
    }
}

// =================================================================================================
// One launch = one time step.  The launch is persistent: one CTA per SM pulls bricks off the work list through
// an atomic counter, heaviest first (host order: C-PML bricks, then long interior bricks, short ones last), so
// that no SM idles while another still holds a long brick and no wave of CTAs ends on a partial wave.  Bricks
// flagged FT_WORK_SLAB run the launch's C-PML code (MODE), the others the C-PML-free instance of the same
// brick routine.  The last CTA to leave resets the queue for the next launch.
template <int MODE>
__global__ void __launch_bounds__(FT_NT, 1)
k_step(const __grid_constant__ CUtensorMap tmS40, const __grid_constant__ CUtensorMap tmS36,
       const __grid_constant__ CUtensorMap tmM37, const __grid_constant__ CUtensorMap tmM36,
       const __grid_constant__ CUtensorMap tmL, const __grid_constant__ CUtensorMap tmS32, const FusedArgs a)
{
    extern __shared__ __align__(1024) float sm[];
    constexpr int SOM = FT_SOM(MODE);
    int* s_next = reinterpret_cast<int*>(sm + FusedMap<SOM>::OFF_TICKET);
    const int n = a.work_end - a.work_begin;
    bool first = true;
    uint32_t tmem_base = 0;
    constexpr bool WT = FT_WT(MODE) != 0;
    constexpr int TMC = WT ? FT_TMEM_COLS_X : FT_TMEM_COLS;
    if (SOM == 2 || WT) {      // tensor memory (parked old stresses, z windows): allocated once per (persistent) CTA by warp 0
        uint32_t* s_tm = reinterpret_cast<uint32_t*>(s_next + 1);
        if (threadIdx.x < 32) {
            asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(s_tm)), "r"(TMC) : "memory");
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
        }
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        tmem_base = *s_tm;
    }
    for (;;) {
        if (threadIdx.x == 0) *s_next = (int)atomicAdd(a.queue, 1u);
        __syncthreads();                 // also: every thread is done with the previous brick's shared memory
        const int b = *s_next;
        if (b >= n) break;
        const int4 wk = __ldg(a.work + a.work_begin + b);
        if (MODE != FM_PLAIN && (wk.x & FT_WORK_SLAB)) fused_brick<MODE, true, SOM, WT>(sm, tmS40, tmS36, tmM37, tmM36, tmL, tmS32, a, wk, first, tmem_base);
        else if (wk.x & FT_WORK_NOEDGE) fused_brick<FM_PLAIN, false, SOM, WT>(sm, tmS40, tmS36, tmM37, tmM36, tmL, tmS32, a, wk, first, tmem_base);
        else fused_brick<FM_PLAIN, true, SOM, WT>(sm, tmS40, tmS36, tmM37, tmM36, tmL, tmS32, a, wk, first, tmem_base);
        first = false;
        // generic-proxy writes of this brick (tables, exchange planes) precede the TMA writes of the next one
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads();                 // *s_next is read by all before thread 0 overwrites it
    }
    if ((SOM == 2 || WT) && threadIdx.x < 32) {   // (every thread left its last brick through the loop's __syncthreads)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(TMC) : "memory");
    }
    if (threadIdx.x == 0) {
        __threadfence();
        if (atomicAdd(a.queue + 1, 1u) == gridDim.x - 1) {   // every CTA has drawn its last (out of range) ticket
            a.queue[0] = 0u;
            a.queue[1] = 0u;
        }
    }
}
