// kernels_acoustic.cuh — the fluid-only specialisation of the fused step: H and H^T of a medium with
// mu = 0 everywhere (the paper's H^dagger_{mu=0}: the skull treated as a fluid).
//
// With mu = 0 the three normal stresses stay equal and the shear stresses stay zero (Eq. 46 with M_jk = 0; DESIGN.md section 3,
// row "mu = 0"), so the state collapses to
// one stress field s (= sigma11 = sigma22 = sigma33, kept in the S11 slot of the state) and the three velocities:
//     u_a <- J_a u_a + B_a (D+_a s + phi_aa)            a = x, y, z          (Eq. 46a,b)
//     s   <- s + Ll (sum_a D-_a u_a + psi_aa)                                (Eq. 46c,d ; lambda only)
// and, on the scaled adjoint variables of DESIGN.md "Adjoint step", W'^T is the same step with the sign of B and Ll
// flipped and the tilde-form transposed C-PML recursions.  4 state fields read + written and 3 material volumes read:
// 44 B per cell-step instead of 88.  The arithmetic is that of the elastic kernel with the vanishing terms dropped
// (0 * e + x = x), so the result equals the elastic path run with mu = 0 to the last bits (1-2 ulp measured).
//
// Same machinery as kernels_fused.cuh: 32 x 32 tiles marching along z, TMA-staged planes, one block barrier per plane,
// mbarriers, work list, shared-memory map (the shear / mu / second-stress regions simply stay idle).  The stress plane is
// fetched once, as a 40 x 40 box (it needs x and y neighbours), into the s22 region; its z window comes from the s33 region.
#pragma once
#include "kernels_fused.cuh"

// Shared-memory map of the acoustic brick (floats; every plane 128-byte aligned).  With one stress field there is room
// to spare, and it goes into latency: a u ring of AC_RING planes lets u_old(c) be requested three iterations ahead
// (the elastic kernel can only ask half an iteration ahead, and waits for it), and the adjoint's exchange planes get
// storage of their own instead of borrowing planes that a TMA refill is waiting for.
#define AC_RING 6
#define AC_OFF_S 0                                   // s(c), 40 x 40, 2 slots
#define AC_OFF_W (AC_OFF_S + 2 * FT_BOX)             // s(c + 2), 40 x 36, 2 slots: feeds the z window
#define AC_OFF_RHO (AC_OFF_W + 2 * FT_UPL)           // 3 slots
#define AC_OFF_ALP (AC_OFF_RHO + 3 * FT_RPL)         // 3 slots
#define AC_OFF_LAM (AC_OFF_ALP + 3 * FT_RPL)         // 2 slots
#define AC_OFF_SO (AC_OFF_LAM + 2 * FT_LPL)          // old s of plane ks (tile only), 2 slots
#define AC_OFF_UR (AC_OFF_SO + 2 * FT_LPL)           // u ring: [component][AC_RING] planes of 40 x 36
#define AC_OFF_BARU (AC_OFF_UR + 3 * AC_RING * FT_UPL)   // 4 mbarriers (32 floats reserved)
#define AC_OFF_SC1 (AC_OFF_BARU + 32)                // adjoint exchange plane of stage 1 (40 x 36)
#define AC_OFF_SC2 (AC_OFF_SC1 + FT_UPL)             // adjoint exchange plane of stage 2
static_assert(AC_OFF_SC2 + FT_BOX <= FT_OFF_END, "acoustic shared-memory map overlaps the barriers / tables");
static_assert(AC_OFF_W % 32 == 0 && AC_OFF_RHO % 32 == 0 && AC_OFF_ALP % 32 == 0 && AC_OFF_LAM % 32 == 0 && AC_OFF_SO % 32 == 0 &&
              AC_OFF_UR % 32 == 0 && AC_OFF_SC1 % 32 == 0, "TMA destinations are 128-byte aligned");

template <int MODE, bool EDGE>
__device__ __forceinline__ void acoustic_brick(float* __restrict__ sm, const CUtensorMap& tmS40, const CUtensorMap& tmS36,
                                               const CUtensorMap& tmM37, const CUtensorMap& tmL, const CUtensorMap& tmS32,
                                               const FusedArgs& a, const int4 wk, const bool first)
{
    uint64_t* bars = reinterpret_cast<uint64_t*>(sm + FT_OFF_END);
    uint64_t* barG = bars;        // [2]  stress plane c, rho / alpha of plane c + 1, z-window plane c + 2
    uint64_t* barM = bars + 2;    // [3]  lambda and old stress of plane j - 1
    uint64_t* barU = reinterpret_cast<uint64_t*>(sm + AC_OFF_BARU);    // [4]  u_old of plane c, requested three iterations ahead

    const int tid = threadIdx.x;
    const int zb = wk.z, ze = wk.w;
    const int x0 = (wk.x & 0xffff) * FT_TX, y0 = wk.y * FT_TY;
    const int itn = ze - zb + 4;

    const bool act1 = tid < 360;
    const int qx = tid % 10, r = tid / 10;
    const int x = x0 - 4 + 4 * qx, y = y0 - 2 + r;
    const bool inner = act1 && qx >= 1 && qx <= 8 && r >= 2 && r < 34 && (!EDGE || (x < a.nx && y < a.ny));
    const int q = tid + 20;                 // quad index in the 40 x 40 stress plane
    const int uq = tid;                     // quad index in a 40 x 36 plane
    const int lq = (r - 2) * 8 + (qx - 1);  // quad index in a 32 x 32 plane (inner threads)
    const bool ld_ok = act1 && (!EDGE || ((y + PACT_HALO_Y < a.ny + 2 * PACT_HALO_Y) && (x + 3 + PACT_HALO_X < (int)a.sy)));
    const long long gxy = (long long)y * a.sy + x;
    const bool yin = (unsigned)y < (unsigned)a.ny;
    const bool m0 = yin && (unsigned)x < (unsigned)a.nx, m1 = yin && (unsigned)(x + 1) < (unsigned)a.nx;
    const bool m2 = yin && (unsigned)(x + 2) < (unsigned)a.nx, m3 = yin && (unsigned)(x + 3) < (unsigned)a.nx;
    const bool edge_xy = EDGE && (x0 == 0 || y0 == 0 || x0 + FT_TX + 4 > a.nx || y0 + FT_TY + 2 > a.ny);

    const bool pml = MODE != FM_PLAIN && a.P > 0;
    const bool bx = pml && (x0 - 8 < a.xl || x0 + FT_TX + 8 > a.xr);
    const bool by = pml && (y0 - 4 < a.P || y0 + FT_TY + 4 > a.ny - 1 - a.P);
    const bool pok = pml && act1 && x >= 0 && x < a.nxq && yin;
    const int colq = pok ? xslab_col(a, x) : -1;
    const int prow = pok ? yzslab_row(y, a.ny, a.P) : -1;
    const bool neary = pok && (y - 2 < a.P || y + 2 >= a.ny - 1 - a.P);
    const int exa = (MODE == FM_ADJ) ? (bx ? 0 : (by ? 1 : -1)) : -1;
    // memory variables: 32-bit running offsets of the own quad at plane kk (x, y slabs), of row 0 of the y slab (adjoint
    // taps) and the plane-independent part in the z slabs (one add per plane instead of 64-bit index products)
    const bool hx = pok && colq >= 0, hy = pok && prow >= 0;
    const int sxp = a.ny * a.wx, syp = a.wyz * a.nxq, szp = a.ny * a.nxq;
    int ox = hx ? ((zb - 2) * a.ny + y) * a.wx + colq : 0;
    int oy = hy ? ((zb - 2) * a.wyz + prow) * a.nxq + x : 0;
    int oyb = pok ? (zb - 2) * a.wyz * a.nxq + x : 0;
    const int ozq = pok ? y * a.nxq + x : 0;

    const float* in = a.in;
    const long long box = a.box;

    if (pml) {
        for (int i = tid; i < 4 * FT_TABW; i += FT_NT) {
            const int t = i / FT_TABW, o = i % FT_TABW - 8;
            sm[FT_OFF_XT + i] = (unsigned)(x0 + o) < (unsigned)a.nx ? __ldg(a.tab[0][t] + x0 + o) : 0.0f;
            sm[FT_OFF_YT + i] = (unsigned)(y0 + o) < (unsigned)a.ny ? __ldg(a.tab[1][t] + y0 + o) : 0.0f;
        }
        if (tid < 4 * 12) {
            const int t = tid / 12, z = zb - 10 + tid % 12;
            sm[FT_OFF_ZT + t * FT_ZRING + (z & (FT_ZRING - 1))] = (unsigned)z < (unsigned)a.nz ? __ldg(a.tab[2][t] + z) : 0.0f;
        }
    }
    if (tid == 0) {
        for (int k = 0; k < 8; ++k) {
            if (!first) mbar_inval(&bars[k]);
            mbar_init(&bars[k], 1);
        }
        for (int k = 0; k < 4; ++k) {
            if (!first) mbar_inval(&barU[k]);
            mbar_init(&barU[k], 1);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();

    const int cx40 = x0 - 4 + PACT_HALO_X, cy40 = y0 - 4 + PACT_HALO_Y, cy36 = y0 - 2 + PACT_HALO_Y;
    const int cxm = x0 + PACT_HALO_X, cym = y0 + PACT_HALO_Y;
    const int cz0 = zb - 2 + PACT_HALO_Z;
    const unsigned char* mfl = a.mflag ? a.mflag + ((size_t)wk.y * a.ntx + (wk.x & 0xffff)) * a.nzp + cz0 : nullptr;
    auto mflag_at = [&](int j) -> unsigned { return mfl ? (unsigned)__ldg(mfl + j) : 0u; };
    auto mz = [&](int j, unsigned f) { return f ? a.mpal + (int)f - 1 : cz0 + j; };
    unsigned long long fh = 0;

    // rho, alpha of plane j -> slot j % 3 (skipped when the slot holds the same palette plane)
    auto issueE = [&](int j, uint64_t* bar, unsigned f, bool keep) {
        if (keep) return;
        const int s = j % 3;
        tma_plane(&tmM37, sm + AC_OFF_RHO + s * FT_RPL, bar, cx40, cy36, mz(j, f), 2);
        tma_plane(&tmM37, sm + AC_OFF_ALP + s * FT_RPL, bar, cx40, cy36, mz(j, f), 3);
    };
    auto issueG = [&](int c, unsigned fE1, unsigned fE0, bool keep) {
        uint64_t* bar = &barG[c & 1];
        const uint32_t mBytes = 2 * FT_BW * FT_RH * 4;
        mbar_expect_tx(bar, (FT_BOX + FT_UPL) * 4 + (keep ? 0 : mBytes) + (c == 0 ? mBytes : 0));
        tma_plane(&tmS40, sm + AC_OFF_S + (c & 1) * FT_BOX, bar, cx40, cy40, cz0 + c, S11);          // s(c), 40 x 40
        issueE(c + 1, bar, fE1, keep);
        tma_plane(&tmS36, sm + AC_OFF_W + (c & 1) * FT_UPL, bar, cx40, cy36, cz0 + c + 2, S11);      // s(c + 2): z window
        if (c == 0) issueE(0, bar, fE0, false);
    };
    auto issueM = [&](int j, unsigned flam, bool keep_lam) {      // lambda and old s of plane j - 1 -> slot (j - 1) & 1
        uint64_t* bar = &barM[j % 3];
        mbar_expect_tx(bar, (keep_lam ? 1 : 2) * FT_LPL * 4);
        if (!keep_lam) tma_plane(&tmL, sm + AC_OFF_LAM + ((j + 1) & 1) * FT_LPL, bar, cxm, cym, mz(j - 1, flam), 0);
        tma_plane(&tmS32, sm + AC_OFF_SO + ((j + 1) & 1) * FT_LPL, bar, cxm, cym, cz0 + j - 1, S11);
    };
    auto issueU = [&](int c) {
        uint64_t* bar = &barU[c & 3];
        mbar_expect_tx(bar, 3 * FT_UPL * 4);
        tma_plane(&tmS36, sm + AC_OFF_UR + (0 * AC_RING + c % AC_RING) * FT_UPL, bar, cx40, cy36, cz0 + c, U1);
        tma_plane(&tmS36, sm + AC_OFF_UR + (1 * AC_RING + c % AC_RING) * FT_UPL, bar, cx40, cy36, cz0 + c, U2);
        tma_plane(&tmS36, sm + AC_OFF_UR + (2 * AC_RING + c % AC_RING) * FT_UPL, bar, cx40, cy36, cz0 + c, U3);
    };

    if (tid == FT_PROD) {
        const unsigned f0 = mflag_at(0), f1 = mflag_at(1), f2 = mflag_at(2);
        fh = (unsigned long long)f2 | ((unsigned long long)f1 << 8) | ((unsigned long long)f0 << 16) | ((unsigned long long)mflag_at(-1) << 24);
        issueG(0, f1, f0, false); issueG(1, f2, 0u, false);
        for (int c = 0; c < 3 && c < itn; ++c) issueU(c);
    }

    // z window of s (own column): planes kk-2 .. kk+1 ; stage 2's oldest u3 taps
    float4 w33a, w33b, w33c, w33d;
    float4 u3m1 = f4(0.0f), u3m2 = f4(0.0f);
    const float4 z4 = f4(0.0f);
    {
        const long long g = (long long)(zb - 2) * a.sz + gxy;
        w33a = ld_ok ? ldg4(in + S11 * box + g - 2 * a.sz) : z4;
        w33b = ld_ok ? ldg4(in + S11 * box + g - a.sz) : z4;
        w33c = ld_ok ? ldg4(in + S11 * box + g) : z4;
        w33d = ld_ok ? ldg4(in + S11 * box + g + a.sz) : z4;
    }

    const float kB = 2.0f * a.sgn * PACT_C2, kL = a.sgn * PACT_C2;
    const float* Rbase = sm + AC_OFF_RHO;
    const float* Abase = sm + AC_OFF_ALP;
    const float* xt0 = sm + FT_OFF_XT + 8 - x0;
    const float* yt0 = sm + FT_OFF_YT + 8 - y0;
    const float* zt0 = sm + FT_OFF_ZT;

    for (int it = 0; it < itn; ++it) {
        const int kk = zb - 2 + it;
        unsigned fnew = 0;
        if (tid == FT_PROD) fnew = mflag_at(it + 3);
        // forward C-PML: phi11 (x), phi22 (y), phi33 (z) of the own quad at plane kk, issued ahead of the wait
        float4 pm0 = z4, pm1 = z4, pm2 = z4;
        if (MODE == FM_FWD) {
            if (bx || by || (pml && (kk - 2 < a.P || kk + 2 >= a.nz - 1 - a.P))) {
                const bool ok = pok && (unsigned)kk < (unsigned)a.nz;
                const int pzk = ok ? yzslab_row(kk, a.nz, a.P) : -1;
                const bool ex = ok && colq >= 0, ey = ok && prow >= 0, ez = pzk >= 0;
                ldg4_into(pm0, a.mvi[0] + (ex ? ox : 0), ex);
                ldg4_into(pm1, a.mvi[4] + (ey ? oy : 0), ey);
                ldg4_into(pm2, a.mvi[8] + (ez ? ozq + pzk * szp : 0), ez);
#if FT_PFMV > 0
                const bool zpf = kk + FT_PFMV < a.nz;
                prefetch_l2(a.mvi[0] + (ox + FT_PFMV * sxp), ex && zpf);
                prefetch_l2(a.mvi[4] + (oy + FT_PFMV * syp), ey && zpf);
                const int pzf = yzslab_row(kk + FT_PFMV, a.nz, a.P);
                if (pzf >= 0) prefetch_l2(a.mvi[8] + (ozq + pzf * szp), pok);
#endif
            }
        }
        // adjoint exchange CTAs: old T of psi_aa (a = exchange axis) of the own quad at plane kk
        float4 e1 = z4;
        long long ie1 = 0;
        bool se1 = false;
        if (MODE == FM_ADJ && exa >= 0) {
            const bool ok = pok && (unsigned)kk < (unsigned)a.nz;
            se1 = ok && (exa == 0 ? colq >= 0 : prow >= 0);
            ie1 = se1 ? (exa == 0 ? ox : oy) : 0;
            ldg4_into(e1, a.mvi[9 + 4 * exa] + ie1, se1);
        }
        mbar_wait(&barG[it & 1], (it >> 1) & 1);

        const int s3 = it % 3, s3n = (it + 1) % 3;
        float4 f33 = z4;
        const bool zin = !EDGE || (unsigned)kk < (unsigned)a.nz;
        const float* PS = sm + AC_OFF_S + (it & 1) * FT_BOX;                          // s(kk), 40 x 40
        // ------------------------------------------------------------------ stage 1: u(kk)
        float* const SC1 = sm + AC_OFF_SC1;
        if (exa >= 0) {
            if (act1) {
                float4 X = z4;
                if (pok && zin) {
                    const bool wr = inner && kk >= zb && kk < ze;
                    const float4 os = ld4s(PS, q);
                    if (exa == 0) X = adj_own_x(e1, a.mvo[9], ie1, se1, tab4(XT(T_A_INT), x), tab4(XT(T_B_INT), x), os, wr);
                    else X = adj_own_x(e1, a.mvo[13], ie1, se1, f4(YT(T_A_INT)[y]), f4(YT(T_B_INT)[y]), os, wr);
                }
                *reinterpret_cast<float4*>(SC1 + 4 * uq) = X;
            }
            __syncthreads();
        }
        const bool yex = exa == 1 && r >= 2 && r < 34;
        if (act1) {
            const float* PR = Rbase + s3 * FT_RPL;
            const float* PA = Abase + s3 * FT_RPL;
            f33 = ld4s(sm + AC_OFF_W + (it & 1) * FT_UPL, uq);   // plane kk+2
            const bool wr1 = inner && kk >= zb && kk < ze;
            const int pz = (pml && zin) ? yzslab_row(kk, a.nz, a.P) : -1;
            const bool bz = pml && (kk - 2 < a.P || kk + 2 >= a.nz - 1 - a.P);
            const bool pml1 = (bx || by || bz) && pok && zin;

            const float4 r0 = ld4s(PR, uq), a0 = ld4s(PA, uq);
            const float4 one = f4(1.0f), mh = f4(-0.5f);
            const float4 cs = ld4s(PS, q);
            float4 n1, n2, n3;
            const int sl = it % AC_RING;
            float* const R1 = sm + AC_OFF_UR + (0 * AC_RING + sl) * FT_UPL + 4 * uq;
            float* const R2 = sm + AC_OFF_UR + (1 * AC_RING + sl) * FT_UPL + 4 * uq;
            float* const R3 = sm + AC_OFF_UR + (2 * AC_RING + sl) * FT_UPL + 4 * uq;
            {   // ---- u1 at (x+1/2, y, z): D+x s
                float4 t1 = dpx(ld2s(PS, 4 * q - 2), cs, ld2s(PS, 4 * q + 4));
                if (MODE == FM_FWD && pml1 && colq >= 0)
                    t1 = pml_fwd_m(pm0, a.mvo[0], ox, tab4(XT(T_A_HALF), x), tab4(XT(T_B_HALF), x), t1, wr1);
                if (MODE == FM_ADJ && pml1 && exa == 0) t1 = t1 + dpx(ld2s(SC1, 4 * uq - 2), ld4s(SC1, uq), ld2s(SC1, 4 * uq + 4));
                const float4 rxp = shl1(r0, PR[4 * uq + 4]), axp = shl1(a0, PA[4 * uq + 4]);
                mbar_wait(&barU[it & 3], (it >> 2) & 1);
                n1 = fma4(fma4(mh, adds(a0, axp), one), *reinterpret_cast<const float4*>(R1), (kB * rcp4(adds(r0, rxp))) * t1);
            }
            {   // ---- u2 at (x, y+1/2, z): D+y s
                const float4 yb = ld4s(PS, q - 10), yc = ld4s(PS, q + 10), yd = ld4s(PS, q + 20);
                float4 t2 = d4(yb, cs, yc, yd);
                if (MODE == FM_FWD && pml1 && prow >= 0)
                    t2 = pml_fwd_m(pm1, a.mvo[4], oy, YT(T_A_HALF)[y], YT(T_B_HALF)[y], t2, wr1);
                if (MODE == FM_ADJ && pml1) {
                    if (yex) t2 = t2 + d4(ld4s(SC1, uq - 10), ld4s(SC1, uq), ld4s(SC1, uq + 10), ld4s(SC1, uq + 20));
                    else if (neary) t2 = t2 + adj_y3(a, a.mvi[13], a.mvo[13], YT(T_A_INT), YT(T_B_INT), oyb, a.nxq, y - 1, 1, yb, cs, yc, yd, wr1 && exa != 1);
                }
                const float4 ryp = ld4s(PR, uq + 10), ayp = ld4s(PA, uq + 10);
                n2 = fma4(fma4(mh, a0 + ayp, one), *reinterpret_cast<const float4*>(R2), (kB * rcp4(r0 + ryp)) * t2);
            }
            {   // ---- u3 at (x, y, z+1/2): D+z s
                float4 t3 = d4(w33b, w33c, w33d, f33);
                if (MODE == FM_FWD && pml1 && pz >= 0)
                    t3 = pml_fwd_m(pm2, a.mvo[8], ozq + pz * szp, ZT(T_A_HALF)[kk & (FT_ZRING - 1)], ZT(T_B_HALF)[kk & (FT_ZRING - 1)], t3, wr1);
                if (MODE == FM_ADJ && pml1 && bz)
                    t3 = t3 + adj_z3(a, a.mvi[17], a.mvo[17], ZT(T_A_INT), ZT(T_B_INT), ozq, szp, kk - 1, 1, w33b, w33c, w33d, f33, wr1);
                const float4 rzp = ld4s(Rbase + s3n * FT_RPL, uq), azp = ld4s(Abase + s3n * FT_RPL, uq);
                n3 = fma4(fma4(mh, a0 + azp, one), *reinterpret_cast<const float4*>(R3), (kB * rcp4(r0 + rzp)) * t3);
            }
            if (EDGE && (edge_xy || !zin)) {
                if (!(zin && m0)) { n1.x = 0.0f; n2.x = 0.0f; n3.x = 0.0f; }
                if (!(zin && m1)) { n1.y = 0.0f; n2.y = 0.0f; n3.y = 0.0f; }
                if (!(zin && m2)) { n1.z = 0.0f; n2.z = 0.0f; n3.z = 0.0f; }
                if (!(zin && m3)) { n1.w = 0.0f; n2.w = 0.0f; n3.w = 0.0f; }
            }
            *reinterpret_cast<float4*>(R1) = n1;
            *reinterpret_cast<float4*>(R2) = n2;
            *reinterpret_cast<float4*>(R3) = n3;
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            const long long g = (long long)kk * a.sz + gxy;
            if (wr1) {
                store_quad<EDGE>(a.out + U1 * box + g, n1, x, a.nx);
                store_quad<EDGE>(a.out + U2 * box + g, n2, x, a.nx);
                store_quad<EDGE>(a.out + U3 * box + g, n3, x, a.nx);
            }
        }
        // forward C-PML: psi11, psi22, psi33 of the quad at plane ks = kk - 2, issued ahead of the barrier
        float4 qm0 = z4, qm1 = z4, qm2 = z4;
        if (MODE == FM_FWD) {
            if (bx || by || (pml && (kk - 4 < a.P || kk >= a.nz - 1 - a.P))) {
                const bool ok = inner && it >= 4;
                const int pzk = ok ? yzslab_row(kk - 2, a.nz, a.P) : -1;
                const bool ex = ok && colq >= 0, ey = ok && prow >= 0, ez = pzk >= 0;
                ldg4_into(qm0, a.mvi[9] + (ex ? ox - 2 * sxp : 0), ex);
                ldg4_into(qm1, a.mvi[13] + (ey ? oy - 2 * syp : 0), ey);
                ldg4_into(qm2, a.mvi[17] + (ez ? ozq + pzk * szp : 0), ez);
#if FT_PFMV > 0
                const bool zpf = kk - 2 + FT_PFMV < a.nz;
                prefetch_l2(a.mvi[9] + (ox + (FT_PFMV - 2) * sxp), ex && zpf);
                prefetch_l2(a.mvi[13] + (oy + (FT_PFMV - 2) * syp), ey && zpf);
                const int pzf = yzslab_row(kk - 2 + FT_PFMV, a.nz, a.P);
                if (pzf >= 0) prefetch_l2(a.mvi[17] + (ozq + pzf * szp), ok);
#endif
            }
        }
        float4 e2 = z4;
        long long i2 = 0;
        bool se2 = false;
        if (MODE == FM_ADJ && exa >= 0 && it >= 4) {
            const bool ok = pok && (unsigned)(kk - 2) < (unsigned)a.nz;
            se2 = ok && (exa == 0 ? colq >= 0 : prow >= 0);
            i2 = se2 ? (exa == 0 ? ox - 2 * sxp : oy - 2 * syp) : 0;
            ldg4_into(e2, a.mvi[4 * exa] + i2, se2);
        }
        if (pml && tid >= 360 && tid < 364) {
            const int t = tid - 360, z = kk + 3;
            sm[FT_OFF_ZT + t * FT_ZRING + (z & (FT_ZRING - 1))] = (unsigned)z < (unsigned)a.nz ? __ldg(a.tab[2][t] + z) : 0.0f;
        }
        __syncthreads();
        unsigned fE = 0, fLam = 0;
        bool kE = false, kLam = false;
        if (tid == FT_PROD) {
            fh = (fh << 8) | fnew;
            fE = (unsigned)fh & 0xffu; fLam = (unsigned)(fh >> 32) & 0xffu;
            const unsigned fIt = (unsigned)(fh >> 24) & 0xffu, fM3 = (unsigned)(fh >> 48) & 0xffu;
            kE = fE != 0 && fE == fIt;
            kLam = it >= 2 && fLam != 0 && fLam == fM3;
            // ring slot of plane it + 3 held plane it - 3, last read in stage 2 of iteration it - 1: free since this barrier
            if (it + 3 < itn) issueU(it + 3);
            if (it + 2 <= itn) issueM(it, fLam, kLam);
            if (it + 2 < itn) issueG(it + 2, fE, 0u, kE);
        }
        if (it >= 1) mbar_wait(&barM[(it - 1) % 3], ((it - 1) / 3) & 1);
        // ------------------------------------------------------------------ stage 2: s(ks), ks = kk - 2
        const int ks = kk - 2;
        float4 cc3 = z4;
        if (inner && it >= 2) cc3 = ld4s(sm + AC_OFF_UR + 2 * AC_RING * FT_UPL + ((it + AC_RING - 2) % AC_RING) * FT_UPL, uq);
        float* const SC2 = sm + AC_OFF_SC2;
        if (exa >= 0) {
            if (act1 && it >= 4) {
                float4 Y = z4;
                if (pok && (unsigned)ks < (unsigned)a.nz) {
                    const int pc = ((it + AC_RING - 2) % AC_RING) * FT_UPL;
                    if (exa == 0) Y = adj_own_x(e2, a.mvo[0], i2, se2, tab4(XT(T_A_HALF), x), tab4(XT(T_B_HALF), x),
                                                ld4s(sm + AC_OFF_UR + 0 * AC_RING * FT_UPL + pc, uq), inner);
                    else Y = adj_own_x(e2, a.mvo[4], i2, se2, f4(YT(T_A_HALF)[y]), f4(YT(T_B_HALF)[y]),
                                       ld4s(sm + AC_OFF_UR + 1 * AC_RING * FT_UPL + pc, uq), inner);
                }
                *reinterpret_cast<float4*>(SC2 + 4 * uq) = Y;
            }
            __syncthreads();
        }
        if (inner && it >= 4) {
            const int j = it - 2;
            const float* U1p = sm + AC_OFF_UR + 0 * AC_RING * FT_UPL;
            const float* U2p = sm + AC_OFF_UR + 1 * AC_RING * FT_UPL;
            const float* U3p = sm + AC_OFF_UR + 2 * AC_RING * FT_UPL;
            const int p0 = (j % AC_RING) * FT_UPL, pp1 = ((j + 1) % AC_RING) * FT_UPL;
            const int pz = pml ? yzslab_row(ks, a.nz, a.P) : -1;
            const bool bz = pml && (ks - 2 < a.P || ks + 2 >= a.nz - 1 - a.P);
            const bool pml2 = bx || by || bz;
            float4 e11, e22, e33;
            {   // D-x u1
                e11 = dmx(ld2s(U1p + p0, 4 * uq - 2), ld4s(U1p + p0, uq), ld2s(U1p + p0, 4 * uq + 4));
                if (MODE == FM_FWD && pml2 && colq >= 0)
                    e11 = pml_fwd_m(qm0, a.mvo[9], ox - 2 * sxp, tab4(XT(T_A_INT), x), tab4(XT(T_B_INT), x), e11, true);
                if (MODE == FM_ADJ && pml2 && exa == 0) e11 = e11 + dmx(ld2s(SC2, 4 * uq - 2), ld4s(SC2, uq), ld2s(SC2, 4 * uq + 4));
            }
            {   // D-y u2
                const float4 ya = ld4s(U2p + p0, uq - 20), yb = ld4s(U2p + p0, uq - 10), c = ld4s(U2p + p0, uq), yd = ld4s(U2p + p0, uq + 10);
                e22 = d4(ya, yb, c, yd);
                if (MODE == FM_FWD && pml2 && prow >= 0)
                    e22 = pml_fwd_m(qm1, a.mvo[13], oy - 2 * syp, YT(T_A_INT)[y], YT(T_B_INT)[y], e22, true);
                if (MODE == FM_ADJ && pml2) {
                    if (exa == 1) e22 = e22 + d4(ld4s(SC2, uq - 20), ld4s(SC2, uq - 10), ld4s(SC2, uq), ld4s(SC2, uq + 10));
                    else if (neary) e22 = e22 + adj_y3(a, a.mvi[4], a.mvo[4], YT(T_A_HALF), YT(T_B_HALF), oyb - 2 * syp, a.nxq, y - 2, 2, ya, yb, c, yd, true);
                }
            }
            {   // D-z u3
                const float4 zd = ld4s(U3p + pp1, uq);
                e33 = d4(u3m2, u3m1, cc3, zd);
                if (MODE == FM_FWD && pml2 && pz >= 0)
                    e33 = pml_fwd_m(qm2, a.mvo[17], ozq + pz * szp, ZT(T_A_INT)[ks & (FT_ZRING - 1)], ZT(T_B_INT)[ks & (FT_ZRING - 1)], e33, true);
                if (MODE == FM_ADJ && pml2 && bz)
                    e33 = e33 + adj_z3(a, a.mvi[8], a.mvo[8], ZT(T_A_HALF), ZT(T_B_HALF), ozq, szp, ks - 2, 2, u3m2, u3m1, cc3, zd, true);
            }
            const float4 lam = ld4s(sm + AC_OFF_LAM + (it & 1) * FT_LPL, lq);
            const float4 ldiv = (kL * lam) * (e11 + e22 + e33);
            const float4 ns = ld4s(sm + AC_OFF_SO + (it & 1) * FT_LPL, lq) + ldiv;
            store_quad<EDGE>(a.out + S11 * box + (long long)ks * a.sz + gxy, ns, x, a.nx);
        }
        u3m2 = u3m1; u3m1 = cc3;
        if (MODE != FM_PLAIN) { ox += sxp; oy += syp; oyb += syp; }
        w33a = w33b; w33b = w33c; w33c = w33d; w33d = f33;
    }
}

// One launch = one time step of the fluid-only operator pair (same persistent work-queue scheme as k_step).
template <int MODE>
__global__ void __launch_bounds__(FT_NT, 1)
k_step_acoustic(const __grid_constant__ CUtensorMap tmS40, const __grid_constant__ CUtensorMap tmS36,
                const __grid_constant__ CUtensorMap tmM37, const __grid_constant__ CUtensorMap tmL,
                const __grid_constant__ CUtensorMap tmS32, const FusedArgs a)
{
    extern __shared__ __align__(1024) float sm[];
    int* s_next = reinterpret_cast<int*>(sm + FT_OFF_ZT + 4 * FT_ZRING);
    const int n = a.work_end - a.work_begin;
    bool first = true;
    for (;;) {
        if (threadIdx.x == 0) *s_next = (int)atomicAdd(a.queue, 1u);
        __syncthreads();
        const int b = *s_next;
        if (b >= n) break;
        const int4 wk = __ldg(a.work + a.work_begin + b);
        if (MODE != FM_PLAIN && (wk.x & FT_WORK_SLAB)) acoustic_brick<MODE, true>(sm, tmS40, tmS36, tmM37, tmL, tmS32, a, wk, first);
        else if (wk.x & FT_WORK_NOEDGE) acoustic_brick<FM_PLAIN, false>(sm, tmS40, tmS36, tmM37, tmL, tmS32, a, wk, first);
        else acoustic_brick<FM_PLAIN, true>(sm, tmS40, tmS36, tmM37, tmL, tmS32, a, wk, first);
        first = false;
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        __threadfence();
        if (atomicAdd(a.queue + 1, 1u) == gridDim.x - 1) {
            a.queue[0] = 0u;
            a.queue[1] = 0u;
        }
    }
}
