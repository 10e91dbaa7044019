// kernels_plain.cuh — variant 1: plain two-kernel in-place time step (one thread per cell).
//
// Forward  (Eq. 46):   k_fwd_vel = 46a + 46b ; k_fwd_str = 46c + 46d
// Adjoint  (Eq. 61; W'^T = S1^T S2^T S3^T S4^T):
//   k_adj_a1 : S4^T, S3^T pointwise part  -> 9 coefficient-scaled fields d_bar (scratch), psi~
//   k_adj_a2 : u_bar <- J u_bar - D(d_bar)                 (transposed differences as gathers)
//   k_adj_b1 : S2^T, S1^T pointwise part  -> 9 fields d_bar (scratch), phi~
//   k_adj_b2 : sigma_bar <- sigma_bar - D(d_bar)
// The adjoint stores u~ (before J) and the memory variables before their b factor ("tilde"
// forms); J and b are applied when the value is next read, which makes every update pointwise.
#pragma once
#include "common.cuh"

#define PLAIN_BX 32
#define PLAIN_BY 8
#define PLAIN_BZ 2

// forward C-PML recursion (Eq. 37/41 + Eq. 36, kappa = 1): mem <- b mem + a d ; return d + mem
__device__ __forceinline__ float cpml_f(float* __restrict__ mem, long long mi, float a, float b, float d)
{
    const float m = fmaf(b, mem[mi], a * d);
    mem[mi] = m;
    return d + m;
}

// transposed recursion in tilde form: T <- b T + g ; return g + a T
__device__ __forceinline__ float cpml_t(float* __restrict__ mem, long long mi, float a, float b, float g)
{
    const float t = fmaf(b, mem[mi], g);
    mem[mi] = t;
    return fmaf(a, t, g);
}

#define PLAIN_THREAD_COORDS                                              \
    const int x = blockIdx.x * PLAIN_BX + threadIdx.x;                   \
    const int y = blockIdx.y * PLAIN_BY + threadIdx.y;                   \
    const int z = blockIdx.z * PLAIN_BZ + threadIdx.z;                   \
    if (x >= g.nx || y >= g.ny || z >= g.nz) return;                     \
    const long long sy = g.sy, sz = g.sz;                                \
    const long long i = (long long)z * sz + (long long)y * sy + x;

#define SLAB_X(q) ((long long)(q) + (long long)g.W * ((long long)y + (long long)g.ny * z))
#define SLAB_Y(q) ((long long)x + (long long)g.nx * ((long long)(q) + (long long)g.W * z))
#define SLAB_Z(q) ((long long)x + (long long)g.nx * ((long long)y + (long long)g.ny * (q)))

// ------------------------------------------------------------------------------------------------
// Eq. 46a + 46b
__global__ void __launch_bounds__(PLAIN_BX* PLAIN_BY* PLAIN_BZ) k_fwd_vel(const DevGrid g)
{
    PLAIN_THREAD_COORDS
    const float* __restrict__ s11 = g.f[S11];
    const float* __restrict__ s22 = g.f[S22];
    const float* __restrict__ s33 = g.f[S33];
    const float* __restrict__ s23 = g.f[S23];
    const float* __restrict__ s13 = g.f[S13];
    const float* __restrict__ s12 = g.f[S12];
    // u1 at (x+1/2,y,z)
    float d11 = DP(s11, i, 1), d12 = DM(s12, i, sy), d13 = DM(s13, i, sz);
    // u2 at (x,y+1/2,z)
    float d21 = DM(s12, i, 1), d22 = DP(s22, i, sy), d23 = DM(s23, i, sz);
    // u3 at (x,y,z+1/2)
    float d31 = DM(s13, i, 1), d32 = DM(s23, i, sy), d33 = DP(s33, i, sz);
    if (g.P > 0) {
        const int qx = slab_pos(x, g.nx, g.P), qy = slab_pos(y, g.ny, g.P), qz = slab_pos(z, g.nz, g.P);
        if (qx >= 0) {
            const long long mi = SLAB_X(qx);
            const float ai = g.tab[0][T_A_INT][x], bi = g.tab[0][T_B_INT][x];
            d11 = cpml_f(g.phi[0], mi, g.tab[0][T_A_HALF][x], g.tab[0][T_B_HALF][x], d11);
            d21 = cpml_f(g.phi[3], mi, ai, bi, d21);
            d31 = cpml_f(g.phi[6], mi, ai, bi, d31);
        }
        if (qy >= 0) {
            const long long mi = SLAB_Y(qy);
            const float ai = g.tab[1][T_A_INT][y], bi = g.tab[1][T_B_INT][y];
            d12 = cpml_f(g.phi[1], mi, ai, bi, d12);
            d22 = cpml_f(g.phi[4], mi, g.tab[1][T_A_HALF][y], g.tab[1][T_B_HALF][y], d22);
            d32 = cpml_f(g.phi[7], mi, ai, bi, d32);
        }
        if (qz >= 0) {
            const long long mi = SLAB_Z(qz);
            const float ai = g.tab[2][T_A_INT][z], bi = g.tab[2][T_B_INT][z];
            d13 = cpml_f(g.phi[2], mi, ai, bi, d13);
            d23 = cpml_f(g.phi[5], mi, ai, bi, d23);
            d33 = cpml_f(g.phi[8], mi, g.tab[2][T_A_HALF][z], g.tab[2][T_B_HALF][z], d33);
        }
    }
    const float r0 = g.Rr[i], a0 = g.Aa[i];
    // J = 1 - dt alpha_b (Eq. 7a), dt/(h rho_b) with rho_b, alpha_b 2-point means
    g.f[U1][i] = fmaf(1.0f - 0.5f * (a0 + g.Aa[i + 1]), g.f[U1][i], 2.0f / (r0 + g.Rr[i + 1]) * (d11 + d12 + d13));
    g.f[U2][i] = fmaf(1.0f - 0.5f * (a0 + g.Aa[i + sy]), g.f[U2][i], 2.0f / (r0 + g.Rr[i + sy]) * (d21 + d22 + d23));
    g.f[U3][i] = fmaf(1.0f - 0.5f * (a0 + g.Aa[i + sz]), g.f[U3][i], 2.0f / (r0 + g.Rr[i + sz]) * (d31 + d32 + d33));
}

// harmonic 4-point mean of mu dt/h from the inverse volume Mi (inf where mu = 0 -> result 0)
__device__ __forceinline__ float mu_shear(const float* __restrict__ Mi, long long i, long long s1, long long s2)
{
    return 4.0f / (Mi[i] + Mi[i + s1] + Mi[i + s2] + Mi[i + s1 + s2]);
}

// ------------------------------------------------------------------------------------------------
// Eq. 46c + 46d (Psi: Eq. 7c)
__global__ void __launch_bounds__(PLAIN_BX* PLAIN_BY* PLAIN_BZ) k_fwd_str(const DevGrid g)
{
    PLAIN_THREAD_COORDS
    const float* __restrict__ u1 = g.f[U1];
    const float* __restrict__ u2 = g.f[U2];
    const float* __restrict__ u3 = g.f[U3];
    float e11 = DM(u1, i, 1), e22 = DM(u2, i, sy), e33 = DM(u3, i, sz);
    float g12 = DP(u1, i, sy), g21 = DP(u2, i, 1);   // s12 at (x+1/2,y+1/2,z)
    float g13 = DP(u1, i, sz), g31 = DP(u3, i, 1);   // s13 at (x+1/2,y,z+1/2)
    float g23 = DP(u2, i, sz), g32 = DP(u3, i, sy);  // s23 at (x,y+1/2,z+1/2)
    if (g.P > 0) {
        const int qx = slab_pos(x, g.nx, g.P), qy = slab_pos(y, g.ny, g.P), qz = slab_pos(z, g.nz, g.P);
        if (qx >= 0) {
            const long long mi = SLAB_X(qx);
            const float ah = g.tab[0][T_A_HALF][x], bh = g.tab[0][T_B_HALF][x];
            e11 = cpml_f(g.psi[0], mi, g.tab[0][T_A_INT][x], g.tab[0][T_B_INT][x], e11);
            g21 = cpml_f(g.psi[3], mi, ah, bh, g21);
            g31 = cpml_f(g.psi[6], mi, ah, bh, g31);
        }
        if (qy >= 0) {
            const long long mi = SLAB_Y(qy);
            const float ah = g.tab[1][T_A_HALF][y], bh = g.tab[1][T_B_HALF][y];
            g12 = cpml_f(g.psi[1], mi, ah, bh, g12);
            e22 = cpml_f(g.psi[4], mi, g.tab[1][T_A_INT][y], g.tab[1][T_B_INT][y], e22);
            g32 = cpml_f(g.psi[7], mi, ah, bh, g32);
        }
        if (qz >= 0) {
            const long long mi = SLAB_Z(qz);
            const float ah = g.tab[2][T_A_HALF][z], bh = g.tab[2][T_B_HALF][z];
            g13 = cpml_f(g.psi[2], mi, ah, bh, g13);
            g23 = cpml_f(g.psi[5], mi, ah, bh, g23);
            e33 = cpml_f(g.psi[8], mi, g.tab[2][T_A_INT][z], g.tab[2][T_B_INT][z], e33);
        }
    }
    const float ll = g.Ll[i], mn2 = 2.0f / g.Mi[i];
    const float ldiv = ll * (e11 + e22 + e33);
    g.f[S11][i] += fmaf(mn2, e11, ldiv);
    g.f[S22][i] += fmaf(mn2, e22, ldiv);
    g.f[S33][i] += fmaf(mn2, e33, ldiv);
    g.f[S12][i] += mu_shear(g.Mi, i, 1, sy) * (g12 + g21);
    g.f[S13][i] += mu_shear(g.Mi, i, 1, sz) * (g13 + g31);
    g.f[S23][i] += mu_shear(g.Mi, i, sy, sz) * (g23 + g32);
}

// ------------------------------------------------------------------------------------------------
// Adjoint, S4^T S3^T pointwise part (Eq. 61a and the Delta^T, G^T coefficients of 61b)
__global__ void __launch_bounds__(PLAIN_BX* PLAIN_BY* PLAIN_BZ) k_adj_a1(const DevGrid g)
{
    PLAIN_THREAD_COORDS
    const float ll = g.Ll[i], mn2 = 2.0f / g.Mi[i];
    const float s11 = g.f[S11][i], s22 = g.f[S22][i], s33 = g.f[S33][i];
    const float ltr = ll * (s11 + s22 + s33);
    float e11 = fmaf(mn2, s11, ltr), e22 = fmaf(mn2, s22, ltr), e33 = fmaf(mn2, s33, ltr);
    const float g12 = mu_shear(g.Mi, i, 1, sy) * g.f[S12][i];
    const float g13 = mu_shear(g.Mi, i, 1, sz) * g.f[S13][i];
    const float g23 = mu_shear(g.Mi, i, sy, sz) * g.f[S23][i];
    float d12 = g12, d21 = g12, d13 = g13, d31 = g13, d23 = g23, d32 = g23;
    if (g.P > 0) {
        const int qx = slab_pos(x, g.nx, g.P), qy = slab_pos(y, g.ny, g.P), qz = slab_pos(z, g.nz, g.P);
        if (qx >= 0) {
            const long long mi = SLAB_X(qx);
            const float ah = g.tab[0][T_A_HALF][x], bh = g.tab[0][T_B_HALF][x];
            e11 = cpml_t(g.psi[0], mi, g.tab[0][T_A_INT][x], g.tab[0][T_B_INT][x], e11);
            d21 = cpml_t(g.psi[3], mi, ah, bh, d21);
            d31 = cpml_t(g.psi[6], mi, ah, bh, d31);
        }
        if (qy >= 0) {
            const long long mi = SLAB_Y(qy);
            const float ah = g.tab[1][T_A_HALF][y], bh = g.tab[1][T_B_HALF][y];
            d12 = cpml_t(g.psi[1], mi, ah, bh, d12);
            e22 = cpml_t(g.psi[4], mi, g.tab[1][T_A_INT][y], g.tab[1][T_B_INT][y], e22);
            d32 = cpml_t(g.psi[7], mi, ah, bh, d32);
        }
        if (qz >= 0) {
            const long long mi = SLAB_Z(qz);
            const float ah = g.tab[2][T_A_HALF][z], bh = g.tab[2][T_B_HALF][z];
            d13 = cpml_t(g.psi[2], mi, ah, bh, d13);
            d23 = cpml_t(g.psi[5], mi, ah, bh, d23);
            e33 = cpml_t(g.psi[8], mi, g.tab[2][T_A_INT][z], g.tab[2][T_B_INT][z], e33);
        }
    }
    g.scr[0][i] = e11; g.scr[1][i] = d12; g.scr[2][i] = d13;
    g.scr[3][i] = d21; g.scr[4][i] = e22; g.scr[5][i] = d23;
    g.scr[6][i] = d31; g.scr[7][i] = d32; g.scr[8][i] = e33;
}

// u~ <- J u~ + E~^T.. : transposed differences, (D-)^T = -D+, (D+)^T = -D- under zero padding
__global__ void __launch_bounds__(PLAIN_BX* PLAIN_BY* PLAIN_BZ) k_adj_a2(const DevGrid g)
{
    PLAIN_THREAD_COORDS
    const float a0 = g.Aa[i];
    g.f[U1][i] = fmaf(1.0f - 0.5f * (a0 + g.Aa[i + 1]), g.f[U1][i],
                      -(DP(g.scr[0], i, 1) + DM(g.scr[1], i, sy) + DM(g.scr[2], i, sz)));
    g.f[U2][i] = fmaf(1.0f - 0.5f * (a0 + g.Aa[i + sy]), g.f[U2][i],
                      -(DM(g.scr[3], i, 1) + DP(g.scr[4], i, sy) + DM(g.scr[5], i, sz)));
    g.f[U3][i] = fmaf(1.0f - 0.5f * (a0 + g.Aa[i + sz]), g.f[U3][i],
                      -(DM(g.scr[6], i, 1) + DM(g.scr[7], i, sy) + DP(g.scr[8], i, sz)));
}

// Adjoint, S2^T S1^T pointwise part (Eq. 61c and the F^T coefficients of 61d)
__global__ void __launch_bounds__(PLAIN_BX* PLAIN_BY* PLAIN_BZ) k_adj_b1(const DevGrid g)
{
    PLAIN_THREAD_COORDS
    const float r0 = g.Rr[i];
    const float g1 = 2.0f / (r0 + g.Rr[i + 1]) * g.f[U1][i];
    const float g2 = 2.0f / (r0 + g.Rr[i + sy]) * g.f[U2][i];
    const float g3 = 2.0f / (r0 + g.Rr[i + sz]) * g.f[U3][i];
    float d11 = g1, d12 = g1, d13 = g1, d21 = g2, d22 = g2, d23 = g2, d31 = g3, d32 = g3, d33 = g3;
    if (g.P > 0) {
        const int qx = slab_pos(x, g.nx, g.P), qy = slab_pos(y, g.ny, g.P), qz = slab_pos(z, g.nz, g.P);
        if (qx >= 0) {
            const long long mi = SLAB_X(qx);
            const float ai = g.tab[0][T_A_INT][x], bi = g.tab[0][T_B_INT][x];
            d11 = cpml_t(g.phi[0], mi, g.tab[0][T_A_HALF][x], g.tab[0][T_B_HALF][x], d11);
            d21 = cpml_t(g.phi[3], mi, ai, bi, d21);
            d31 = cpml_t(g.phi[6], mi, ai, bi, d31);
        }
        if (qy >= 0) {
            const long long mi = SLAB_Y(qy);
            const float ai = g.tab[1][T_A_INT][y], bi = g.tab[1][T_B_INT][y];
            d12 = cpml_t(g.phi[1], mi, ai, bi, d12);
            d22 = cpml_t(g.phi[4], mi, g.tab[1][T_A_HALF][y], g.tab[1][T_B_HALF][y], d22);
            d32 = cpml_t(g.phi[7], mi, ai, bi, d32);
        }
        if (qz >= 0) {
            const long long mi = SLAB_Z(qz);
            const float ai = g.tab[2][T_A_INT][z], bi = g.tab[2][T_B_INT][z];
            d13 = cpml_t(g.phi[2], mi, ai, bi, d13);
            d23 = cpml_t(g.phi[5], mi, ai, bi, d23);
            d33 = cpml_t(g.phi[8], mi, g.tab[2][T_A_HALF][z], g.tab[2][T_B_HALF][z], d33);
        }
    }
    g.scr[0][i] = d11; g.scr[1][i] = d12; g.scr[2][i] = d13;
    g.scr[3][i] = d21; g.scr[4][i] = d22; g.scr[5][i] = d23;
    g.scr[6][i] = d31; g.scr[7][i] = d32; g.scr[8][i] = d33;
}

__global__ void __launch_bounds__(PLAIN_BX* PLAIN_BY* PLAIN_BZ) k_adj_b2(const DevGrid g)
{
    PLAIN_THREAD_COORDS
    g.f[S11][i] -= DM(g.scr[0], i, 1);
    g.f[S22][i] -= DM(g.scr[4], i, sy);
    g.f[S33][i] -= DM(g.scr[8], i, sz);
    g.f[S12][i] -= DP(g.scr[1], i, sy) + DP(g.scr[3], i, 1);
    g.f[S13][i] -= DP(g.scr[2], i, sz) + DP(g.scr[6], i, 1);
    g.f[S23][i] -= DP(g.scr[5], i, sz) + DP(g.scr[7], i, sy);
}
