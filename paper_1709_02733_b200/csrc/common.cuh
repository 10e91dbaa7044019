// common.cuh — device-side view of a context, shared by all kernels of libpact.
//
// Layout in HBM: every field is fp32, x fastest, stored in a padded box
//   [nz + 2*HALO_Z][ny + 2*HALO_Y][pitch],  pitch = round_up(nx + HALO_X + 4, 32)
// with node (0,0,0) at element offset `org`, so that element (x,y,z) is at org + x + sy*y + sz*z
// and x = 0 is 128-byte aligned.  The halo holds zeros for state fields ("samples outside the
// index range are zero", reading G9) and edge-replicated values for material volumes
// (clamp at the last index, reading G10), so stencils need no bounds checks.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define PACT_HALO_X 32
#define PACT_HALO_Y 4
#define PACT_HALO_Z 4
#define PACT_NPAL 4     // palette planes behind every material volume (kernels_fused.cuh, material elision)

// state field order
enum { U1 = 0, U2, U3, S11, S22, S33, S23, S13, S12, NFIELD };

// PML table order per axis
enum { T_A_INT = 0, T_B_INT, T_A_HALF, T_B_HALF };

struct DevGrid {
    int nx, ny, nz;
    int P;            // npml
    int W;            // slab width 2P+1 (0 if P == 0)
    long long sy, sz; // strides of the padded box (elements)
    float* f[NFIELD]; // state (pointers to node (0,0,0))
    float* scr[9];    // adjoint scratch fields (same padded layout)
    // scaled material volumes (same padded layout, halo edge-replicated):
    //   Ll = lambda dt/h ; Mi = h/(mu dt) (inf where mu = 0) ; Rr = rho h/dt ; Aa = alpha dt
    const float *Ll, *Mi, *Rr, *Aa;
    // C-PML tables per axis, T_* order, each of length n_axis (Eq. 38)
    const float* tab[3][4];
    // memory variables, slab-confined along their derivative axis b:
    //   b = x: [nz][ny][W] ; b = y: [nz][W][nx] ; b = z: [W][ny][nx]
    // phi[3a+b]: memory of d_b sigma^{ab} at u^a ; psi[3a+b]: memory of d_b u^a at sigma^{ab}
    float* phi[9];
    float* psi[9];
};

// Eq. 8 without the 1/h factor (folded into the scaled material volumes)
#define PACT_C1 1.125f
#define PACT_C2 (-1.0f / 24.0f)

// D+ : integer -> half positions (result at i + 1/2) ; D- : half -> integer (result at i)
#define DP(f, i, s) (PACT_C1 * ((f)[(i) + (s)] - (f)[(i)]) + PACT_C2 * ((f)[(i) + 2 * (s)] - (f)[(i) - (s)]))
#define DM(f, i, s) (PACT_C1 * ((f)[(i)] - (f)[(i) - (s)]) + PACT_C2 * ((f)[(i) + (s)] - (f)[(i) - 2 * (s)]))

// position of index i inside the boundary slab of an axis of length n, or -1
__device__ __forceinline__ int slab_pos(int i, int n, int P)
{
    if (i < P) return i;
    if (i >= n - 1 - P) return i - (n - 1 - P) + P;
    return -1;
}
