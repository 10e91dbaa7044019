// kernels_pgd.cuh — element-wise and reduction kernels of the projected-gradient reconstruction built on the pair
// (H, H^T): the use the paper builds the pair for ("iterative image reconstruction", PAPER.md:357;
// BASELINE.json config 5).  SURVEY 8(f)-1:  p <- max(0, p - s H^T (H p - d)),  s = 1/||H||^2 from a power iteration.
//
// Norms are accumulated in fp64 and are bit-reproducible: every block sums its grid-stride share in a fixed order
// and writes one partial; a single block then adds the partials in index order (no atomics).
#pragma once
#include "common.cuh"

#define PGD_BLOCK 256
#define PGD_MAXBLOCKS 1184     // 148 SMs x 8: upper bound on partial sums

__device__ __forceinline__ double block_sum(double v)
{
    __shared__ double sh[PGD_BLOCK / 32];
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);     // fixed butterfly order
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    double s = 0.0;
    if (threadIdx.x == 0)
        for (int w = 0; w < PGD_BLOCK / 32; ++w) s += sh[w];
    __syncthreads();
    return s;    // valid in thread 0
}

// r <- r - d (the residual H p - d, in place over the nt x L samples) ; partial[b] = sum over the block's share of r^2
__global__ void k_pgd_residual(float* __restrict__ r, const float* __restrict__ d, long long n, double* __restrict__ partial)
{
    double acc = 0.0;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const float v = r[i] - d[i];
        r[i] = v;
        acc += (double)v * (double)v;
    }
    const double s = block_sum(acc);
    if (threadIdx.x == 0) partial[blockIdx.x] = s;
}

// p <- max(0, p - s g) (nonneg) or p - s g ; partial[b] = sum of (p_new - p_old)^2
__global__ void k_pgd_update(float* __restrict__ p, const float* __restrict__ g, float s, int nonneg, long long n,
                             double* __restrict__ partial)
{
    double acc = 0.0;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const float o = p[i];
        float v = fmaf(-s, g[i], o);
        if (nonneg) v = fmaxf(v, 0.0f);
        p[i] = v;
        const double dlt = (double)v - (double)o;
        acc += dlt * dlt;
    }
    const double t = block_sum(acc);
    if (threadIdx.x == 0) partial[blockIdx.x] = t;
}

// partial[b] = sum of v^2 over the block's share
__global__ void k_pgd_norm2(const float* __restrict__ v, long long n, double* __restrict__ partial)
{
    double acc = 0.0;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        acc += (double)v[i] * (double)v[i];
    const double s = block_sum(acc);
    if (threadIdx.x == 0) partial[blockIdx.x] = s;
}

// out[slot] = sqrt(sum of partial[0..nb)), added in index order by one thread (bit-reproducible)
__global__ void k_pgd_finish(const double* __restrict__ partial, int nb, double* __restrict__ out, int slot)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        double s = 0.0;
        for (int b = 0; b < nb; ++b) s += partial[b];
        out[slot] = sqrt(s);
    }
}

// v <- v / norms[slot] (power iteration: normalise with the norm a previous kernel left on the device)
__global__ void k_pgd_scale_by_inverse(float* __restrict__ v, long long n, const double* __restrict__ norms, int slot)
{
    const double nrm = norms[slot];
    const float inv = nrm > 0.0 ? (float)(1.0 / nrm) : 0.0f;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        v[i] *= inv;
}
