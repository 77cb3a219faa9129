// order_kernels.cuh -- spatial ordering of the packed particle arrays (EWALD_TABLE mode).
//
// The table kernels (pair_table_*.cuh) gather four (CIC) or nine (TSC) nodes of the correction table D(rho, |r_z|) of
// Eq. 17 per pair.  A warp handles 32 targets x 32 sources per ring pass; when both groups are
// spatially compact all their separations -- hence all their table nodes -- fall in one small patch of the table,
// and the gathers of a warp touch a few cache lines instead of 32 different ones.  Measured at N = 1 048 576
// (config 3): double-node CIC 4.66 s -> 2.65 s per evaluation, TSC 9.5 s -> 5.0 s (profiles/r2_table_ordering.md).
//
// The order is a Morton (Z-order) curve through (x, y, z) quantised to 11 + 11 + 10 bits, x and y first mapped by
// asinh(x / s), s = R_max / 64, so that the resolution follows the radial compactification of the particle load
// (constant-resolution core, density ~ r^-2 outside: PAPER.md:215-231).  It is only a locality hint: ANY
// permutation gives the same sums, so it is recomputed every kReorderEvery evaluations, not every step.
// Keys are (morton << 32 | caller index): unique, so the bitonic network below -- compare-exchange passes, no
// atomics -- yields the same permutation on every run (the DETERMINISTIC kernels stay bit-reproducible).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace steps {

constexpr int kReorderEvery = 64;          // force evaluations between two re-orderings

// max(|x|, |y|) over the particles, as the bit pattern of a non-negative double (orders like an integer).
__global__ void extent_kernel(const double *__restrict__ x, const double *__restrict__ y, int n,
                              unsigned long long *__restrict__ rmax_bits)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    double v = 0.0;
    if (i < n) v = fmax(fabs(x[i]), fabs(y[i]));
    if (!(v < 1.0e300)) v = 0.0;                       // NaN / Inf coordinates do not set the scale
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    if ((threadIdx.x & 31) == 0 && v > 0.0) atomicMax(rmax_bits, (unsigned long long)__double_as_longlong(v));
}

__device__ __forceinline__ uint32_t spread3(uint32_t v)        // abcd -> a00b00c00d (up to 11 bits)
{
    v &= 0x7ffu;
    v = (v | (v << 16)) & 0x070000ffu;
    v = (v | (v << 8)) & 0x0700f00fu;
    v = (v | (v << 4)) & 0x430c30c3u;
    v = (v | (v << 2)) & 0x49249249u;
    return v;
}

// key[i] = morton(x_i, y_i, z_i) << 32 | i for i < n; the padding up to the power of two sorts last.
__global__ void order_key_kernel(const double *__restrict__ x, const double *__restrict__ y,
                                 const double *__restrict__ z, int n, int n_pow2, double L,
                                 const unsigned long long *__restrict__ rmax_bits,
                                 unsigned long long *__restrict__ keys)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_pow2) return;
    if (i >= n) { keys[i] = ~0ull; return; }
    double R = __longlong_as_double((long long)*rmax_bits);
    if (!(R > 0.0)) R = 1.0;
    const double s = R / 64.0, inv = 1.0 / asinh(64.0);
    const double fx = asinh(x[i] / s) * inv, fy = asinh(y[i] / s) * inv;      // in [-1, 1]
    double fz = z[i] / L;
    fz -= floor(fz);                                                          // in [0, 1)
    const int ix = min(max((int)((fx + 1.0) * 1023.5), 0), 2047);
    const int iy = min(max((int)((fy + 1.0) * 1023.5), 0), 2047);
    const int iz = min(max((int)(fz * 1024.0), 0), 1023);
    // z takes every third bit from bit 2 up (10 bits), x and y the other two (11 bits each): 32 bits in all
    const uint32_t mkey = spread3((uint32_t)ix) | (spread3((uint32_t)iy) << 1) | ((spread3((uint32_t)iz) & 0x09249249u) << 2);
    keys[i] = ((unsigned long long)mkey << 32) | (unsigned)i;
}

// One compare-exchange pass of the bitonic sorting network (ascending), stride j inside sequences of length k.
__global__ void bitonic_pass_kernel(unsigned long long *__restrict__ keys, int n_pow2, int j, int k)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;             // one thread per pair
    if (t >= n_pow2 / 2) return;
    const int i = ((t & ~(j - 1)) << 1) | (t & (j - 1));             // lower element of the pair (bit j clear)
    const int q = i | j;
    const unsigned long long a = keys[i], b = keys[q];
    const bool up = (i & k) == 0;
    if ((a > b) == up) { keys[i] = b; keys[q] = a; }
}

// All passes with stride < 2 * blockDim.x of the merges k = k0 .. k1 (k <= 2 * blockDim.x: the whole merge; larger k:
// its tail) on one 2 * blockDim.x chunk held in shared memory.
template <int THREADS>
__global__ void __launch_bounds__(THREADS)
bitonic_chunk_kernel(unsigned long long *__restrict__ keys, int k0, int k1)
{
    __shared__ unsigned long long s[2 * THREADS];
    const int base = blockIdx.x * 2 * THREADS;
    s[threadIdx.x] = keys[base + threadIdx.x];
    s[threadIdx.x + THREADS] = keys[base + threadIdx.x + THREADS];
    __syncthreads();
    for (int k = k0; k <= k1; k <<= 1) {
        for (int j = min(k >> 1, THREADS); j > 0; j >>= 1) {
            const int t = threadIdx.x;
            const int i = ((t & ~(j - 1)) << 1) | (t & (j - 1));
            const int q = i | j;
            const unsigned long long a = s[i], b = s[q];
            const bool up = ((base + i) & k) == 0;
            if ((a > b) == up) { s[i] = b; s[q] = a; }
            __syncthreads();
        }
        if (k == k1) break;                                          // k1 may be the largest int power of two
    }
    keys[base + threadIdx.x] = s[threadIdx.x];
    keys[base + threadIdx.x + THREADS] = s[threadIdx.x + THREADS];
}

__global__ void order_perm_kernel(const unsigned long long *__restrict__ keys, int n, int *__restrict__ perm)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) perm[i] = (int)(unsigned)(keys[i] & 0xffffffffull);
}

}  // namespace steps
