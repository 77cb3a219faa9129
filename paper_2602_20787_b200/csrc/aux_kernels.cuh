// aux_kernels.cuh -- the O(N) kernels around the all-pairs sum: pack + wrap (a1), partial-sum
// reduction (a5), homogeneous-cylinder background force (a6, Eq. 9/10), KDK kick/drift (a7,
// Eq. 11), and the FP64-pipe ceiling probe used for the roofline denominator.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "pair_fp64.cuh"

namespace steps {

// z reduced to [0, L)  (periodicity along z).
__device__ __forceinline__ double wrap_z(double z, double L)
{
    double w = z - L * floor(z / L);
    if (w >= L) w -= L;        // floor() round-off when z is a tiny negative number
    if (w < 0.0) w = 0.0;
    return w;
}

// a6: homogeneous cylinder, Eq. 9 in the corrected form of DESIGN.md reading G3:
//   F_h = 2 G rho0 int_0^R { 2 ln[(w+ + L)/(w- + L)] - ln(a+/a-) } dY,
//   a+- = R^2 + rho^2 +- 2 rho sqrt(R^2 - Y^2),  w+- = sqrt(L^2 + a+-),  L = N_cut L_z,
// by double-exponential quadrature: nodes Y_k = R - e_k, stored as (Y_k, e_k, weight_k) so that
// sqrt(R^2 - Y^2) = sqrt(e (R + Y)) is cancellation free at the nodes that crowd Y = R and Y = 0.
// The two logarithms are merged: integrand = ln{ [(w+ + L)/(w- + L)]^2 a-/a+ }.
struct QuadNode { double Y, e, wgt; };

// Quadrature sum of the nodes kq = k0, k0 + stride, ... for a particle at radius rho.
__device__ __forceinline__ double background_nodes(double rho, double R, double Lhalf,
                                                   const QuadNode *__restrict__ nodes, int n_nodes,
                                                   int k0, int stride)
{
    const double L2 = Lhalf * Lhalf;
    double acc = 0.0;
    for (int kq = k0; kq < n_nodes; kq += stride) {
        const QuadNode q = nodes[kq];
        const double X  = sqrt(q.e * (R + q.Y));
        // a+- = (rho +- X)^2 + Y^2  (R^2 = X^2 + Y^2): no cancellation for rho ~ R, Y ~ 0
        const double Y2 = q.Y * q.Y, sp = rho + X, sm = rho - X;
        const double ap = fma(sp, sp, Y2), am = fma(sm, sm, Y2);
        if (am <= 0.0) continue;                                      // rho == R, Y == 0: measure zero
        const double wp = sqrt(L2 + ap), wm = sqrt(L2 + am);
        const double ratio = (wp + Lhalf) / (wm + Lhalf);
        acc = fma(q.wgt, log(ratio * ratio * (am / ap)), acc);
    }
    return acc;
}

// ---------------------------------------------------------------------------------------------
// The O(N) work of a force evaluation / KDK step is two launches around the all-pairs kernel:
//   prestep_kernel  : [b(x_n), kick 1, drift]  pack + wrap (a1), zero the accumulators, max(h), h <= 0
//   poststep_kernel : partial-sum reduction (a5)  [b(x_n+1), kick 2]
// (the bracketed parts only inside steps_cyl_kdk_step).
//   LANES = 1 : one thread per particle, one 128-thread CTA per tile;
//   LANES = 32: one WARP per particle, 8 particles per 256-thread CTA -- the Eq. 9 quadrature (361 nodes, ~100 FP64
//               instructions each) is then spread over the lanes and over every SM; with a thread per particle it would
//               outlast the pair kernel at small n (n = 2048: 128 particles x 361 nodes on each of 16 SMs).
struct BgParams {
    double R, Lhalf, G, rho0;
    int infinite;                    // Eq. 10 instead of Eq. 9
    int n_nodes;
    const QuadNode *nodes;
};
struct KickParams { double inv_a3, H, dt; };
// Single-writer slabs of the deterministic symmetric kernel (pair_fp64_sym.cuh, SLAB): rows = CTA rows of the pair
// kernel (tr target tiles each), then chunks x split target-side slabs; tpc = source tiles per chunk.  rows == 0: off.
struct SlabLayout { int rows, tr, tpc, chunks, split; };

template <int LANES> struct OnStep {
    static constexpr int kParticlesPerBlock = (LANES == 32) ? 8 : PAIR_THREADS;
    static constexpr int kThreads = (LANES == 32) ? 256 : PAIR_THREADS;
};

// s with b = s (x, y): s = -F_h(rho)/rho (Eq. 11 subtracts F_h < 0: outward push); 0 when disabled or on the axis.
// LANES == 32: called by a whole warp for ONE particle, every lane returns the sum.
template <int LANES>
__device__ __forceinline__ double background_scale(double xv, double yv, const BgParams &bg, int lane)
{
    if (bg.rho0 == 0.0) return 0.0;
    const double rho = sqrt(fma(xv, xv, yv * yv));
    if (rho == 0.0) return 0.0;
    double Fh;
    if (bg.infinite) {
        Fh = -2.0 * 3.141592653589793238 * bg.G * bg.rho0 * rho;          // Eq. 10
    } else {
        double acc = background_nodes(rho, bg.R, bg.Lhalf, bg.nodes, bg.n_nodes, LANES == 32 ? lane : 0, LANES);
        if (LANES == 32) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        }
        Fh = 2.0 * bg.G * bg.rho0 * acc;
    }
    return -Fh / rho;
}

__device__ __forceinline__ void atomic_max_positive(double *addr, double v)      // v > 0: bit patterns order like values
{
    atomicMax(reinterpret_cast<unsigned long long *>(addr), (unsigned long long)__double_as_longlong(v));
}

// a1 (+ a6, a7 first half when KICK).  KICK (reading S4):
//   v <- v + (dt/2)[(g + b)/a_n^3 - 2 H_n v];  x <- x + v dt;  z reduced to [0, L)
// then, for the positions the force is wanted at: SoA -> packed, padded source arrays (massless far-away dummies
// beyond n), float hi/lo splits for the mixed kernels, per-tile max h (bounds h_i + h_j in the spline pre-test;
// tile_hmax is zero on entry -- poststep_kernel clears it), global max h and the h <= 0 flag, and zeroed
// accumulator rows part[0 .. zero_rows) x [n_pad].   grid = n_pad / particles per block.
template <int LANES, bool KICK>
__global__ void __launch_bounds__(OnStep<LANES>::kThreads)
prestep_kernel(double *__restrict__ x, double *__restrict__ y, double *__restrict__ z,
               double *__restrict__ vx, double *__restrict__ vy, double *__restrict__ vz,
               const double *__restrict__ gx, const double *__restrict__ gy, const double *__restrict__ gz,
               const double *__restrict__ m, const double *__restrict__ h, int n, int n_pad, double L,
               BgParams bg, KickParams kp,
               double2 *__restrict__ xy, double2 *__restrict__ zm, double *__restrict__ hs,
               float4 *__restrict__ f_hi, float4 *__restrict__ f_lo, double *__restrict__ tile_hmax,
               DevFlags *__restrict__ flags, int *__restrict__ bad_h_sticky,
               double *__restrict__ part, int zero_rows, const int *__restrict__ perm)
{
    const int lane = threadIdx.x & 31;
    const int i = (LANES == 32) ? blockIdx.x * OnStep<LANES>::kParticlesPerBlock + (threadIdx.x >> 5)
                                : blockIdx.x * PAIR_THREADS + threadIdx.x;           // < n_pad
    // i: slot in the packed arrays; p: the caller's index of the particle that sits there (perm: the spatial
    // ordering of the EWALD_TABLE kernels, order_kernels.cuh; nullptr = caller order)
    const int p = (perm != nullptr && i < n) ? perm[i] : i;
    double xv, yv, zv, mv, hv;
    if (i < n) {
        xv = x[p]; yv = y[p];
        double sb = 0.0;
        if (KICK) sb = background_scale<LANES>(xv, yv, bg, lane);
        if (LANES == 32 && lane != 0) return;
        zv = z[p]; mv = m[p]; hv = h[p];
        if (KICK) {
            const double hdt = 0.5 * kp.dt;
            double ux = vx[p], uy = vy[p], uz = vz[p];
            ux = ux + hdt * ((gx[p] + sb * xv) * kp.inv_a3 - 2.0 * kp.H * ux);
            uy = uy + hdt * ((gy[p] + sb * yv) * kp.inv_a3 - 2.0 * kp.H * uy);
            uz = uz + hdt * (gz[p] * kp.inv_a3 - 2.0 * kp.H * uz);
            vx[p] = ux; vy[p] = uy; vz[p] = uz;
            xv = xv + ux * kp.dt;
            yv = yv + uy * kp.dt;
            zv = wrap_z(zv + uz * kp.dt, L);
            x[p] = xv; y[p] = yv; z[p] = zv;
        } else {
            zv = wrap_z(zv, L);
        }
        if (!(hv > 0.0)) { atomicOr(&flags->bad_h, 1); atomicOr(bad_h_sticky, 1); }
    } else {                   // massless dummy far outside any particle load
        if (LANES == 32 && lane != 0) return;
        xv = 1.0e60; yv = 1.0e60; zv = 0.0; mv = 0.0; hv = 1.0;
    }
    xy[i] = make_double2(xv, yv);
    zm[i] = make_double2(zv, mv);
    hs[i] = hv;
    for (int r = 0; r < zero_rows; ++r) part[(size_t)r * n_pad + i] = 0.0;
    const double hm = (i < n && hv > 0.0) ? hv : 0.0;         // dummies count as 0
    if (LANES == 32) {
        if (hm > 0.0) {
            atomic_max_positive(tile_hmax + i / PAIR_THREADS, hm);
            atomicMax(&flags->hmax_bits, (unsigned long long)__double_as_longlong(hm));
        }
    } else {                   // the CTA is the tile: shuffle / shared-memory reduction, one store
        __shared__ double s_max[PAIR_THREADS / 32];
        double t = hm;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t = fmax(t, __shfl_xor_sync(0xffffffffu, t, o));
        if (lane == 0) s_max[threadIdx.x >> 5] = t;
        __syncthreads();
        if (threadIdx.x == 0) {
            for (int wq = 1; wq < PAIR_THREADS / 32; ++wq) t = fmax(t, s_max[wq]);
            tile_hmax[blockIdx.x] = t;
            if (t > 0.0) atomicMax(&flags->hmax_bits, (unsigned long long)__double_as_longlong(t));
        }
    }
    if (f_hi) {
        // x = hi + lo with hi = fl32(x), lo = fl32(x - hi): the difference of two such pairs,
        // (hi_i - hi_j) + (lo_i - lo_j), keeps ~2^-24 RELATIVE accuracy of the separation
        // even for close pairs at large radius (Sterbenz: the hi difference is then exact).
        if (i >= n) { xv = 1.0e18; yv = 1.0e18; }
        const float xh = (float)xv, yh = (float)yv, zh = (float)zv;
        f_hi[i] = make_float4(xh, yh, zh, (float)mv);
        f_lo[i] = make_float4((float)(xv - (double)xh), (float)(yv - (double)yh),
                              (float)(zv - (double)zh), (float)hv);
    }
}

// a5 (+ a6, a7 second half when KICK): g = -G (A_x, A_y, A_z1 - L A_z2), the partial sums added over the n_slabs
// slabs the pair kernel wrote, in fixed order; KICK:  v <- [v + (dt/2)(g' + b')/a_{n+1}^3] / (1 + H_{n+1} dt).
// Also clears what the NEXT evaluation's prestep accumulates into with atomics: the other flag block (flags
// alternate between two blocks, so that no memset sits between the launches) and tile_hmax.
template <int LANES, bool KICK>
__global__ void __launch_bounds__(OnStep<LANES>::kThreads)
poststep_kernel(const double *__restrict__ part, int n, int n_pad, int n_slabs, double G, double L,
                DevFlags *__restrict__ flags_next, double *__restrict__ tile_hmax,
                double *__restrict__ gx, double *__restrict__ gy, double *__restrict__ gz,
                const double *__restrict__ x, const double *__restrict__ y,
                double *__restrict__ vx, double *__restrict__ vy, double *__restrict__ vz,
                BgParams bg, KickParams kp, const int *__restrict__ perm, SlabLayout sl)
{
    const int lane = threadIdx.x & 31;
    const int i = (LANES == 32) ? blockIdx.x * OnStep<LANES>::kParticlesPerBlock + (threadIdx.x >> 5)
                                : blockIdx.x * PAIR_THREADS + threadIdx.x;           // < n_pad
    if (blockIdx.x == 0 && threadIdx.x == 0) { flags_next->hmax_bits = 0ull; flags_next->bad_h = 0; }
    if ((i % PAIR_THREADS) == 0 && lane == 0) tile_hmax[i / PAIR_THREADS] = 0.0;
    if (i >= n) return;
    const int p = (perm != nullptr) ? perm[i] : i;      // slot i of the packed arrays holds the caller's particle p
    double sb = 0.0, xv = 0.0, yv = 0.0;
    if (KICK) {
        xv = x[p]; yv = y[p];
        sb = background_scale<LANES>(xv, yv, bg, lane);
    }
    if (LANES == 32 && lane != 0) return;
    double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
    if (sl.rows > 0) {
        // the slots of particle i that were written, in fixed order: source-side sums from every CTA row at or
        // below its tile's row, target-side sums from every non-empty CTA (chunk, sub-tile) of its own row
        const size_t slab = 3 * (size_t)n_pad;
        const int tile = i / PAIR_THREADS, row = tile / sl.tr;
        for (int bx = 0; bx <= row; ++bx) {
            const double *p = part + (size_t)bx * slab + i;
            a0 += p[0];
            a1 += p[(size_t)n_pad];
            a2 += p[2 * (size_t)n_pad];
        }
        for (int c = (row * sl.tr) / sl.tpc; c < sl.chunks; ++c)
            for (int z = 0; z < sl.split; ++z) {
                const double *p = part + ((size_t)sl.rows + (size_t)c * sl.split + z) * slab + i;
                a0 += p[0];
                a1 += p[(size_t)n_pad];
                a2 += p[2 * (size_t)n_pad];
            }
    } else
    for (int c = 0; c < n_slabs; ++c) {
        const double *p = part + (size_t)c * 4 * n_pad + i;
        a0 += p[0];
        a1 += p[(size_t)n_pad];
        a2 += p[2 * (size_t)n_pad];
        a3 += p[3 * (size_t)n_pad];
    }
    const double g0 = -G * a0, g1 = -G * a1, g2 = -G * fma(-L, a3, a2);
    gx[p] = g0; gy[p] = g1; gz[p] = g2;
    if (KICK) {
        const double hdt = 0.5 * kp.dt, den = 1.0 + kp.H * kp.dt;
        vx[p] = (vx[p] + hdt * (g0 + sb * xv) * kp.inv_a3) / den;
        vy[p] = (vy[p] + hdt * (g1 + sb * yv) * kp.inv_a3) / den;
        vz[p] = (vz[p] + hdt * g2 * kp.inv_a3) / den;
    }
}

// steps_cyl_background: LANES = 1: one thread per particle.  LANES = 32: one warp per particle.
template <int LANES>
__global__ void background_kernel(const double *__restrict__ x, const double *__restrict__ y,
                                  int n, BgParams bg, double *__restrict__ bx, double *__restrict__ by)
{
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    const int i = tid / LANES, lane = tid % LANES;
    if (i >= n) return;                                               // uniform over a warp when LANES == 32
    const double xv = x[i], yv = y[i];
    const double s = background_scale<LANES>(xv, yv, bg, lane);
    if (lane != 0) return;
    bx[i] = s * xv;
    by[i] = s * yv;
}

// FP64-pipe ceiling: 16 independent DFMA chains per thread, `iters` x 16 DFMAs each.
__global__ void __launch_bounds__(256) dfma_peak_kernel(double *out, int iters, double a, double b)
{
    double r[16];
#pragma unroll
    for (int q = 0; q < 16; ++q) r[q] = (double)(threadIdx.x + q);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int q = 0; q < 16; ++q) r[q] = fma(r[q], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int q = 0; q < 16; ++q) s += r[q];
    if (s == 123.456) out[0] = s;     // never true for the a, b used; keeps the chain alive
}

}  // namespace steps
