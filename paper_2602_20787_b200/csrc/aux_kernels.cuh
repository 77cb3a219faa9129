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

// a1: SoA inputs -> packed, padded source arrays; records max(h) and h <= 0.
// Mixed mode additionally gets float hi/lo splits (see pair_mixed.cuh).
__global__ void pack_kernel(const double *__restrict__ x, const double *__restrict__ y,
                            const double *__restrict__ z, const double *__restrict__ m,
                            const double *__restrict__ h, int n, int n_pad, double L,
                            double2 *__restrict__ xy, double2 *__restrict__ zm,
                            double *__restrict__ hs,
                            float4 *__restrict__ f_hi, float4 *__restrict__ f_lo,
                            double *__restrict__ tile_hmax, DevFlags *__restrict__ flags)
{
    // launched with PAIR_THREADS threads per block: block b == source tile b (n_pad = tiles * 128)
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    double xv, yv, zv, mv, hv;
    if (i < n) {
        xv = x[i]; yv = y[i]; zv = wrap_z(z[i], L); mv = m[i]; hv = h[i];
        if (!(hv > 0.0)) atomicOr(&flags->bad_h, 1);
        else atomicMax(&flags->hmax_bits, (unsigned long long)__double_as_longlong(hv));
    } else {                   // massless dummy far outside any particle load
        xv = 1.0e60; yv = 1.0e60; zv = 0.0; mv = 0.0; hv = 1.0;
    }
    xy[i] = make_double2(xv, yv);
    zm[i] = make_double2(zv, mv);
    hs[i] = hv;
    {   // max h of the tile (dummies count as 0): bounds h_i + h_j in the pair kernels' spline pre-test
        __shared__ double s_max[PAIR_THREADS / 32];
        double hm = (i < n && hv > 0.0) ? hv : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) hm = fmax(hm, __shfl_xor_sync(0xffffffffu, hm, o));
        if ((threadIdx.x & 31) == 0) s_max[threadIdx.x >> 5] = hm;
        __syncthreads();
        if (threadIdx.x == 0) {
            double t = s_max[0];
            for (int wq = 1; wq < PAIR_THREADS / 32; ++wq) t = fmax(t, s_max[wq]);
            tile_hmax[blockIdx.x] = t;
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

// a5: g = -G (A_x, A_y, A_z1 - L A_z2), partial sums added over source chunks in fixed order.
// n_chunks_fast: chunks written by the fast-path kernel that ran (1 for the symmetric kernel);
// n_chunks_general: chunks of the general kernel, which ran instead iff 2 max(h) > L/2.
__global__ void finalize_kernel(const double *__restrict__ part, int n, int n_pad,
                                int n_chunks_fast, int n_chunks_general, double halfL,
                                const DevFlags *__restrict__ flags, double G, double L,
                                double *__restrict__ gx, double *__restrict__ gy,
                                double *__restrict__ gz)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double hmax = __longlong_as_double((long long)flags->hmax_bits);
    const int n_chunks = ((2.0 * hmax > halfL) || flags->bad_h) ? n_chunks_general : n_chunks_fast;
    double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
    for (int c = 0; c < n_chunks; ++c) {
        const double *p = part + (size_t)c * 4 * n_pad + i;
        a0 += p[0];
        a1 += p[(size_t)n_pad];
        a2 += p[2 * (size_t)n_pad];
        a3 += p[3 * (size_t)n_pad];
    }
    gx[i] = -G * a0;
    gy[i] = -G * a1;
    gz[i] = -G * fma(-L, a3, a2);
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

// LANES = 1: one thread per particle.  LANES = 32: one warp per particle (nodes strided over the lanes,
// fixed-order butterfly sum) -- for small n, where one thread per particle leaves most SMs empty and the
// 361-node loop (~120 us) would outlast the pair kernel.
template <int LANES>
__global__ void background_kernel(const double *__restrict__ x, const double *__restrict__ y,
                                  int n, double R, double Lhalf, double G, double rho0,
                                  int infinite, const QuadNode *__restrict__ nodes, int n_nodes,
                                  double *__restrict__ bx, double *__restrict__ by)
{
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    const int i = tid / LANES, lane = tid % LANES;
    if (i >= n) return;                                               // uniform over a warp when LANES == 32
    const double xv = x[i], yv = y[i];
    const double rho = sqrt(fma(xv, xv, yv * yv));
    if (rho0 == 0.0 || rho == 0.0) {
        if (lane == 0) { bx[i] = 0.0; by[i] = 0.0; }
        return;
    }
    double Fh;
    if (infinite) {
        Fh = -2.0 * 3.141592653589793238 * G * rho0 * rho;          // Eq. 10
    } else {
        double acc = background_nodes(rho, R, Lhalf, nodes, n_nodes, lane, LANES);
        if (LANES == 32) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        }
        Fh = 2.0 * G * rho0 * acc;
    }
    if (lane != 0) return;
    const double s = -Fh / rho;      // Eq. 11 subtracts F_h (F_h < 0): outward push
    bx[i] = s * xv;
    by[i] = s * yv;
}

// a7, first half of the KDK step (reading S4):
//   v <- v + (dt/2)[(g + b)/a_n^3 - 2 H_n v];  x <- x + v dt;  z reduced to [0, L).
__global__ void kick1_drift_kernel(double *__restrict__ x, double *__restrict__ y,
                                   double *__restrict__ z, double *__restrict__ vx,
                                   double *__restrict__ vy, double *__restrict__ vz,
                                   const double *__restrict__ gx, const double *__restrict__ gy,
                                   const double *__restrict__ gz, const double *__restrict__ bx,
                                   const double *__restrict__ by, int n, double inv_a3,
                                   double H, double dt, double L)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double hdt = 0.5 * dt;
    double ux = vx[i], uy = vy[i], uz = vz[i];
    ux = ux + hdt * ((gx[i] + bx[i]) * inv_a3 - 2.0 * H * ux);
    uy = uy + hdt * ((gy[i] + by[i]) * inv_a3 - 2.0 * H * uy);
    uz = uz + hdt * (gz[i] * inv_a3 - 2.0 * H * uz);
    vx[i] = ux; vy[i] = uy; vz[i] = uz;
    x[i] = x[i] + ux * dt;
    y[i] = y[i] + uy * dt;
    z[i] = wrap_z(z[i] + uz * dt, L);
}

// a7, second half:  v <- [v + (dt/2)(g' + b')/a_{n+1}^3] / (1 + H_{n+1} dt).
__global__ void kick2_kernel(double *__restrict__ vx, double *__restrict__ vy,
                             double *__restrict__ vz, const double *__restrict__ gx,
                             const double *__restrict__ gy, const double *__restrict__ gz,
                             const double *__restrict__ bx, const double *__restrict__ by, int n,
                             double inv_a3, double H, double dt)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double hdt = 0.5 * dt, den = 1.0 + H * dt;
    vx[i] = (vx[i] + hdt * (gx[i] + bx[i]) * inv_a3) / den;
    vy[i] = (vy[i] + hdt * (gy[i] + by[i]) * inv_a3) / den;
    vz[i] = (vz[i] + hdt * gz[i] * inv_a3) / den;
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
