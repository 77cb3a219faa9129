// pair_fp64.cuh -- all-pairs S^1 x R^2 acceleration, every pair term in double precision.
//
// Computes, for each target i, the four partial sums over a chunk of sources j
//     A_x  = sum_j m_j S_ij r_x,   A_y = sum_j m_j S_ij r_y,
//     A_z1 = sum_j m_j S_ij r_z,   A_z2 = sum_j m_j T_ij,
// where r = x_i - x_j with r_z reduced to the nearest image, and over the image set of
// Eq. 8 (readings G2/S1)
//     S_ij = sum_n w_n,   T_ij = sum_n n w_n,   w_n = F(s_n, h_i + h_j)/s_n,
//     s_n^2 = rho^2 + (r_z - n L)^2,
// F the spline of Eq. 3 (reading G1).  Because sum_n w_n (r_z - n L) =
// r_z S - L T, the acceleration of Eq. 1/4/8 is g = -G (A_x, A_y, A_z1 - L A_z2); that last
// step is done by finalize_kernel (aux_kernels.cuh).
//
// FP64-pipe bound: the design goal is the fewest FP64-pipe instructions per image term.
//   * images +n and -n share B_n = q + n^2 L^2 (q = rho^2 + r_z^2):
//         s_{+-n}^2 = fma(-+2 n L, r_z, B_n)                       3 instr / 2 images
//   * w = (s^2)^(-3/2) from MUFU.RSQ64H (XU pipe, 20-bit seed y0, low word zero so y0^2 is
//     exact) and one third-order step:  e = 1 - s^2 y0^2,  w = y0^3 (1 + 3e/2 + 15e^2/8)
//                                                                    6 instr / image
//   * S += w, T += n (w_+ - w_-)                                     2 instr / image
//   * the spline can only act on the nearest image when 2 max(h) <= L/2 (checked on the
//     device); it is a divergent slow path taken only by warps with a pair inside the support.
// Sources are staged per CTA in shared memory and read as warp-wide broadcasts.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace steps {

constexpr int PAIR_THREADS = 128;   // targets per CTA (one per thread) == sources per tile
constexpr int MAX_NCUT_UNROLLED = 8;
#ifndef STEPS_RT_UNROLL
#define STEPS_RT_UNROLL 2
#endif
constexpr int kRtUnroll = STEPS_RT_UNROLL;      // image-loop unroll of the run-time N_cut fp64 kernels (1/2/3/4 at
                                                // N_cut = 10: 490 / 478 / 480 / 486 ms per evaluation at N = 262144)
constexpr int MAX_NCUT_TABLE = 64;  // run-time N_cut up to here reads its per-image constants from PairConsts

struct WrapConsts {           // what the nearest-image reduction needs (all the general path reads)
    double L;                 // period
    double halfL;
    int L_hi, L_lo, halfL_hi; // integer views of L and L/2 (ALU-pipe wrap test)
};
struct PairConsts : WrapConsts {
    double c2nL[MAX_NCUT_TABLE + 1];      // 2 n L
    double n2L2[MAX_NCUT_TABLE + 1];      // (n L)^2
    double dn[MAX_NCUT_TABLE + 1];        // n
};

struct DevFlags {             // written by pack_kernel, read by the pair kernels
    unsigned long long hmax_bits;   // bit pattern of max_i h_i (positive doubles order as integers)
    int bad_h;                      // some h_i <= 0 or NaN
    int pad;
};

__device__ __forceinline__ double rsqrt_seed(double x)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));   // MUFU.RSQ64H: 20-bit, low word 0
    return y;
}

// (x)^(-3/2) for normal positive x, ~1.5 ulp.  Series remainder 35/16 e^3 < 2^-55 for |e| < 2^-19 (measured:
// |e| <= 1.84e-6 = 2^-19.05 for the RSQ64H seed).
// Operand forms matter on this pipe (measured, profiles/r2_fp64_pipe_microbench.md): an FP64 instruction with THREE
// distinct register sources takes three issue cycles instead of two, so the last step is written c * (1 + e p)
// (DFMA with an immediate addend, then DMUL) rather than fma(c e, p, c).
__device__ __forceinline__ double inv_cube_sqrt(double x)
{
    const double y0 = rsqrt_seed(x);
    const double y2 = y0 * y0;                 // exact (21-bit operands)
    const double e  = fma(-x, y2, 1.0);
    const double c  = y2 * y0;
    const double p  = fma(1.875, e, 1.5);
    const double g  = fma(e, p, 1.0);
    return c * g;
}

// The same with the series cut after the linear term, w = y0^3 (1 + d0 + 3e/2): 5 FP64 instructions.
// Measured on the B200 (4 M arguments per decade range): the RSQ64H seed leaves e in [-1.13e-6, 1.84e-6] with
// mean(e^2) = 3.04e-13, so the dropped 15 e^2/8 is at most 6.3e-12 and 5.7e-13 on average; d0 = 5.7e-13 puts that
// average back, which leaves a zero-mean residual (a uniform deficit would scale the whole far field).
// Used for the far images only, and only under STEPS_FLAG_FAR_ORDER2: see DESIGN.md section 5.
__device__ __forceinline__ double inv_cube_sqrt_o2(double x)
{
    const double y0 = rsqrt_seed(x);
    const double y2 = y0 * y0;
    const double e  = fma(-x, y2, 1.0);
    const double c  = y2 * y0;
    return c * fma(1.5, e, 1.0 + 5.7e-13);
}

template <bool O2>
__device__ __forceinline__ double inv_cube_sqrt_far(double x)
{
    return O2 ? inv_cube_sqrt_o2(x) : inv_cube_sqrt(x);
}

// w = F(s, h)/s of Eq. 3 for s^2 = q < h^2, h = h_i + h_j  (slow path).
__device__ __noinline__ double spline_w(double q, double hh)
{
    const double s   = sqrt(q);
    const double ih  = 1.0 / hh;
    const double u   = s * ih;
    const double ih3 = ih * ih * ih;
    if (u < 0.5)
        return fma(u * u, fma(32.0, u, -38.4), 32.0 / 3.0) * ih3;
    const double u3 = u * u * u;
    double poly = fma(u, fma(u, fma(u, -32.0 / 3.0, 38.4), -48.0), 64.0 / 3.0);
    poly -= 1.0 / (15.0 * u3);
    return poly * ih3;
}

// Integer views of a double: the FP64 pipe is the bottleneck, so sign / magnitude tests that do
// not need a rounded result are done on the ALU pipe (high-word compares of positive doubles
// order like the doubles themselves).
__device__ __forceinline__ int hi32(double v) { return __double2hiint(v); }
__device__ __forceinline__ int lo32(double v) { return __double2loint(v); }

// Pair geometry (a2): r = x_i - x_j with r_z brought to the nearest image.  The decision uses
// the high word only: |r_z| may stay above L/2 by a relative 2^-20, which leaves the image SET
// {d = r_z - nL : |d| < N_cut L} and every formula below unchanged (reading S2).
__device__ __forceinline__ double nearest_image(double rz, const WrapConsts &k)
{
    const int h = hi32(rz);
    const bool wrap = (h & 0x7fffffff) > k.halfL_hi;
    const int sh = wrap ? (k.L_hi | (h & 0x80000000)) : 0;     // copysign(L, rz) or 0
    const int sl = wrap ? k.L_lo : 0;
    return rz - __hiloint2double(sh, sl);
}

// Image sum of one pair (a3/a4): S = sum_n w_n, T = sum_n n w_n over the window of Eq. 8.
// soft_hi: high word of an upper bound of (h_i + h_j)^2 over the source tile; only pairs with
// hi32(q) <= soft_hi can be inside the spline support and take the exact test.
// NC > 0: image loop fully unrolled for N_cut == NC; NC == 0: run-time N_cut.
template <int NC, bool O2 = false>
__device__ __forceinline__ void image_sum(double rz, double q, double hi, double hj, int soft_hi,
                                          const PairConsts &k, int ncut_rt, double &S, double &T)
{
    // nearest image n = 0 (the only one the spline can touch on this path)
    double w0 = inv_cube_sqrt(q);
    if (hi32(q) <= soft_hi) {
        const double hh = hi + hj;
        if (q < hh * hh) w0 = spline_w(q, hh);
    }
    S = w0;
    T = 0.0;
    const bool rz_nonzero = ((hi32(rz) & 0x7fffffff) | lo32(rz)) != 0;
    if (NC > 0) {
#pragma unroll
        for (int n = 1; n < NC; ++n) {
            const double B  = q + k.n2L2[n];
            const double wp = inv_cube_sqrt_far<O2>(fma(-k.c2nL[n], rz, B));   // image +n: d = rz - nL
            const double wm = inv_cube_sqrt_far<O2>(fma(k.c2nL[n], rz, B));    // image -n: d = rz + nL
            S += wp;
            S += wm;
            T = (n == 1) ? (wp - wm) : fma((double)n, wp - wm, T);
        }
        // end image n = sign(rz) N_cut (absent when rz == 0): d = -sign(rz)(N L - |rz|)
        double we = inv_cube_sqrt_far<O2>(fma(-k.c2nL[NC], fabs(rz), q + k.n2L2[NC]));
        we = rz_nonzero ? we : 0.0;
        S += we;
        T = (NC == 1) ? copysign(we, rz) : fma(copysign((double)NC, rz), we, T);

    } else if (ncut_rt <= MAX_NCUT_TABLE) {
        // run-time N_cut: the same arithmetic as the unrolled instances, the per-image constants
        // (uniform across the warp) indexed out of the kernel-parameter bank
#pragma unroll 2
        for (int n = 1; n < ncut_rt; ++n) {
            const double B  = q + k.n2L2[n];
            const double wp = inv_cube_sqrt_far<O2>(fma(-k.c2nL[n], rz, B));
            const double wm = inv_cube_sqrt_far<O2>(fma(k.c2nL[n], rz, B));
            S += wp;
            S += wm;
            T = fma(k.dn[n], wp - wm, T);
        }
        double we = inv_cube_sqrt_far<O2>(fma(-k.c2nL[ncut_rt], fabs(rz), q + k.n2L2[ncut_rt]));
        we = rz_nonzero ? we : 0.0;
        S += we;
        T = fma(copysign(k.dn[ncut_rt], rz), we, T);
    } else {
        for (int n = 1; n < ncut_rt; ++n) {
            const double nL = (double)n * k.L;
            const double B  = fma(nL, nL, q);
            const double t  = 2.0 * nL;
            const double wp = inv_cube_sqrt(fma(-t, rz, B));
            const double wm = inv_cube_sqrt(fma(t, rz, B));
            S += wp;
            S += wm;
            T = fma((double)n, wp - wm, T);
        }
        const double NL = (double)ncut_rt * k.L;
        double we = inv_cube_sqrt(fma(-2.0 * NL, fabs(rz), fma(NL, NL, q)));
        we = rz_nonzero ? we : 0.0;
        S += we;
        T = fma(copysign((double)ncut_rt, rz), we, T);
    }
}

// Image sums of R pairs that share the source (the ring kernels: R targets of a lane), written for |r_z|:
//     S = sum_n w_n (as above),   Ta = sum_n n w_n evaluated at |r_z|  ( = sign(r_z) T ),
// so that the end image always sits at n = +N_cut (an immediate instead of a copysign'd register) and
// sum_n w_n (r_z - n L) = sign(r_z) (S |r_z| - L Ta).  arz = |r_z|, q = rho^2 + r_z^2.
// The spline pre-test of the R pairs is ONE warp-level branch.  NC > 0: unrolled; NC == 0: run-time N_cut with the
// image loop outside the targets (2 R independent rsqrt chains per trip, per-image constants read once).
template <int NC, int R, bool O2>
__device__ __forceinline__ void image_sums(const double (&arz)[R], const double (&q)[R],
                                           const double (&hi)[R], double hj, const int (&soft_hi)[R],
                                           const PairConsts &k, int ncut_rt, double (&S)[R], double (&Ta)[R])
{
    bool any_soft = false;
#pragma unroll
    for (int r = 0; r < R; ++r) {
        S[r] = inv_cube_sqrt(q[r]);                       // nearest image n = 0 (the only one the spline can touch)
        any_soft |= hi32(q[r]) <= soft_hi[r];
    }
    if (any_soft) {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const double hh = hi[r] + hj;
            if (q[r] < hh * hh) S[r] = spline_w(q[r], hh);
        }
    }
    if (NC > 0) {
#pragma unroll
        for (int n = 1; n < NC; ++n) {
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const double B  = q[r] + k.n2L2[n];
                const double wp = inv_cube_sqrt_far<O2>(fma(-k.c2nL[n], arz[r], B));   // image +n: d = |rz| - nL
                const double wm = inv_cube_sqrt_far<O2>(fma(k.c2nL[n], arz[r], B));    // image -n: d = |rz| + nL
                S[r] = __dadd_rn(S[r], wp);          // not contracted with w = c g: that DFMA would have three register sources
                S[r] = __dadd_rn(S[r], wm);
                Ta[r] = (n == 1) ? (wp - wm) : fma((double)n, wp - wm, Ta[r]);
            }
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            // end image n = +N_cut (absent when rz == 0): d = -(N L - |rz|)
            double we = inv_cube_sqrt_far<O2>(fma(-k.c2nL[NC], arz[r], q[r] + k.n2L2[NC]));
            we = ((hi32(arz[r]) & 0x7fffffff) | lo32(arz[r])) != 0 ? we : 0.0;
            S[r] = __dadd_rn(S[r], we);
            Ta[r] = (NC == 1) ? we : fma((double)NC, we, Ta[r]);
        }
    } else if (ncut_rt <= MAX_NCUT_TABLE) {
#pragma unroll
        for (int r = 0; r < R; ++r) Ta[r] = 0.0;
#pragma unroll kRtUnroll
        for (int n = 1; n < ncut_rt; ++n) {
            const double c = k.c2nL[n], b = k.n2L2[n], d = k.dn[n];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const double B  = q[r] + b;
                const double wp = inv_cube_sqrt_far<O2>(fma(-c, arz[r], B));
                const double wm = inv_cube_sqrt_far<O2>(fma(c, arz[r], B));
                S[r] = __dadd_rn(S[r], wp);          // not contracted with w = c g: that DFMA would have three register sources
                S[r] = __dadd_rn(S[r], wm);
                Ta[r] = fma(d, wp - wm, Ta[r]);
            }
        }
        const double ce = k.c2nL[ncut_rt], be = k.n2L2[ncut_rt], de = k.dn[ncut_rt];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            double we = inv_cube_sqrt_far<O2>(fma(-ce, arz[r], q[r] + be));
            we = ((hi32(arz[r]) & 0x7fffffff) | lo32(arz[r])) != 0 ? we : 0.0;
            S[r] = __dadd_rn(S[r], we);
            Ta[r] = fma(de, we, Ta[r]);
        }
    } else {
        // N_cut beyond the tabulated constants: they are formed in the loop
#pragma unroll
        for (int r = 0; r < R; ++r) Ta[r] = 0.0;
        for (int n = 1; n < ncut_rt; ++n) {
            const double nL = (double)n * k.L, t = 2.0 * nL;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const double B  = fma(nL, nL, q[r]);
                const double wp = inv_cube_sqrt(fma(-t, arz[r], B));
                const double wm = inv_cube_sqrt(fma(t, arz[r], B));
                S[r] = __dadd_rn(S[r], wp);          // not contracted with w = c g: that DFMA would have three register sources
                S[r] = __dadd_rn(S[r], wm);
                Ta[r] = fma((double)n, wp - wm, Ta[r]);
            }
        }
        const double NL = (double)ncut_rt * k.L;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            double we = inv_cube_sqrt(fma(-2.0 * NL, arz[r], fma(NL, NL, q[r])));
            we = ((hi32(arz[r]) & 0x7fffffff) | lo32(arz[r])) != 0 ? we : 0.0;
            S[r] = __dadd_rn(S[r], we);
            Ta[r] = fma((double)ncut_rt, we, Ta[r]);
        }
    }
}

// One source j against one target i: adds into (ax, ay, az1, az2).
template <int NC>
__device__ __forceinline__ void pair_term(double xi, double yi, double zi, double hi,
                                          double xj, double yj, double zj, double mj, double hj,
                                          int soft_hi, const PairConsts &k, int ncut_rt,
                                          double &ax, double &ay, double &az1, double &az2)
{
    const double rx = xi - xj, ry = yi - yj;
    const double rz = nearest_image(zi - zj, k);          // zi - zj in (-L, L): both z in [0, L)
    const double rho2 = fma(ry, ry, rx * rx);
    const double q = fma(rz, rz, rho2);
    double S, T;
    image_sum<NC>(rz, q, hi, hj, soft_hi, k, ncut_rt, S, T);
    const double Sm = mj * S;
    ax  = fma(Sm, rx, ax);
    ay  = fma(Sm, ry, ay);
    az1 = fma(Sm, rz, az1);
    az2 = fma(mj, T, az2);
}

// General path (2 max(h) > L/2, reading S7): every image of the window of Eq. 8 is formed directly and sent
// through the spline test, exactly as the equation is written.  S = sum_n w_n, T = sum_n n w_n as in image_sum.
__device__ __forceinline__ void image_sum_general(double rz, double rho2, double hh, const WrapConsts &k,
                                                  int ncut, double &S, double &T)
{
    const double hh2 = hh * hh;
    int nlo = -ncut + 1, nhi = ncut - 1;
    if (rz > 0.0) nhi = ncut;
    if (rz < 0.0) nlo = -ncut;
    S = 0.0;
    T = 0.0;
    for (int n = nlo; n <= nhi; ++n) {
        const double d = rz - (double)n * k.L;
        const double s2 = fma(d, d, rho2);
        const double w = (s2 < hh2) ? spline_w(s2, hh) : inv_cube_sqrt(s2);
        S += w;
        T = fma((double)n, w, T);
    }
}

__device__ __forceinline__ void pair_term_general(double xi, double yi, double zi, double hi,
                                                  double xj, double yj, double zj, double mj,
                                                  double hj, const WrapConsts &k, int ncut,
                                                  double &ax, double &ay, double &az1, double &az2)
{
    const double rx = xi - xj, ry = yi - yj;
    const double rz = nearest_image(zi - zj, k);
    const double rho2 = fma(ry, ry, rx * rx);
    double S, T;
    image_sum_general(rz, rho2, hi + hj, k, ncut, S, T);
    const double Sm = mj * S;
    ax  = fma(Sm, rx, ax);
    ay  = fma(Sm, ry, ay);
    az1 = fma(Sm, rz, az1);
    az2 = fma(mj, T, az2);
}

// True when the fast kernels' precondition fails: some far image can fall inside a spline support
// (2 max h > L/2), or some h <= 0 (outputs then unspecified, reported through steps_cyl_check).
__device__ __forceinline__ bool need_general_path(const DevFlags *flags, double halfL)
{
    const double hmax = __longlong_as_double((long long)flags->hmax_bits);
    return (2.0 * hmax > halfL) || flags->bad_h;
}

// Packed source layout (written by prestep_kernel, padded to a multiple of PAIR_THREADS with
// massless far-away dummies): xy[j] = {x, y}, zm[j] = {z in [0,L), m}, hs[j] = h.
//
// Ordered pairs, the literal form of Eq. 1 (STEPS_FLAG_ORDERED_PAIRS): grid = (n_tiles, n_chunks); CTA (bx, by)
// handles targets [bx*128, bx*128+128) against source tiles [by*tiles_per_chunk, (by+1)*tiles_per_chunk).
// part layout: part[((chunk*4 + comp) * n_pad) + i].
struct OrdSmem { double2 xy[PAIR_THREADS]; double2 zm[PAIR_THREADS]; double h[PAIR_THREADS]; };

template <int NC, bool GENERAL, class KC>
__device__ __forceinline__ void ordered_body(const double2 *__restrict__ xy, const double2 *__restrict__ zm,
                                             const double *__restrict__ hs, const double *__restrict__ tile_hmax,
                                             int n_pad, int n_tiles, int tiles_per_chunk, int ncut_rt,
                                             const KC &k, double *__restrict__ part, OrdSmem &sm)
{
    const int i = blockIdx.x * PAIR_THREADS + threadIdx.x;      // < n_pad always
    const double2 pi = xy[i], qi = zm[i];
    const double xi = pi.x, yi = pi.y, zi = qi.x, hi = hs[i];
    double ax = 0.0, ay = 0.0, az1 = 0.0, az2 = 0.0;

    const int t0 = blockIdx.y * tiles_per_chunk;
    const int t1 = min(t0 + tiles_per_chunk, n_tiles);
    for (int t = t0; t < t1; ++t) {
        const int j = t * PAIR_THREADS + threadIdx.x;
        __syncthreads();
        sm.xy[threadIdx.x] = xy[j];
        sm.zm[threadIdx.x] = zm[j];
        sm.h[threadIdx.x]  = hs[j];
        __syncthreads();
        int soft_hi;
        {
            const double b = hi + tile_hmax[t];          // >= h_i + h_j for every j of the tile
            soft_hi = hi32(b * b);
        }
#pragma unroll 1
        for (int jj = 0; jj < PAIR_THREADS; ++jj) {
            const double2 a = sm.xy[jj], b = sm.zm[jj];
            const double hj = sm.h[jj];
            if constexpr (GENERAL)
                pair_term_general(xi, yi, zi, hi, a.x, a.y, b.x, b.y, hj, k, ncut_rt, ax, ay, az1, az2);
            else
                pair_term<NC>(xi, yi, zi, hi, a.x, a.y, b.x, b.y, hj, soft_hi, k, ncut_rt, ax, ay, az1, az2);
        }
    }
    double *p = part + (size_t)blockIdx.y * 4 * n_pad + i;
    p[0] = ax;
    p[(size_t)n_pad] = ay;
    p[2 * (size_t)n_pad] = az1;
    p[3 * (size_t)n_pad] = az2;
}

// The general path of the ordered kernels (fp64 and mixed), out of line so that it costs the fast path nothing.
__device__ __noinline__ void ordered_body_general(const double2 *xy, const double2 *zm, const double *hs,
                                                  const double *tile_hmax, int n_pad, int n_tiles,
                                                  int tiles_per_chunk, int ncut_rt, WrapConsts k,
                                                  double *part, OrdSmem &sm)
{
    ordered_body<0, true>(xy, zm, hs, tile_hmax, n_pad, n_tiles, tiles_per_chunk, ncut_rt, k, part, sm);
}

template <int NC>
__global__ void __launch_bounds__(PAIR_THREADS)
pair_fp64_kernel(const double2 *__restrict__ xy, const double2 *__restrict__ zm,
                 const double *__restrict__ hs, const double *__restrict__ tile_hmax, int n_pad,
                 int n_tiles, int tiles_per_chunk, int ncut_rt, PairConsts k,
                 const DevFlags *__restrict__ flags, double *__restrict__ part)
{
    __shared__ OrdSmem sm;
    if (need_general_path(flags, k.halfL)) {
        ordered_body_general(xy, zm, hs, tile_hmax, n_pad, n_tiles, tiles_per_chunk, ncut_rt, k, part, sm);
        return;
    }
    ordered_body<NC, false>(xy, zm, hs, tile_hmax, n_pad, n_tiles, tiles_per_chunk, ncut_rt, k, part, sm);
}

}  // namespace steps
