// pair_fp64_sym.cuh -- all-pairs S^1 x R^2 acceleration in double precision, each UNORDERED
// pair evaluated once (the default fp64 kernel).
//
// The pair law of Eq. 8 is antisymmetric: with r = x_i - x_j the image sums
// S = sum_n w_n and T = sum_n n w_n (pair_fp64.cuh) are the same for (i,j) and (j,i) up to
// T -> -T, r -> -r, and h_i + h_j is symmetric (Eq. 1).  So one evaluation of (S, T) -- the
// ~95 FP64-pipe instructions of the image sum -- serves both particles:
//     target i :  A_i += m_j (S r_x, S r_y, S r_z, T)
//     target j :  A_j -= m_i (S r_x, S r_y, S r_z, T)
// which nearly halves the FP64-pipe work per ordered pair interaction.
//
// Mapping (no cross-lane reduction anywhere): a warp owns 32 targets i (one per lane, in
// registers) and walks a 32-source sub-tile as a ring: at step s lane l meets source
// (l + s) mod 32, whose data it reads from the shared-memory tile and whose accumulator is in
// lane l's registers; after the step the four source accumulators move one lane down
// (8 SHFL), so that after 32 steps every accumulator is back in its home lane and has met all
// 32 targets.  Home accumulators go to a per-warp shared slab, the four slabs of the CTA are
// summed at the end of the tile and leave with one RED.ADD.F64 per value.
//
// Work decomposition: CTA (bi, c) = target block bi x source tiles [c*tpc, (c+1)*tpc) with
// tile >= bi (upper triangle).  In the diagonal tile, warp w takes sub-tiles js > w both ways,
// js == w target-side only (every ordered pair of the 32x32 block once; j == i contributes
// exactly 0), and skips js < w.
//
// Results are accumulated with floating-point atomics, so the summation ORDER (not the set of
// terms) can differ from run to run: results are reproducible to round-off (~1e-16 relative),
// not bit for bit.  STEPS_FLAG_DETERMINISTIC selects pair_fp64_kernel instead.
#pragma once
#include <cuda_runtime.h>

#include "pair_fp64.cuh"

namespace steps {

// 32 ring steps of one warp against one 32-source sub-tile.  SYM: also accumulate on the sources.
template <int NC, bool SYM>
__device__ __forceinline__ void ring_subtile(double xi, double yi, double zi, double hi, double mi,
                                             const double2 *s_xy, const double2 *s_zm,
                                             const double *s_h, int jbase, int lane, int soft_hi,
                                             const PairConsts &k, int ncut_rt,
                                             double &ax, double &ay, double &az1, double &az2,
                                             double &bx, double &by, double &bz1, double &bz2)
{
    bx = by = bz1 = bz2 = 0.0;
#pragma unroll 1
    for (int s = 0; s < 32; ++s) {
        const int jj = jbase + ((lane + s) & 31);
        const double2 a = s_xy[jj], b = s_zm[jj];
        const double hj = s_h[jj];
        const double rx = xi - a.x, ry = yi - a.y;
        const double rz = nearest_image(zi - b.x, k);
        const double rho2 = fma(ry, ry, rx * rx);
        const double q = fma(rz, rz, rho2);
        double S, T;
        image_sum<NC>(rz, q, hi, hj, soft_hi, k, ncut_rt, S, T);
        const double Sj = b.y * S;
        ax  = fma(Sj, rx, ax);
        ay  = fma(Sj, ry, ay);
        az1 = fma(Sj, rz, az1);
        az2 = fma(b.y, T, az2);
        if (SYM) {
            const double Si = mi * S;
            bx  = fma(Si, rx, bx);
            by  = fma(Si, ry, by);
            bz1 = fma(Si, rz, bz1);
            bz2 = fma(mi, T, bz2);
            const int src = (lane + 1) & 31;
            bx  = __shfl_sync(0xffffffffu, bx, src);
            by  = __shfl_sync(0xffffffffu, by, src);
            bz1 = __shfl_sync(0xffffffffu, bz1, src);
            bz2 = __shfl_sync(0xffffffffu, bz2, src);
        }
    }
}

// acc layout: acc[comp * n_pad + particle], comp = 0..3 (A_x, A_y, A_z1, A_z2), zeroed by the host
// before the launch.  grid = (n_tiles, n_chunks_sym).
template <int NC>
__global__ void __launch_bounds__(PAIR_THREADS, 4)
pair_fp64_sym_kernel(const double2 *__restrict__ xy, const double2 *__restrict__ zm,
                     const double *__restrict__ hs, const double *__restrict__ tile_hmax,
                     int n_pad, int n_tiles, int tiles_per_chunk, int ncut_rt, PairConsts k,
                     const DevFlags *__restrict__ flags, double *__restrict__ acc)
{
    const int bi = blockIdx.x;
    const int t0 = max(blockIdx.y * tiles_per_chunk, bi);
    const int t1 = min((blockIdx.y + 1) * tiles_per_chunk, n_tiles);
    if (t0 >= t1) return;
    {
        const double hmax = __longlong_as_double((long long)flags->hmax_bits);
        if ((2.0 * hmax > k.halfL) || flags->bad_h) return;      // general kernel's job
    }
    __shared__ double2 s_xy[PAIR_THREADS];
    __shared__ double2 s_zm[PAIR_THREADS];
    __shared__ double  s_h[PAIR_THREADS];
    __shared__ double  s_b[PAIR_THREADS / 32][4][PAIR_THREADS];   // per-warp source accumulators

    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int i = bi * PAIR_THREADS + threadIdx.x;
    const double2 pi = xy[i], qi = zm[i];
    const double xi = pi.x, yi = pi.y, zi = qi.x, mi = qi.y, hi = hs[i];
    double ax = 0.0, ay = 0.0, az1 = 0.0, az2 = 0.0;

    for (int t = t0; t < t1; ++t) {
        const int j = t * PAIR_THREADS + threadIdx.x;
        __syncthreads();                                   // previous tile's flush has read s_b
        s_xy[threadIdx.x] = xy[j];
        s_zm[threadIdx.x] = zm[j];
        s_h[threadIdx.x]  = hs[j];
        __syncthreads();
        int soft_hi;
        {
            const double b = hi + tile_hmax[t];
            soft_hi = hi32(b * b);
        }
        const bool diag = (t == bi);
#pragma unroll 1
        for (int js = 0; js < PAIR_THREADS / 32; ++js) {
            double bx = 0.0, by = 0.0, bz1 = 0.0, bz2 = 0.0;
            if (!diag || js > w)
                ring_subtile<NC, true>(xi, yi, zi, hi, mi, s_xy, s_zm, s_h, js * 32, lane, soft_hi,
                                       k, ncut_rt, ax, ay, az1, az2, bx, by, bz1, bz2);
            else if (js == w)
                ring_subtile<NC, false>(xi, yi, zi, hi, mi, s_xy, s_zm, s_h, js * 32, lane, soft_hi,
                                        k, ncut_rt, ax, ay, az1, az2, bx, by, bz1, bz2);
            const int jl = js * 32 + lane;
            s_b[w][0][jl] = bx;
            s_b[w][1][jl] = by;
            s_b[w][2][jl] = bz1;
            s_b[w][3][jl] = bz2;
        }
        __syncthreads();
        {
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                double v = s_b[0][c][threadIdx.x];
#pragma unroll
                for (int ww = 1; ww < PAIR_THREADS / 32; ++ww) v += s_b[ww][c][threadIdx.x];
                if (v != 0.0) atomicAdd(acc + (size_t)c * n_pad + j, -v);
            }
        }
    }
    atomicAdd(acc + i, ax);
    atomicAdd(acc + (size_t)n_pad + i, ay);
    atomicAdd(acc + 2 * (size_t)n_pad + i, az1);
    atomicAdd(acc + 3 * (size_t)n_pad + i, az2);
}

}  // namespace steps
