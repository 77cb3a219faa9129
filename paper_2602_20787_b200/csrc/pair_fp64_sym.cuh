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
// Mapping (no cross-lane reduction anywhere): a lane holds SYM_R = 2 targets in registers (one from
// each of the CTA's two target tiles), and its warp walks a 32-source sub-tile as a ring: at step
// s lane l meets source (l + s) mod 32, whose record it reads from the shared-memory tile and
// whose three accumulators (sum m_i S r_x, sum m_i S r_y, sum m_i (S r_z - L T)) are in lane l's
// registers; after the step they move one lane down (6 SHFL), so that after 32 steps every
// accumulator is back in its home lane having met all 2 x 32 targets of the warp.  Home
// accumulators go to a per-warp shared slab; the four slabs of the CTA are summed at the end of the
// tile and leave with one RED.ADD.F64 per value.
//
// Work decomposition: CTA (b, c) = target tiles 2b, 2b+1 x source tiles [c*tpc, (c+1)*tpc) from 2b
// on (upper triangle).  In one of its own tiles, target tile tt meets source tile t only if
// t >= tt; for t == tt warp w takes sub-tiles js > w both ways, js == w target-side only (every
// ordered pair of the 32 x 32 block once; j == i contributes exactly 0), and skips js < w.
//
// Results are accumulated with floating-point atomics, so the summation ORDER (not the set of
// terms) can differ from run to run: results are reproducible to round-off (~1e-16 relative),
// not bit for bit.  STEPS_FLAG_DETERMINISTIC selects pair_fp64_round_kernel (end of this file).
//
// If 2 max(h) > L/2 (a far image can be softened, reading S7) the same CTA runs the general pair law instead --
// same ring, same decomposition, every image through the spline test -- decided on the device from the flag
// block prestep_kernel wrote.
#pragma once
#include <cuda_runtime.h>

#include "pair_fp64.cuh"

namespace steps {

#ifndef STEPS_SYM_UNROLL
#define STEPS_SYM_UNROLL 2
#endif
// ring-loop unroll of every ring pass.  Measured at N = 1 048 576, N_cut = 5 (pair kernel, ms per evaluation):
// 1 / 2 / 4 -> 3679.7 / 3640.4 / 3657.4.  (Unrolling ONLY the two-target main pass and leaving the single-target
// passes of the diagonal tiles rolled measured 3700.0: the gain is in how ptxas schedules the whole kernel.)
constexpr int kSymUnroll = STEPS_SYM_UNROLL;
#ifndef STEPS_SYM_MINBLOCKS
#define STEPS_SYM_MINBLOCKS 4      // resident CTAs per SM the register allocation aims at
#endif

// One staged source: 48 bytes, read with two LDS.128 and one LDS.64 off a single address.
struct __align__(16) SymSrc { double x, y, z, m, h, pad; };

// Targets a lane keeps in registers (R = SYM_R of them, one per target tile of the CTA).
struct SymTgt { double x, y, z, h, m; };

// 32 ring steps of one warp against one 32-source sub-tile.  R targets per lane meet the same
// source in a step, so the source record is loaded and its accumulators are shuffled once per R
// pairs.  SYM: also accumulate on the sources.  Per pair, with (S, T) the image sums,
//     P = (S r_x, S r_y, S r_z - L T)          -- the pair's acceleration per unit G m, sign included
//     target i:  a   += m_j P        source j (rotating accumulators):  b += m_i P   (subtracted at the flush)
// so the three products P are formed once and serve both particles, and only three values travel.
// (FP64 instructions with three distinct register sources -- the six multiply-adds above -- take three issue
// cycles, all others two: profiles/r2_fp64_pipe_microbench.md.)
template <int NC, int R, bool SYM, bool O2, bool GENERAL = false, class KC = PairConsts>
__device__ __forceinline__ void ring_subtile(const SymTgt (&ti)[R], const int (&soft_hi)[R],
                                             const SymSrc *s_src, int lane, const KC &k,
                                             int ncut_rt, double (&a)[R][3], double &bx,
                                             double &by, double &bz)
{
    bx = by = bz = 0.0;
#pragma unroll kSymUnroll
    for (int s = 0; s < 32; ++s) {
        const SymSrc *sj = s_src + ((lane + s) & 31);
        const double2 pa = *reinterpret_cast<const double2 *>(&sj->x);
        const double2 pb = *reinterpret_cast<const double2 *>(&sj->z);
        const double hj = sj->h;
        double rx[R], ry[R], rz[R], U[R], S[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            rx[r] = ti[r].x - pa.x;
            ry[r] = ti[r].y - pa.y;
            rz[r] = nearest_image(ti[r].z - pb.x, k);
        }
        if constexpr (GENERAL) {
            // general path (2 max h > L/2): the literal image loop of Eq. 8 with every image through the spline
            // test; (S, T) serve both particles of the pair exactly as on the fast path
#pragma unroll
            for (int r = 0; r < R; ++r) {
                double T;
                image_sum_general(rz[r], fma(ry[r], ry[r], rx[r] * rx[r]), ti[r].h + hj, k, ncut_rt, S[r], T);
                U[r] = fma(-k.L, T, S[r] * rz[r]);
            }
        } else {
            double arz[R], q[R], hi[R], Ta[R];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                arz[r] = fabs(rz[r]);
                q[r] = fma(rz[r], rz[r], fma(ry[r], ry[r], rx[r] * rx[r]));
                hi[r] = ti[r].h;
            }
            image_sums<NC, R, O2>(arz, q, hi, hj, soft_hi, k, ncut_rt, S, Ta);
#pragma unroll
            for (int r = 0; r < R; ++r) {
                // sign(r_z) (S |r_z| - L Ta): the sign goes back on with one integer op on the high word
                const double Ua = fma(-k.L, Ta[r], S[r] * arz[r]);
                U[r] = __hiloint2double(hi32(Ua) ^ (hi32(rz[r]) & 0x80000000), lo32(Ua));
            }
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const double Px = S[r] * rx[r], Py = S[r] * ry[r];
            a[r][0] = fma(pb.y, Px, a[r][0]);
            a[r][1] = fma(pb.y, Py, a[r][1]);
            a[r][2] = fma(pb.y, U[r], a[r][2]);
            if (SYM) {
                bx = fma(ti[r].m, Px, bx);
                by = fma(ti[r].m, Py, by);
                bz = fma(ti[r].m, U[r], bz);
            }
        }
        if (SYM) {
            const int src = (lane + 1) & 31;
            bx = __shfl_sync(0xffffffffu, bx, src);
            by = __shfl_sync(0xffffffffu, by, src);
            bz = __shfl_sync(0xffffffffu, bz, src);
        }
    }
}

#ifndef STEPS_SYM_R
#define STEPS_SYM_R 2
#endif
constexpr int SYM_R = STEPS_SYM_R;     // target tiles per CTA (n_tiles is kept a multiple of SYM_R by the host)

// Shared memory of a symmetric CTA: one staged source tile and the per-warp source accumulators.
struct SymSmem {
    SymSrc src[PAIR_THREADS];
    double b[PAIR_THREADS / 32][3][PAIR_THREADS];
};

// acc layout: acc[comp * n_pad + particle], comp = 0..3 (A_x, A_y, A_z1, A_z2), zeroed by prestep_kernel
// before the launch; these kernels add the combined z sum S r_z - L T to A_z1 and leave A_z2 zero.
// grid = (n_tiles / SYM_R, chunks).  CTA (bi, c): target tiles SYM_R*bi + r (lane holds particle
// tid of each), source tiles [c*tpc, (c+1)*tpc) from SYM_R*bi on.
// GENERAL: the same decomposition with the general pair law (ring_subtile<..., GENERAL>).
// SLAB (STEPS_FLAG_DETERMINISTIC up to N = 131 072): instead of atomics every sum goes to a slot with exactly one
// writer -- source-side sums of CTA row bx to slab bx (each (row, source tile) is handled by one CTA), target-side
// sums of CTA (bx, c, z) to slab gridDim.x + c * gridDim.z + z -- and poststep_kernel adds the slots that were
// written (a rule on indices, no zeroing) in fixed order: bit-reproducible at the speed of the atomic kernel.
template <int NC, bool O2, bool GENERAL, int TR, bool SLAB, class KC>
__device__ __forceinline__ void sym_body(const double2 *__restrict__ xy, const double2 *__restrict__ zm,
                                         const double *__restrict__ hs, const double *__restrict__ tile_hmax,
                                         int n_pad, int n_tiles, int tiles_per_chunk, int ncut_rt,
                                         const KC &k, double *__restrict__ acc, SymSmem &sm)
{
    const int tb = blockIdx.x * TR;                       // first target tile of this CTA
    const int t0 = max(blockIdx.y * tiles_per_chunk, tb);
    const int t1 = min((blockIdx.y + 1) * tiles_per_chunk, n_tiles);
    if (t0 >= t1) return;
    SymSrc *s_src = sm.src;
    double (*s_b)[3][PAIR_THREADS] = sm.b;
    double *slab_src = acc, *slab_tgt = acc;
    if (SLAB) {
        slab_src = acc + (size_t)blockIdx.x * 3 * n_pad;
        slab_tgt = acc + ((size_t)gridDim.x + (size_t)blockIdx.y * gridDim.z + blockIdx.z) * 3 * n_pad;
    }

    // gridDim.z == 4 (small N: fewer tile pairs than the GPU has schedulers): CTA z takes source sub-tile z only
    const bool split = gridDim.z == PAIR_THREADS / 32;
    const int js0 = split ? blockIdx.z : 0, js1 = split ? blockIdx.z + 1 : PAIR_THREADS / 32;
    const bool mine = (int)threadIdx.x >= js0 * 32 && (int)threadIdx.x < js1 * 32;   // sources this CTA takes
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    SymTgt ti[TR];
    double a[TR][3];
#pragma unroll
    for (int r = 0; r < TR; ++r) {
        const int i = (tb + r) * PAIR_THREADS + threadIdx.x;
        const double2 pi = xy[i], qi = zm[i];
        ti[r].x = pi.x; ti[r].y = pi.y; ti[r].z = qi.x; ti[r].m = qi.y; ti[r].h = hs[i];
        a[r][0] = a[r][1] = a[r][2] = 0.0;
    }

    for (int t = t0; t < t1; ++t) {
        const int j = t * PAIR_THREADS + threadIdx.x;
        __syncthreads();                                   // previous tile's flush has read s_b
        {
            const double2 pj = xy[j], qj = zm[j];
            SymSrc v;
            v.x = pj.x; v.y = pj.y; v.z = qj.x; v.m = qj.y; v.h = hs[j]; v.pad = 0.0;
            s_src[threadIdx.x] = v;
        }
        __syncthreads();
        int soft_hi[TR];
        {
            const double hm = tile_hmax[t];
#pragma unroll
            for (int r = 0; r < TR; ++r) {
                const double b = ti[r].h + hm;
                soft_hi[r] = hi32(b * b);
            }
        }
#pragma unroll 1
        for (int js = js0; js < js1; ++js) {
            double bx = 0.0, by = 0.0, bz = 0.0;
            const SymSrc *sub = s_src + js * 32;
            if (t >= tb + TR) {
                // off-diagonal tile: every target of the CTA meets every source, both ways
                ring_subtile<NC, TR, true, O2, GENERAL, KC>(ti, soft_hi, sub, lane, k, ncut_rt, a, bx, by, bz);
            } else {
                // one of the CTA's own tiles: target tile tb + r meets source tile t only if
                // t >= tb + r; in its own tile (t == tb + r) warp w takes sub-tiles js > w both
                // ways, js == w target-side only, and leaves js < w to the warp that owns them.
#pragma unroll
                for (int r = 0; r < TR; ++r) {
                    if (tb + r > t) continue;
                    const SymTgt (&t1r)[1] = reinterpret_cast<const SymTgt (&)[1]>(ti[r]);
                    const int (&s1r)[1] = reinterpret_cast<const int (&)[1]>(soft_hi[r]);
                    double (&a1r)[1][3] = reinterpret_cast<double (&)[1][3]>(a[r]);
                    double cx = 0.0, cy = 0.0, cz = 0.0;
                    if (tb + r < t || js > w)
                        ring_subtile<NC, 1, true, O2, GENERAL, KC>(t1r, s1r, sub, lane, k, ncut_rt, a1r, cx, cy, cz);
                    else if (js == w)
                        ring_subtile<NC, 1, false, O2, GENERAL, KC>(t1r, s1r, sub, lane, k, ncut_rt, a1r, cx, cy, cz);
                    bx += cx; by += cy; bz += cz;
                }
            }
            const int jl = js * 32 + lane;
            s_b[w][0][jl] = bx;
            s_b[w][1][jl] = by;
            s_b[w][2][jl] = bz;
        }
        __syncthreads();
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            double v = s_b[0][c][threadIdx.x];
#pragma unroll
            for (int ww = 1; ww < PAIR_THREADS / 32; ++ww) v += s_b[ww][c][threadIdx.x];
            if (SLAB) {
                if (mine) slab_src[(size_t)c * n_pad + j] = -v;
            } else {
                if (mine && v != 0.0) atomicAdd(acc + (size_t)c * n_pad + j, -v);
            }
        }
    }
#pragma unroll
    for (int r = 0; r < TR; ++r) {
        const int i = (tb + r) * PAIR_THREADS + threadIdx.x;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            if (SLAB) slab_tgt[(size_t)c * n_pad + i] = a[r][c];
            else atomicAdd(acc + (size_t)c * n_pad + i, a[r][c]);
        }
    }
}

// The general path of the symmetric kernels (fp64 and mixed), out of line: it costs the fast path no registers.
template <int TR, bool SLAB = false>
__device__ __noinline__ void sym_body_general(const double2 *xy, const double2 *zm, const double *hs,
                                              const double *tile_hmax, int n_pad, int n_tiles,
                                              int tiles_per_chunk, int ncut_rt, WrapConsts k,
                                              double *acc, SymSmem &sm)
{
    sym_body<0, false, true, TR, SLAB>(xy, zm, hs, tile_hmax, n_pad, n_tiles, tiles_per_chunk, ncut_rt, k, acc, sm);
}

// TR = target tiles per CTA: SYM_R = 2 in general; 1 in the small-N split mode (gridDim.z = 4), where the kernel
// time is one CTA's critical path -- a CTA of the diagonal then walks one single-target ring pass instead of two.
template <int NC, bool O2, int TR = SYM_R, bool SLAB = false>
__global__ void __launch_bounds__(PAIR_THREADS, STEPS_SYM_MINBLOCKS)
pair_fp64_sym_kernel(const double2 *__restrict__ xy, const double2 *__restrict__ zm,
                     const double *__restrict__ hs, const double *__restrict__ tile_hmax,
                     int n_pad, int n_tiles, int tiles_per_chunk, int ncut_rt, PairConsts k,
                     const DevFlags *__restrict__ flags, double *__restrict__ acc)
{
    __shared__ SymSmem sm;
    if (need_general_path(flags, k.halfL)) {          // decided on the device: no host synchronisation
        sym_body_general<TR, SLAB>(xy, zm, hs, tile_hmax, n_pad, n_tiles, tiles_per_chunk, ncut_rt, k, acc, sm);
        return;
    }
    sym_body<NC, O2, false, TR, SLAB>(xy, zm, hs, tile_hmax, n_pad, n_tiles, tiles_per_chunk, ncut_rt, k, acc, sm);
}

// ---------------------------------------------------------------------------------------------
// Deterministic variant (STEPS_FLAG_DETERMINISTIC): the same unordered-pair evaluation, scheduled in
// ROUNDS so that no two CTAs ever update the same accumulator in one launch, and plain
// read-modify-writes replace the atomics.  With T tiles (T even) and CTA b owning target tiles 2b and
// 2b+1, round r gives CTA b the source tile t = (2b + r) mod T: distinct CTAs get distinct source
// tiles, so the source-side sums acc_j[.][tile t] have one writer per round, and the target-side sums
// acc_i[.][tiles 2b, 2b+1] only ever have their owner.  A tile pair (tt, t) with cyclic offset
// o = (t - tt) mod T is taken when 0 < o < T/2, or o == T/2 and tt < t, or o == 0 (the tile against
// itself, sub-tile rules as above); the other half of the offsets is the same pair seen from t.
// Rounds r = 0 .. min(T/2 + 1, T - 1) are launched one after the other on the stream, so every
// accumulator receives its contributions in a fixed order: bit-reproducible results at ~97 % of the
// atomic kernel's speed (one tile of work per CTA per launch; T/2 + 2 launches per evaluation).
// acc_i: gridDim.y slabs of [4][n_pad], acc_j: [3][n_pad], all zeroed by the host before round 0.
template <int NC, bool SPLIT, bool GENERAL, class KC>
__device__ __forceinline__ void round_body(const double2 *__restrict__ xy, const double2 *__restrict__ zm,
                                           const double *__restrict__ hs, const double *__restrict__ tile_hmax,
                                           int n_pad, int n_tiles, int round, int ncut_rt, const KC &k,
                                           double *__restrict__ acc_i, double *__restrict__ acc_j, SymSmem &sm)
{
    static_assert(SYM_R == 2, "round scheduling is written for two target tiles per CTA");
    const int tb = blockIdx.x * SYM_R;
    const int t = (tb + round) % n_tiles;
    int mode[SYM_R];                                      // 0 skip, 1 both ways, 2 the tile against itself
    {
        const int half = n_tiles / 2;
#pragma unroll
        for (int r = 0; r < SYM_R; ++r) {
            const int tt = tb + r, o = (t - tt + n_tiles) % n_tiles;
            mode[r] = (o == 0) ? 2 : ((o < half || (o == half && tt < t)) ? 1 : 0);
        }
    }
    if (mode[0] == 0 && mode[1] == 0) return;
    SymSrc *s_src = sm.src;
    double (*s_b)[3][PAIR_THREADS] = sm.b;

    // SPLIT (gridDim.y == 4; small N: a round has fewer items than the GPU has schedulers): CTA y takes source
    // sub-tile y only and adds its target-side sums into its own slab y of acc_i
    const int js0 = SPLIT ? blockIdx.y : 0, js1 = SPLIT ? blockIdx.y + 1 : PAIR_THREADS / 32;
    if (SPLIT) acc_i += (size_t)blockIdx.y * 4 * n_pad;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    SymTgt ti[SYM_R];
    double a[SYM_R][3];
    int soft_hi[SYM_R];
    const double hm = tile_hmax[t];
#pragma unroll
    for (int r = 0; r < SYM_R; ++r) {
        const int i = (tb + r) * PAIR_THREADS + threadIdx.x;
        const double2 pi = xy[i], qi = zm[i];
        ti[r].x = pi.x; ti[r].y = pi.y; ti[r].z = qi.x; ti[r].m = qi.y; ti[r].h = hs[i];
        a[r][0] = a[r][1] = a[r][2] = 0.0;
        const double b = ti[r].h + hm;
        soft_hi[r] = hi32(b * b);
    }
    const int j = t * PAIR_THREADS + threadIdx.x;
    {
        const double2 pj = xy[j], qj = zm[j];
        SymSrc v;
        v.x = pj.x; v.y = pj.y; v.z = qj.x; v.m = qj.y; v.h = hs[j]; v.pad = 0.0;
        s_src[threadIdx.x] = v;
    }
    __syncthreads();
#pragma unroll 1
    for (int js = js0; js < js1; ++js) {
        double bx = 0.0, by = 0.0, bz = 0.0;
        const SymSrc *sub = s_src + js * 32;
        if (mode[0] == 1 && mode[1] == 1) {
            ring_subtile<NC, SYM_R, true, false, GENERAL, KC>(ti, soft_hi, sub, lane, k, ncut_rt, a, bx, by, bz);
        } else {
#pragma unroll
            for (int r = 0; r < SYM_R; ++r) {
                if (mode[r] == 0) continue;
                const SymTgt (&t1r)[1] = reinterpret_cast<const SymTgt (&)[1]>(ti[r]);
                const int (&s1r)[1] = reinterpret_cast<const int (&)[1]>(soft_hi[r]);
                double (&a1r)[1][3] = reinterpret_cast<double (&)[1][3]>(a[r]);
                double cx = 0.0, cy = 0.0, cz = 0.0;
                if (mode[r] == 1 || js > w)
                    ring_subtile<NC, 1, true, false, GENERAL, KC>(t1r, s1r, sub, lane, k, ncut_rt, a1r, cx, cy, cz);
                else if (js == w)
                    ring_subtile<NC, 1, false, false, GENERAL, KC>(t1r, s1r, sub, lane, k, ncut_rt, a1r, cx, cy, cz);
                bx += cx; by += cy; bz += cz;
            }
        }
        const int jl = js * 32 + lane;
        s_b[w][0][jl] = bx;
        s_b[w][1][jl] = by;
        s_b[w][2][jl] = bz;
    }
    __syncthreads();
    const bool mine = !SPLIT || (int)(threadIdx.x >> 5) == js0;                      // sources this CTA took
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        double v = s_b[0][c][threadIdx.x];
#pragma unroll
        for (int ww = 1; ww < PAIR_THREADS / 32; ++ww) v += s_b[ww][c][threadIdx.x];
        double *p = acc_j + (size_t)c * n_pad + j;            // this CTA is the tile's only writer this round
        if (mine) *p = *p - v;
    }
#pragma unroll
    for (int r = 0; r < SYM_R; ++r) {
        if (mode[r] == 0) continue;
        const int i = (tb + r) * PAIR_THREADS + threadIdx.x;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            double *p = acc_i + (size_t)c * n_pad + i;        // only the owner CTA ever writes these
            *p = *p + a[r][c];
        }
    }
}

// The general path of the round-scheduled kernels (fp64 and mixed), out of line; bit-reproducible like the fast one.
template <bool SPLIT>
__device__ __noinline__ void round_body_general(const double2 *xy, const double2 *zm, const double *hs,
                                                const double *tile_hmax, int n_pad, int n_tiles, int round,
                                                int ncut_rt, WrapConsts k, double *acc_i, double *acc_j,
                                                SymSmem &sm)
{
    round_body<0, SPLIT, true>(xy, zm, hs, tile_hmax, n_pad, n_tiles, round, ncut_rt, k, acc_i, acc_j, sm);
}

template <int NC, bool SPLIT>
__global__ void __launch_bounds__(PAIR_THREADS, STEPS_SYM_MINBLOCKS)
pair_fp64_round_kernel(const double2 *__restrict__ xy, const double2 *__restrict__ zm,
                       const double *__restrict__ hs, const double *__restrict__ tile_hmax,
                       int n_pad, int n_tiles, int round, int ncut_rt, PairConsts k,
                       const DevFlags *__restrict__ flags, double *__restrict__ acc_i,
                       double *__restrict__ acc_j)
{
    __shared__ SymSmem sm;
    if (need_general_path(flags, k.halfL)) {
        round_body_general<SPLIT>(xy, zm, hs, tile_hmax, n_pad, n_tiles, round, ncut_rt, k, acc_i, acc_j, sm);
        return;
    }
    round_body<NC, SPLIT, false>(xy, zm, hs, tile_hmax, n_pad, n_tiles, round, ncut_rt, k, acc_i, acc_j, sm);
}

}  // namespace steps
