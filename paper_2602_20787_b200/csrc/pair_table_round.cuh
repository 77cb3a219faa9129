// pair_table_round.cuh -- EWALD_TABLE mode under STEPS_FLAG_DETERMINISTIC: the round scheduling of
// pair_fp64_round_kernel (pair_fp64_sym.cuh) with the pair law of pair_table_sym.cuh.
//
// Round r pairs target group b (tiles 2b, 2b+1) with source tile t = (2b + r) mod T; within a round
// every source tile belongs to exactly one group, so the source-side sums are stored with a plain
// read-modify-write, the target-side sums only ever by the group's owner, and the result is
// bit-reproducible.  One launch per round, r = 0 .. min(T/2 + 1, T - 1).  A work item (one group
// against one source tile) is taken by a QUAD of four warps; with the float table in shared memory a
// CTA is persistent (one per SM, four quads) and strides over the round's items, so the 152 KB table
// is staged once per CTA and round (~1 % of a round at N = 1 M).  Quads synchronise on their own
// named barrier.
#pragma once
#include <cuda_runtime.h>

#include "pair_table_mixed_sym.cuh"

namespace steps {

__device__ __forceinline__ void quad_sync(int quad)
{
    asm volatile("bar.sync %0, 128;" ::"r"(quad + 1) : "memory");
}

// Target tile tt against source tile t: 0 = not this CTA's pair (the mirrored item takes it),
// 1 = both ways, 2 = the tile against itself.  Same rule as pair_fp64_round_kernel.
__device__ __forceinline__ int round_mode(int tt, int t, int n_tiles)
{
    const int half = n_tiles / 2, o = (t - tt + n_tiles) % n_tiles;
    return (o == 0) ? 2 : ((o < half || (o == half && tt < t)) ? 1 : 0);
}

// acc_i: [4][n_pad] (row 3 stays 0), acc_j: [3][n_pad], both zeroed by the host before round 0.
// grid = any number of CTAs (items are strided); dynamic shared memory as pair_table_sym_kernel.
template <int INTERP, int TW, bool SMEM_TABLE>
__global__ void __launch_bounds__(TW * 32, SMEM_TABLE ? 1 : 4)
pair_table_round_kernel(const double2 *__restrict__ xy, const double2 *__restrict__ zm,
                        const double *__restrict__ hs, const double *__restrict__ tile_hmax,
                        int n_pad, int n_tiles, int round, PairConsts k, TableConsts tc,
                        const float2 *__restrict__ table_f32, double *__restrict__ acc_i,
                        double *__restrict__ acc_j)
{
    static_assert(SYM_R == 2, "round scheduling is written for two target tiles per group");
    constexpr int QUADS = TW / 4;
    __shared__ SymSrc s_src[QUADS][PAIR_THREADS];
    extern __shared__ double s_dyn[];
    double (*s_b)[3][PAIR_THREADS] = reinterpret_cast<double (*)[3][PAIR_THREADS]>(s_dyn);
    float2 *s_table = reinterpret_cast<float2 *>(s_dyn + TW * 3 * PAIR_THREADS);
    if (SMEM_TABLE) {
        stage_table_halo(s_table, table_f32, tc.nrho, tc.nz, TW * 32);
        __syncthreads();
    }
    GlobalTable gtab{tc.D};
    SharedTableF32 stab{s_table};

    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, wq = w & 3, quad = w >> 2;
    const int tq = wq * 32 + lane;                             // thread index within the quad
    for (int b = blockIdx.x * QUADS + quad; b < n_tiles / SYM_R; b += gridDim.x * QUADS) {
        const int tb = b * SYM_R, t = (tb + round) % n_tiles;
        const int mode[SYM_R] = {round_mode(tb, t, n_tiles), round_mode(tb + 1, t, n_tiles)};
        if (mode[0] == 0 && mode[1] == 0) continue;             // uniform over the quad
        SymTgt ti[SYM_R];
        double a[SYM_R][3];
        int soft_hi[SYM_R];
        const double hm = tile_hmax[t];
#pragma unroll
        for (int r = 0; r < SYM_R; ++r) {
            const int i = (tb + r) * PAIR_THREADS + tq;
            const double2 pi = xy[i], qi = zm[i];
            ti[r].x = pi.x; ti[r].y = pi.y; ti[r].z = qi.x; ti[r].m = qi.y; ti[r].h = hs[i];
            a[r][0] = a[r][1] = a[r][2] = 0.0;
            const double bb = ti[r].h + hm;
            soft_hi[r] = hi32(bb * bb);
        }
        const int j = t * PAIR_THREADS + tq;
        {
            const double2 pj = xy[j], qj = zm[j];
            SymSrc v;
            v.x = pj.x; v.y = pj.y; v.z = qj.x; v.m = qj.y; v.h = hs[j]; v.pad = 0.0;
            s_src[quad][tq] = v;
        }
        quad_sync(quad);
#pragma unroll 1
        for (int js = 0; js < PAIR_THREADS / 32; ++js) {
            double bx = 0.0, by = 0.0, bz = 0.0;
            const SymSrc *sub = s_src[quad] + js * 32;
            if (mode[0] == 1 && mode[1] == 1) {
                if (SMEM_TABLE)
                    ring_subtile_table<INTERP, SYM_R, true>(ti, soft_hi, sub, lane, k, tc, stab, a, bx, by, bz);
                else
                    ring_subtile_table<INTERP, SYM_R, true>(ti, soft_hi, sub, lane, k, tc, gtab, a, bx, by, bz);
            } else {
#pragma unroll
                for (int r = 0; r < SYM_R; ++r) {
                    if (mode[r] == 0) continue;
                    const SymTgt (&t1r)[1] = reinterpret_cast<const SymTgt (&)[1]>(ti[r]);
                    const int (&s1r)[1] = reinterpret_cast<const int (&)[1]>(soft_hi[r]);
                    double (&a1r)[1][3] = reinterpret_cast<double (&)[1][3]>(a[r]);
                    double cx = 0.0, cy = 0.0, cz = 0.0;
                    const bool both = (mode[r] == 1) || (js > wq);
                    if (both || js == wq) {
                        if (SMEM_TABLE) {
                            if (both) ring_subtile_table<INTERP, 1, true>(t1r, s1r, sub, lane, k, tc, stab, a1r, cx, cy, cz);
                            else      ring_subtile_table<INTERP, 1, false>(t1r, s1r, sub, lane, k, tc, stab, a1r, cx, cy, cz);
                        } else {
                            if (both) ring_subtile_table<INTERP, 1, true>(t1r, s1r, sub, lane, k, tc, gtab, a1r, cx, cy, cz);
                            else      ring_subtile_table<INTERP, 1, false>(t1r, s1r, sub, lane, k, tc, gtab, a1r, cx, cy, cz);
                        }
                    }
                    bx += cx; by += cy; bz += cz;
                }
            }
            const int jl = js * 32 + lane;
            s_b[w][0][jl] = bx;
            s_b[w][1][jl] = by;
            s_b[w][2][jl] = bz;
        }
        quad_sync(quad);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            double v = s_b[quad * 4][c][tq];
#pragma unroll
            for (int ww = 1; ww < 4; ++ww) v += s_b[quad * 4 + ww][c][tq];
            double *p = acc_j + (size_t)c * n_pad + j;          // this quad is the tile's only writer this round
            *p = *p - v;
        }
#pragma unroll
        for (int r = 0; r < SYM_R; ++r) {
            if (mode[r] == 0) continue;
            const int i = (tb + r) * PAIR_THREADS + tq;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                double *p = acc_i + (size_t)c * n_pad + i;      // only the group's owner ever writes these
                *p = *p + a[r][c];
            }
        }
        quad_sync(quad);                                        // s_src / s_b are reused by the next item
    }
}

// Mixed precision: float pair terms and interpolation (pair_table_mixed_sym.cuh), double sums.
template <int INTERP>
__global__ void __launch_bounds__(TABLE_MIXED_WARPS * 32, 1)
pair_table_mixed_round_kernel(const float4 *__restrict__ f_hi, const float4 *__restrict__ f_lo,
                              const double *__restrict__ tile_hmax, int n_pad, int n_tiles, int round,
                              MixedConsts k, TableConstsF32 tc, const float2 *__restrict__ table_f32,
                              double *__restrict__ acc_i, double *__restrict__ acc_j)
{
    static_assert(SYM_R == 2, "round scheduling is written for two target tiles per group");
    constexpr int TW = TABLE_MIXED_WARPS, QUADS = TW / 4;
    __shared__ float4 s_hi[QUADS][PAIR_THREADS];
    __shared__ float4 s_lo[QUADS][PAIR_THREADS];
    extern __shared__ float s_dynf[];
    float (*s_b)[3][PAIR_THREADS] = reinterpret_cast<float (*)[3][PAIR_THREADS]>(s_dynf);
    float2 *s_table = reinterpret_cast<float2 *>(s_dynf + TW * 3 * PAIR_THREADS);
    stage_table_halo(s_table, table_f32, tc.nrho, tc.nz, TW * 32);
    __syncthreads();

    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, wq = w & 3, quad = w >> 2;
    const int tq = wq * 32 + lane;
    for (int b = blockIdx.x * QUADS + quad; b < n_tiles / SYM_R; b += gridDim.x * QUADS) {
        const int tb = b * SYM_R, t = (tb + round) % n_tiles;
        const int mode[SYM_R] = {round_mode(tb, t, n_tiles), round_mode(tb + 1, t, n_tiles)};
        if (mode[0] == 0 && mode[1] == 0) continue;
        MixTgt ti[SYM_R];
        double A[SYM_R][3];
        int soft_bits[SYM_R];
        const float hm = (float)tile_hmax[t] * 1.0001f;
#pragma unroll
        for (int r = 0; r < SYM_R; ++r) {
            const int i = (tb + r) * PAIR_THREADS + tq;
            const float4 h4 = f_hi[i], l4 = f_lo[i];
            ti[r].xh = h4.x; ti[r].yh = h4.y; ti[r].zh = h4.z; ti[r].m = h4.w;
            ti[r].xl = l4.x; ti[r].yl = l4.y; ti[r].zl = l4.z; ti[r].h = l4.w;
            ti[r].mL = 0.0f;
            A[r][0] = A[r][1] = A[r][2] = 0.0;
            const float bb = (ti[r].h + hm) * 1.0001f;
            soft_bits[r] = __float_as_int(bb * bb);
        }
        const int j = t * PAIR_THREADS + tq;
        s_hi[quad][tq] = f_hi[j];
        s_lo[quad][tq] = f_lo[j];
        quad_sync(quad);
#pragma unroll 1
        for (int js = 0; js < PAIR_THREADS / 32; ++js) {
            float bx = 0.0f, by = 0.0f, bz = 0.0f;
            const float4 *sh = s_hi[quad] + js * 32, *sl = s_lo[quad] + js * 32;
            if (mode[0] == 1 && mode[1] == 1) {
                float a[SYM_R][3];
                ring_subtile_table_f32<INTERP, SYM_R, true>(ti, soft_bits, sh, sl, lane, k, tc, s_table, a,
                                                            bx, by, bz);
#pragma unroll
                for (int r = 0; r < SYM_R; ++r)
#pragma unroll
                    for (int c = 0; c < 3; ++c) A[r][c] += (double)a[r][c];
            } else {
#pragma unroll
                for (int r = 0; r < SYM_R; ++r) {
                    if (mode[r] == 0) continue;
                    const MixTgt (&t1r)[1] = reinterpret_cast<const MixTgt (&)[1]>(ti[r]);
                    const int (&s1r)[1] = reinterpret_cast<const int (&)[1]>(soft_bits[r]);
                    float a1[1][3] = {{0.0f, 0.0f, 0.0f}};
                    float cx = 0.0f, cy = 0.0f, cz = 0.0f;
                    if (mode[r] == 1 || js > wq)
                        ring_subtile_table_f32<INTERP, 1, true>(t1r, s1r, sh, sl, lane, k, tc, s_table, a1, cx, cy, cz);
                    else if (js == wq)
                        ring_subtile_table_f32<INTERP, 1, false>(t1r, s1r, sh, sl, lane, k, tc, s_table, a1, cx, cy, cz);
#pragma unroll
                    for (int c = 0; c < 3; ++c) A[r][c] += (double)a1[0][c];
                    bx += cx; by += cy; bz += cz;
                }
            }
            const int jl = js * 32 + lane;
            s_b[w][0][jl] = bx;
            s_b[w][1][jl] = by;
            s_b[w][2][jl] = bz;
        }
        quad_sync(quad);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            double v = (double)s_b[quad * 4][c][tq];
#pragma unroll
            for (int ww = 1; ww < 4; ++ww) v += (double)s_b[quad * 4 + ww][c][tq];
            double *p = acc_j + (size_t)c * n_pad + j;
            *p = *p - v;
        }
#pragma unroll
        for (int r = 0; r < SYM_R; ++r) {
            if (mode[r] == 0) continue;
            const int i = (tb + r) * PAIR_THREADS + tq;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                double *p = acc_i + (size_t)c * n_pad + i;
                *p = *p + A[r][c];
            }
        }
        quad_sync(quad);
    }
}

}  // namespace steps
