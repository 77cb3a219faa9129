// pair_mixed_sym.cuh -- mixed precision (STEPS_PREC_MIXED), each UNORDERED pair evaluated once:
// the float analogue of pair_fp64_sym.cuh (same ring exchange, same CTA decomposition, same
// atomics into acc[4][n_pad]).
//
// Precision contract of the mode: every pair term (separation, image sum of Eq. 8, spline of
// Eq. 3) is evaluated in float, with the cancellation-safe hi/lo separations of pair_mixed.cuh;
// the contributions of one 32-source ring (32 pair terms per particle) are summed in float and
// each such partial sum is then added in DOUBLE -- across rings, tiles and CTAs the accumulation
// is fp64.  (A float sum of 32 terms adds ~2^-24 sqrt(32) relative error, the size of one pair
// term's own rounding.)  This keeps F2F conversions and DADDs out of the per-pair loop, which is
// bound by the XU pipe (one MUFU.RSQ per image) and by instruction issue.
#pragma once
#include <cuda_runtime.h>

#include "pair_fp64_sym.cuh"
#include "pair_mixed.cuh"

namespace steps {

struct MixTgt { float xh, yh, zh, xl, yl, zl, h, m, mL; };      // mL = -L m

// S = sum_n w_n, T = sum_n n w_n in float (same image window and pairing as image_sum<NC>).
template <int NC>
__device__ __forceinline__ void image_sum_f32(float rz, float q, float hi, float hj, int soft_bits,
                                              const MixedConsts &k, int ncut_rt, float &S, float &T)
{
    float w0 = inv_cube_sqrt_f32(q);
    if (__float_as_int(q) <= soft_bits) {
        const float hh = hi + hj;
        if (q < hh * hh) w0 = spline_w_f32(q, hh);
    }
    S = w0;
    T = 0.0f;
    if (NC > 0) {
#pragma unroll
        for (int n = 1; n < NC; ++n) {
            const float B  = q + k.n2L2[n];
            const float wp = inv_cube_sqrt_f32(fmaf(-k.c2nL[n], rz, B));
            const float wm = inv_cube_sqrt_f32(fmaf(k.c2nL[n], rz, B));
            S += wp;
            S += wm;
            T = (n == 1) ? (wp - wm) : fmaf((float)n, wp - wm, T);
        }
        float we = inv_cube_sqrt_f32(fmaf(-k.c2nL[NC], fabsf(rz), q + k.n2L2[NC]));
        we = (rz == 0.0f) ? 0.0f : we;
        S += we;
        T = (NC == 1) ? copysignf(we, rz) : fmaf(copysignf((float)NC, rz), we, T);
    } else {
        const float L = k.Lh;
        for (int n = 1; n < ncut_rt; ++n) {
            const float nL = (float)n * L;
            const float B  = fmaf(nL, nL, q);
            const float t  = 2.0f * nL;
            const float wp = inv_cube_sqrt_f32(fmaf(-t, rz, B));
            const float wm = inv_cube_sqrt_f32(fmaf(t, rz, B));
            S += wp;
            S += wm;
            T = fmaf((float)n, wp - wm, T);
        }
        const float NL = (float)ncut_rt * L;
        float we = inv_cube_sqrt_f32(fmaf(-2.0f * NL, fabsf(rz), fmaf(NL, NL, q)));
        we = (rz == 0.0f) ? 0.0f : we;
        S += we;
        T = fmaf(copysignf((float)ncut_rt, rz), we, T);
    }
}

// 32 ring steps; a[r][0..3] and (bx, by, bz) are FLOAT partial sums of this ring only.
template <int NC, int R, bool SYM>
__device__ __forceinline__ void ring_subtile_f32(const MixTgt (&ti)[R], const int (&soft_bits)[R],
                                                 const float4 *s_hi, const float4 *s_lo, int lane,
                                                 const MixedConsts &k, int ncut_rt,
                                                 float (&a)[R][4], float &bx, float &by, float &bz)
{
    bx = by = bz = 0.0f;
#pragma unroll
    for (int r = 0; r < R; ++r) a[r][0] = a[r][1] = a[r][2] = a[r][3] = 0.0f;
#pragma unroll 1
    for (int s = 0; s < 32; ++s) {
        const int jj = (lane + s) & 31;
        const float4 jh = s_hi[jj], jl = s_lo[jj];          // {x_hi,y_hi,z_hi,m}, {x_lo,y_lo,z_lo,h}
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const float rx = (ti[r].xh - jh.x) + (ti[r].xl - jl.x);
            const float ry = (ti[r].yh - jh.y) + (ti[r].yl - jl.y);
            float rzh = ti[r].zh - jh.z, rzl = ti[r].zl - jl.z;
            const float sgn = (fabsf(rzh) > k.halfL) ? copysignf(1.0f, rzh) : 0.0f;
            rzh = fmaf(-sgn, k.Lh, rzh);
            rzl = fmaf(-sgn, k.Ll, rzl);
            const float rz = rzh + rzl;
            const float rho2 = fmaf(ry, ry, rx * rx);
            const float q = fmaf(rz, rz, rho2);
            float S, T;
            image_sum_f32<NC>(rz, q, ti[r].h, jl.w, soft_bits[r], k, ncut_rt, S, T);
            const float Sj = jh.w * S;
            a[r][0] = fmaf(Sj, rx, a[r][0]);
            a[r][1] = fmaf(Sj, ry, a[r][1]);
            a[r][2] = fmaf(Sj, rz, a[r][2]);
            a[r][3] = fmaf(jh.w, T, a[r][3]);
            if (SYM) {
                const float Si = ti[r].m * S;
                bx = fmaf(Si, rx, bx);
                by = fmaf(Si, ry, by);
                bz = fmaf(Si, rz, bz);
                bz = fmaf(ti[r].mL, T, bz);
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

// Same grid / decomposition / acc layout as pair_fp64_sym_kernel.
template <int NC>
__global__ void __launch_bounds__(PAIR_THREADS, 4)
pair_mixed_sym_kernel(const float4 *__restrict__ f_hi, const float4 *__restrict__ f_lo,
                      const double *__restrict__ tile_hmax, int n_pad, int n_tiles,
                      int tiles_per_chunk, int ncut_rt, MixedConsts k, double halfL,
                      const DevFlags *__restrict__ flags, double *__restrict__ acc)
{
    const int tb = blockIdx.x * SYM_R;
    const int t0 = max(blockIdx.y * tiles_per_chunk, tb);
    const int t1 = min((blockIdx.y + 1) * tiles_per_chunk, n_tiles);
    if (t0 >= t1) return;
    {
        const double hmax = __longlong_as_double((long long)flags->hmax_bits);
        if ((2.0 * hmax > halfL) || flags->bad_h) return;        // fp64 general kernel's job
    }
    __shared__ float4 s_hi[PAIR_THREADS];
    __shared__ float4 s_lo[PAIR_THREADS];
    __shared__ float  s_b[PAIR_THREADS / 32][3][PAIR_THREADS];

    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    MixTgt ti[SYM_R];
    double A[SYM_R][4];
#pragma unroll
    for (int r = 0; r < SYM_R; ++r) {
        const int i = (tb + r) * PAIR_THREADS + threadIdx.x;
        const float4 h4 = f_hi[i], l4 = f_lo[i];
        ti[r].xh = h4.x; ti[r].yh = h4.y; ti[r].zh = h4.z; ti[r].m = h4.w;
        ti[r].xl = l4.x; ti[r].yl = l4.y; ti[r].zl = l4.z; ti[r].h = l4.w;
        ti[r].mL = -k.Lh * h4.w;
        A[r][0] = A[r][1] = A[r][2] = A[r][3] = 0.0;
    }

    for (int t = t0; t < t1; ++t) {
        const int j = t * PAIR_THREADS + threadIdx.x;
        __syncthreads();
        s_hi[threadIdx.x] = f_hi[j];
        s_lo[threadIdx.x] = f_lo[j];
        __syncthreads();
        int soft_bits[SYM_R];
        {
            const float hm = (float)tile_hmax[t] * 1.0001f;   // rounded up: bound must not shrink
#pragma unroll
            for (int r = 0; r < SYM_R; ++r) {
                const float b = (ti[r].h + hm) * 1.0001f;
                soft_bits[r] = __float_as_int(b * b);
            }
        }
#pragma unroll 1
        for (int js = 0; js < PAIR_THREADS / 32; ++js) {
            float bx = 0.0f, by = 0.0f, bz = 0.0f;
            const float4 *sh = s_hi + js * 32, *sl = s_lo + js * 32;
            if (t >= tb + SYM_R) {
                float a[SYM_R][4];
                ring_subtile_f32<NC, SYM_R, true>(ti, soft_bits, sh, sl, lane, k, ncut_rt, a, bx, by, bz);
#pragma unroll
                for (int r = 0; r < SYM_R; ++r)
#pragma unroll
                    for (int c = 0; c < 4; ++c) A[r][c] += (double)a[r][c];
            } else {
#pragma unroll
                for (int r = 0; r < SYM_R; ++r) {
                    if (tb + r > t) continue;
                    const MixTgt (&t1r)[1] = reinterpret_cast<const MixTgt (&)[1]>(ti[r]);
                    const int (&s1r)[1] = reinterpret_cast<const int (&)[1]>(soft_bits[r]);
                    float a1[1][4] = {{0.0f, 0.0f, 0.0f, 0.0f}};
                    float cx = 0.0f, cy = 0.0f, cz = 0.0f;
                    if (tb + r < t || js > w)
                        ring_subtile_f32<NC, 1, true>(t1r, s1r, sh, sl, lane, k, ncut_rt, a1, cx, cy, cz);
                    else if (js == w)
                        ring_subtile_f32<NC, 1, false>(t1r, s1r, sh, sl, lane, k, ncut_rt, a1, cx, cy, cz);
#pragma unroll
                    for (int c = 0; c < 4; ++c) A[r][c] += (double)a1[0][c];
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
            double v = (double)s_b[0][c][threadIdx.x];
#pragma unroll
            for (int ww = 1; ww < PAIR_THREADS / 32; ++ww) v += (double)s_b[ww][c][threadIdx.x];
            if (v != 0.0) atomicAdd(acc + (size_t)c * n_pad + j, -v);
        }
    }
#pragma unroll
    for (int r = 0; r < SYM_R; ++r) {
        const int i = (tb + r) * PAIR_THREADS + threadIdx.x;
#pragma unroll
        for (int c = 0; c < 4; ++c) atomicAdd(acc + (size_t)c * n_pad + i, A[r][c]);
    }
}

}  // namespace steps
