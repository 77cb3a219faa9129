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
    } else if (ncut_rt <= MAX_NCUT_TABLE) {
        // run-time N_cut: per-image constants indexed out of the kernel-parameter bank
#pragma unroll 2
        for (int n = 1; n < ncut_rt; ++n) {
            const float B  = q + k.n2L2[n];
            const float wp = inv_cube_sqrt_f32(fmaf(-k.c2nL[n], rz, B));
            const float wm = inv_cube_sqrt_f32(fmaf(k.c2nL[n], rz, B));
            S += wp;
            S += wm;
            T = fmaf(k.dn[n], wp - wm, T);
        }
        float we = inv_cube_sqrt_f32(fmaf(-k.c2nL[ncut_rt], fabsf(rz), q + k.n2L2[ncut_rt]));
        we = (rz == 0.0f) ? 0.0f : we;
        S += we;
        T = fmaf(copysignf(k.dn[ncut_rt], rz), we, T);
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

// ---------------------------------------------------------------------------------------------
// Packed path: sm_100 has two-wide FP32 instructions (PTX add/sub/mul/fma .f32x2 -> SASS FADD2 /
// FMUL2 / FFMA2, scalar operands broadcast for free).  The kernel is bound by instruction issue, and
// the two targets a lane holds go through identical arithmetic against the same source, so they are
// processed as the two halves of one packed value: half the FP32 instructions per pair.  MUFU.RSQ
// (one per image per target), the compares and the sign / mask bit operations stay scalar.
#ifndef STEPS_MIXED_UNROLL
#define STEPS_MIXED_UNROLL 1
#endif
#ifndef STEPS_MIXED_MINBLOCKS
#define STEPS_MIXED_MINBLOCKS 4
#endif
constexpr int kMixedUnroll = STEPS_MIXED_UNROLL;
typedef unsigned long long u64;
__device__ __forceinline__ u64 pk(float2 a) { return *reinterpret_cast<u64 *>(&a); }
__device__ __forceinline__ float2 upk(u64 a) { return *reinterpret_cast<float2 *>(&a); }
__device__ __forceinline__ float2 bc(float s) { return make_float2(s, s); }
__device__ __forceinline__ float2 add2(float2 a, float2 b)
{
    u64 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(pk(a)), "l"(pk(b)));
    return upk(d);
}
__device__ __forceinline__ float2 sub2(float2 a, float2 b)
{
    u64 d;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(pk(a)), "l"(pk(b)));
    return upk(d);
}
__device__ __forceinline__ float2 mul2(float2 a, float2 b)
{
    u64 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(pk(a)), "l"(pk(b)));
    return upk(d);
}
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c)
{
    u64 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(pk(a)), "l"(pk(b)), "l"(pk(c)));
    return upk(d);
}
__device__ __forceinline__ float2 rsqrt2(float2 x) { return make_float2(rsqrt_f32(x.x), rsqrt_f32(x.y)); }
__device__ __forceinline__ float2 cube2(float2 y) { return mul2(mul2(y, y), y); }

struct MixTgt2 { float2 xh, yh, zh, xl, yl, zl, h, m, mL; };       // .x: target tile r = 0, .y: r = 1

// 32 ring steps, both targets of the lane at once, symmetric (source side accumulated too).
// a[c] (c = 0..3: A_x, A_y, A_z1, A_z2) and bx, by, bz are FLOAT partial sums of this ring, the two
// halves belonging to the two targets; the caller adds the halves of b.
// SIMPLE (decided per warp and source sub-tile from bounding boxes, pass_is_simple below): every pair of the pass
// (a) has the same nearest-image shift zshift in {0, +L, -L}, (b) lies outside every spline support, and (c) is
// far apart compared with the size of the source sub-tile and with the coordinates' magnitude.  Then positions are
// taken relative to the sub-tile's centre O: the sources' offsets (x_hi - O) + x_lo were stored as single floats
// when the tile was staged (s_rel; error 2^-24 of the sub-tile's size), the two targets' offsets are formed once per
// pass, and a separation is ONE packed subtraction -- 3 packed operations of geometry instead of 13, one LDS.128
// instead of two, no spline pre-test.  What is lost is the targets' lo part relative to their distance from O
// (2^-24 d): an error common to all sources of the pass, which the sum tolerates (measured: parity unchanged),
// unlike independent per-source roundings of 2^-24 |x| (measured: 10x the error at r ~ 2000).
// Possible because the packed arrays are in Morton order (order_kernels.cuh).
template <int NC, bool SIMPLE = false>
__device__ __forceinline__ void ring_subtile_f32x2(const MixTgt2 &ti, const int (&soft_bits)[2],
                                                   const float4 *s_hi, const float4 *s_lo, int lane,
                                                   const MixedConsts &k, int ncut_rt, float2 (&a)[4],
                                                   float2 &bx, float2 &by, float2 &bz,
                                                   const float4 *s_rel = nullptr, float ox = 0.0f, float oy = 0.0f,
                                                   float oz = 0.0f, float zshift = 0.0f)
{
    float2 Tx = bc(0.0f), Ty = bc(0.0f), Tz = bc(0.0f);
    if constexpr (SIMPLE) {
        Tx = add2(sub2(ti.xh, bc(ox)), ti.xl);
        Ty = add2(sub2(ti.yh, bc(oy)), ti.yl);
        Tz = add2(sub2(sub2(ti.zh, bc(oz)), bc(zshift)), ti.zl);
    }
    bx = by = bz = bc(0.0f);
#pragma unroll
    for (int c = 0; c < 4; ++c) a[c] = bc(0.0f);
    const float invL = 1.0f / k.Lh, magic = 12582912.0f;          // 1.5 * 2^23: round-to-nearest-integer
#pragma unroll kMixedUnroll
    for (int s = 0; s < 32; ++s) {
        const int jj = (lane + s) & 31;
        float2 rx, ry, rz;
        float hj = 0.0f, jm;
        if constexpr (SIMPLE) {
            const float4 jr = s_rel[jj];                     // {x, y, z relative to the sub-tile's centre, m}
            jm = jr.w;
            rx = sub2(Tx, bc(jr.x));
            ry = sub2(Ty, bc(jr.y));
            rz = sub2(Tz, bc(jr.z));
        } else {
            const float4 jh = s_hi[jj], jl = s_lo[jj];       // {x_hi,y_hi,z_hi,m}, {x_lo,y_lo,z_lo,h}
            hj = jl.w;
            jm = jh.w;
            rx = add2(sub2(ti.xh, bc(jh.x)), sub2(ti.xl, bc(jl.x)));
            ry = add2(sub2(ti.yh, bc(jh.y)), sub2(ti.yl, bc(jl.y)));
            float2 rzh = sub2(ti.zh, bc(jh.z)), rzl = sub2(ti.zl, bc(jl.z));
            // nearest image: k = rint(rz / L) by the magic-number trick (|rz| < L, so k in {-1, 0, 1});
            // a tie at |rz| = L/2 may go either way (the image set is symmetric then)
            const float2 kk = sub2(fma2(rzh, bc(invL), bc(magic)), bc(magic));
            rzh = fma2(kk, bc(-k.Lh), rzh);
            rzl = fma2(kk, bc(-k.Ll), rzl);
            rz = add2(rzh, rzl);
        }
        const float2 rho2 = fma2(ry, ry, mul2(rx, rx));
        const float2 q = fma2(rz, rz, rho2);
        float2 w0 = cube2(rsqrt2(q));
        if constexpr (!SIMPLE) {
            if (__float_as_int(q.x) <= soft_bits[0] || __float_as_int(q.y) <= soft_bits[1]) {
                const float h0 = ti.h.x + hj, h1 = ti.h.y + hj;
                if (q.x < h0 * h0) w0.x = spline_w_f32(q.x, h0);
                if (q.y < h1 * h1) w0.y = spline_w_f32(q.y, h1);
            }
        }
        float2 S = w0, T = bc(0.0f);
        const int n_img = (NC > 0) ? NC : ncut_rt;
        if (NC > 0) {
#pragma unroll
            for (int n = 1; n < NC; ++n) {
                const float2 B  = add2(q, bc(k.n2L2[n]));
                const float2 wp = cube2(rsqrt2(fma2(bc(-k.c2nL[n]), rz, B)));
                const float2 wm = cube2(rsqrt2(fma2(bc(k.c2nL[n]), rz, B)));
                S = add2(add2(S, wp), wm);
                T = (n == 1) ? sub2(wp, wm) : fma2(bc((float)n), sub2(wp, wm), T);
            }
        } else if (ncut_rt <= MAX_NCUT_TABLE) {
#pragma unroll kRtUnrollMixed
            for (int n = 1; n < ncut_rt; ++n) {
                const float2 B  = add2(q, bc(k.n2L2[n]));
                const float2 wp = cube2(rsqrt2(fma2(bc(-k.c2nL[n]), rz, B)));
                const float2 wm = cube2(rsqrt2(fma2(bc(k.c2nL[n]), rz, B)));
                S = add2(add2(S, wp), wm);
                T = fma2(bc(k.dn[n]), sub2(wp, wm), T);
            }
        } else {
            for (int n = 1; n < ncut_rt; ++n) {
                const float nL = (float)n * k.Lh;
                const float2 B  = fma2(bc(nL), bc(nL), q);
                const float2 wp = cube2(rsqrt2(fma2(bc(-2.0f * nL), rz, B)));
                const float2 wm = cube2(rsqrt2(fma2(bc(2.0f * nL), rz, B)));
                S = add2(add2(S, wp), wm);
                T = fma2(bc((float)n), sub2(wp, wm), T);
            }
        }
        {   // end image n = sign(rz) N_cut, absent when rz == 0
            const bool tab = NC > 0 || n_img <= MAX_NCUT_TABLE;         // constants from MixedConsts
            const float NL = (float)n_img * k.Lh;
            const float2 arz = make_float2(fabsf(rz.x), fabsf(rz.y));
            const float2 Be = tab ? add2(q, bc(k.n2L2[tab ? n_img : 0])) : fma2(bc(NL), bc(NL), q);
            float2 we = cube2(rsqrt2(fma2(bc(tab ? -k.c2nL[tab ? n_img : 0] : -2.0f * NL), arz, Be)));
            we.x = (rz.x == 0.0f) ? 0.0f : we.x;
            we.y = (rz.y == 0.0f) ? 0.0f : we.y;
            S = add2(S, we);
            const float2 ns = make_float2(copysignf((float)n_img, rz.x), copysignf((float)n_img, rz.y));
            T = fma2(ns, we, T);
        }
        const float2 Sj = mul2(bc(jm), S);
        a[0] = fma2(Sj, rx, a[0]);
        a[1] = fma2(Sj, ry, a[1]);
        a[2] = fma2(Sj, rz, a[2]);
        a[3] = fma2(bc(jm), T, a[3]);
        const float2 Si = mul2(ti.m, S);
        bx = fma2(Si, rx, bx);
        by = fma2(Si, ry, by);
        bz = fma2(Si, rz, bz);
        bz = fma2(ti.mL, T, bz);
        const int src = (lane + 1) & 31;
        bx = upk(__shfl_sync(0xffffffffu, pk(bx), src));
        by = upk(__shfl_sync(0xffffffffu, pk(by), src));
        bz = upk(__shfl_sync(0xffffffffu, pk(bz), src));
    }
}

// Bounding box (of the float hi parts) of a group of particles, with their largest softening and largest |x|, |y|.
struct MixBox { float xlo, xhi, ylo, yhi, zlo, zhi, hmax, cmax; };

__device__ __forceinline__ MixBox box_of(float x, float y, float z, float h)
{
    MixBox b;
    b.xlo = b.xhi = x; b.ylo = b.yhi = y; b.zlo = b.zhi = z; b.hmax = h;
    b.cmax = fmaxf(fabsf(x), fabsf(y));
    return b;
}
__device__ __forceinline__ MixBox box_join(const MixBox &a, const MixBox &b)
{
    MixBox c;
    c.xlo = fminf(a.xlo, b.xlo); c.xhi = fmaxf(a.xhi, b.xhi);
    c.ylo = fminf(a.ylo, b.ylo); c.yhi = fmaxf(a.yhi, b.yhi);
    c.zlo = fminf(a.zlo, b.zlo); c.zhi = fmaxf(a.zhi, b.zhi);
    c.hmax = fmaxf(a.hmax, b.hmax); c.cmax = fmaxf(a.cmax, b.cmax);
    return c;
}
__device__ __forceinline__ MixBox box_warp(MixBox b)            // union over the lanes of the warp
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        MixBox c;
        c.xlo = __shfl_xor_sync(0xffffffffu, b.xlo, o); c.xhi = __shfl_xor_sync(0xffffffffu, b.xhi, o);
        c.ylo = __shfl_xor_sync(0xffffffffu, b.ylo, o); c.yhi = __shfl_xor_sync(0xffffffffu, b.yhi, o);
        c.zlo = __shfl_xor_sync(0xffffffffu, b.zlo, o); c.zhi = __shfl_xor_sync(0xffffffffu, b.zhi, o);
        c.hmax = __shfl_xor_sync(0xffffffffu, b.hmax, o); c.cmax = __shfl_xor_sync(0xffffffffu, b.cmax, o);
        b = box_join(b, c);
    }
    return b;
}

// Can every pair (target in t, source in s) take the SIMPLE form of ring_subtile_f32x2?  (a) one nearest-image
// shift for all of them, (b) box distance d beyond every spline support, (c) d >= half the source box's largest
// extent (the stored offsets from its centre are then good to 2^-23 d) and d >= c / 8 with c the largest
// coordinate magnitude (x, y of both boxes; z < L) -- thresholds in MixedConsts, set by the host.  Margins cover
// the lo parts the boxes do not see.
__device__ __forceinline__ bool pass_is_simple(const MixBox &t, const MixBox &s, const MixedConsts &k, float &zshift)
{
    const float eps = 1.0e-5f * k.Lh;
    float dlo = t.zlo - s.zhi - eps, dhi = t.zhi - s.zlo + eps;          // range of the raw r_z = z_i - z_j
    if (dlo > -k.halfL && dhi < k.halfL) zshift = 0.0f;
    else if (dlo > k.halfL) zshift = k.Lh;
    else if (dhi < -k.halfL) zshift = -k.Lh;
    else return false;
    dlo -= zshift;
    dhi -= zshift;
    const float gz = fmaxf(0.0f, fmaxf(dlo, -dhi));
    const float gx = fmaxf(0.0f, fmaxf(t.xlo - s.xhi, s.xlo - t.xhi));
    const float gy = fmaxf(0.0f, fmaxf(t.ylo - s.yhi, s.ylo - t.yhi));
    const float d2 = fmaf(gx, gx, fmaf(gy, gy, gz * gz));
    const float c = fmaxf(fmaxf(t.cmax, s.cmax), k.Lh);
    const float hh = t.hmax + s.hmax;
    const float ext = fmaxf(fmaxf(s.xhi - s.xlo, s.yhi - s.ylo), s.zhi - s.zlo);
    return d2 > 1.01f * hh * hh && k.simple_ratio2 * d2 >= 1.01f * c * c && d2 >= k.simple_ext2 * ext * ext;   // false for NaN / padding
}

// Same grid / decomposition / acc layout as pair_fp64_sym_kernel.
template <int NC>
__global__ void __launch_bounds__(PAIR_THREADS, STEPS_MIXED_MINBLOCKS)
pair_mixed_sym_kernel(const float4 *__restrict__ f_hi, const float4 *__restrict__ f_lo,
                      const double2 *__restrict__ xy, const double2 *__restrict__ zm,
                      const double *__restrict__ hs,
                      const double *__restrict__ tile_hmax, int n_pad, int n_tiles,
                      int tiles_per_chunk, int ncut_rt, MixedConsts k, PairConsts kd,
                      const DevFlags *__restrict__ flags, double *__restrict__ acc,
                      unsigned long long *__restrict__ pass_stats)
{
    __shared__ SymSmem sm;
    if (need_general_path(flags, kd.halfL)) {         // the fp64 general path (xy, zm, hs are only read here)
        sym_body_general<SYM_R>(xy, zm, hs, tile_hmax, n_pad, n_tiles, tiles_per_chunk, ncut_rt, kd, acc, sm);
        return;
    }
    const int tb = blockIdx.x * SYM_R;
    const int t0 = max(blockIdx.y * tiles_per_chunk, tb);
    const int t1 = min((blockIdx.y + 1) * tiles_per_chunk, n_tiles);
    if (t0 >= t1) return;
    float4 *s_hi = reinterpret_cast<float4 *>(sm.src), *s_lo = s_hi + PAIR_THREADS, *s_rel = s_lo + PAIR_THREADS;
    float (*s_b)[3][PAIR_THREADS] = reinterpret_cast<float (*)[3][PAIR_THREADS]>(sm.b);

    // gridDim.z == 4 (small N): CTA z takes source sub-tile z only (see pair_fp64_sym_kernel)
    const bool split = gridDim.z == PAIR_THREADS / 32;
    const int js0 = split ? blockIdx.z : 0, js1 = split ? blockIdx.z + 1 : PAIR_THREADS / 32;
    const bool mine = (int)threadIdx.x >= js0 * 32 && (int)threadIdx.x < js1 * 32;
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
    static_assert(SYM_R == 2, "the packed path holds exactly two targets per lane");
    MixTgt2 ti2;
    ti2.xh = make_float2(ti[0].xh, ti[1].xh); ti2.yh = make_float2(ti[0].yh, ti[1].yh);
    ti2.zh = make_float2(ti[0].zh, ti[1].zh); ti2.xl = make_float2(ti[0].xl, ti[1].xl);
    ti2.yl = make_float2(ti[0].yl, ti[1].yl); ti2.zl = make_float2(ti[0].zl, ti[1].zl);
    ti2.h = make_float2(ti[0].h, ti[1].h);    ti2.m = make_float2(ti[0].m, ti[1].m);
    ti2.mL = make_float2(ti[0].mL, ti[1].mL);
    // bounding box of this warp's 64 targets, and (per staged tile) of each 32-source sub-tile
    const MixBox tbox = box_warp(box_join(box_of(ti[0].xh, ti[0].yh, ti[0].zh, ti[0].h),
                                          box_of(ti[1].xh, ti[1].yh, ti[1].zh, ti[1].h)));
    __shared__ MixBox s_box[PAIR_THREADS / 32];
    unsigned n_simple = 0, n_pass = 0;                 // two-way ring passes of this warp: SIMPLE / all

    for (int t = t0; t < t1; ++t) {
        const int j = t * PAIR_THREADS + threadIdx.x;
        __syncthreads();
        {
            const float4 vh = f_hi[j], vl = f_lo[j];
            s_hi[threadIdx.x] = vh;
            s_lo[threadIdx.x] = vl;
            const MixBox sb = box_warp(box_of(vh.x, vh.y, vh.z, vl.w));
            if (lane == 0) s_box[w] = sb;
            // offsets from the sub-tile's centre as single floats (SIMPLE passes)
            const float ox = 0.5f * (sb.xlo + sb.xhi), oy = 0.5f * (sb.ylo + sb.yhi), oz = 0.5f * (sb.zlo + sb.zhi);
            s_rel[threadIdx.x] = make_float4((vh.x - ox) + vl.x, (vh.y - oy) + vl.y, (vh.z - oz) + vl.z, vh.w);
        }
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
        for (int js = js0; js < js1; ++js) {
            float bx = 0.0f, by = 0.0f, bz = 0.0f;
            const float4 *sh = s_hi + js * 32, *sl = s_lo + js * 32;
            if (t >= tb + SYM_R) {
                float2 a2[4], b2x, b2y, b2z;
                float zshift;
                n_pass += 1;
                const MixBox sb = s_box[js];
                if (pass_is_simple(tbox, sb, k, zshift)) {              // warp-uniform
                    n_simple += 1;
                    ring_subtile_f32x2<NC, true>(ti2, soft_bits, sh, sl, lane, k, ncut_rt, a2, b2x, b2y, b2z,
                                                 s_rel + js * 32, 0.5f * (sb.xlo + sb.xhi), 0.5f * (sb.ylo + sb.yhi),
                                                 0.5f * (sb.zlo + sb.zhi), zshift);
                } else {
                    ring_subtile_f32x2<NC, false>(ti2, soft_bits, sh, sl, lane, k, ncut_rt, a2, b2x, b2y, b2z);
                }
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    A[0][c] += (double)a2[c].x;
                    A[1][c] += (double)a2[c].y;
                }
                bx = b2x.x + b2x.y;
                by = b2y.x + b2y.y;
                bz = b2z.x + b2z.y;
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
            if (mine && v != 0.0) atomicAdd(acc + (size_t)c * n_pad + j, -v);
        }
    }
#pragma unroll
    for (int r = 0; r < SYM_R; ++r) {
        const int i = (tb + r) * PAIR_THREADS + threadIdx.x;
#pragma unroll
        for (int c = 0; c < 4; ++c) atomicAdd(acc + (size_t)c * n_pad + i, A[r][c]);
    }
    if (lane == 0 && n_pass != 0) {                    // cumulative statistics (steps_cyl_pass_stats)
        atomicAdd(pass_stats, (unsigned long long)n_simple);
        atomicAdd(pass_stats + 1, (unsigned long long)n_pass);
    }
}

// Deterministic variant in rounds: the scheduling of pair_fp64_round_kernel (pair_fp64_sym.cuh) with the
// float pair arithmetic of this file.  acc_i: [4][n_pad], acc_j: [3][n_pad], zeroed before round 0.
template <int NC, bool SPLIT>
__global__ void __launch_bounds__(PAIR_THREADS, STEPS_MIXED_MINBLOCKS)
pair_mixed_round_kernel(const float4 *__restrict__ f_hi, const float4 *__restrict__ f_lo,
                        const double2 *__restrict__ xy, const double2 *__restrict__ zm,
                        const double *__restrict__ hs,
                        const double *__restrict__ tile_hmax, int n_pad, int n_tiles, int round,
                        int ncut_rt, MixedConsts k, PairConsts kd, const DevFlags *__restrict__ flags,
                        double *__restrict__ acc_i, double *__restrict__ acc_j)
{
    static_assert(SYM_R == 2, "round scheduling is written for two target tiles per CTA");
    __shared__ SymSmem sm;
    if (need_general_path(flags, kd.halfL)) {         // the fp64 general path, same round scheduling
        round_body_general<SPLIT>(xy, zm, hs, tile_hmax, n_pad, n_tiles, round, ncut_rt, kd, acc_i, acc_j, sm);
        return;
    }
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
    float4 *s_hi = reinterpret_cast<float4 *>(sm.src), *s_lo = s_hi + PAIR_THREADS;
    float (*s_b)[3][PAIR_THREADS] = reinterpret_cast<float (*)[3][PAIR_THREADS]>(sm.b);
    // SPLIT (gridDim.y == 4): one source sub-tile per CTA, own acc_i slab (see pair_fp64_round_kernel)
    const int js0 = SPLIT ? blockIdx.y : 0, js1 = SPLIT ? blockIdx.y + 1 : PAIR_THREADS / 32;
    if (SPLIT) acc_i += (size_t)blockIdx.y * 4 * n_pad;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    MixTgt ti[SYM_R];
    double A[SYM_R][4];
    int soft_bits[SYM_R];
    const float hm = (float)tile_hmax[t] * 1.0001f;
#pragma unroll
    for (int r = 0; r < SYM_R; ++r) {
        const int i = (tb + r) * PAIR_THREADS + threadIdx.x;
        const float4 h4 = f_hi[i], l4 = f_lo[i];
        ti[r].xh = h4.x; ti[r].yh = h4.y; ti[r].zh = h4.z; ti[r].m = h4.w;
        ti[r].xl = l4.x; ti[r].yl = l4.y; ti[r].zl = l4.z; ti[r].h = l4.w;
        ti[r].mL = -k.Lh * h4.w;
        A[r][0] = A[r][1] = A[r][2] = A[r][3] = 0.0;
        const float b = (ti[r].h + hm) * 1.0001f;
        soft_bits[r] = __float_as_int(b * b);
    }
    MixTgt2 ti2;
    ti2.xh = make_float2(ti[0].xh, ti[1].xh); ti2.yh = make_float2(ti[0].yh, ti[1].yh);
    ti2.zh = make_float2(ti[0].zh, ti[1].zh); ti2.xl = make_float2(ti[0].xl, ti[1].xl);
    ti2.yl = make_float2(ti[0].yl, ti[1].yl); ti2.zl = make_float2(ti[0].zl, ti[1].zl);
    ti2.h = make_float2(ti[0].h, ti[1].h);    ti2.m = make_float2(ti[0].m, ti[1].m);
    ti2.mL = make_float2(ti[0].mL, ti[1].mL);
    const int j = t * PAIR_THREADS + threadIdx.x;
    s_hi[threadIdx.x] = f_hi[j];
    s_lo[threadIdx.x] = f_lo[j];
    __syncthreads();
#pragma unroll 1
    for (int js = js0; js < js1; ++js) {
        float bx = 0.0f, by = 0.0f, bz = 0.0f;
        const float4 *sh = s_hi + js * 32, *sl = s_lo + js * 32;
        if (mode[0] == 1 && mode[1] == 1) {
            float2 a2[4], b2x, b2y, b2z;
            ring_subtile_f32x2<NC>(ti2, soft_bits, sh, sl, lane, k, ncut_rt, a2, b2x, b2y, b2z);
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                A[0][c] += (double)a2[c].x;
                A[1][c] += (double)a2[c].y;
            }
            bx = b2x.x + b2x.y;
            by = b2y.x + b2y.y;
            bz = b2z.x + b2z.y;
        } else {
#pragma unroll
            for (int r = 0; r < SYM_R; ++r) {
                if (mode[r] == 0) continue;
                const MixTgt (&t1r)[1] = reinterpret_cast<const MixTgt (&)[1]>(ti[r]);
                const int (&s1r)[1] = reinterpret_cast<const int (&)[1]>(soft_bits[r]);
                float a1[1][4] = {{0.0f, 0.0f, 0.0f, 0.0f}};
                float cx = 0.0f, cy = 0.0f, cz = 0.0f;
                if (mode[r] == 1 || js > w)
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
    const bool mine = !SPLIT || (int)(threadIdx.x >> 5) == js0;                      // sources this CTA took
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        double v = (double)s_b[0][c][threadIdx.x];
#pragma unroll
        for (int ww = 1; ww < PAIR_THREADS / 32; ++ww) v += (double)s_b[ww][c][threadIdx.x];
        double *p = acc_j + (size_t)c * n_pad + j;
        if (mine) *p = *p - v;
    }
#pragma unroll
    for (int r = 0; r < SYM_R; ++r) {
        if (mode[r] == 0) continue;
        const int i = (tb + r) * PAIR_THREADS + threadIdx.x;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            double *p = acc_i + (size_t)c * n_pad + i;
            *p = *p + A[r][c];
        }
    }
}

}  // namespace steps
