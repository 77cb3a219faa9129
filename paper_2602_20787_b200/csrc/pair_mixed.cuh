// pair_mixed.cuh -- all-pairs S^1 x R^2 acceleration, pair terms in float, sums over sources
// in double (precision == STEPS_PREC_MIXED).
//
// Same sums as pair_fp64.cuh (A_x, A_y, A_z1, A_z2; Eq. 1/3/4/8 of the paper), with three
// differences dictated by single precision:
//   * separations: positions reach r ~ 2000 where fl32 has ulp 1.2e-4, comparable to close-pair
//     distances.  Each coordinate is carried as hi + lo floats (pack_kernel) and the separation
//     is (hi_i - hi_j) + (lo_i - lo_j): the hi difference is exact for close pairs (Sterbenz),
//     so the separation keeps ~2^-24 relative accuracy at any radius.  The period is split the
//     same way (L = Lh + Ll) so the nearest-image shift is exact too.
//   * rsqrt: MUFU.RSQ (rsqrt.approx.f32, 2^-22) cubed; no refinement.
//   * each pair's contribution is converted to double before it is added (fp64 accumulate).
// The XU pipe (one MUFU per image) and instruction issue bound this kernel, not the FMA pipes.
#pragma once
#include <cuda_runtime.h>

#include "pair_fp64.cuh"

namespace steps {

#ifndef STEPS_RT_UNROLL_MIXED
#define STEPS_RT_UNROLL_MIXED 3
#endif
constexpr int kRtUnrollMixed = STEPS_RT_UNROLL_MIXED;   // run-time N_cut image loop of the packed mixed kernel
                                                        // (1/2/3/4 at N_cut = 10: 237 / 223 / 214 / 215 ms)

struct MixedConsts {
    float Lh, Ll, halfL;
    float simple_ratio2;                  // SIMPLE ring pass (pair_mixed_sym.cuh) needs d^2 * simple_ratio2 >= c^2
    float simple_ext2;                    // ... and d^2 >= simple_ext2 * (source box extent)^2
    float c2nL[MAX_NCUT_TABLE + 1];       // 2 n L
    float n2L2[MAX_NCUT_TABLE + 1];       // (n L)^2
    float dn[MAX_NCUT_TABLE + 1];         // n
};

__device__ __forceinline__ float rsqrt_f32(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__device__ __forceinline__ float inv_cube_sqrt_f32(float x)
{
    const float y = rsqrt_f32(x);
    // explicit roundings: a product left open to FMA contraction would make w(+n) - w(-n) != 0
    // for r_z = 0 (one side fused into the subtraction, the other rounded)
    return __fmul_rn(__fmul_rn(y, y), y);
}

__device__ __noinline__ float spline_w_f32(float q, float hh)
{
    const float s   = sqrtf(q);
    const float ih  = 1.0f / hh;
    const float u   = s * ih;
    const float ih3 = ih * ih * ih;
    if (u < 0.5f)
        return fmaf(u * u, fmaf(32.0f, u, -38.4f), 32.0f / 3.0f) * ih3;
    const float u3 = u * u * u;
    float poly = fmaf(u, fmaf(u, fmaf(u, -32.0f / 3.0f, 38.4f), -48.0f), 64.0f / 3.0f);
    poly -= 1.0f / (15.0f * u3);
    return poly * ih3;
}

template <int NC>
__device__ __forceinline__ void pair_term_mixed(const float4 &ih, const float4 &il,
                                                const float4 &jh, const float4 &jl,
                                                const MixedConsts &k, int ncut_rt,
                                                double &ax, double &ay, double &az1, double &az2)
{
    // *h = {x_hi, y_hi, z_hi, m}, *l = {x_lo, y_lo, z_lo, h}
    const float rx = (ih.x - jh.x) + (il.x - jl.x);
    const float ry = (ih.y - jh.y) + (il.y - jl.y);
    float rzh = ih.z - jh.z, rzl = il.z - jl.z;
    const float sgn = (fabsf(rzh) > k.halfL) ? copysignf(1.0f, rzh) : 0.0f;
    rzh = fmaf(-sgn, k.Lh, rzh);
    rzl = fmaf(-sgn, k.Ll, rzl);
    const float rz = rzh + rzl;
    const float rho2 = fmaf(ry, ry, rx * rx);
    const float q = fmaf(rz, rz, rho2);
    const float hh = il.w + jl.w;

    float w0 = inv_cube_sqrt_f32(q);
    if (q < hh * hh) w0 = spline_w_f32(q, hh);
    float S = w0, T = 0.0f;
    if (NC > 0) {
#pragma unroll
        for (int n = 1; n < NC; ++n) {
            const float B  = q + k.n2L2[n];
            const float wp = inv_cube_sqrt_f32(fmaf(-k.c2nL[n], rz, B));
            const float wm = inv_cube_sqrt_f32(fmaf(k.c2nL[n], rz, B));
            S += wp;
            S += wm;
            T = fmaf((float)n, wp - wm, T);
        }
        float we = inv_cube_sqrt_f32(fmaf(-k.c2nL[NC], fabsf(rz), q + k.n2L2[NC]));
        we = (rz == 0.0f) ? 0.0f : we;
        S += we;
        T = fmaf(copysignf((float)NC, rz), we, T);
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
    const float Sm = jh.w * S;
    ax  += (double)(Sm * rx);
    ay  += (double)(Sm * ry);
    az1 += (double)(Sm * rz);
    az2 += (double)(jh.w * T);
}

// Same grid / chunk / partial-sum layout as pair_fp64_kernel.  The fast path's precondition
// (2 max h <= L/2) is required in mixed mode; otherwise the fp64 general path does the work (xy, zm, hs are
// only read then).
template <int NC>
__global__ void __launch_bounds__(PAIR_THREADS)
pair_mixed_kernel(const float4 *__restrict__ f_hi, const float4 *__restrict__ f_lo,
                  const double2 *__restrict__ xy, const double2 *__restrict__ zm,
                  const double *__restrict__ hs, const double *__restrict__ tile_hmax, int n_pad,
                  int n_tiles, int tiles_per_chunk, int ncut_rt, MixedConsts k, PairConsts kd,
                  const DevFlags *__restrict__ flags, double *__restrict__ part)
{
    __shared__ OrdSmem sm;
    if (need_general_path(flags, kd.halfL)) {
        ordered_body_general(xy, zm, hs, tile_hmax, n_pad, n_tiles, tiles_per_chunk, ncut_rt, kd, part, sm);
        return;
    }
    float4 *s_hi = reinterpret_cast<float4 *>(sm.xy), *s_lo = reinterpret_cast<float4 *>(sm.zm);
    const int i = blockIdx.x * PAIR_THREADS + threadIdx.x;
    const float4 ih = f_hi[i], il = f_lo[i];
    double ax = 0.0, ay = 0.0, az1 = 0.0, az2 = 0.0;
    const int t0 = blockIdx.y * tiles_per_chunk;
    const int t1 = min(t0 + tiles_per_chunk, n_tiles);
    for (int t = t0; t < t1; ++t) {
        const int j = t * PAIR_THREADS + threadIdx.x;
        __syncthreads();
        s_hi[threadIdx.x] = f_hi[j];
        s_lo[threadIdx.x] = f_lo[j];
        __syncthreads();
#pragma unroll 2
        for (int jj = 0; jj < PAIR_THREADS; ++jj)
            pair_term_mixed<NC>(ih, il, s_hi[jj], s_lo[jj], k, ncut_rt, ax, ay, az1, az2);
    }
    double *p = part + (size_t)blockIdx.y * 4 * n_pad + i;
    p[0] = ax;
    p[(size_t)n_pad] = ay;
    p[2 * (size_t)n_pad] = az1;
    p[3 * (size_t)n_pad] = az2;
}

}  // namespace steps
