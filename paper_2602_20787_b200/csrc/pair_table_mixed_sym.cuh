// pair_table_mixed_sym.cuh -- EWALD_TABLE mode in mixed precision: pair terms and the table
// interpolation in float, sums across rings / tiles / CTAs in double (the precision contract of
// pair_mixed_sym.cuh), float table in shared memory, 512-thread CTAs (the layout of
// pair_table_sym_kernel<., 16, true>).  Pair law: see pair_table_sym.cuh.
#pragma once
#include <cuda_runtime.h>

#include "pair_mixed_sym.cuh"
#include "pair_table_sym.cuh"

namespace steps {

struct TableConstsF32 {
    int nrho, nz;
    float rho_max2, inv_drho, inv_dz, two_over_L;
};

// floor(x) and frac(x) of 0 <= x < 2^22 without the quarter-rate conversion instructions.
__device__ __forceinline__ void floor_frac_f32(float x, int &i, float &f)
{
    const float t = __fadd_rd(x, 8388608.0f);               // 2^23 + floor(x), exact
    i = __float_as_int(t) - 0x4b000000;
    f = x - (t - 8388608.0f);
}

// Interpolated {D_rho, D_z} in float; nodes from the shared-memory float2 table.
template <int INTERP>
__device__ __forceinline__ float2 table_lookup_f32(const TableConstsF32 &tc, const float2 *tab, float rho,
                                                  float az, bool live)
{
    const float xr = rho * tc.inv_drho, xz = az * tc.inv_dz;
    const int nzs = tc.nz + 2;
    if (INTERP == 0) {
        int i0, j0;
        float fr, fz;
        floor_frac_f32(xr, i0, fr);
        floor_frac_f32(xz, j0, fz);
        // lanes beyond rho_max (and the padding particles) arrive here too: any node will do for them
        i0 = min(max(i0, 0), tc.nrho - 1);
        j0 = min(max(j0, 0), tc.nz - 1);
        // haloed table (stage_table_halo); lanes whose value is discarded all read node (-1, -1): a broadcast
        const float2 *d = tab + (live ? (i0 + 1) * nzs + j0 + 1 : 0);
        const float2 d00 = d[0], d01 = d[1], d10 = d[nzs], d11 = d[nzs + 1];
        const float ax = fmaf(fz, d01.x - d00.x, d00.x), bx = fmaf(fz, d11.x - d10.x, d10.x);
        const float ay = fmaf(fz, d01.y - d00.y, d00.y), by = fmaf(fz, d11.y - d10.y, d10.y);
        return make_float2(fmaf(fr, bx - ax, ax), fmaf(fr, by - ay, ay));
    }
    int ic, jc;
    float dr, dz;
    floor_frac_f32(xr + 0.5f, ic, dr);
    floor_frac_f32(xz + 0.5f, jc, dz);
    dr -= 0.5f;
    dz -= 0.5f;
    ic = min(max(ic, 0), tc.nrho - 1);
    jc = min(max(jc, 0), tc.nz - 1);
    const float2 *d = tab + (live ? ic * nzs + jc : 0);     // node (ic - 1, jc - 1)
    const float wr[3] = {0.5f * (0.5f - dr) * (0.5f - dr), 0.75f - dr * dr, 0.5f * (0.5f + dr) * (0.5f + dr)};
    const float wz[3] = {0.5f * (0.5f - dz) * (0.5f - dz), 0.75f - dz * dz, 0.5f * (0.5f + dz) * (0.5f + dz)};
    float ox = 0.0f, oy = 0.0f;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        float rx = 0.0f, ry = 0.0f;
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            const float2 v = d[a * nzs + b];
            rx = fmaf(wz[b], v.x, rx);
            ry = fmaf(wz[b], v.y, ry);
        }
        ox = fmaf(wr[a], rx, ox);
        oy = fmaf(wr[a], ry, oy);
    }
    return make_float2(ox, oy);
}

template <int INTERP, int R, bool SYM>
__device__ __forceinline__ void ring_subtile_table_f32(const MixTgt (&ti)[R], const int (&soft_bits)[R],
                                                       const float4 *s_hi, const float4 *s_lo, int lane,
                                                       const MixedConsts &k, const TableConstsF32 &tc,
                                                       const float2 *tab, float (&a)[R][3], float &bx,
                                                       float &by, float &bz)
{
    bx = by = bz = 0.0f;
#pragma unroll
    for (int r = 0; r < R; ++r) a[r][0] = a[r][1] = a[r][2] = 0.0f;
#pragma unroll 1
    for (int s = 0; s < 32; ++s) {
        const int jj = (lane + s) & 31;
        const float4 jh = s_hi[jj], jl = s_lo[jj];
        // three phases per source, as in ring_subtile_table (pair_table_sym.cuh): branch-free geometry +
        // lookup for all R targets, then the rare spline correction, then selects and accumulation
        float rx[R], ry[R], rz[R], q[R], w0[R], y[R];
        float2 Dv[R];
        bool near[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            rx[r] = (ti[r].xh - jh.x) + (ti[r].xl - jl.x);
            ry[r] = (ti[r].yh - jh.y) + (ti[r].yl - jl.y);
            const float rz0 = (ti[r].zh - jh.z) + (ti[r].zl - jl.z);
            // exact nearest image: |rz| <= L/2 afterwards
            const float sg = (fabsf(rz0) > k.halfL) ? copysignf(1.0f, rz0) : 0.0f;
            rz[r] = fmaf(-sg, k.Ll, fmaf(-sg, k.Lh, rz0));
            // + 1e-36: keeps 1/rho finite for rho = 0 (see ring_subtile_table)
            const float rho2 = fmaf(ry[r], ry[r], fmaf(rx[r], rx[r], 1.0e-36f));
            y[r] = rsqrt_f32(rho2);
            near[r] = rho2 < tc.rho_max2;
            q[r] = fmaf(rz[r], rz[r], rho2);
            w0[r] = inv_cube_sqrt_f32(q[r]);
            Dv[r] = table_lookup_f32<INTERP>(tc, tab, rho2 * y[r], fabsf(rz[r]), near[r]);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            if (__float_as_int(q[r]) <= soft_bits[r]) {
                const float hh = ti[r].h + jl.w;
                if (q[r] < hh * hh) w0[r] = spline_w_f32(q[r], hh);
            }
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const float cn = fmaf(-Dv[r].x, y[r], w0[r]);
            const float cf = tc.two_over_L * y[r] * y[r];
            const float dz = __int_as_float(__float_as_int(Dv[r].y) ^ (~__float_as_int(rz[r]) & 0x80000000));
            const float zn = fmaf(w0[r], rz[r], dz);           // w0 r_z - sign(r_z) D_z
            const float cr = near[r] ? cn : cf;
            const float px = cr * rx[r], py = cr * ry[r], pz = near[r] ? zn : 0.0f;
            a[r][0] = fmaf(jh.w, px, a[r][0]);
            a[r][1] = fmaf(jh.w, py, a[r][1]);
            a[r][2] = fmaf(jh.w, pz, a[r][2]);
            if (SYM) {
                bx = fmaf(ti[r].m, px, bx);
                by = fmaf(ti[r].m, py, by);
                bz = fmaf(ti[r].m, pz, bz);
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

constexpr int TABLE_MIXED_WARPS = 16;

// grid = (n_tiles / 8, chunks), 512 threads; dynamic shared memory = 16*3*128 floats + (nrho+2)(nz+2)*8 bytes.
template <int INTERP>
__global__ void __launch_bounds__(TABLE_MIXED_WARPS * 32, 1)
pair_table_mixed_sym_kernel(const float4 *__restrict__ f_hi, const float4 *__restrict__ f_lo,
                            const double *__restrict__ tile_hmax, int n_pad, int n_tiles,
                            int tiles_per_chunk, MixedConsts k, TableConstsF32 tc,
                            const float2 *__restrict__ table_f32, double *__restrict__ acc)
{
    constexpr int TW = TABLE_MIXED_WARPS, TILES_PER_CTA = (TW / 4) * SYM_R;
    const int tb = blockIdx.x * TILES_PER_CTA;
    const int t0 = max(blockIdx.y * tiles_per_chunk, tb);
    const int t1 = min((blockIdx.y + 1) * tiles_per_chunk, n_tiles);
    if (t0 >= t1) return;
    __shared__ float4 s_hi[PAIR_THREADS];
    __shared__ float4 s_lo[PAIR_THREADS];
    extern __shared__ float s_dynf[];
    float (*s_b)[3][PAIR_THREADS] = reinterpret_cast<float (*)[3][PAIR_THREADS]>(s_dynf);
    float2 *s_table = reinterpret_cast<float2 *>(s_dynf + TW * 3 * PAIR_THREADS);
    stage_table_halo(s_table, table_f32, tc.nrho, tc.nz, TW * 32);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, wq = w & 3;
    const int tgt0 = tb + (w >> 2) * SYM_R;
    MixTgt ti[SYM_R];
    double A[SYM_R][3];
#pragma unroll
    for (int r = 0; r < SYM_R; ++r) {
        const int i = (tgt0 + r) * PAIR_THREADS + wq * 32 + lane;
        const float4 h4 = f_hi[i], l4 = f_lo[i];
        ti[r].xh = h4.x; ti[r].yh = h4.y; ti[r].zh = h4.z; ti[r].m = h4.w;
        ti[r].xl = l4.x; ti[r].yl = l4.y; ti[r].zl = l4.z; ti[r].h = l4.w;
        ti[r].mL = 0.0f;
        A[r][0] = A[r][1] = A[r][2] = 0.0;
    }
    for (int t = t0; t < t1; ++t) {
        __syncthreads();
        if (threadIdx.x < PAIR_THREADS) {
            const int j = t * PAIR_THREADS + threadIdx.x;
            s_hi[threadIdx.x] = f_hi[j];
            s_lo[threadIdx.x] = f_lo[j];
        }
        __syncthreads();
        int soft_bits[SYM_R];
        {
            const float hm = (float)tile_hmax[t] * 1.0001f;
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
            if (t >= tgt0 + SYM_R) {
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
                    if (tgt0 + r > t) continue;
                    const MixTgt (&t1r)[1] = reinterpret_cast<const MixTgt (&)[1]>(ti[r]);
                    const int (&s1r)[1] = reinterpret_cast<const int (&)[1]>(soft_bits[r]);
                    float a1[1][3] = {{0.0f, 0.0f, 0.0f}};
                    float cx = 0.0f, cy = 0.0f, cz = 0.0f;
                    const bool both = (tgt0 + r < t) || (js > wq);
                    if (both)
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
        __syncthreads();
        for (int q = threadIdx.x; q < 3 * PAIR_THREADS; q += TW * 32) {
            const int c = q / PAIR_THREADS, jl = q % PAIR_THREADS;
            double v = (double)s_b[0][c][jl];
#pragma unroll
            for (int ww = 1; ww < TW; ++ww) v += (double)s_b[ww][c][jl];
            if (v != 0.0) atomicAdd(acc + (size_t)c * n_pad + t * PAIR_THREADS + jl, -v);
        }
    }
#pragma unroll
    for (int r = 0; r < SYM_R; ++r) {
        const int i = (tgt0 + r) * PAIR_THREADS + wq * 32 + lane;
#pragma unroll
        for (int c = 0; c < 3; ++c) atomicAdd(acc + (size_t)c * n_pad + i, A[r][c]);
    }
}

}  // namespace steps
