// pair_table_sym.cuh -- all-pairs acceleration in STEPS_PERIODIC_EWALD_TABLE mode, fp64, each
// unordered pair once (same ring exchange / CTA decomposition / atomics as pair_fp64_sym.cuh).
//
// Pair law (Eq. 17; readings T1-T3), r = x_i - x_j, r_z nearest image,
// rho = |(r_x, r_y)|, per unit G m_i m_j:
//     rho <  rho_max :  f = -F(s, h_i + h_j)/s r  +  D_rho(rho, |r_z|) (r_x, r_y)/rho
//                          +  sign(r_z) D_z(rho, |r_z|) e_z
//     rho >= rho_max :  f = -2/(L rho^2) (r_x, r_y)            (line-mass term, Eq. 16, alpha -> inf)
// F the spline force of Eq. 3, D the host-built table of Eq. 17 ({D_rho, D_z} interleaved, node
// (i, j) at rho = i d_rho, z = j d_z), interpolated by cloud-in-cell (bilinear, 4 gathers of 16 B)
// or by triangular-shaped cloud (3 x 3 nodes, boundary nodes by the symmetries of D).
// The kernel accumulates A = -sum m f so that finalize_kernel's g = -G (A_x, A_y, A_z1 - L A_z2)
// applies unchanged with A_z2 = 0.
#pragma once
#include <cuda_runtime.h>

#include "pair_fp64_sym.cuh"

namespace steps {

struct TableConsts {
    const double2 *D;          // device table, nrho * nz nodes
    int nrho, nz, interp;
    double rho_max2;           // rho_max^2
    double inv_drho, inv_dz;   // 1 / node spacing
    double two_over_L;
};

// Exact nearest image, |r_z| <= L/2.  The high-word test of nearest_image() may leave |r_z| above
// L/2 by a relative 2^-20 -- harmless for the symmetric image window of Eq. 8, but here the single
// image that is kept, and the sign given to D_z, depend on it.
__device__ __forceinline__ double nearest_image_exact(double rz, const PairConsts &k)
{
    return (fabs(rz) > k.halfL) ? rz - copysign(k.L, rz) : rz;
}

// 1/sqrt(x) to ~1 ulp for normal positive x (RSQ64H seed + one third-order step).
__device__ __forceinline__ double rsqrt_full(double x)
{
    const double y0 = rsqrt_seed(x);
    const double y2 = y0 * y0;
    const double e  = fma(-x, y2, 1.0);
    const double p  = fma(0.375, e, 0.5);
    return fma(y0 * e, p, y0);
}

__device__ __forceinline__ double2 table_node(const TableConsts &tc, int i, int j)
{
    // boundary rules: D_rho odd in rho / even in z, D_z even in rho / odd in z, both periodic in z
    double sr = 1.0, sz = 1.0;
    if (i < 0) { i = -i; sr = -1.0; }
    if (i > tc.nrho - 1) i = tc.nrho - 1;
    if (j < 0) { j = -j; sz = -1.0; }
    if (j > tc.nz - 1) { j = 2 * (tc.nz - 1) - j; sz = -sz; }
    const double2 v = __ldg(tc.D + (size_t)i * tc.nz + j);
    return make_double2(sr * v.x, sz * v.y);
}

// Interpolated {D_rho, D_z} at (rho, az = |r_z|), rho < rho_max.
template <int INTERP>
__device__ __forceinline__ double2 table_lookup(const TableConsts &tc, double rho, double az)
{
    const double xr = rho * tc.inv_drho, xz = az * tc.inv_dz;
    if (INTERP == 0) {
        int i0 = __double2int_rd(xr), j0 = __double2int_rd(xz);
        const double fr = xr - (double)i0, fz = xz - (double)j0;
        // a weight of exactly 0 multiplies the clamped node when rho or |r_z| sits on the last node
        const int i1 = min(i0 + 1, tc.nrho - 1), j1 = min(j0 + 1, tc.nz - 1);
        i0 = min(i0, tc.nrho - 1);
        j0 = min(j0, tc.nz - 1);
        const double2 d00 = __ldg(tc.D + (size_t)i0 * tc.nz + j0);
        const double2 d01 = __ldg(tc.D + (size_t)i0 * tc.nz + j1);
        const double2 d10 = __ldg(tc.D + (size_t)i1 * tc.nz + j0);
        const double2 d11 = __ldg(tc.D + (size_t)i1 * tc.nz + j1);
        const double ax = fma(fz, d01.x - d00.x, d00.x), bx = fma(fz, d11.x - d10.x, d10.x);
        const double ay = fma(fz, d01.y - d00.y, d00.y), by = fma(fz, d11.y - d10.y, d10.y);
        return make_double2(fma(fr, bx - ax, ax), fma(fr, by - ay, ay));
    }
    const int ic = __double2int_rd(xr + 0.5), jc = __double2int_rd(xz + 0.5);
    const double dr = xr - (double)ic, dz = xz - (double)jc;
    const double wr[3] = {0.5 * (0.5 - dr) * (0.5 - dr), 0.75 - dr * dr, 0.5 * (0.5 + dr) * (0.5 + dr)};
    const double wz[3] = {0.5 * (0.5 - dz) * (0.5 - dz), 0.75 - dz * dz, 0.5 * (0.5 + dz) * (0.5 + dz)};
    double ox = 0.0, oy = 0.0;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        double rx = 0.0, ry = 0.0;
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            const double2 v = table_node(tc, ic - 1 + a, jc - 1 + b);
            rx = fma(wz[b], v.x, rx);
            ry = fma(wz[b], v.y, ry);
        }
        ox = fma(wr[a], rx, ox);
        oy = fma(wr[a], ry, oy);
    }
    return make_double2(ox, oy);
}

// -f of one pair (see the header): (px, py, pz).
template <int INTERP>
__device__ __forceinline__ void table_pair(double rx, double ry, double rz, double hi, double hj,
                                           int soft_hi, const TableConsts &tc, double &px,
                                           double &py, double &pz)
{
    const double rho2 = fma(ry, ry, rx * rx);
    // rho2 == 0: y = 0 kills the radial table term (D_rho(0) = 0 and no direction)
    const double y = (rho2 > 0.0) ? rsqrt_full(rho2) : 0.0;
    if (rho2 < tc.rho_max2) {
        const double q = fma(rz, rz, rho2);
        double w0 = inv_cube_sqrt(q);
        if (hi32(q) <= soft_hi) {
            const double hh = hi + hj;
            if (q < hh * hh) w0 = spline_w(q, hh);
        }
        const double2 Dv = table_lookup<INTERP>(tc, rho2 * y, fabs(rz));
        const double cr = fma(-Dv.x, y, w0);               // w0 - D_rho / rho
        px = cr * rx;
        py = cr * ry;
        pz = fma(w0, rz, (rz < 0.0) ? Dv.y : -Dv.y);       // w0 r_z - sign(r_z) D_z;  D_z(rho, 0) = 0
    } else {
        const double cr = tc.two_over_L * y * y;
        px = cr * rx;
        py = cr * ry;
        pz = 0.0;
    }
}

template <int INTERP, int R, bool SYM>
__device__ __forceinline__ void ring_subtile_table(const SymTgt (&ti)[R], const int (&soft_hi)[R],
                                                   const SymSrc *s_src, int lane,
                                                   const PairConsts &k, const TableConsts &tc,
                                                   double (&a)[R][3], double &bx, double &by,
                                                   double &bz)
{
    bx = by = bz = 0.0;
#pragma unroll 1
    for (int s = 0; s < 32; ++s) {
        const SymSrc *sj = s_src + ((lane + s) & 31);
        const double2 pa = *reinterpret_cast<const double2 *>(&sj->x);
        const double2 pb = *reinterpret_cast<const double2 *>(&sj->z);
        const double hj = sj->h;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const double rx = ti[r].x - pa.x, ry = ti[r].y - pa.y;
            const double rz = nearest_image_exact(ti[r].z - pb.x, k);
            double px, py, pz;
            table_pair<INTERP>(rx, ry, rz, ti[r].h, hj, soft_hi[r], tc, px, py, pz);
            a[r][0] = fma(pb.y, px, a[r][0]);
            a[r][1] = fma(pb.y, py, a[r][1]);
            a[r][2] = fma(pb.y, pz, a[r][2]);
            if (SYM) {
                bx = fma(ti[r].m, px, bx);
                by = fma(ti[r].m, py, by);
                bz = fma(ti[r].m, pz, bz);
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

// Same grid, decomposition and acc layout as pair_fp64_sym_kernel (A_z2 stays 0).  The spline
// pre-test needs no restriction on max(h): only the nearest image is ever evaluated here.
template <int INTERP>
__global__ void __launch_bounds__(PAIR_THREADS, 4)
pair_table_sym_kernel(const double2 *__restrict__ xy, const double2 *__restrict__ zm,
                      const double *__restrict__ hs, const double *__restrict__ tile_hmax,
                      int n_pad, int n_tiles, int tiles_per_chunk, PairConsts k, TableConsts tc,
                      double *__restrict__ acc)
{
    const int tb = blockIdx.x * SYM_R;
    const int t0 = max(blockIdx.y * tiles_per_chunk, tb);
    const int t1 = min((blockIdx.y + 1) * tiles_per_chunk, n_tiles);
    if (t0 >= t1) return;
    __shared__ SymSrc s_src[PAIR_THREADS];
    __shared__ double s_b[PAIR_THREADS / 32][3][PAIR_THREADS];

    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    SymTgt ti[SYM_R];
    double a[SYM_R][3];
#pragma unroll
    for (int r = 0; r < SYM_R; ++r) {
        const int i = (tb + r) * PAIR_THREADS + threadIdx.x;
        const double2 pi = xy[i], qi = zm[i];
        ti[r].x = pi.x; ti[r].y = pi.y; ti[r].z = qi.x; ti[r].m = qi.y; ti[r].h = hs[i];
        ti[r].mL = 0.0;
        a[r][0] = a[r][1] = a[r][2] = 0.0;
    }
    for (int t = t0; t < t1; ++t) {
        const int j = t * PAIR_THREADS + threadIdx.x;
        __syncthreads();
        {
            const double2 pj = xy[j], qj = zm[j];
            SymSrc v;
            v.x = pj.x; v.y = pj.y; v.z = qj.x; v.m = qj.y; v.h = hs[j]; v.pad = 0.0;
            s_src[threadIdx.x] = v;
        }
        __syncthreads();
        int soft_hi[SYM_R];
        {
            const double hm = tile_hmax[t];
#pragma unroll
            for (int r = 0; r < SYM_R; ++r) {
                const double b = ti[r].h + hm;
                soft_hi[r] = hi32(b * b);
            }
        }
#pragma unroll 1
        for (int js = 0; js < PAIR_THREADS / 32; ++js) {
            double bx = 0.0, by = 0.0, bz = 0.0;
            const SymSrc *sub = s_src + js * 32;
            if (t >= tb + SYM_R) {
                ring_subtile_table<INTERP, SYM_R, true>(ti, soft_hi, sub, lane, k, tc, a, bx, by, bz);
            } else {
#pragma unroll
                for (int r = 0; r < SYM_R; ++r) {
                    if (tb + r > t) continue;
                    const SymTgt (&t1r)[1] = reinterpret_cast<const SymTgt (&)[1]>(ti[r]);
                    const int (&s1r)[1] = reinterpret_cast<const int (&)[1]>(soft_hi[r]);
                    double (&a1r)[1][3] = reinterpret_cast<double (&)[1][3]>(a[r]);
                    double cx = 0.0, cy = 0.0, cz = 0.0;
                    if (tb + r < t || js > w)
                        ring_subtile_table<INTERP, 1, true>(t1r, s1r, sub, lane, k, tc, a1r, cx, cy, cz);
                    else if (js == w)
                        ring_subtile_table<INTERP, 1, false>(t1r, s1r, sub, lane, k, tc, a1r, cx, cy, cz);
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
            if (v != 0.0) atomicAdd(acc + (size_t)c * n_pad + j, -v);
        }
    }
#pragma unroll
    for (int r = 0; r < SYM_R; ++r) {
        const int i = (tb + r) * PAIR_THREADS + threadIdx.x;
#pragma unroll
        for (int c = 0; c < 3; ++c) atomicAdd(acc + (size_t)c * n_pad + i, a[r][c]);
    }
}

}  // namespace steps
