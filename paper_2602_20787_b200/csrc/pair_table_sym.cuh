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
    const double2 *Dh;         // the same with a one-node halo on every side, (nrho + 2) * (nz + 2) nodes, the
                               // boundary symmetries of D (reading T3) baked in: node (i, j), -1 <= i <= nrho,
                               // -1 <= j <= nz, at Dh[(i + 1) * (nz + 2) + j + 1]  (TSC lookups in double)
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

// Where the nodes live: double2 in global memory (read through L1), or float2 in shared memory.
struct GlobalTable {
    static constexpr bool kLookupAlways = false;   // gathers from L1: only lanes that need the node
    const double2 *D;
    __device__ __forceinline__ double2 node(int idx) const { return __ldg(D + idx); }
};
struct SharedTableF32 {
    static constexpr bool kLookupAlways = true;    // shared memory: cheaper than a divergent branch
    const float2 *D;
};

// floor(x) and 1 + frac(x) (truncated to float) of 0 <= x < 2^31 from three FP64 additions and two
// integer instructions: the conversion instructions (F2I.F64, I2F.F64, F2F) issue at a quarter of
// the FP64 rate and were what bounded this kernel.
__device__ __forceinline__ void floor_frac(double x, int &i, double &f)
{
    const double t = __dadd_rd(x, 4503599627370496.0);            // 2^52 + floor(x), exact
    i = lo32(t);
    f = x - (t - 4503599627370496.0);
}

// floor(x) and 1 + frac(x) as a float in [1, 2), for 0 <= x < 2^28, from ONE FP64 addition: x + 1.5 * 2^29 (rounded
// down) lies in [2^29, 2^30), where a double's ulp is 2^-23, so its 52 mantissa bits are
// [2^28 + floor(x) : 29 bits][frac(x) : 23 bits] -- the fraction truncated to 2^-23 of a cell, far below the float
// nodes' own rounding.  A funnel shift and a mask give floor(x), one LOP3 the float.  (Any other x, NaN included,
// gives SOME i in [0, 2^28) and SOME f1 in [1, 2): the callers clamp i from above and discard such lanes.)
__device__ __forceinline__ void floor_frac1(double x, int &i, float &f1)
{
    const double t = __dadd_rd(x, 805306368.0);                  // 1.5 * 2^29
    const unsigned lo = (unsigned)lo32(t), hi = (unsigned)hi32(t);
    i = (int)(__funnelshift_r(lo, hi, 23) & 0x0fffffffu);
    f1 = __uint_as_float(0x3f800000u | (lo & 0x007fffffu));
}

template <class Tab>
__device__ __forceinline__ double2 table_node(const TableConsts &tc, const Tab &tab, int i, int j)
{
    // boundary rules: D_rho odd in rho / even in z, D_z even in rho / odd in z, both periodic in z
    double sr = 1.0, sz = 1.0;
    if (i < 0) { i = -i; sr = -1.0; }
    if (i > tc.nrho - 1) i = tc.nrho - 1;
    if (j < 0) { j = -j; sz = -1.0; }
    if (j > tc.nz - 1) { j = 2 * (tc.nz - 1) - j; sz = -sz; }
    const double2 v = tab.node(i * tc.nz + j);
    return make_double2(sr * v.x, sz * v.y);
}

// Interpolated {D_rho, D_z} at (rho, az = |r_z|), rho < rho_max.
template <int INTERP>
__device__ __forceinline__ double2 table_lookup(const TableConsts &tc, const GlobalTable &tab, double rho,
                                                double az, bool /*live*/)
{
    const double xr = rho * tc.inv_drho, xz = az * tc.inv_dz;
    if (INTERP == 0) {
        int i0, j0;
        double fr, fz;
        floor_frac(xr, i0, fr);
        floor_frac(xz, j0, fz);
        // a weight of exactly 0 multiplies the clamped node when rho or |r_z| sits on the last node;
        // lanes beyond rho_max (and the padding particles) arrive here too: any node will do for them
        i0 = min(max(i0, 0), tc.nrho - 1);
        j0 = min(max(j0, 0), tc.nz - 1);
        const int i1 = min(i0 + 1, tc.nrho - 1), j1 = min(j0 + 1, tc.nz - 1);
        const double2 d00 = tab.node(i0 * tc.nz + j0);
        const double2 d01 = tab.node(i0 * tc.nz + j1);
        const double2 d10 = tab.node(i1 * tc.nz + j0);
        const double2 d11 = tab.node(i1 * tc.nz + j1);
        const double ax = fma(fz, d01.x - d00.x, d00.x), bx = fma(fz, d11.x - d10.x, d10.x);
        const double ay = fma(fz, d01.y - d00.y, d00.y), by = fma(fz, d11.y - d10.y, d10.y);
        return make_double2(fma(fr, bx - ax, ax), fma(fr, by - ay, ay));
    }
    int ic, jc;
    double dr, dz;
    floor_frac(xr + 0.5, ic, dr);
    floor_frac(xz + 0.5, jc, dz);
    dr -= 0.5;
    dz -= 0.5;
    ic = min(max(ic, 0), tc.nrho - 1);
    jc = min(max(jc, 0), tc.nz - 1);
    const double wr[3] = {0.5 * (0.5 - dr) * (0.5 - dr), 0.75 - dr * dr, 0.5 * (0.5 + dr) * (0.5 + dr)};
    const double wz[3] = {0.5 * (0.5 - dz) * (0.5 - dz), 0.75 - dz * dz, 0.5 * (0.5 + dz) * (0.5 + dz)};
    double ox = 0.0, oy = 0.0;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        double rx = 0.0, ry = 0.0;
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            // the haloed table: no reflection, clamp or sign per node (9 sign multiplications and ~20 integer
            // instructions less per lookup than table_node(); the values, hence the sums, are bit for bit the same)
            const double2 v = __ldg(tc.Dh + (ic + a) * (tc.nz + 2) + jc + b);
            rx = fma(wz[b], v.x, rx);
            ry = fma(wz[b], v.y, ry);
        }
        ox = fma(wr[a], rx, ox);
        oy = fma(wr[a], ry, oy);
    }
    return make_double2(ox, oy);
}

// Copy of the float table in shared memory with a one-node halo on every side, filled by the boundary rules
// (D_rho odd in rho / even in z, D_z even in rho / odd in z about z = 0 and z = L/2, clamped beyond
// rho_max): node (i, j), -1 <= i <= nrho, -1 <= j <= nz, sits at s_table[(i + 1) * (nz + 2) + j + 1], so
// neither interpolation needs an index clamp, a reflection or a sign.
__host__ __device__ inline size_t table_halo_nodes(int nrho, int nz) { return (size_t)(nrho + 2) * (nz + 2); }

__device__ __forceinline__ void stage_table_halo(float2 *s_table, const float2 *__restrict__ table_f32,
                                                 int nrho, int nz, int nthreads)
{
    const int nzs = nz + 2, total = (nrho + 2) * nzs;
    for (int q = threadIdx.x; q < total; q += nthreads) {
        int i = q / nzs - 1, j = q % nzs - 1;
        float sr = 1.0f, sz = 1.0f;
        if (i < 0) { i = -i; sr = -1.0f; }
        if (i > nrho - 1) i = nrho - 1;
        if (j < 0) { j = -j; sz = -1.0f; }
        if (j > nz - 1) { j = 2 * (nz - 1) - j; sz = -sz; }
        const float2 v = table_f32[i * nz + j];
        s_table[q] = make_float2(sr * v.x, sz * v.y);
    }
}

// The float table in shared memory: node indices and weights from the fp64 (rho, |r_z|), the weighted sum
// of the float nodes in fp32 (its rounding, ~1e-7 of D, is of the size of the nodes' own), two conversions.
template <int INTERP>
__device__ __forceinline__ double2 table_lookup(const TableConsts &tc, const SharedTableF32 &tab,
                                                double rho, double az, bool live)
{
    const float2 *D = tab.D;
    const int nzs = tc.nz + 2;
    float ox, oy;
    if (INTERP == 0) {
        int i0, j0;
        float fr1, fz1;
        floor_frac1(rho * tc.inv_drho, i0, fr1);
        floor_frac1(az * tc.inv_dz, j0, fz1);
        const float fr = fr1 - 1.0f, fz = fz1 - 1.0f;
        // lanes beyond rho_max (and the padding particles) arrive here too: any node will do for them
        // (j0 is in range for finite input; the clamp keeps a NaN coordinate from reading out of bounds;
        // floor_frac1 never returns a negative index)
        i0 = min(i0, tc.nrho - 1);
        j0 = min(j0, tc.nz - 1);
        // (this loop is bound by issue slots: redirecting the discarded lanes' gathers to one broadcast
        // address, as the TSC branch does, costs more in its SEL than it saves in bank conflicts)
        const float2 *d = D + (i0 + 1) * nzs + j0 + 1;
        const float2 d00 = d[0], d01 = d[1], d10 = d[nzs], d11 = d[nzs + 1];
        const float ax = fmaf(fz, d01.x - d00.x, d00.x), bx = fmaf(fz, d11.x - d10.x, d10.x);
        const float ay = fmaf(fz, d01.y - d00.y, d00.y), by = fmaf(fz, d11.y - d10.y, d10.y);
        ox = fmaf(fr, bx - ax, ax);
        oy = fmaf(fr, by - ay, ay);
    } else {
        int ic, jc;
        float fr1, fz1;
        floor_frac1(fma(rho, tc.inv_drho, 0.5), ic, fr1);
        floor_frac1(fma(az, tc.inv_dz, 0.5), jc, fz1);
        const float dr = fr1 - 1.5f, dz = fz1 - 1.5f;
        ic = min(ic, tc.nrho - 1);
        jc = min(jc, tc.nz - 1);
        // node (ic - 1, jc - 1); lanes whose value is discarded all read node (-1, -1): one broadcast, no bank
        // conflicts (the nine gathers per pair make this loop shared-memory bound)
        const float2 *d = D + (live ? ic * nzs + jc : 0);
        const float wr[3] = {0.5f * (0.5f - dr) * (0.5f - dr), 0.75f - dr * dr, 0.5f * (0.5f + dr) * (0.5f + dr)};
        const float wz[3] = {0.5f * (0.5f - dz) * (0.5f - dz), 0.75f - dz * dz, 0.5f * (0.5f + dz) * (0.5f + dz)};
        ox = oy = 0.0f;
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
    }
    return make_double2((double)ox, (double)oy);
}

// One ring pass.  Per source the R pairs go through three phases so that the long part is one
// branch-free block the scheduler can interleave across the R targets (with one 16-warp CTA per SM
// there are only four warps per scheduler to hide the FP64 latencies):
//   1. geometry, unsoftened w0 = q^-3/2, 1/rho, and the table lookup -- no branches when the table is in
//      shared memory: lanes beyond rho_max look up a clamped node and discard it;
//   2. the spline correction of w0 (rare; also takes the coincident / self pair q = 0);
//   3. -f of the pair (see the header) by selects, and the accumulation.
template <int INTERP, int R, bool SYM, class Tab>
__device__ __forceinline__ void ring_subtile_table(const SymTgt (&ti)[R], const int (&soft_hi)[R],
                                                   const SymSrc *s_src, int lane,
                                                   const PairConsts &k, const TableConsts &tc,
                                                   const Tab &tab,
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
        double rx[R], ry[R], rz[R], q[R], w0[R], y[R];
        double2 Dv[R];
        bool near[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            rx[r] = ti[r].x - pa.x;
            ry[r] = ti[r].y - pa.y;
            rz[r] = nearest_image_exact(ti[r].z - pb.x, k);
            // + 1e-300 (below half an ulp of any rho^2 that matters): keeps 1/rho finite for rho = 0, where
            // the interpolated D_rho underflows to D_rho(0) = 0 and (r_x, r_y) = 0 removes the direction
            const double rho2 = fma(ry[r], ry[r], fma(rx[r], rx[r], 1.0e-300));
            y[r] = rsqrt_full(rho2);
            near[r] = rho2 < tc.rho_max2;
            q[r] = fma(rz[r], rz[r], rho2);
            w0[r] = inv_cube_sqrt(q[r]);
            if (Tab::kLookupAlways || near[r]) Dv[r] = table_lookup<INTERP>(tc, tab, rho2 * y[r], fabs(rz[r]), near[r]);
            else Dv[r] = make_double2(0.0, 0.0);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            if (hi32(q[r]) <= soft_hi[r]) {
                const double hh = ti[r].h + hj;
                if (q[r] < hh * hh) w0[r] = spline_w(q[r], hh);
            }
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const double cn = fma(-Dv[r].x, y[r], w0[r]);                 // w0 - D_rho / rho
            const double cf = tc.two_over_L * y[r] * y[r];                // line mass beyond rho_max
            // w0 r_z - sign(r_z) D_z: the sign of D_z flipped unless r_z < 0, on the high word (D_z(rho, 0) = 0)
            const double dz = __hiloint2double(hi32(Dv[r].y) ^ (~hi32(rz[r]) & 0x80000000), lo32(Dv[r].y));
            const double zn = fma(w0[r], rz[r], dz);
            const double cr = near[r] ? cn : cf;
            const double px = cr * rx[r], py = cr * ry[r], pz = near[r] ? zn : 0.0;
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

// Same decomposition and acc layout as pair_fp64_sym_kernel (A_z2 stays 0), generalised to TW warps:
// a CTA owns (TW/4) * SYM_R target tiles -- warp w holds sub-block w % 4 of target tiles
// tb + (w/4) * SYM_R + r -- and streams 128-source tiles.  grid = (n_tiles / tiles_per_cta, chunks).
//   SMEM_TABLE = false: TW = 4, the table is read from global memory (double2 nodes);
//   SMEM_TABLE = true : TW = 16 (one CTA per SM), the float2 table is copied to shared memory first,
//                       dynamic shared memory = TW*3*128*8 bytes of accumulators + (nrho+2)(nz+2) * 8 bytes.
// The spline pre-test needs no restriction on max(h): only the nearest image is evaluated here.
template <int INTERP, int TW, bool SMEM_TABLE>
__global__ void __launch_bounds__(TW * 32, SMEM_TABLE ? 1 : 4)
pair_table_sym_kernel(const double2 *__restrict__ xy, const double2 *__restrict__ zm,
                      const double *__restrict__ hs, const double *__restrict__ tile_hmax,
                      int n_pad, int n_tiles, int tiles_per_chunk, PairConsts k, TableConsts tc,
                      const float2 *__restrict__ table_f32, double *__restrict__ acc)
{
    constexpr int TILES_PER_CTA = (TW / 4) * SYM_R;
    const int tb = blockIdx.x * TILES_PER_CTA;
    // CTA (bx, c) takes the source tiles t = c, c + chunks, c + 2 chunks, ... from its first target tile on: the
    // packed arrays are in Morton order (order_kernels.cuh), and a CTA walking CONTIGUOUS tiles would add up one
    // compact region after the other -- long one-sided partial sums that cost the cancellation accuracy of the
    // total (measured: 1e-14 -> 2e-11 for core particles).  Strided tiles visit the volume in scattered order.
    const int t_stride = gridDim.y;
    const int t0 = tb + ((int)blockIdx.y - tb % t_stride + t_stride) % t_stride;       // first t >= tb, t = c mod chunks
    const int t1 = n_tiles;
    (void)tiles_per_chunk;
    if (t0 >= t1) return;
    __shared__ SymSrc s_src[PAIR_THREADS];
    // dynamic shared memory: per-warp source accumulators s_b[TW][3][128], then the float2 table
    extern __shared__ double s_dyn[];
    double (*s_b)[3][PAIR_THREADS] = reinterpret_cast<double (*)[3][PAIR_THREADS]>(s_dyn);
    float2 *s_table = reinterpret_cast<float2 *>(s_dyn + TW * 3 * PAIR_THREADS);

    if (SMEM_TABLE) stage_table_halo(s_table, table_f32, tc.nrho, tc.nz, TW * 32);
    GlobalTable gtab{tc.D};
    SharedTableF32 stab{s_table};

    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int wq = w & 3;                                   // sub-block of the target tiles
    const int tgt0 = tb + (w >> 2) * SYM_R;                 // this warp's first target tile
    SymTgt ti[SYM_R];
    double a[SYM_R][3];
#pragma unroll
    for (int r = 0; r < SYM_R; ++r) {
        const int i = (tgt0 + r) * PAIR_THREADS + wq * 32 + lane;
        const double2 pi = xy[i], qi = zm[i];
        ti[r].x = pi.x; ti[r].y = pi.y; ti[r].z = qi.x; ti[r].m = qi.y; ti[r].h = hs[i];
        a[r][0] = a[r][1] = a[r][2] = 0.0;
    }
    for (int t = t0; t < t1; t += t_stride) {
        __syncthreads();                                    // previous flush done (and the table is in)
        if (threadIdx.x < PAIR_THREADS) {
            const int j = t * PAIR_THREADS + threadIdx.x;
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
            if (t >= tgt0 + SYM_R) {
                if (SMEM_TABLE)
                    ring_subtile_table<INTERP, SYM_R, true>(ti, soft_hi, sub, lane, k, tc, stab, a, bx, by, bz);
                else
                    ring_subtile_table<INTERP, SYM_R, true>(ti, soft_hi, sub, lane, k, tc, gtab, a, bx, by, bz);
            } else {
                // a tile at or below this warp's own target tiles: target tile tgt0 + r meets source tile t
                // only if t >= tgt0 + r; in its own tile the warp takes sub-tiles above its own both ways,
                // its own target-side only, and leaves the ones below to their owners
#pragma unroll
                for (int r = 0; r < SYM_R; ++r) {
                    if (tgt0 + r > t) continue;
                    const SymTgt (&t1r)[1] = reinterpret_cast<const SymTgt (&)[1]>(ti[r]);
                    const int (&s1r)[1] = reinterpret_cast<const int (&)[1]>(soft_hi[r]);
                    double (&a1r)[1][3] = reinterpret_cast<double (&)[1][3]>(a[r]);
                    double cx = 0.0, cy = 0.0, cz = 0.0;
                    const bool both = (tgt0 + r < t) || (js > wq);
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
        __syncthreads();
        for (int q = threadIdx.x; q < 3 * PAIR_THREADS; q += TW * 32) {
            const int c = q / PAIR_THREADS, jl = q % PAIR_THREADS;
            double v = s_b[0][c][jl];
#pragma unroll
            for (int ww = 1; ww < TW; ++ww) v += s_b[ww][c][jl];
            if (v != 0.0) atomicAdd(acc + (size_t)c * n_pad + t * PAIR_THREADS + jl, -v);
        }
    }
#pragma unroll
    for (int r = 0; r < SYM_R; ++r) {
        const int i = (tgt0 + r) * PAIR_THREADS + wq * 32 + lane;
#pragma unroll
        for (int c = 0; c < 3; ++c) atomicAdd(acc + (size_t)c * n_pad + i, a[r][c]);
    }
}

}  // namespace steps
