// steps_cyl.cu -- host side of libsteps_cyl.so: context, validation, scratch ownership, kernel
// launches, and the C ABI declared in include/steps_cyl.h.  No torch types, no CPU fallback.
#include "../../include/steps_cyl.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "aux_kernels.cuh"
#include "order_kernels.cuh"
#include "pair_fp64.cuh"
#include "pair_fp64_sym.cuh"
#include "pair_mixed.cuh"
#include "pair_mixed_sym.cuh"
#include "pair_table_sym.cuh"
#include "pair_table_mixed_sym.cuh"
#include "pair_table_round.cuh"
#include "ewald_table.h"

using namespace steps;

struct GraphSlot {
    cudaGraphExec_t exec = nullptr;
    cudaGraph_t graph = nullptr;
    cudaGraphNode_t pre = nullptr, post = nullptr;      // the prestep / poststep nodes (re-parameterised per step)
    const void *key[11] = {};                           // the caller's pointers the graph was captured with
    int n_kernels = 0;
};

struct steps_cyl_ctx {
    steps_cyl_params p;
    int n, n_pad, n_tiles;
    int n_chunks, tiles_per_chunk;
    int sym_chunks, sym_tiles_per_chunk;          // decomposition of the symmetric kernel
    bool use_sym;                                 // !STEPS_FLAG_DETERMINISTIC
    int sym_split = 1;                            // gridDim.z of the symmetric image-mode kernels (1 or 4)
    bool sym_small = false;                       // fp64 image mode at small N: one target tile per CTA (TR = 1)
    bool use_slabs = false;                       // DETERMINISTIC fp64 image mode up to N = 131072: single-writer slabs
    int sym_tr() const { return sym_small ? 1 : SYM_R; }
    int round_split = 1;                          // gridDim.y of the image-mode round kernels (1 or 4)
    bool use_rounds;                              // DETERMINISTIC: round-scheduled symmetric kernels
    int sm_count;
    PairConsts kc;
    MixedConsts mc;
    // device scratch (owned)
    double2 *xy = nullptr, *zm = nullptr;
    double *hs = nullptr, *tile_hmax = nullptr;
    float4 *f_hi = nullptr, *f_lo = nullptr;
    double *part = nullptr;
    DevFlags *flags = nullptr;                     // two blocks used by alternate force evaluations (+ a sticky word)
    DevFlags *cur_flags = nullptr;                 // the block of the evaluation being enqueued
    int *bad_h_sticky = nullptr;                   // h <= 0 seen since the last steps_cyl_check
    unsigned eval_count = 0;
    // spatial ordering of the packed arrays (EWALD_TABLE mode, order_kernels.cuh)
    bool use_order = false;
    int n_pow2 = 0;
    int *perm = nullptr;                           // packed slot -> caller index
    unsigned long long *order_keys = nullptr, *rmax_bits = nullptr;
    unsigned long long *pass_stats = nullptr;      // mixed kernel: SIMPLE / all ring passes since init
    GraphSlot gslot[2];                            // STEPS_FLAG_GRAPH: one captured evaluation per flag-block parity
    QuadNode *nodes = nullptr;
    double2 *d_table = nullptr;                    // EWALD_TABLE mode: D(rho, z), Eq. 17
    double2 *d_table_halo = nullptr;               // the same with the symmetry halo (TableConsts::Dh)
    float2 *d_table_f32 = nullptr;                 // the same rounded to float (tab_fp32), staged in smem
    size_t table_smem_bytes = 0, table_mixed_smem_bytes = 0;
    TableConstsF32 tcf;
    TableConsts tc;
    bool table_mode = false;
    int n_nodes = 0;
    double *host_io = nullptr;                     // device staging for the *_host entry points
    double *peak_out = nullptr;
    cudaStream_t own_stream = nullptr;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    bool ev_valid = false;
    int64_t launches = 0;
    char kernel_name[96];                          // the all-pairs kernel launch_pair() selects (sassmix.py naming)
    char cuda_msg[256];
};

namespace {

int cuda_fail(steps_cyl_ctx *c, cudaError_t e)
{
    if (c) snprintf(c->cuda_msg, sizeof c->cuda_msg, "%s: %s", cudaGetErrorName(e), cudaGetErrorString(e));
    return STEPS_ECUDA;
}

#define CK(call)                                                     \
    do {                                                             \
        cudaError_t e_ = (call);                                     \
        if (e_ != cudaSuccess) return cuda_fail(ctx, e_);            \
    } while (0)

// Makes the context's device current for the duration of an API call and puts the caller's back afterwards.
struct DeviceGuard {
    int prev = -1;
    cudaError_t err = cudaSuccess;
    explicit DeviceGuard(int dev)
    {
        int cur = -1;
        err = cudaGetDevice(&cur);
        if (err == cudaSuccess && cur != dev) {
            err = cudaSetDevice(dev);
            if (err == cudaSuccess) prev = cur;
        }
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};
#define ON_DEVICE(ctx_)                                              \
    DeviceGuard dev_guard_((ctx_)->p.device);                        \
    if (dev_guard_.err != cudaSuccess) return cuda_fail((ctx_), dev_guard_.err)

template <typename T>
cudaError_t dev_alloc(T **p, size_t count)
{
    return cudaMalloc((void **)p, count * sizeof(T));
}

// Double-exponential (tanh-sinh) nodes on [0, R]: Y = R/2 (1 + tanh(pi/2 sinh t)), stored with
// the distance to the nearer end point computed without cancellation.
std::vector<QuadNode> make_nodes(double R)
{
    std::vector<QuadNode> v;
    const double step = 1.0 / 24.0, half = 0.5 * R, hpi = 1.57079632679489661923;
    for (int k = -180; k <= 180; ++k) {
        const double t = k * step;
        const double u = hpi * std::sinh(t);
        const double ch = std::cosh(u);
        const double wgt = step * half * hpi * std::cosh(t) / (ch * ch);
        const double d = half * std::exp(-std::fabs(u)) / ch;       // distance to nearer end
        if (!(wgt > 0.0) || !(d > 0.0) || wgt < 1e-40 * R) continue;
        QuadNode q;
        if (u >= 0.0) { q.Y = R - d; q.e = d; }                      // near Y = R
        else          { q.Y = d;     q.e = R - d; }                  // near Y = 0
        q.wgt = wgt;
        v.push_back(q);
    }
    return v;
}

// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-function, process-wide setting: contexts with tables of
// different sizes can be alive together, so the limits are only ever raised (to the largest table seen).
cudaError_t raise_table_smem_limits(size_t fp64_bytes, size_t mixed_bytes)
{
    static std::mutex mu;
    static size_t cur_fp64 = 0, cur_mixed = 0;
    std::lock_guard<std::mutex> lock(mu);
    cudaError_t e = cudaSuccess;
    auto set = [&](auto *kernel, size_t bytes) {
        if (e == cudaSuccess) e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    };
    if (fp64_bytes > cur_fp64) {
        set(pair_table_sym_kernel<0, 16, true>, fp64_bytes);
        set(pair_table_sym_kernel<1, 16, true>, fp64_bytes);
        set(pair_table_round_kernel<0, 16, true>, fp64_bytes);
        set(pair_table_round_kernel<1, 16, true>, fp64_bytes);
        if (e == cudaSuccess) cur_fp64 = fp64_bytes;
    }
    if (mixed_bytes > cur_mixed) {
        set(pair_table_mixed_sym_kernel<0>, mixed_bytes);
        set(pair_table_mixed_sym_kernel<1>, mixed_bytes);
        set(pair_table_mixed_round_kernel<0>, mixed_bytes);
        set(pair_table_mixed_round_kernel<1>, mixed_bytes);
        if (e == cudaSuccess) cur_mixed = mixed_bytes;
    }
    return e;
}

void choose_chunks(steps_cyl_ctx *c)
{
    // Enough CTAs for ~24 waves of 4 resident CTAs per SM, at least one source tile per chunk.
    const int i_blocks = c->n_tiles;
    const int target = 24 * 4 * c->sm_count;
    int chunks = (target + i_blocks - 1) / i_blocks;
    chunks = std::max(1, std::min(chunks, c->n_tiles));
    chunks = std::min(chunks, 64);
    c->tiles_per_chunk = (c->n_tiles + chunks - 1) / chunks;
    c->n_chunks = (c->n_tiles + c->tiles_per_chunk - 1) / c->tiles_per_chunk;
    // symmetric kernel: CTAs cover the upper triangle of (target block, source tile); aim at
    // >= 8 waves of non-empty CTAs, at most 64 tiles (~2 ms) per CTA.
    const double tri = 0.5 * (double)c->n_tiles * (double)(c->n_tiles + 1);
    int tpc = (int)(tri / (8.0 * 4.0 * c->sm_count));
    tpc = std::max(1, std::min(tpc, 64));
    c->sym_tiles_per_chunk = tpc;
    c->sym_chunks = (c->n_tiles + tpc - 1) / tpc;
    // small N: fewer (target pair, source tile) items than two per SM -> split them by source sub-tile
    c->sym_split = (tri / SYM_R < 2.0 * c->sm_count) ? PAIR_THREADS / 32 : 1;
}

template <int NC>
void launch_pair_fp64_nc(steps_cyl_ctx *c, cudaStream_t s)
{
    dim3 grid(c->n_tiles, c->n_chunks);
    pair_fp64_kernel<NC><<<grid, PAIR_THREADS, 0, s>>>(c->xy, c->zm, c->hs, c->tile_hmax, c->n_pad, c->n_tiles,
                                                         c->tiles_per_chunk, c->p.n_cut, c->kc,
                                                         c->cur_flags, c->part);
}

template <int NC>
void launch_pair_sym_nc(steps_cyl_ctx *c, cudaStream_t s)
{
    const bool o2 = (c->p.flags & STEPS_FLAG_FAR_ORDER2) != 0;
#define SYM_LAUNCH(O2, TR, GRID)                                                                            \
    pair_fp64_sym_kernel<NC, O2, TR><<<GRID, PAIR_THREADS, 0, s>>>(c->xy, c->zm, c->hs, c->tile_hmax, c->n_pad, \
                                                                  c->n_tiles, c->sym_tiles_per_chunk, c->p.n_cut, \
                                                                  c->kc, c->cur_flags, c->part)
    if (c->use_slabs) {
        // DETERMINISTIC: the same kernel with single-writer slots instead of atomics
        const dim3 grid(c->n_tiles / c->sym_tr(), c->sym_chunks, c->sym_split);
        if (c->sym_small)
            pair_fp64_sym_kernel<NC, false, 1, true><<<grid, PAIR_THREADS, 0, s>>>(
                c->xy, c->zm, c->hs, c->tile_hmax, c->n_pad, c->n_tiles, c->sym_tiles_per_chunk, c->p.n_cut, c->kc,
                c->cur_flags, c->part);
        else
            pair_fp64_sym_kernel<NC, false, SYM_R, true><<<grid, PAIR_THREADS, 0, s>>>(
                c->xy, c->zm, c->hs, c->tile_hmax, c->n_pad, c->n_tiles, c->sym_tiles_per_chunk, c->p.n_cut, c->kc,
                c->cur_flags, c->part);
    } else if (c->sym_small) {
        // small N: one target tile and one source sub-tile per CTA (the kernel time is one CTA's critical path)
        const dim3 grid(c->n_tiles, c->sym_chunks, c->sym_split);
        if (o2) SYM_LAUNCH(true, 1, grid); else SYM_LAUNCH(false, 1, grid);
    } else {
        const dim3 grid(c->n_tiles / SYM_R, c->sym_chunks, c->sym_split);
        if (o2) SYM_LAUNCH(true, SYM_R, grid); else SYM_LAUNCH(false, SYM_R, grid);
    }
#undef SYM_LAUNCH
}

// Deterministic fp64 path: rounds of the symmetric evaluation, one launch each (pair_fp64_sym.cuh).
template <int NC>
void launch_pair_rounds_nc(steps_cyl_ctx *c, cudaStream_t s)
{
    const int T = c->n_tiles, last = std::min(T / 2 + 1, T - 1);
    double *acc_i = c->part, *acc_j = c->part + 4 * (size_t)c->n_pad * c->round_split;
    for (int r = 0; r <= last; ++r) {
        if (c->round_split > 1)
            pair_fp64_round_kernel<NC, true><<<dim3(T / SYM_R, c->round_split), PAIR_THREADS, 0, s>>>(
                c->xy, c->zm, c->hs, c->tile_hmax, c->n_pad, T, r, c->p.n_cut, c->kc, c->cur_flags, acc_i, acc_j);
        else
            pair_fp64_round_kernel<NC, false><<<T / SYM_R, PAIR_THREADS, 0, s>>>(
                c->xy, c->zm, c->hs, c->tile_hmax, c->n_pad, T, r, c->p.n_cut, c->kc, c->cur_flags, acc_i, acc_j);
    }
    c->launches += last;      // launch_pair() adds the remaining one
}

template <int NC>
void launch_pair_mixed_rounds_nc(steps_cyl_ctx *c, cudaStream_t s)
{
    const int T = c->n_tiles, last = std::min(T / 2 + 1, T - 1);
    double *acc_i = c->part, *acc_j = c->part + 4 * (size_t)c->n_pad * c->round_split;
    for (int r = 0; r <= last; ++r) {
        if (c->round_split > 1)
            pair_mixed_round_kernel<NC, true><<<dim3(T / SYM_R, c->round_split), PAIR_THREADS, 0, s>>>(
                c->f_hi, c->f_lo, c->xy, c->zm, c->hs, c->tile_hmax, c->n_pad, T, r, c->p.n_cut, c->mc, c->kc, c->cur_flags,
                acc_i, acc_j);
        else
            pair_mixed_round_kernel<NC, false><<<T / SYM_R, PAIR_THREADS, 0, s>>>(
                c->f_hi, c->f_lo, c->xy, c->zm, c->hs, c->tile_hmax, c->n_pad, T, r, c->p.n_cut, c->mc, c->kc, c->cur_flags,
                acc_i, acc_j);
    }
    c->launches += last;
}

template <int NC>
void launch_pair_mixed_nc(steps_cyl_ctx *c, cudaStream_t s)
{
    dim3 grid(c->n_tiles, c->n_chunks);
    pair_mixed_kernel<NC><<<grid, PAIR_THREADS, 0, s>>>(c->f_hi, c->f_lo, c->xy, c->zm, c->hs, c->tile_hmax,
                                                       c->n_pad, c->n_tiles, c->tiles_per_chunk, c->p.n_cut,
                                                       c->mc, c->kc, c->cur_flags, c->part);
}

template <int NC>
void launch_pair_mixed_sym_nc(steps_cyl_ctx *c, cudaStream_t s)
{
    dim3 grid(c->n_tiles / SYM_R, c->sym_chunks, c->sym_split);
    pair_mixed_sym_kernel<NC><<<grid, PAIR_THREADS, 0, s>>>(c->f_hi, c->f_lo, c->xy, c->zm, c->hs, c->tile_hmax,
                                                           c->n_pad, c->n_tiles, c->sym_tiles_per_chunk,
                                                           c->p.n_cut, c->mc, c->kc, c->cur_flags, c->part, c->pass_stats);
}

// EWALD_TABLE + DETERMINISTIC: one launch per round (pair_table_round.cuh).
void launch_table_rounds(steps_cyl_ctx *c, cudaStream_t s)
{
    const int T = c->n_tiles, last = std::min(T / 2 + 1, T - 1), groups = T / SYM_R;
    double *acc_i = c->part, *acc_j = c->part + 4 * (size_t)c->n_pad;
    const bool cic = c->tc.interp == STEPS_INTERP_CIC;
    const int g16 = std::min(c->sm_count, (groups + 3) / 4), g4 = std::min(groups, 8 * c->sm_count);
    const size_t sb4 = 4 * 3 * PAIR_THREADS * sizeof(double);
    for (int r = 0; r <= last; ++r) {
        if (c->p.precision == STEPS_PREC_MIXED) {
            if (cic)
                pair_table_mixed_round_kernel<0><<<g16, 512, c->table_mixed_smem_bytes, s>>>(
                    c->f_hi, c->f_lo, c->tile_hmax, c->n_pad, T, r, c->mc, c->tcf, c->d_table_f32, acc_i, acc_j);
            else
                pair_table_mixed_round_kernel<1><<<g16, 512, c->table_mixed_smem_bytes, s>>>(
                    c->f_hi, c->f_lo, c->tile_hmax, c->n_pad, T, r, c->mc, c->tcf, c->d_table_f32, acc_i, acc_j);
        } else if (c->d_table_f32) {
            if (cic)
                pair_table_round_kernel<0, 16, true><<<g16, 512, c->table_smem_bytes, s>>>(
                    c->xy, c->zm, c->hs, c->tile_hmax, c->n_pad, T, r, c->kc, c->tc, c->d_table_f32, acc_i, acc_j);
            else
                pair_table_round_kernel<1, 16, true><<<g16, 512, c->table_smem_bytes, s>>>(
                    c->xy, c->zm, c->hs, c->tile_hmax, c->n_pad, T, r, c->kc, c->tc, c->d_table_f32, acc_i, acc_j);
        } else {
            if (cic)
                pair_table_round_kernel<0, 4, false><<<g4, PAIR_THREADS, sb4, s>>>(
                    c->xy, c->zm, c->hs, c->tile_hmax, c->n_pad, T, r, c->kc, c->tc, nullptr, acc_i, acc_j);
            else
                pair_table_round_kernel<1, 4, false><<<g4, PAIR_THREADS, sb4, s>>>(
                    c->xy, c->zm, c->hs, c->tile_hmax, c->n_pad, T, r, c->kc, c->tc, nullptr, acc_i, acc_j);
        }
    }
    c->launches += last + 1;
}

// The kernel launch_pair() selects, spelled as sassmix.py spells the template instances.
void name_pair_kernel(steps_cyl_ctx *c)
{
    const bool mixed = c->p.precision == STEPS_PREC_MIXED, det = c->use_rounds,
               ord = !c->use_sym && !c->use_rounds && !c->use_slabs;
    const int nc = c->p.n_cut <= MAX_NCUT_UNROLLED ? c->p.n_cut : 0;
    char *o = c->kernel_name;
    const size_t cap = sizeof c->kernel_name;
    if (c->table_mode) {
        const int ip = c->tc.interp == STEPS_INTERP_CIC ? 0 : 1;
        if (mixed) snprintf(o, cap, "pair_table_mixed_%s_kernel<%d>", det ? "round" : "sym", ip);
        else snprintf(o, cap, "pair_table_%s_kernel<%d,%s>", det ? "round" : "sym", ip, c->d_table_f32 ? "16,true" : "4,false");
    } else if (ord) {
        if (mixed) snprintf(o, cap, "pair_mixed_kernel<%d>", nc);
        else snprintf(o, cap, "pair_fp64_kernel<%d>", nc);
    } else if (c->use_slabs) {
        snprintf(o, cap, "pair_fp64_sym_kernel<%d,false,%d,true>", nc, c->sym_tr());
    } else if (det) {
        snprintf(o, cap, "pair_%s_round_kernel<%d,%s>", mixed ? "mixed" : "fp64", nc, c->round_split > 1 ? "true" : "false");
    } else if (mixed) {
        snprintf(o, cap, "pair_mixed_sym_kernel<%d>", nc);
    } else {
        snprintf(o, cap, "pair_fp64_sym_kernel<%d,%s,%d,false>", nc, (c->p.flags & STEPS_FLAG_FAR_ORDER2) ? "true" : "false",
                 c->sym_tr());
    }
}

void launch_pair(steps_cyl_ctx *c, cudaStream_t s)
{
    if (c->table_mode && c->use_rounds) {
        launch_table_rounds(c, s);
        return;
    }
    if (c->table_mode) {
        dim3 grid(c->n_tiles / SYM_R, c->sym_chunks);
        const size_t sb4 = 4 * 3 * PAIR_THREADS * sizeof(double);
        if (c->p.precision == STEPS_PREC_MIXED) {
            dim3 g16(c->n_tiles / (4 * SYM_R), c->sym_chunks);
            if (c->tc.interp == STEPS_INTERP_CIC)
                pair_table_mixed_sym_kernel<0><<<g16, 512, c->table_mixed_smem_bytes, s>>>(
                    c->f_hi, c->f_lo, c->tile_hmax, c->n_pad, c->n_tiles, c->sym_tiles_per_chunk, c->mc,
                    c->tcf, c->d_table_f32, c->part);
            else
                pair_table_mixed_sym_kernel<1><<<g16, 512, c->table_mixed_smem_bytes, s>>>(
                    c->f_hi, c->f_lo, c->tile_hmax, c->n_pad, c->n_tiles, c->sym_tiles_per_chunk, c->mc,
                    c->tcf, c->d_table_f32, c->part);
        } else if (c->d_table_f32) {
            dim3 g16(c->n_tiles / (4 * SYM_R), c->sym_chunks);
            if (c->tc.interp == STEPS_INTERP_CIC)
                pair_table_sym_kernel<0, 16, true><<<g16, 512, c->table_smem_bytes, s>>>(
                    c->xy, c->zm, c->hs, c->tile_hmax, c->n_pad, c->n_tiles, c->sym_tiles_per_chunk, c->kc,
                    c->tc, c->d_table_f32, c->part);
            else
                pair_table_sym_kernel<1, 16, true><<<g16, 512, c->table_smem_bytes, s>>>(
                    c->xy, c->zm, c->hs, c->tile_hmax, c->n_pad, c->n_tiles, c->sym_tiles_per_chunk, c->kc,
                    c->tc, c->d_table_f32, c->part);
        } else if (c->tc.interp == STEPS_INTERP_CIC) {
            pair_table_sym_kernel<0, 4, false><<<grid, PAIR_THREADS, sb4, s>>>(
                c->xy, c->zm, c->hs, c->tile_hmax, c->n_pad, c->n_tiles, c->sym_tiles_per_chunk, c->kc, c->tc,
                nullptr, c->part);
        } else {
            pair_table_sym_kernel<1, 4, false><<<grid, PAIR_THREADS, sb4, s>>>(
                c->xy, c->zm, c->hs, c->tile_hmax, c->n_pad, c->n_tiles, c->sym_tiles_per_chunk, c->kc, c->tc,
                nullptr, c->part);
        }
        c->launches += 1;
        return;
    }
    const bool mixed = c->p.precision == STEPS_PREC_MIXED;
    switch (c->p.n_cut) {
#define CASE_NC(N)                                               \
    case N:                                                      \
        if (mixed && c->use_sym) launch_pair_mixed_sym_nc<N>(c, s); \
        else if (mixed && c->use_rounds) launch_pair_mixed_rounds_nc<N>(c, s); \
        else if (mixed) launch_pair_mixed_nc<N>(c, s);           \
        else if (c->use_sym || c->use_slabs) launch_pair_sym_nc<N>(c, s); \
        else if (c->use_rounds) launch_pair_rounds_nc<N>(c, s);  \
        else launch_pair_fp64_nc<N>(c, s);                       \
        break;
        CASE_NC(1) CASE_NC(2) CASE_NC(3) CASE_NC(4) CASE_NC(5) CASE_NC(6) CASE_NC(7) CASE_NC(8)
#undef CASE_NC
    default:
        if (mixed && c->use_sym) launch_pair_mixed_sym_nc<0>(c, s);
        else if (mixed && c->use_rounds) launch_pair_mixed_rounds_nc<0>(c, s);
        else if (mixed) launch_pair_mixed_nc<0>(c, s);
        else if (c->use_sym || c->use_slabs) launch_pair_sym_nc<0>(c, s);
        else if (c->use_rounds) launch_pair_rounds_nc<0>(c, s);
        else launch_pair_fp64_nc<0>(c, s);
    }
    c->launches += 1;
}

BgParams bg_params(const steps_cyl_ctx *c)
{
    BgParams b;
    b.R = c->p.R_sim;
    b.Lhalf = (double)c->p.n_cut * c->p.Lz;
    b.G = c->p.G;
    b.rho0 = c->p.rho0;
    b.infinite = c->p.background == STEPS_BG_INFINITE;
    b.n_nodes = c->n_nodes;
    b.nodes = c->nodes;
    return b;
}

// Eq. 9 per particle is a 361-node quadrature: below this n one warp takes a particle (see aux_kernels.cuh)
bool bg_warp_per_particle(const steps_cyl_ctx *c)
{
    return c->p.rho0 != 0.0 && c->p.background == STEPS_BG_FINITE && c->n <= 256 * 1024;
}

// One force evaluation = three launches: prestep (pack), the all-pairs kernel, poststep (reduction).  Inside a KDK
// step (kick != nullptr) the first carries b(x_n), kick 1 and the drift, the last b(x_n+1) and kick 2.
struct KdkArgs { double *vx, *vy, *vz; KickParams k1, k2; };

// Argument blocks of the two O(N) kernels, in parameter order (launched through cudaLaunchKernel so that the same
// blocks can re-parameterise the nodes of a captured graph, STEPS_FLAG_GRAPH).
struct PreVals {
    double *x, *y, *z, *vx, *vy, *vz;
    const double *gx, *gy, *gz, *m, *h;
    int n, n_pad;
    double L;
    BgParams bg;
    KickParams kp;
    double2 *xy, *zm;
    double *hs;
    float4 *f_hi, *f_lo;
    double *tile_hmax;
    DevFlags *fl;
    int *sticky;
    double *part;
    int zero_rows;
    const int *perm;
    void *args[27];
    void bind()
    {
        void *a[27] = {&x, &y, &z, &vx, &vy, &vz, &gx, &gy, &gz, &m, &h, &n, &n_pad, &L, &bg, &kp, &xy, &zm, &hs,
                       &f_hi, &f_lo, &tile_hmax, &fl, &sticky, &part, &zero_rows, &perm};
        std::memcpy(args, a, sizeof a);
    }
};
struct PostVals {
    const double *part;
    int n, n_pad, n_slabs;
    double G, L;
    DevFlags *fl_next;
    double *tile_hmax;
    double *gx, *gy, *gz;
    const double *x, *y;
    double *vx, *vy, *vz;
    BgParams bg;
    KickParams kp;
    const int *perm;
    SlabLayout sl;
    void *args[20];
    void bind()
    {
        void *a[20] = {&part, &n, &n_pad, &n_slabs, &G, &L, &fl_next, &tile_hmax, &gx, &gy, &gz, &x, &y, &vx, &vy, &vz,
                       &bg, &kp, &perm, &sl};
        std::memcpy(args, a, sizeof a);
    }
};

const void *prestep_func(bool kick, bool wpp)
{
    if (!kick) return (const void *)prestep_kernel<1, false>;
    return wpp ? (const void *)prestep_kernel<32, true> : (const void *)prestep_kernel<1, true>;
}
const void *poststep_func(bool kick, bool wpp)
{
    if (!kick) return (const void *)poststep_kernel<1, false>;
    return wpp ? (const void *)poststep_kernel<32, true> : (const void *)poststep_kernel<1, true>;
}

// launch geometry of prestep / poststep (aux_kernels.cuh: OnStep<LANES>)
int onstep_block(const steps_cyl_ctx *c, bool kick)
{
    return (kick && bg_warp_per_particle(c)) ? OnStep<32>::kThreads : OnStep<1>::kThreads;
}
int onstep_grid(const steps_cyl_ctx *c, bool kick)
{
    return c->n_pad / ((kick && bg_warp_per_particle(c)) ? OnStep<32>::kParticlesPerBlock : OnStep<1>::kParticlesPerBlock);
}

struct ForceArgs {
    double *x, *y, *z;
    const double *m, *h;
    double *gx, *gy, *gz;
    const KdkArgs *kick;
};

void fill_vals(steps_cyl_ctx *ctx, const ForceArgs &f, unsigned parity, PreVals &pre, PostVals &post)
{
    const KdkArgs *kick = f.kick;
    const KickParams none = {0.0, 0.0, 0.0};
    pre.x = f.x; pre.y = f.y; pre.z = f.z;
    pre.vx = kick ? kick->vx : nullptr; pre.vy = kick ? kick->vy : nullptr; pre.vz = kick ? kick->vz : nullptr;
    pre.gx = f.gx; pre.gy = f.gy; pre.gz = f.gz; pre.m = f.m; pre.h = f.h;
    pre.n = ctx->n; pre.n_pad = ctx->n_pad; pre.L = ctx->p.Lz;
    pre.bg = bg_params(ctx);
    pre.kp = kick ? kick->k1 : none;
    pre.xy = ctx->xy; pre.zm = ctx->zm; pre.hs = ctx->hs; pre.f_hi = ctx->f_hi; pre.f_lo = ctx->f_lo;
    pre.tile_hmax = ctx->tile_hmax;
    pre.fl = ctx->flags + (parity & 1u);
    pre.sticky = ctx->bad_h_sticky;
    pre.part = ctx->part;
    // accumulator rows the pair kernel adds into (the ordered kernels overwrite theirs)
    pre.zero_rows = ctx->use_sym ? 4 : (ctx->use_rounds ? 4 * (ctx->round_split + 1) : 0);
    post.part = ctx->part; post.n = ctx->n; post.n_pad = ctx->n_pad;
    post.n_slabs = ctx->use_sym ? 1 : (ctx->use_rounds ? ctx->round_split + 1 : ctx->n_chunks);
    post.G = ctx->p.G; post.L = ctx->p.Lz;
    post.fl_next = ctx->flags + ((parity + 1u) & 1u);
    post.tile_hmax = ctx->tile_hmax;
    post.gx = f.gx; post.gy = f.gy; post.gz = f.gz; post.x = f.x; post.y = f.y;
    post.vx = pre.vx; post.vy = pre.vy; post.vz = pre.vz;
    post.bg = pre.bg;
    post.kp = kick ? kick->k2 : none;
    pre.perm = post.perm = ctx->use_order ? ctx->perm : nullptr;
    post.sl = {0, 1, 1, 1, 1};
    if (ctx->use_slabs) {
        post.sl = {ctx->n_tiles / ctx->sym_tr(), ctx->sym_tr(), ctx->sym_tiles_per_chunk, ctx->sym_chunks, ctx->sym_split};
        pre.zero_rows = 0;
    }
}

int enqueue_force_plain(steps_cyl_ctx *ctx, const ForceArgs &f, unsigned parity, bool timed, cudaStream_t s)
{
    PreVals pre;
    PostVals post;
    fill_vals(ctx, f, parity, pre, post);
    pre.bind();
    post.bind();
    const bool wpp = bg_warp_per_particle(ctx), kick = f.kick != nullptr;
    const dim3 grid(onstep_grid(ctx, kick)), block(onstep_block(ctx, kick));
    ctx->cur_flags = pre.fl;
    CK(cudaLaunchKernel(prestep_func(kick, wpp), grid, block, pre.args, 0, s));
    ctx->launches += 1;
    if (timed) CK(cudaEventRecord(ctx->ev0, s));
    launch_pair(ctx, s);
    if (timed) CK(cudaEventRecord(ctx->ev1, s));
    ctx->ev_valid = timed;
    CK(cudaLaunchKernel(poststep_func(kick, wpp), grid, block, post.args, 0, s));
    ctx->launches += 1;
    CK(cudaGetLastError());
    return STEPS_OK;
}

// STEPS_FLAG_GRAPH: the evaluation captured once per (flag-block parity, pointer set) as a CUDA graph; later calls
// with the same pointers re-parameterise the two O(N) nodes (the kick scalars change every step) and replay it --
// one launch per step instead of three.  The all-pairs kernel is not timed in this mode (no event nodes).
void drop_graph(GraphSlot &g)
{
    if (g.exec) cudaGraphExecDestroy(g.exec);
    if (g.graph) cudaGraphDestroy(g.graph);
    g = GraphSlot();
}

int enqueue_force_graph(steps_cyl_ctx *ctx, const ForceArgs &f, unsigned parity, cudaStream_t s)
{
    GraphSlot &g = ctx->gslot[parity & 1u];
    const void *key[11] = {f.x, f.y, f.z, f.m, f.h, f.gx, f.gy, f.gz, f.kick ? f.kick->vx : nullptr,
                           f.kick ? f.kick->vy : nullptr, f.kick ? f.kick->vz : nullptr};
    const bool wpp = bg_warp_per_particle(ctx), kick = f.kick != nullptr;
    if (g.exec && std::memcmp(key, g.key, sizeof key) != 0) drop_graph(g);
    if (!g.exec) {
        const int64_t before = ctx->launches;
        // captured on the context's own stream (the caller's may be the legacy default stream, which cannot
        // capture); the graph is launched on the caller's stream
        cudaStream_t cs = ctx->own_stream;
        CK(cudaStreamBeginCapture(cs, cudaStreamCaptureModeThreadLocal));
        int rc = enqueue_force_plain(ctx, f, parity, false, cs);
        cudaGraph_t graph = nullptr;
        cudaError_t e = cudaStreamEndCapture(cs, &graph);
        if (rc != STEPS_OK || e != cudaSuccess) {
            if (graph) cudaGraphDestroy(graph);
            return rc != STEPS_OK ? rc : cuda_fail(ctx, e);
        }
        g.graph = graph;
        g.n_kernels = (int)(ctx->launches - before);
        ctx->launches = before;
        size_t n_nodes = 0;
        CK(cudaGraphGetNodes(graph, nullptr, &n_nodes));
        std::vector<cudaGraphNode_t> nodes(n_nodes);
        CK(cudaGraphGetNodes(graph, nodes.data(), &n_nodes));
        for (cudaGraphNode_t nd : nodes) {
            cudaGraphNodeType ty;
            CK(cudaGraphNodeGetType(nd, &ty));
            if (ty != cudaGraphNodeTypeKernel) continue;
            cudaKernelNodeParams kp;
            CK(cudaGraphKernelNodeGetParams(nd, &kp));
            if (kp.func == prestep_func(kick, wpp)) g.pre = nd;
            if (kp.func == poststep_func(kick, wpp)) g.post = nd;
        }
        if (!g.pre || !g.post) { drop_graph(g); return STEPS_ECUDA; }
        CK(cudaGraphInstantiate(&g.exec, graph, 0));
        std::memcpy(g.key, key, sizeof key);
    } else {
        PreVals pre;
        PostVals post;
        fill_vals(ctx, f, parity, pre, post);
        pre.bind();
        post.bind();
        cudaKernelNodeParams kp = {};
        kp.gridDim = dim3(onstep_grid(ctx, kick));
        kp.blockDim = dim3(onstep_block(ctx, kick));
        kp.func = const_cast<void *>(prestep_func(kick, wpp));
        kp.kernelParams = pre.args;
        CK(cudaGraphExecKernelNodeSetParams(g.exec, g.pre, &kp));
        kp.func = const_cast<void *>(poststep_func(kick, wpp));
        kp.kernelParams = post.args;
        CK(cudaGraphExecKernelNodeSetParams(g.exec, g.post, &kp));
    }
    CK(cudaGraphLaunch(g.exec, s));
    ctx->launches += g.n_kernels;
    ctx->ev_valid = false;
    return STEPS_OK;
}

// perm <- the particles' order along a Morton curve through their current positions (order_kernels.cuh): key
// generation, a bitonic sort of the (key, index) words -- chunks of 1024 in shared memory, larger strides one pass
// per launch -- and the extraction of the indices.  O(N log^2 N), a few ms at N = 4 M, once per kReorderEvery calls.
int enqueue_reorder(steps_cyl_ctx *ctx, const double *x, const double *y, const double *z, cudaStream_t s)
{
    constexpr int T = 512, CHUNK = 2 * T;
    const int tb = 256, np2 = ctx->n_pow2;
    CK(cudaMemsetAsync(ctx->rmax_bits, 0, sizeof(unsigned long long), s));
    extent_kernel<<<(ctx->n + tb - 1) / tb, tb, 0, s>>>(x, y, ctx->n, ctx->rmax_bits);
    order_key_kernel<<<(np2 + tb - 1) / tb, tb, 0, s>>>(x, y, z, ctx->n, np2, ctx->p.Lz, ctx->rmax_bits,
                                                       ctx->order_keys);
    bitonic_chunk_kernel<T><<<np2 / CHUNK, T, 0, s>>>(ctx->order_keys, 2, CHUNK);
    ctx->launches += 3;
    for (long long k = 2LL * CHUNK; k <= np2; k <<= 1) {
        for (long long j = k >> 1; j >= CHUNK; j >>= 1) {
            bitonic_pass_kernel<<<(np2 / 2 + tb - 1) / tb, tb, 0, s>>>(ctx->order_keys, np2, (int)j, (int)k);
            ctx->launches += 1;
        }
        bitonic_chunk_kernel<T><<<np2 / CHUNK, T, 0, s>>>(ctx->order_keys, (int)k, (int)k);
        ctx->launches += 1;
    }
    order_perm_kernel<<<(ctx->n + tb - 1) / tb, tb, 0, s>>>(ctx->order_keys, ctx->n, ctx->perm);
    ctx->launches += 1;
    CK(cudaGetLastError());
    return STEPS_OK;
}

int enqueue_force(steps_cyl_ctx *ctx, double *x, double *y, double *z, const double *m, const double *h,
                  double *gx, double *gy, double *gz, const KdkArgs *kick, cudaStream_t s)
{
    const ForceArgs f = {x, y, z, m, h, gx, gy, gz, kick};
    const unsigned parity = ctx->eval_count & 1u;      // which of the two flag blocks this evaluation uses
    // the ordering is a locality hint: refreshed now and then (inside a replayed graph: taken once, before capture)
    if (ctx->use_order && (ctx->eval_count == 0 ||
                           (!(ctx->p.flags & STEPS_FLAG_GRAPH) && ctx->eval_count % kReorderEvery == 0))) {
        int rc = enqueue_reorder(ctx, x, y, z, s);
        if (rc != STEPS_OK) return rc;
    }
    ctx->eval_count += 1;
    if (ctx->p.flags & STEPS_FLAG_GRAPH) return enqueue_force_graph(ctx, f, parity, s);
    return enqueue_force_plain(ctx, f, parity, true, s);
}

int enqueue_background(steps_cyl_ctx *ctx, const double *x, const double *y, double *bx, double *by,
                       cudaStream_t s)
{
    const int tb = 128;
    const BgParams bg = bg_params(ctx);
    if (bg_warp_per_particle(ctx))
        background_kernel<32><<<(ctx->n * 32 + tb - 1) / tb, tb, 0, s>>>(x, y, ctx->n, bg, bx, by);
    else
        background_kernel<1><<<(ctx->n + tb - 1) / tb, tb, 0, s>>>(x, y, ctx->n, bg, bx, by);
    ctx->launches += 1;
    CK(cudaGetLastError());
    return STEPS_OK;
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// steps_cyl_accel_noalloc: one force evaluation (fp64, image mode, default symmetric kernel) that allocates
// NOTHING -- for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses
// that forbid it).  Everything steps_cyl_init would allocate for such an evaluation lives in ONE file-scope device
// array of a fixed, modest size (every GPU that loads the library holds it until the process exits):
//     xy[16 B] zm[16 B] hs[8 B] part[4 x 8 B] per particle slot, tile_hmax[8 B] per 128 slots, three flag blocks.
// In HOST code the array's name is a host-side stand-in, not a device address, so its address is taken once per
// device with cudaGetSymbolAddress (that device current) and only that pointer is ever handed to a kernel.
// The array is shared by every call and keeps the last call's contents: what must start at zero (the flag blocks)
// is cleared on the stream at the start of every call, the accumulator rows by prestep_kernel as in the ordinary path.
constexpr int64_t kNoallocMaxN = STEPS_CYL_NOALLOC_MAX_N;
static_assert(kNoallocMaxN % (SYM_R * PAIR_THREADS) == 0, "the limit is a whole number of CTA target groups");
constexpr size_t kNoallocOffXy = 0;
constexpr size_t kNoallocOffZm = kNoallocOffXy + sizeof(double2) * (size_t)kNoallocMaxN;
constexpr size_t kNoallocOffHs = kNoallocOffZm + sizeof(double2) * (size_t)kNoallocMaxN;
constexpr size_t kNoallocOffPart = kNoallocOffHs + sizeof(double) * (size_t)kNoallocMaxN;
constexpr size_t kNoallocOffHmax = kNoallocOffPart + 4 * sizeof(double) * (size_t)kNoallocMaxN;
constexpr size_t kNoallocOffFlags = kNoallocOffHmax + sizeof(double) * (size_t)(kNoallocMaxN / PAIR_THREADS);
constexpr size_t kNoallocBytes = ((kNoallocOffFlags + 3 * sizeof(DevFlags) + 255) / 256) * 256;
static_assert(kNoallocOffZm % 256 == 0 && kNoallocOffHs % 256 == 0 && kNoallocOffPart % 256 == 0 &&
              kNoallocOffHmax % 256 == 0 && kNoallocOffFlags % 256 == 0, "every sub-array starts 256-byte aligned");

static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoallocBytes];      // 2.25 MiB per GPU

namespace {

struct NoallocDevice {
    unsigned char *scratch = nullptr;      // DEVICE address of g_noalloc_scratch on this device
    int sm_count = 0;
    bool ready = false;
};
constexpr int kNoallocMaxDevices = 64;
NoallocDevice g_noalloc_dev[kNoallocMaxDevices];
std::mutex g_noalloc_mu;

// Set-up, once per device, with that device current: the device address of the scratch array and the SM count.
// Neither call allocates.  Returns cudaSuccess or the failing call's error.
cudaError_t noalloc_setup(int dev, NoallocDevice **out)
{
    std::lock_guard<std::mutex> lock(g_noalloc_mu);
    NoallocDevice &d = g_noalloc_dev[dev];
    if (!d.ready) {
        void *ptr = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&ptr, g_noalloc_scratch);
        if (e != cudaSuccess) return e;
        int sms = 0;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return e;
        if (ptr == nullptr || sms <= 0) return cudaErrorUnknown;
        d.scratch = static_cast<unsigned char *>(ptr);
        d.sm_count = sms;
        d.ready = true;
    }
    *out = &d;
    return cudaSuccess;
}

}  // namespace

extern "C" {

int steps_cyl_init(const steps_cyl_params *p, steps_cyl_ctx **out)
{
    if (!p || !out) return STEPS_EINVAL;
    *out = nullptr;
    // upper limit: the symmetric kernels put source chunks of <= 64 tiles on gridDim.y (<= 65535)
    if (p->n < 1 || p->n > STEPS_CYL_MAX_N) return STEPS_EINVAL;
    if (!(p->Lz > 0.0) || !std::isfinite(p->Lz) || !std::isfinite(p->G)) return STEPS_EINVAL;
    if (p->n_cut < 1 || p->n_cut > 1000000) return STEPS_EINVAL;
    if (p->periodic_mode != STEPS_PERIODIC_IMAGES && p->periodic_mode != STEPS_PERIODIC_EWALD_TABLE)
        return STEPS_EINVAL;
    if (p->precision != STEPS_PREC_FP64 && p->precision != STEPS_PREC_MIXED) return STEPS_EINVAL;
    if (p->background != STEPS_BG_FINITE && p->background != STEPS_BG_INFINITE) return STEPS_EINVAL;
    if ((p->flags & ~(STEPS_FLAG_DETERMINISTIC | STEPS_FLAG_FAR_ORDER2 | STEPS_FLAG_ORDERED_PAIRS | STEPS_FLAG_GRAPH)) != 0 ||
        p->device < 0)
        return STEPS_EINVAL;
    if (!std::isfinite(p->rho0) || !std::isfinite(p->R_sim)) return STEPS_EINVAL;
    if (p->rho0 != 0.0 && p->background == STEPS_BG_FINITE && !(p->R_sim > 0.0)) return STEPS_EINVAL;
    if (p->tab_fp32 != 0 && p->tab_fp32 != 1) return STEPS_EINVAL;
    steps_cyl_params pp = *p;                      // table parameters with defaults filled in
    if (p->periodic_mode == STEPS_PERIODIC_EWALD_TABLE) {
        if (pp.ew_nmax == 0) pp.ew_nmax = 5;
        if (pp.ew_mmax == 0) pp.ew_mmax = 12;
        if (pp.ew_alpha == 0.0) pp.ew_alpha = 2.0 / p->Lz;
        if (pp.tab_nrho == 0) pp.tab_nrho = 144;
        if (pp.tab_nz == 0) pp.tab_nz = 128;
        if (pp.tab_rho_max == 0.0) pp.tab_rho_max = 5.0 * p->Lz;
        if (pp.ew_nmax < 0 || pp.ew_mmax < 0 || !(pp.ew_alpha > 0.0) || !std::isfinite(pp.ew_alpha) ||
            pp.tab_nrho < 2 || pp.tab_nz < 2 || pp.tab_nrho > 16384 || pp.tab_nz > 16384 ||
            !(pp.tab_rho_max > 0.0) || !std::isfinite(pp.tab_rho_max) ||
            (pp.interp != STEPS_INTERP_CIC && pp.interp != STEPS_INTERP_TSC))
            return STEPS_EINVAL;
        if (p->flags & STEPS_FLAG_ORDERED_PAIRS) return STEPS_EUNSUPPORTED;
        if (p->precision == STEPS_PREC_MIXED) pp.tab_fp32 = 1;      // mixed mode always uses the float table
    }

    steps_cyl_ctx *ctx = new (std::nothrow) steps_cyl_ctx();
    if (!ctx) return STEPS_ENOMEM;
    ctx->cuda_msg[0] = 0;
    ctx->p = pp;
    int rc = STEPS_OK;
    auto fail = [&](int code) { steps_cyl_destroy(ctx); return code; };

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || p->device >= ndev) { delete ctx; return STEPS_ECUDA; }
    DeviceGuard dev_guard(p->device);               // the caller's current device is restored on return
    if (dev_guard.err != cudaSuccess) { delete ctx; return STEPS_ECUDA; }
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, p->device) != cudaSuccess) { delete ctx; return STEPS_ECUDA; }
    ctx->sm_count = prop.multiProcessorCount;

    ctx->n = (int)p->n;
    // a multiple of SYM_R tiles: the symmetric kernel's CTAs own SYM_R target tiles each
    {
        const int tile_group = (pp.periodic_mode == STEPS_PERIODIC_EWALD_TABLE && pp.tab_fp32) ? 4 * SYM_R : SYM_R;
        ctx->n_tiles = tile_group * ((ctx->n + tile_group * PAIR_THREADS - 1) / (tile_group * PAIR_THREADS));
    }
    ctx->n_pad = ctx->n_tiles * PAIR_THREADS;
    choose_chunks(ctx);
    ctx->use_sym = !(p->flags & (STEPS_FLAG_DETERMINISTIC | STEPS_FLAG_ORDERED_PAIRS));
    ctx->sym_small = ctx->use_sym && ctx->sym_split > 1 && pp.precision == STEPS_PREC_FP64 &&
                     pp.periodic_mode == STEPS_PERIODIC_IMAGES;
    ctx->use_rounds = (p->flags & STEPS_FLAG_DETERMINISTIC) && !(p->flags & STEPS_FLAG_ORDERED_PAIRS);
    // DETERMINISTIC, fp64 image mode, N <= 131072: the symmetric kernel with single-writer slabs instead of atomics
    // (n_tiles / TR + chunks x split slabs of 24 B x n_pad: 1.7 GB at the limit); above, and in the other modes, the
    // round-scheduled kernels (within 3 % of the atomic ones from N ~ 260 000 up)
    if (ctx->use_rounds && pp.precision == STEPS_PREC_FP64 && pp.periodic_mode == STEPS_PERIODIC_IMAGES &&
        ctx->n <= 131072) {
        ctx->use_rounds = false;
        ctx->use_slabs = true;
        ctx->sym_small = ctx->sym_split > 1;
    }

    // small N: a round has n_tiles / 2 items of four warps; below ~1.5 warps per scheduler (measured break-even:
    // N ~ 260 000) split the items by source sub-tile
    if (ctx->use_rounds && pp.periodic_mode == STEPS_PERIODIC_IMAGES && ctx->n_tiles / SYM_R < 6 * ctx->sm_count)
        ctx->round_split = PAIR_THREADS / 32;

    const double L = p->Lz;
    ctx->kc.L = L;
    ctx->kc.halfL = 0.5 * L;
    {
        uint64_t bits;
        std::memcpy(&bits, &L, 8);
        ctx->kc.L_hi = (int)(bits >> 32);
        ctx->kc.L_lo = (int)(bits & 0xffffffffu);
        const double hl = 0.5 * L;
        std::memcpy(&bits, &hl, 8);
        ctx->kc.halfL_hi = (int)(bits >> 32);
    }
    ctx->mc.Lh = (float)L;
    ctx->mc.Ll = (float)(L - (double)ctx->mc.Lh);
    ctx->mc.halfL = (float)(0.5 * L);
    // SIMPLE ring passes of the mixed kernel (pair_mixed_sym.cuh: pass_is_simple): box distance d >= c / 8 and
    // d >= (source box extent) / 2 -- measured at configs 1-3: parity as without them, 87 % of the passes at N = 1 M
    ctx->mc.simple_ratio2 = 64.0f;
    ctx->mc.simple_ext2 = 0.25f;
    for (int n = 0; n <= MAX_NCUT_TABLE; ++n) {
        const double nL = (double)n * L;
        ctx->kc.c2nL[n] = 2.0 * nL;
        ctx->kc.n2L2[n] = nL * nL;
        ctx->kc.dn[n] = (double)n;
        ctx->mc.c2nL[n] = (float)(2.0 * nL);
        ctx->mc.n2L2[n] = (float)(nL * nL);
        ctx->mc.dn[n] = (float)n;
    }

    auto A = [&](cudaError_t e) { if (e != cudaSuccess && rc == STEPS_OK) { rc = (e == cudaErrorMemoryAllocation) ? STEPS_ENOMEM : STEPS_ECUDA; cuda_fail(ctx, e); } };
    const size_t np = (size_t)ctx->n_pad;
    A(dev_alloc(&ctx->xy, np));
    A(dev_alloc(&ctx->zm, np));
    A(dev_alloc(&ctx->hs, np));
    A(dev_alloc(&ctx->tile_hmax, (size_t)ctx->n_tiles));
    if (rc == STEPS_OK) A(cudaMemset(ctx->tile_hmax, 0, (size_t)ctx->n_tiles * sizeof(double)));
    A(dev_alloc(&ctx->f_hi, np));
    A(dev_alloc(&ctx->f_lo, np));
    {
        size_t part_doubles = np * 4 * (size_t)std::max(ctx->n_chunks, 5);
        if (ctx->use_slabs)
            part_doubles = std::max(part_doubles, np * 3 * ((size_t)ctx->n_tiles / ctx->sym_tr() +
                                                           (size_t)ctx->sym_chunks * ctx->sym_split));
        A(dev_alloc(&ctx->part, part_doubles));
    }
    A(dev_alloc(&ctx->pass_stats, 2));
    if (rc == STEPS_OK) A(cudaMemset(ctx->pass_stats, 0, 2 * sizeof(unsigned long long)));
    A(dev_alloc(&ctx->flags, 3));                   // two alternating blocks + the sticky h <= 0 word
    A(dev_alloc(&ctx->peak_out, 1));
    A(cudaStreamCreateWithFlags(&ctx->own_stream, cudaStreamNonBlocking));
    A(cudaEventCreate(&ctx->ev0));
    A(cudaEventCreate(&ctx->ev1));
    if (rc != STEPS_OK) return fail(rc);

    if (p->rho0 != 0.0 && p->background == STEPS_BG_FINITE) {
        std::vector<QuadNode> v = make_nodes(p->R_sim);
        ctx->n_nodes = (int)v.size();
        A(dev_alloc(&ctx->nodes, v.size()));
        if (rc == STEPS_OK) A(cudaMemcpy(ctx->nodes, v.data(), v.size() * sizeof(QuadNode), cudaMemcpyHostToDevice));
        if (rc != STEPS_OK) return fail(rc);
    }
    if (pp.periodic_mode == STEPS_PERIODIC_EWALD_TABLE) {
        ctx->table_mode = true;
        const size_t nodes = (size_t)pp.tab_nrho * pp.tab_nz;
        std::vector<double> D(nodes * 2);
        build_ewald_table(pp.Lz, pp.ew_alpha, pp.ew_nmax, pp.ew_mmax, pp.tab_nrho, pp.tab_nz,
                          pp.tab_rho_max, D.data());
        A(dev_alloc(&ctx->d_table, nodes));
        if (rc == STEPS_OK) A(cudaMemcpy(ctx->d_table, D.data(), nodes * sizeof(double2), cudaMemcpyHostToDevice));
        {
            // haloed copy for the double-precision TSC stencil: nodes outside the grid by the symmetries of D
            // (D_rho odd in rho / even in z, D_z even in rho / odd in z about z = 0 and z = L/2; beyond the last
            // radial node the last node) -- the rules of table_node() / stage_table_halo(), applied once here
            const int nr = pp.tab_nrho, nzz = pp.tab_nz, nzs = nzz + 2;
            std::vector<double> H((size_t)(nr + 2) * nzs * 2);
            for (int i = -1; i <= nr; ++i)
                for (int j = -1; j <= nzz; ++j) {
                    int ii = i, jj = j;
                    double sr = 1.0, sz = 1.0;
                    if (ii < 0) { ii = -ii; sr = -1.0; }
                    if (ii > nr - 1) ii = nr - 1;
                    if (jj < 0) { jj = -jj; sz = -1.0; }
                    if (jj > nzz - 1) { jj = 2 * (nzz - 1) - jj; sz = -sz; }
                    const size_t src = ((size_t)ii * nzz + jj) * 2, dst = ((size_t)(i + 1) * nzs + (j + 1)) * 2;
                    H[dst] = sr * D[src];
                    H[dst + 1] = sz * D[src + 1];
                }
            A(dev_alloc(&ctx->d_table_halo, H.size() / 2));
            if (rc == STEPS_OK) A(cudaMemcpy(ctx->d_table_halo, H.data(), H.size() * sizeof(double), cudaMemcpyHostToDevice));
        }
        if (rc != STEPS_OK) return fail(rc);
        if (pp.tab_fp32) {
            // table rounded to float and staged in shared memory by a 512-thread CTA per SM
            const size_t halo_bytes = table_halo_nodes(pp.tab_nrho, pp.tab_nz) * sizeof(float2);
            ctx->table_smem_bytes = 16 * 3 * PAIR_THREADS * sizeof(double) + halo_bytes;
            // static shared memory: one source tile (four, one per quad, in the round-scheduled kernels)
            if (ctx->table_smem_bytes + (ctx->use_rounds ? 4 : 1) * sizeof(SymSrc) * PAIR_THREADS >
                (size_t)prop.sharedMemPerBlockOptin)
                return fail(STEPS_EUNSUPPORTED);
            std::vector<float> Df(nodes * 2);
            for (size_t q = 0; q < nodes * 2; ++q) Df[q] = (float)D[q];
            A(dev_alloc(&ctx->d_table_f32, nodes));
            if (rc == STEPS_OK) A(cudaMemcpy(ctx->d_table_f32, Df.data(), nodes * sizeof(float2), cudaMemcpyHostToDevice));
            ctx->table_mixed_smem_bytes = 16 * 3 * PAIR_THREADS * sizeof(float) + halo_bytes;
            ctx->tcf.nrho = pp.tab_nrho;
            ctx->tcf.nz = pp.tab_nz;
            ctx->tcf.rho_max2 = (float)(pp.tab_rho_max * pp.tab_rho_max);
            ctx->tcf.inv_drho = (float)((double)(pp.tab_nrho - 1) / pp.tab_rho_max);
            ctx->tcf.inv_dz = (float)((double)(pp.tab_nz - 1) / (0.5 * pp.Lz));
            ctx->tcf.two_over_L = (float)(2.0 / pp.Lz);
            A(raise_table_smem_limits(ctx->table_smem_bytes, ctx->table_mixed_smem_bytes));
            if (rc != STEPS_OK) return fail(rc);
        }
        ctx->tc.D = ctx->d_table;
        ctx->tc.Dh = ctx->d_table_halo;
        ctx->tc.nrho = pp.tab_nrho;
        ctx->tc.nz = pp.tab_nz;
        ctx->tc.interp = pp.interp;
        ctx->tc.rho_max2 = pp.tab_rho_max * pp.tab_rho_max;
        ctx->tc.inv_drho = (double)(pp.tab_nrho - 1) / pp.tab_rho_max;
        ctx->tc.inv_dz = (double)(pp.tab_nz - 1) / (0.5 * pp.Lz);
        ctx->tc.two_over_L = 2.0 / pp.Lz;
        // spatially ordered packed arrays: the gathers of a warp then fall in one patch of the table
        ctx->use_order = true;
        ctx->n_pow2 = 1024;
        while (ctx->n_pow2 < ctx->n) ctx->n_pow2 <<= 1;
        A(dev_alloc(&ctx->perm, (size_t)ctx->n));
        A(dev_alloc(&ctx->order_keys, (size_t)ctx->n_pow2));
        A(dev_alloc(&ctx->rmax_bits, 1));
        if (rc != STEPS_OK) return fail(rc);
    }
    if (!ctx->use_order && ctx->use_sym && pp.precision == STEPS_PREC_MIXED && ctx->n >= 16384) {
        // mixed image-sum kernel: with spatially ordered packed arrays most ring passes are between far-apart groups
        // and take the SIMPLE form (pair_mixed_sym.cuh: pass_is_simple); at small n the groups are too extended for
        // that and the sort would only cost latency.  The fp64 image-sum kernel stays in caller order: measured, the
        // analogous far-pass form gains nothing there (FP64-issue bound either way), and summing the sources in
        // spatial order costs cancellation accuracy (1e-14 -> 1e-12 for core particles, kappa ~ 1e3).
        ctx->use_order = true;
        ctx->n_pow2 = 1024;
        while (ctx->n_pow2 < ctx->n) ctx->n_pow2 <<= 1;
        A(dev_alloc(&ctx->perm, (size_t)ctx->n));
        A(dev_alloc(&ctx->order_keys, (size_t)ctx->n_pow2));
        A(dev_alloc(&ctx->rmax_bits, 1));
    }
    A(cudaMemset(ctx->flags, 0, 3 * sizeof(DevFlags)));
    if (rc != STEPS_OK) return fail(rc);
    ctx->bad_h_sticky = reinterpret_cast<int *>(ctx->flags + 2);
    ctx->cur_flags = ctx->flags;
    name_pair_kernel(ctx);
    *out = ctx;
    return STEPS_OK;
}

void steps_cyl_destroy(steps_cyl_ctx *c)
{
    if (!c) return;
    for (GraphSlot &g : c->gslot) {
        if (g.exec) cudaGraphExecDestroy(g.exec);
        if (g.graph) cudaGraphDestroy(g.graph);
    }
    cudaFree(c->xy); cudaFree(c->zm); cudaFree(c->hs); cudaFree(c->tile_hmax); cudaFree(c->f_hi); cudaFree(c->f_lo);
    cudaFree(c->part); cudaFree(c->flags); cudaFree(c->perm); cudaFree(c->order_keys); cudaFree(c->rmax_bits); cudaFree(c->pass_stats); cudaFree(c->nodes); cudaFree(c->d_table); cudaFree(c->d_table_halo); cudaFree(c->d_table_f32);
    cudaFree(c->host_io); cudaFree(c->peak_out);
    if (c->ev0) cudaEventDestroy(c->ev0);
    if (c->ev1) cudaEventDestroy(c->ev1);
    if (c->own_stream) cudaStreamDestroy(c->own_stream);
    delete c;
}

int steps_cyl_accel(steps_cyl_ctx *ctx, const double *x, const double *y, const double *z,
                    const double *m, const double *h, double *gx, double *gy, double *gz,
                    void *cuda_stream)
{
    if (!ctx || !x || !y || !z || !m || !h || !gx || !gy || !gz) return STEPS_EINVAL;
    ON_DEVICE(ctx);
    return enqueue_force(ctx, const_cast<double *>(x), const_cast<double *>(y), const_cast<double *>(z), m, h,
                         gx, gy, gz, nullptr, (cudaStream_t)cuda_stream);
}

int steps_cyl_check(steps_cyl_ctx *ctx, void *cuda_stream)
{
    if (!ctx) return STEPS_EINVAL;
    ON_DEVICE(ctx);
    CK(cudaStreamSynchronize((cudaStream_t)cuda_stream));
    int bad = 0;
    CK(cudaMemcpy(&bad, ctx->bad_h_sticky, sizeof bad, cudaMemcpyDeviceToHost));
    if (bad) CK(cudaMemset(ctx->bad_h_sticky, 0, sizeof bad));          // reported once, then cleared
    CK(cudaGetLastError());
    return bad ? STEPS_ESOFT : STEPS_OK;
}

int steps_cyl_accel_host(steps_cyl_ctx *ctx, const double *x, const double *y, const double *z,
                         const double *m, const double *h, double *gx, double *gy, double *gz)
{
    if (!ctx || !x || !y || !z || !m || !h || !gx || !gy || !gz) return STEPS_EINVAL;
    ON_DEVICE(ctx);
    const size_t n = (size_t)ctx->n, B = n * sizeof(double);
    if (!ctx->host_io) {
        cudaError_t e = dev_alloc(&ctx->host_io, 11 * n);
        if (e != cudaSuccess) { cuda_fail(ctx, e); return e == cudaErrorMemoryAllocation ? STEPS_ENOMEM : STEPS_ECUDA; }
    }
    cudaStream_t s = ctx->own_stream;
    double *d = ctx->host_io;
    const double *src[5] = {x, y, z, m, h};
    for (int k = 0; k < 5; ++k) CK(cudaMemcpyAsync(d + k * n, src[k], B, cudaMemcpyHostToDevice, s));
    int rc = enqueue_force(ctx, d, d + n, d + 2 * n, d + 3 * n, d + 4 * n, d + 5 * n, d + 6 * n, d + 7 * n, nullptr, s);
    if (rc != STEPS_OK) return rc;
    double *dst[3] = {gx, gy, gz};
    for (int k = 0; k < 3; ++k) CK(cudaMemcpyAsync(dst[k], d + (5 + k) * n, B, cudaMemcpyDeviceToHost, s));
    return steps_cyl_check(ctx, (void *)s);
}

int steps_cyl_background(steps_cyl_ctx *ctx, const double *x, const double *y, double *bx, double *by,
                         void *cuda_stream)
{
    if (!ctx || !x || !y || !bx || !by) return STEPS_EINVAL;
    ON_DEVICE(ctx);
    return enqueue_background(ctx, x, y, bx, by, (cudaStream_t)cuda_stream);
}

int steps_cyl_kdk_step(steps_cyl_ctx *ctx, double *x, double *y, double *z, double *vx, double *vy,
                       double *vz, const double *m, const double *h, double *gx, double *gy,
                       double *gz, double a_n, double H_n, double a_np1, double H_np1, double dt,
                       void *cuda_stream)
{
    if (!ctx || !x || !y || !z || !vx || !vy || !vz || !m || !h || !gx || !gy || !gz) return STEPS_EINVAL;
    if (!(a_n > 0.0) || !(a_np1 > 0.0) || !std::isfinite(dt)) return STEPS_EINVAL;
    ON_DEVICE(ctx);
    KdkArgs k;
    k.vx = vx; k.vy = vy; k.vz = vz;
    k.k1 = {1.0 / (a_n * a_n * a_n), H_n, dt};
    k.k2 = {1.0 / (a_np1 * a_np1 * a_np1), H_np1, dt};
    // b(x_n) is recomputed inside prestep_kernel: the caller may have moved the particles since the last step
    return enqueue_force(ctx, x, y, z, m, h, gx, gy, gz, &k, (cudaStream_t)cuda_stream);
}

int steps_cyl_kdk_step_host(steps_cyl_ctx *ctx, double *x, double *y, double *z, double *vx,
                            double *vy, double *vz, const double *m, const double *h, double *gx,
                            double *gy, double *gz, double a_n, double H_n, double a_np1,
                            double H_np1, double dt)
{
    if (!ctx || !x || !y || !z || !vx || !vy || !vz || !m || !h || !gx || !gy || !gz) return STEPS_EINVAL;
    ON_DEVICE(ctx);
    const size_t n = (size_t)ctx->n, B = n * sizeof(double);
    if (!ctx->host_io) {
        cudaError_t e = dev_alloc(&ctx->host_io, 11 * n);
        if (e != cudaSuccess) { cuda_fail(ctx, e); return e == cudaErrorMemoryAllocation ? STEPS_ENOMEM : STEPS_ECUDA; }
    }
    cudaStream_t s = ctx->own_stream;
    double *d = ctx->host_io;
    const double *src[11] = {x, y, z, vx, vy, vz, m, h, gx, gy, gz};
    for (int k = 0; k < 11; ++k) CK(cudaMemcpyAsync(d + k * n, src[k], B, cudaMemcpyHostToDevice, s));
    int rc = steps_cyl_kdk_step(ctx, d, d + n, d + 2 * n, d + 3 * n, d + 4 * n, d + 5 * n, d + 6 * n,
                                d + 7 * n, d + 8 * n, d + 9 * n, d + 10 * n, a_n, H_n, a_np1, H_np1,
                                dt, (void *)s);
    if (rc != STEPS_OK) return rc;
    double *dst[11] = {x, y, z, vx, vy, vz, nullptr, nullptr, gx, gy, gz};
    for (int k = 0; k < 11; ++k)
        if (dst[k]) CK(cudaMemcpyAsync(dst[k], d + k * n, B, cudaMemcpyDeviceToHost, s));
    return steps_cyl_check(ctx, (void *)s);
}

static double hubble_of_a(double a, double H0, double Om, double Or, double Ok, double OL)
{
    const double ia = 1.0 / a;
    return H0 * std::sqrt(((Or * ia + Om) * ia + Ok) * ia * ia + OL);
}

int steps_cyl_friedmann_step(double a, double dt, double H0, double Om, double Or, double Ok,
                             double OL, double *a_next, double *H_next)
{
    if (!a_next || !H_next || !(a > 0.0)) return STEPS_EINVAL;
    auto f = [&](double s) { return s * hubble_of_a(s, H0, Om, Or, Ok, OL); };
    const double k1 = f(a);
    const double k2 = f(a + 0.5 * dt * k1);
    const double k3 = f(a + 0.5 * dt * k2);
    const double k4 = f(a + dt * k3);
    const double an = a + dt / 6.0 * (k1 + 2.0 * (k2 + k3) + k4);
    *a_next = an;
    *H_next = hubble_of_a(an, H0, Om, Or, Ok, OL);
    return STEPS_OK;
}

// Eq. 19-20 in closed form: int_1^a (1 + w0 + wa (1 - a'))/a' da' = (1 + w0 + wa) ln a - wa (a - 1).
static double hubble_cpl_of_a(double a, double H0, double Om, double Or, double Ok, double ODE,
                              double w0, double wa)
{
    const double ia = 1.0 / a;
    const double de = ODE * std::pow(a, -3.0 * (1.0 + w0 + wa)) * std::exp(3.0 * wa * (a - 1.0));
    return H0 * std::sqrt(((Or * ia + Om) * ia + Ok) * ia * ia + de);
}

int steps_cyl_friedmann_step_cpl(double a, double dt, double H0, double Om, double Or, double Ok,
                                 double ODE, double w0, double wa, double *a_next, double *H_next)
{
    if (!a_next || !H_next || !(a > 0.0)) return STEPS_EINVAL;
    auto f = [&](double s) { return s * hubble_cpl_of_a(s, H0, Om, Or, Ok, ODE, w0, wa); };
    const double k1 = f(a);
    const double k2 = f(a + 0.5 * dt * k1);
    const double k3 = f(a + 0.5 * dt * k2);
    const double k4 = f(a + dt * k3);
    const double an = a + dt / 6.0 * (k1 + 2.0 * (k2 + k3) + k4);
    *a_next = an;
    *H_next = hubble_cpl_of_a(an, H0, Om, Or, Ok, ODE, w0, wa);
    return STEPS_OK;
}

int steps_cyl_ewald_table(double Lz, double alpha, int32_t nmax, int32_t mmax, int32_t nrho,
                          int32_t nz, double rho_max, double *out)
{
    if (!out || !(Lz > 0.0) || !(alpha > 0.0) || nrho < 2 || nz < 2 || nmax < 0 || mmax < 0 ||
        !(rho_max > 0.0))
        return STEPS_EINVAL;
    build_ewald_table(Lz, alpha, nmax, mmax, nrho, nz, rho_max, out);
    return STEPS_OK;
}

int steps_cyl_fp64_peak(steps_cyl_ctx *ctx, double ms, double *dfma_per_s)
{
    if (!ctx || !dfma_per_s || !(ms > 0.0)) return STEPS_EINVAL;
    ON_DEVICE(ctx);
    cudaStream_t s = ctx->own_stream;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    cudaError_t err = cudaEventCreate(&e0);
    if (err == cudaSuccess) err = cudaEventCreate(&e1);
    const int blocks = ctx->sm_count * 8, threads = 256;
    int iters = 4096;
    double best = 0.0;
    for (int rep = 0; rep < 4 && err == cudaSuccess; ++rep) {
        float t = 0.f;
        err = cudaEventRecord(e0, s);
        if (err == cudaSuccess) {
            dfma_peak_kernel<<<blocks, threads, 0, s>>>(ctx->peak_out, iters, 0.999999, 1.0e-3);
            err = cudaEventRecord(e1, s);
        }
        if (err == cudaSuccess) err = cudaEventSynchronize(e1);
        if (err == cudaSuccess) err = cudaEventElapsedTime(&t, e0, e1);
        if (err != cudaSuccess) break;
        ctx->launches += 1;
        const double rate = (double)blocks * threads * 16.0 * iters / (t * 1e-3);
        if (rep > 0) best = std::max(best, rate);
        // aim the next repetition at `ms`
        const double scale = ms / std::max((double)t, 1e-3);
        iters = (int)std::min(4.0e6, std::max(1024.0, iters * scale));
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (err != cudaSuccess) return cuda_fail(ctx, err);
    *dfma_per_s = best;
    return STEPS_OK;
}

int steps_cyl_last_pair_kernel_ms(steps_cyl_ctx *ctx, float *ms)
{
    if (!ctx || !ms || !ctx->ev_valid) return STEPS_EINVAL;
    CK(cudaEventSynchronize(ctx->ev1));
    CK(cudaEventElapsedTime(ms, ctx->ev0, ctx->ev1));
    return STEPS_OK;
}

int steps_cyl_accel_noalloc(int64_t n, double Lz, double G, int32_t n_cut, const double *x, const double *y,
                            const double *z, const double *m, const double *h, double *gx, double *gy,
                            double *gz, void *cuda_stream)
{
    if (!x || !y || !z || !m || !h || !gx || !gy || !gz) return STEPS_EINVAL;
    if (n < 1 || !(Lz > 0.0) || !std::isfinite(Lz) || !std::isfinite(G) || n_cut < 1 || n_cut > 1000000)
        return STEPS_EINVAL;
    if (n > kNoallocMaxN) return STEPS_ETOOBIG;          // before any CUDA call: the scratch array is fixed
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kNoallocMaxDevices) return STEPS_ECUDA;
    NoallocDevice *nd = nullptr;
    if (noalloc_setup(dev, &nd) != cudaSuccess) return STEPS_ECUDA;

    // A throw-away context on the host stack whose scratch pointers all lie inside the static array; the launches
    // are the ordinary ones (prestep_kernel, pair_fp64_sym_kernel, poststep_kernel through enqueue_force_plain).
    steps_cyl_ctx c;
    steps_cyl_ctx *ctx = &c;
    c.cuda_msg[0] = 0;
    c.kernel_name[0] = 0;
    std::memset(&c.p, 0, sizeof c.p);
    c.p.n = n; c.p.Lz = Lz; c.p.G = G; c.p.n_cut = n_cut; c.p.device = dev;
    c.p.periodic_mode = STEPS_PERIODIC_IMAGES; c.p.precision = STEPS_PREC_FP64; c.p.background = STEPS_BG_FINITE;
    c.sm_count = nd->sm_count;
    c.n = (int)n;
    c.n_tiles = SYM_R * ((c.n + SYM_R * PAIR_THREADS - 1) / (SYM_R * PAIR_THREADS));
    c.n_pad = c.n_tiles * PAIR_THREADS;                  // <= kNoallocMaxN (a multiple of SYM_R * 128)
    choose_chunks(ctx);
    c.use_sym = true;
    c.use_rounds = false;
    c.sym_small = c.sym_split > 1;
    unsigned char *base = nd->scratch;
    c.xy = reinterpret_cast<double2 *>(base + kNoallocOffXy);
    c.zm = reinterpret_cast<double2 *>(base + kNoallocOffZm);
    c.hs = reinterpret_cast<double *>(base + kNoallocOffHs);
    c.part = reinterpret_cast<double *>(base + kNoallocOffPart);
    c.tile_hmax = reinterpret_cast<double *>(base + kNoallocOffHmax);
    c.flags = reinterpret_cast<DevFlags *>(base + kNoallocOffFlags);
    c.bad_h_sticky = reinterpret_cast<int *>(c.flags + 2);
    c.cur_flags = c.flags;
    c.kc.L = Lz;
    c.kc.halfL = 0.5 * Lz;
    {
        uint64_t bits;
        std::memcpy(&bits, &Lz, 8);
        c.kc.L_hi = (int)(bits >> 32);
        c.kc.L_lo = (int)(bits & 0xffffffffu);
        const double hl = 0.5 * Lz;
        std::memcpy(&bits, &hl, 8);
        c.kc.halfL_hi = (int)(bits >> 32);
    }
    for (int k = 0; k <= MAX_NCUT_TABLE; ++k) {
        const double kL = (double)k * Lz;
        c.kc.c2nL[k] = 2.0 * kL;
        c.kc.n2L2[k] = kL * kL;
        c.kc.dn[k] = (double)k;
    }
    cudaStream_t s = (cudaStream_t)cuda_stream;
    // the array keeps the previous call's contents: the flag blocks (max h, h <= 0) must start at zero
    CK(cudaMemsetAsync(c.flags, 0, 3 * sizeof(DevFlags), s));
    const ForceArgs f = {const_cast<double *>(x), const_cast<double *>(y), const_cast<double *>(z), m, h,
                         gx, gy, gz, nullptr};
    return enqueue_force_plain(ctx, f, 0u, false, s);
}

const char *steps_cyl_strerror(int code)
{
    switch (code) {
    case STEPS_OK: return "ok";
    case STEPS_EINVAL: return "invalid argument";
    case STEPS_ESOFT: return "softening precondition violated (some h_i <= 0)";
    case STEPS_ECUDA: return "CUDA runtime error (see steps_cyl_last_cuda_error)";
    case STEPS_ENOMEM: return "out of memory";
    case STEPS_ETOOBIG: return "n exceeds STEPS_CYL_NOALLOC_MAX_N, the fixed capacity of steps_cyl_accel_noalloc";
    case STEPS_EUNSUPPORTED: return "combination not built (EWALD_TABLE with the ORDERED_PAIRS flag, or a float table too large for shared memory)";
    default: return "unknown status";
    }
}

const char *steps_cyl_last_cuda_error(steps_cyl_ctx *ctx) { return ctx ? ctx->cuda_msg : ""; }

const char *steps_cyl_pair_kernel_name(steps_cyl_ctx *ctx) { return ctx ? ctx->kernel_name : ""; }

int steps_cyl_pass_stats(steps_cyl_ctx *ctx, void *cuda_stream, uint64_t *simple, uint64_t *total)
{
    if (!ctx || !simple || !total) return STEPS_EINVAL;
    ON_DEVICE(ctx);
    CK(cudaStreamSynchronize((cudaStream_t)cuda_stream));
    unsigned long long v[2] = {0, 0};
    CK(cudaMemcpy(v, ctx->pass_stats, sizeof v, cudaMemcpyDeviceToHost));
    *simple = v[0];
    *total = v[1];
    return STEPS_OK;
}

int64_t steps_cyl_launch_count(steps_cyl_ctx *ctx) { return ctx ? ctx->launches : 0; }

}  // extern "C"
