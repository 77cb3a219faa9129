// ubench_fp64_pipe.cu -- what one FP64-pipe issue slot costs on B200 (sm_100a), measured.
//
//     python -m paper_2602_20787_b200.ubench            (compiles this file with nvcc, runs it on cuda:0)
//
// The all-pairs kernels of this library are bound by the FP64 pipe (64 lanes per SM: a warp-wide DFMA / DMUL / DADD
// holds a scheduler's pipe for two cycles).  This program times loops of independent FP64 chains, alone and mixed
// with other instructions, and prints the achieved fraction of 64 lanes x clock.  What the pair kernels' design
// takes from it (numbers in profiles/r2_fp64_pipe_microbench.md):
//   * an FP64 instruction with at most TWO distinct 64-bit register sources (the third a constant, an immediate,
//     or a repeated register) sustains 99.8 % of the nominal rate; one with THREE distinct register sources
//     sustains 66.7 % -- three issue cycles instead of two;
//   * nothing is issued under the FP64 instruction's second cycle: every other instruction (FFMA, integer, MOV,
//     MUFU, SHFL = 2) adds about one issue cycle of its own.
// Not part of the library: nothing links against it.
#include <cstdio>
#include <cuda_runtime.h>

#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { printf("%s at line %d\n", cudaGetErrorString(e_), __LINE__); return 1; } } while (0)

enum Mode {
    DFMA_2REG_CONST, DFMA_1REG_2UNIFORM, DFMA_3REG, DFMA_3REG_SHARED, DFMA_REG_IMM, DMUL_2REG, DADD_2REG, DADD_CONST,
    MIX_FFMA_1_1, MIX_FFMA_4_1, MIX_INT_4_3, MIX_SHFL_4_1, MIX_RSQ64H_8_1, MIX_MOV_8_1
};

template <int CH, int MODE>
__global__ void __launch_bounds__(256) chain_kernel(double *out, int iters, double a, double b, float fa)
{
    double r[CH], p[CH];
#pragma unroll
    for (int q = 0; q < CH; ++q) {
        r[q] = (double)(threadIdx.x + q) * 1e-3 + 1.0;
        p[q] = 1.0 - (double)(threadIdx.x + q) * 1e-9;
    }
    const double mreg = 1.0 + 1e-12 * threadIdx.x;     // a per-thread value: lives in a register, not a constant
    float f = fa * threadIdx.x;
    int n = threadIdx.x;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int q = 0; q < CH; ++q) {
            if (MODE == DFMA_2REG_CONST)    r[q] = fma(r[q], r[(q + 1) % CH], b);
            if (MODE == DFMA_1REG_2UNIFORM) r[q] = fma(r[q], a, b);
            if (MODE == DFMA_3REG)          r[q] = fma(r[q], r[(q + 1) % CH], r[(q + 2) % CH]);
            if (MODE == DFMA_3REG_SHARED)   r[q] = fma(mreg, p[q], r[q]);       // a += m P: one source common to all
            if (MODE == DFMA_REG_IMM)       r[q] = fma(r[q], 1.875, r[(q + 1) % CH]);
            if (MODE == DMUL_2REG)          r[q] = r[q] * p[q];
            if (MODE == DADD_2REG)          r[q] = r[q] + p[q];
            if (MODE == DADD_CONST)         r[q] = r[q] + a;
            if (MODE >= MIX_FFMA_1_1)       r[q] = fma(r[q], r[(q + 1) % CH], b);
            if (MODE == MIX_FFMA_1_1)       f = fmaf(f, fa, 1.0f);
            if (MODE == MIX_FFMA_4_1 && (q & 3) == 0) f = fmaf(f, fa, 1.0f);
            if (MODE == MIX_INT_4_3 && (q & 3) == 0)  n = (n ^ (n >> 3)) + q;   // SHF + LOP3 + IADD
            if (MODE == MIX_SHFL_4_1 && (q & 3) == 0) n = __shfl_sync(0xffffffffu, n, (threadIdx.x + 1) & 31);
            if (MODE == MIX_RSQ64H_8_1 && (q & 7) == 0) {
                double y;
                asm volatile("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(r[q]));     // MUFU.RSQ64H + low-word MOV
                r[q] = y;
            }
            if (MODE == MIX_MOV_8_1 && (q & 7) == 0) r[q] = __hiloint2double(__double2hiint(r[q]) ^ n, 0);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int q = 0; q < CH; ++q) s += r[q] + p[q];
    if (s == 123.456 || f == 77.0f || n == 12345) out[0] = s + f + n;
}

template <int CH, int MODE>
int run(const char *name, double *out, int blocks_per_sm, int sms, double ghz)
{
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0));
    CK(cudaEventCreate(&e1));
    const int iters = 20000, threads = 256;
    chain_kernel<CH, MODE><<<sms * blocks_per_sm, threads>>>(out, 1000, 0.999999, 1e-3, 0.99f);
    CK(cudaEventRecord(e0));
    chain_kernel<CH, MODE><<<sms * blocks_per_sm, threads>>>(out, iters, 0.999999, 1e-3, 0.99f);
    CK(cudaEventRecord(e1));
    CK(cudaEventSynchronize(e1));
    float ms;
    CK(cudaEventElapsedTime(&ms, e0, e1));
    const double warps_per_sm = blocks_per_sm * threads / 32.0;
    const double cycles = ms * 1e-3 * ghz * 1e9;
    // per SM: 4 schedulers, 2 pipe cycles per FP64 warp instruction
    const double util = warps_per_sm * iters * (double)CH * 2.0 / 4.0 / cycles;
    printf("| %-52s | %2.0f | %8.3f | %5.3f | %5.2f |\n", name, warps_per_sm / 4, ms, util, 2.0 / util);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return 0;
}

int main()
{
    cudaDeviceProp p;
    CK(cudaGetDeviceProperties(&p, 0));
    int khz = 0;
    CK(cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, 0));
    const double ghz = khz * 1e-6;
    printf("%s, %d SMs, SM clock %.3f GHz (attribute; the run must hold it: check nvidia-smi)\n\n", p.name,
           p.multiProcessorCount, ghz);
    printf("| loop body (16 independent FP64 chains per thread)           | warps/scheduler | ms | FP64 pipe utilisation | cycles per FP64 instruction (incl. what rides along) |\n");
    printf("|---|---:|---:|---:|---:|\n");
    double *out;
    CK(cudaMalloc(&out, 8));
    const int sms = p.multiProcessorCount;
    run<16, DFMA_2REG_CONST>("DFMA reg * reg + const", out, 8, sms, ghz);
    run<16, DFMA_REG_IMM>("DFMA reg * imm + reg", out, 8, sms, ghz);
    run<16, DMUL_2REG>("DMUL reg * reg", out, 8, sms, ghz);
    run<16, DADD_2REG>("DADD reg + reg", out, 8, sms, ghz);
    run<16, DADD_CONST>("DADD reg + const", out, 8, sms, ghz);
    run<16, DFMA_1REG_2UNIFORM>("DFMA reg * uniform + uniform (kernel parameters)", out, 8, sms, ghz);
    run<16, DFMA_3REG>("DFMA reg * reg + reg (three distinct registers)", out, 8, sms, ghz);
    run<16, DFMA_3REG_SHARED>("DFMA m * P[q] + a[q] (three registers, m shared)", out, 8, sms, ghz);
    run<16, DFMA_2REG_CONST>("DFMA reg * reg + const, 4 warps per scheduler", out, 2, sms, ghz);
    run<16, DFMA_2REG_CONST>("DFMA reg * reg + const, 2 warps per scheduler", out, 1, sms, ghz);
    run<16, MIX_FFMA_1_1>("16 DFMA + 16 FFMA", out, 8, sms, ghz);
    run<16, MIX_FFMA_4_1>("16 DFMA + 4 FFMA", out, 8, sms, ghz);
    run<16, MIX_INT_4_3>("16 DFMA + 4 x (SHF, LOP3, IADD)", out, 8, sms, ghz);
    run<16, MIX_SHFL_4_1>("16 DFMA + 4 SHFL", out, 8, sms, ghz);
    run<16, MIX_RSQ64H_8_1>("16 DFMA + 2 x (MUFU.RSQ64H, MOV)", out, 8, sms, ghz);
    run<16, MIX_MOV_8_1>("16 DFMA + 2 x (LOP3, MOV)", out, 8, sms, ghz);
    cudaFree(out);
    return 0;
}
