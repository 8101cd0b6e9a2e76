// fp64_microbench.cu -- stand-alone FP64-pipe microbenchmarks for sm_100a (the evidence behind DESIGN.md section 6 and
// profiles/r1_fp64_microbench.md).  Not part of libmipwa.so.  Build and run:
//     python -m paper_1703_03284_b200.build --microbench && ./paper_1703_03284_b200/fp64_microbench
// Every kernel keeps C independent dependent-chains per thread in registers, W warps per SM sub-partition, 16-fold
// unrolled; the result is FP64 thread-instructions per clock per SM at the SM clock given on the command line
// (default 1965 MHz), best of 3 launches timed with CUDA events.  The FP64 pipe's peak is 64 (16 lanes x 4).
#include <cstdio>
#include <cstdlib>
#include <cuda_runtime.h>

enum Mode {
    DFMA_3REG,      // x = fma(x, ar, br): three distinct register operands
    DFMA_IMM,       // x = fma(x, ar, 1.0): two register operands + immediate
    DFMA_SELF,      // x = fma(x, x, x): one distinct register operand
    DMUL_2REG,      // x = x * ar
    DADD_2REG,      // x = x + br
    DMUL_DFMA,      // t = x * ar; x = fma(t, t, br): two-operand mix
    DFMA_1ALU,      // DFMA_IMM + one integer ALU instruction
    DFMA_3ALU,      // DFMA_IMM + three integer ALU instructions
    RSQ64H,         // MUFU.RSQ64H chain
    RSQ_4DFMA       // one MUFU.RSQ64H + four DFMA_IMM
};

template <int MODE, int CHAINS>
__global__ void __launch_bounds__(256) k_chain(double* out, long long iters, double a, double b, int ia)
{
    double x[CHAINS];
    int z[CHAINS];
    const double ar = a + threadIdx.x * 1e-9, br = b + threadIdx.x * 1e-12;
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) { x[c] = threadIdx.x * 1e-3 + c + 1.0; z[c] = threadIdx.x + c; }
    for (long long i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 16; ++u) {
#pragma unroll
            for (int c = 0; c < CHAINS; ++c) {
                if (MODE == DFMA_3REG) x[c] = fma(x[c], ar, br);
                if (MODE == DFMA_IMM) x[c] = fma(x[c], ar, 1.0);
                if (MODE == DFMA_SELF) x[c] = fma(x[c], x[c], x[c]);
                if (MODE == DMUL_2REG) x[c] = x[c] * ar;
                if (MODE == DADD_2REG) x[c] = x[c] + br;
                if (MODE == DMUL_DFMA) { const double t = x[c] * ar; x[c] = fma(t, t, br); }
                if (MODE == DFMA_1ALU) { x[c] = fma(x[c], ar, 1.0); z[c] = (z[c] ^ ia) + u; }
                if (MODE == DFMA_3ALU) { x[c] = fma(x[c], ar, 1.0); z[c] = (z[c] ^ ia) + u; z[c] = (z[c] & 0x55555) | u; z[c] = (z[c] ^ 0x3333) + ia; }
                if (MODE == RSQ64H) { double y; asm volatile("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x[c])); x[c] = y; }
                if (MODE == RSQ_4DFMA) {
                    double y;
                    asm volatile("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x[c]));
                    x[c] = fma(y, ar, 1.0); x[c] = fma(x[c], ar, 1.0); x[c] = fma(x[c], ar, 1.0); x[c] = fma(x[c], ar, 1.0);
                }
            }
        }
    }
    double s = 0;
    int t = 0;
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) { s += x[c]; t += z[c]; }
    if (s == 123.456 || t == 0x7fffffff) out[0] = s + t;      // keeps the chains alive
}

static double g_mhz = 1965.0;

template <int MODE, int CHAINS>
static void run(const char* name, int warps_per_smsp, double counted_per_step)
{
    cudaDeviceProp p;
    cudaGetDeviceProperties(&p, 0);
    double* d;
    cudaMalloc(&d, 64);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const long long iters = 20000;
    const int threads = warps_per_smsp >= 2 ? 256 : 128;
    const int blocks_per_sm = warps_per_smsp * 128 / threads, grid = p.multiProcessorCount * blocks_per_sm;
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0);
        k_chain<MODE, CHAINS><<<grid, threads>>>(d, iters, 0.999999, 1e-9, 3);
        cudaEventRecord(e1);
        cudaEventSynchronize(e1);
        float ms;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep && ms < best) best = ms;
    }
    const double inst = counted_per_step * 16.0 * CHAINS * iters * (double)grid * threads;
    const double per_clk_sm = inst / (best * 1e-3) / (g_mhz * 1e6 * p.multiProcessorCount);
    printf("%-44s chains %2d  warps/SMSP %2d  %9.3f ms  %6.2f counted inst/clk/SM\n", name, CHAINS, warps_per_smsp, best,
           per_clk_sm);
    cudaFree(d);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
}

int main(int argc, char** argv)
{
    if (argc > 1) g_mhz = atof(argv[1]);
    printf("FP64 microbenchmarks, SM clock assumed %.0f MHz; FP64 instructions counted unless stated\n", g_mhz);
    run<DFMA_3REG, 8>("DFMA 3 register operands", 16, 1);
    run<DMUL_2REG, 8>("DMUL", 16, 1);
    run<DADD_2REG, 8>("DADD", 16, 1);
    run<DFMA_3REG, 1>("DFMA 3 regs, latency (1 warp, 1 chain)", 1, 1);
    run<DFMA_3REG, 1>("DFMA 3 regs, 1 chain", 4, 1);
    run<DFMA_3REG, 1>("DFMA 3 regs, 1 chain", 8, 1);
    run<DFMA_3REG, 1>("DFMA 3 regs, 1 chain", 16, 1);
    run<DFMA_3REG, 2>("DFMA 3 regs, 2 chains", 4, 1);
    run<DFMA_3REG, 4>("DFMA 3 regs, 4 chains", 4, 1);
    run<DFMA_3REG, 6>("DFMA 3 regs, 6 chains", 4, 1);
    run<DFMA_IMM, 1>("DFMA 2 regs + immediate, 1 chain", 8, 1);
    run<DFMA_SELF, 1>("DFMA x*x+x, 1 chain", 8, 1);
    run<DMUL_2REG, 1>("DMUL 2 regs, 1 chain", 8, 1);
    run<DADD_2REG, 1>("DADD 2 regs, 1 chain", 8, 1);
    run<DMUL_DFMA, 2>("DMUL + DFMA(t,t,b), 2 chains", 4, 2);
    run<DFMA_IMM, 8>("DFMA imm only, 8 chains", 4, 1);
    run<DFMA_1ALU, 8>("DFMA imm + 1 integer ALU op (FP64 counted)", 4, 1);
    run<DFMA_3ALU, 8>("DFMA imm + 3 integer ALU ops (FP64 counted)", 4, 1);
    run<RSQ64H, 8>("MUFU.RSQ64H (MUFU counted)", 8, 1);
    run<RSQ_4DFMA, 8>("MUFU.RSQ64H + 4 DFMA (DFMA counted)", 8, 4);
    return 0;
}
