// ubench_fp64.cu -- what the FP64 pipe of one B200 SM sustains, as DFMA and as DMMA (mma.sync.m8n8k4.f64), alone and
// mixed. Stand-alone (no library code): `python -m paper_2503_00264_b200.ubench` builds and runs it. The numbers are
// the denominator of bench.py's "alu" roofline and the evidence behind north_star's "FP64 DMMA
// only if ncu shows a gain": one DMMA carries 8 fused multiply-adds per lane in ONE issue slot at the full rate of the
// pipe, from a single warp per SM sub-partition (profiles/r02_fp64_pipe.md).
#include <cstdio>
#include <cuda_runtime.h>

__device__ __forceinline__ void dmma(double &c0, double &c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// MODE 0: DMMA only, ILP independent accumulator pairs; 1: DFMA only (8 per slot = the FMAs of one DMMA per lane);
// 2: one DMMA + 8 DFMA per slot
template <int ILP, int MODE>
__global__ void k(double *out, long long *cyc, double y, double z, int iters)
{
    double c[ILP][2];
    double f[8];
#pragma unroll
    for (int i = 0; i < ILP; ++i) { c[i][0] = threadIdx.x * 1e-3 + i; c[i][1] = 0.5 * i; }
#pragma unroll
    for (int i = 0; i < 8; ++i) f[i] = threadIdx.x * 1e-4 + i;
    const double a = y + threadIdx.x * 1e-9, b = z;
    __syncthreads();
    long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < ILP; ++i) {
            if (MODE == 0 || MODE == 2) dmma(c[i][0], c[i][1], a, b);
            if (MODE == 1 || MODE == 2) {
#pragma unroll
                for (int q = 0; q < 8; ++q) f[q] = fma(f[q], y, z);
            }
        }
    }
    long long t1 = clock64();
    double s = 0;
#pragma unroll
    for (int i = 0; i < ILP; ++i) s += c[i][0] + c[i][1];
#pragma unroll
    for (int i = 0; i < 8; ++i) s += f[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0) cyc[blockIdx.x] = t1 - t0;
}

template <int ILP, int MODE> void run(int blocks, int warps, double *out, long long *cyc)
{
    const int iters = 2048;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    k<ILP, MODE><<<blocks, warps * 32>>>(out, cyc, 0.999, 0.001, iters);
    cudaEventRecord(e0);
    k<ILP, MODE><<<blocks, warps * 32>>>(out, cyc, 0.999, 0.001, iters);
    cudaEventRecord(e1);
    cudaDeviceSynchronize();
    float ms;
    cudaEventElapsedTime(&ms, e0, e1);
    long long h;
    cudaMemcpy(&h, cyc, 8, cudaMemcpyDeviceToHost);
    const double per_slot = (MODE == 2 ? 16.0 : 8.0); // FMAs per lane per slot
    const double eq_per_clk = (double)warps * 32 * ILP * iters * per_slot / h;
    const double tf = (double)blocks * warps * 32 * ILP * iters * per_slot * 2 / (ms * 1e-3) / 1e12;
    const char *name = MODE == 0 ? "DMMA     " : (MODE == 1 ? "DFMA     " : "DMMA+DFMA");
    printf("%s CTAs %3d warps/CTA %2d ILP %d: %7.2f cycles per slot per warp, %5.1f FMA/clk/SM, %6.2f TFLOP/s (CUDA events)\n",
           name, blocks, warps, ILP, (double)h / (ILP * iters), eq_per_clk, tf);
}

int main()
{
    double *out;
    long long *cyc;
    cudaMalloc(&out, 8 * 148 * 1024 * 2);
    cudaMalloc(&cyc, 8 * 1024);
    printf("# dependent-issue latency (one warp, one accumulator): cycles per slot = latency of a DMMA / of 8 chained DFMAs\n");
    run<1, 0>(1, 1, out, cyc);
    run<1, 1>(1, 1, out, cyc);
    printf("# one SM\n");
    for (int w : {1, 4, 8, 16}) {
        run<2, 0>(1, w, out, cyc);
        run<8, 0>(1, w, out, cyc);
        run<4, 1>(1, w, out, cyc);
        run<4, 2>(1, w, out, cyc);
    }
    printf("# whole chip (148 CTAs)\n");
    for (int w : {4, 8, 16}) {
        run<8, 0>(148, w, out, cyc);
        run<4, 1>(148, w, out, cyc);
        run<4, 2>(148, w, out, cyc);
    }
    return 0;
}
