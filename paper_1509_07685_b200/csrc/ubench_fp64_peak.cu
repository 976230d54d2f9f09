// Microbenchmark behind the fp64 roof that DESIGN.md sections 6 / 7 use for P3 (the one pass that is bound by fp64 issue, not by HBM):
// how many DFMA lanes per SM and clock does this GPU retire?  Not part of the library (paper_1509_07685_b200/build.py does not
// compile it).  Build and run on the GPU box:
//     nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o /tmp/ubench_fp64_peak paper_1509_07685_b200/csrc/ubench_fp64_peak.cu
//     /tmp/ubench_fp64_peak
// Every thread runs CHAINS independent dependent-FMA chains (enough to cover the pipe latency at every warp count tried);
// the kernel reads clock64() on entry and exit of each block, so lanes / SM / clock comes from SM cycles and does not depend on
// the clock frequency the board happens to run at; the rate in instructions per second comes from CUDA events.
#include <cstdio>
#include <cuda_runtime.h>

constexpr int CHAINS = 8, ITERS = 4096;

__global__ void dfma_chains(double *out, long long *cycles, double a, double b)
{
    double v[CHAINS];
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) v[c] = threadIdx.x + c;
    const long long t0 = clock64();
#pragma unroll 1
    for (int i = 0; i < ITERS; ++i) {
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int c = 0; c < CHAINS; ++c) v[c] = fma(v[c], a, b);
    }
    const long long t1 = clock64();
    double s = 0;
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) s += v[c];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

int main()
{
    cudaDeviceProp prop;
    cudaGetDeviceProperties(&prop, 0);
    const int sms = prop.multiProcessorCount;
    double *out;
    long long *cyc, *hcyc = new long long[sms * 8];
    cudaMalloc(&out, sizeof(double) * sms * 8 * 1024);
    cudaMalloc(&cyc, sizeof(long long) * sms * 8);
    printf("%s, %d SMs; %d chains x %d x 4 DFMA per thread\n", prop.name, sms, CHAINS, ITERS);
    printf("%12s %10s %14s %18s %16s\n", "warps/SM", "ms", "DFMA lane/s", "lanes/SM/clk(cyc)", "SM MHz (implied)");
    const int threads_per_block[] = { 128, 256, 384, 512, 1024 };
    for (int tpb : threads_per_block) {
        cudaEvent_t e0, e1;
        cudaEventCreate(&e0); cudaEventCreate(&e1);
        for (int rep = 0; rep < 3; ++rep) {                     // the last repetition is reported
            cudaEventRecord(e0);
            dfma_chains<<<sms, tpb>>>(out, cyc, 0.999999, 1e-9);
            cudaEventRecord(e1);
            cudaEventSynchronize(e1);
        }
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        cudaMemcpy(hcyc, cyc, sizeof(long long) * sms, cudaMemcpyDeviceToHost);
        double mean_cyc = 0;
        for (int i = 0; i < sms; ++i) mean_cyc += (double)hcyc[i] / sms;
        const double lane_ops = (double)sms * tpb * CHAINS * ITERS * 4.0;
        printf("%12d %10.4f %14.4e %18.2f %16.0f\n", tpb / 32, ms, lane_ops / (ms * 1e-3), lane_ops / sms / mean_cyc, mean_cyc / (ms * 1e-3) / 1e6);
    }
    if (cudaGetLastError() != cudaSuccess) { printf("CUDA error\n"); return 1; }
    return 0;
}
