// probe: do DMMA / DFMA hold the warp scheduler's issue port?  Mix them with FFMA work.
#include <cstdio>
#include <cuda_runtime.h>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("err %s line %d\n",cudaGetErrorString(e),__LINE__);return 1;}}while(0)
__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
template <int NMMA, int NDF, int NFF>
__global__ void __launch_bounds__(512) k(double* sink, int iters, double seed)
{
    double c[8][2]; double f[8]; float g[16];
#pragma unroll
    for (int i = 0; i < 8; ++i) { c[i][0] = seed + i; c[i][1] = seed - i; f[i] = seed + threadIdx.x * 1e-9 + i; }
#pragma unroll
    for (int i = 0; i < 16; ++i) g[i] = (float)seed + i;
    double a = 1.0 - 1e-9 * seed, b = 1e-9 * (threadIdx.x + 1);
    float fa = 1.0f - 1e-6f * (float)seed, fb = 1e-6f;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
#pragma unroll
            for (int i = 0; i < NMMA; ++i) dmma(c[i % 8][0], c[i % 8][1], a, b);
#pragma unroll
            for (int i = 0; i < NDF; ++i) f[i % 8] = fma(f[i % 8], a, b);
#pragma unroll
            for (int i = 0; i < NFF; ++i) g[i % 16] = fmaf(g[i % 16], fa, fb);
        }
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += c[i][0] + c[i][1] + f[i];
#pragma unroll
    for (int i = 0; i < 16; ++i) s += g[i];
    if (s == 123.456) sink[threadIdx.x] = s;
}
template <int NMMA, int NDF, int NFF>
int run(const char* name)
{
    cudaDeviceProp p; CK(cudaGetDeviceProperties(&p, 0));
    double* sink; CK(cudaMalloc(&sink, 8 * 1024));
    cudaEvent_t e0, e1; CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
    int blocks = p.multiProcessorCount, iters = 2048;   // 16 warps per SM = 4 per scheduler
    k<NMMA, NDF, NFF><<<blocks, 512>>>(sink, 64, 1.0);
    CK(cudaEventRecord(e0));
    k<NMMA, NDF, NFF><<<blocks, 512>>>(sink, iters, 1.0);
    CK(cudaEventRecord(e1));
    CK(cudaEventSynchronize(e1));
    float ms; CK(cudaEventElapsedTime(&ms, e0, e1));
    // cycles per scheduler per unrolled unit (4 warps per scheduler), at 1.965 GHz
    double cyc = ms * 1e-3 * 1.965e9 / (iters * 4.0) / 4.0;
    printf("%-40s %8.3f ms   %7.1f cycles per (warp, unit): pipe need %d, ffma %d\n", name, ms, cyc, NMMA * 16 + NDF * 2, NFF);
    cudaFree(sink);
    return 0;
}
int main()
{
    run<4, 0, 0>("4 dmma");
    run<4, 0, 32>("4 dmma + 32 ffma");
    run<4, 0, 64>("4 dmma + 64 ffma");
    run<4, 0, 128>("4 dmma + 128 ffma");
    run<0, 32, 0>("32 dfma");
    run<0, 32, 32>("32 dfma + 32 ffma");
    run<0, 32, 64>("32 dfma + 64 ffma");
    run<0, 32, 128>("32 dfma + 128 ffma");
    run<0, 0, 128>("128 ffma");
    run<2, 16, 64>("2 dmma + 16 dfma + 64 ffma");
    return 0;
}
