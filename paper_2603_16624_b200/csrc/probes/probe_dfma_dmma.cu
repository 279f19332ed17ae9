// probe: DFMA vs DMMA m8n8k4 throughput and whether they overlap (B200)
#include <cstdio>
#include <cuda_runtime.h>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("err %s line %d\n",cudaGetErrorString(e),__LINE__);return 1;}}while(0)

__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

template <int NMMA, int NFMA>
__global__ void __launch_bounds__(256) k(double* sink, int iters, double seed)
{
    double c[8][2];
    double f[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) { c[i][0] = seed + i; c[i][1] = seed - i; f[i] = seed + threadIdx.x * 1e-9 + i; }
    double a = 1.0 - 1e-9 * seed, b = 1e-9 * (threadIdx.x + 1);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
#pragma unroll
            for (int i = 0; i < NMMA; ++i) dmma(c[i][0], c[i][1], a, b);
#pragma unroll
            for (int i = 0; i < NFMA; ++i) f[i % 8] = fma(f[i % 8], a, b);
        }
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += c[i][0] + c[i][1] + f[i];
    if (s == 123.456) sink[threadIdx.x] = s;
}

template <int NMMA, int NFMA>
int run(const char* name, int blocks_per_sm)
{
    cudaDeviceProp p; CK(cudaGetDeviceProperties(&p, 0));
    double* sink; CK(cudaMalloc(&sink, 8 * 1024));
    cudaEvent_t e0, e1; CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
    int blocks = p.multiProcessorCount * blocks_per_sm, iters = 4096;
    k<NMMA, NFMA><<<blocks, 256>>>(sink, 64, 1.0);
    CK(cudaEventRecord(e0));
    k<NMMA, NFMA><<<blocks, 256>>>(sink, iters, 1.0);
    CK(cudaEventRecord(e1));
    CK(cudaEventSynchronize(e1));
    float ms; CK(cudaEventElapsedTime(&ms, e0, e1));
    double warps = (double)blocks * 8;
    double fl_mma = 2.0 * 256 * NMMA * 4 * iters * warps, fl_fma = 2.0 * 32 * NFMA * 4 * iters * warps;
    printf("%-28s bps=%d  %8.3f ms  dmma %7.2f TF  dfma %7.2f TF  total %7.2f TF\n", name, blocks_per_sm, ms,
           fl_mma / ms * 1e-9, fl_fma / ms * 1e-9, (fl_mma + fl_fma) / ms * 1e-9);
    cudaFree(sink);
    return 0;
}

int main()
{
    for (int bps = 1; bps <= 8; bps *= 2) {
        run<0, 32>("dfma only (32/iter)", bps);
        run<8, 0>("dmma only (8/iter)", bps);
        run<4, 0>("dmma only (4 chains)", bps);
        run<8, 32>("dmma 8 + dfma 32", bps);
        run<8, 64>("dmma 8 + dfma 64", bps);
        run<4, 64>("dmma 4 + dfma 64", bps);
    }
    return 0;
}
