// probe: which instruction classes issue underneath DMMA / DFMA?  (4 warps per scheduler)
#include <cstdio>
#include <cuda_runtime.h>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("err %s line %d\n",cudaGetErrorString(e),__LINE__);return 1;}}while(0)
__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
// KIND: 0 none, 1 FFMA, 2 LOP3/IADD (alu pipe), 3 LDS, 4 IMAD
template <int NMMA, int NDF, int KIND, int NX>
__global__ void __launch_bounds__(512) k(double* sink, int iters, double seed, const unsigned* zero)
{
    __shared__ double sm[1024];
    sm[threadIdx.x] = threadIdx.x; sm[threadIdx.x + 512] = seed;
    __syncthreads();
    double c[8][2]; double f[8]; float g[16]; unsigned u[16]; double ld = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) { c[i][0] = seed + i; c[i][1] = seed - i; f[i] = seed + threadIdx.x * 1e-9 + i; }
#pragma unroll
    for (int i = 0; i < 16; ++i) { g[i] = (float)seed + i; u[i] = threadIdx.x * 7 + i + zero[0]; }
    double a = 1.0 - 1e-9 * seed, b = 1e-9 * (threadIdx.x + 1);
    float fa = 1.0f - 1e-6f * (float)seed, fb = 1e-6f;
    unsigned ua = zero[1] + 0x9e3779b9u, ub = zero[2] + 3u;
    unsigned idx = threadIdx.x & 511; unsigned smaddr = (unsigned)__cvta_generic_to_shared(sm) + (idx & 31) * 8;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r) {
#pragma unroll
            for (int i = 0; i < NMMA; ++i) dmma(c[i % 8][0], c[i % 8][1], a, b);
#pragma unroll
            for (int i = 0; i < NDF; ++i) f[i % 8] = fma(f[i % 8], a, b);
#pragma unroll
            for (int i = 0; i < NX; ++i) {
                if (KIND == 1) g[i % 16] = fmaf(g[i % 16], fa, fb);
                if (KIND == 2) u[i % 16] = (u[i % 16] ^ ua) + ub;          // LOP3 + IADD3
                if (KIND == 3) { double t; asm volatile("ld.shared.f64 %0, [%1];" : "=d"(t) : "r"(smaddr + ((i * 256) & 4095))); u[i % 16] ^= (unsigned)__double2loint(t); }
                if (KIND == 4) u[i % 16] = u[i % 16] * ua + ub;            // IMAD
            }
        }
    }
    double s = ld;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += c[i][0] + c[i][1] + f[i];
#pragma unroll
    for (int i = 0; i < 16; ++i) s += g[i] + u[i];
    if (s == 123.456) sink[threadIdx.x] = s;
}
template <int NMMA, int NDF, int KIND, int NX>
int run(const char* name, const unsigned* zero)
{
    cudaDeviceProp p; CK(cudaGetDeviceProperties(&p, 0));
    double* sink; CK(cudaMalloc(&sink, 8 * 1024));
    cudaEvent_t e0, e1; CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
    int blocks = p.multiProcessorCount, iters = 2048;
    k<NMMA, NDF, KIND, NX><<<blocks, 512>>>(sink, 64, 1.0, zero);
    CK(cudaEventRecord(e0));
    k<NMMA, NDF, KIND, NX><<<blocks, 512>>>(sink, iters, 1.0, zero);
    CK(cudaEventRecord(e1));
    CK(cudaEventSynchronize(e1));
    float ms; CK(cudaEventElapsedTime(&ms, e0, e1));
    double cyc = ms * 1e-3 * 1.965e9 / (iters * 4.0) / 4.0;
    printf("%-34s %8.3f ms  %7.1f cycles per (warp, unit): fp64 pipe need %d, other instr %d\n", name, ms, cyc, NMMA * 16 + NDF * 2, NX);
    cudaFree(sink);
    return 0;
}
int main()
{
    unsigned* zero; cudaMalloc(&zero, 16); cudaMemset(zero, 0, 16);
    run<4, 0, 0, 0>("4 dmma", zero);
    run<0, 0, 2, 64>("64 lop3+iadd3 pairs", zero);
    run<4, 0, 2, 64>("4 dmma + 64 lop3+iadd3 pairs", zero);
    run<0, 0, 4, 64>("64 imad", zero);
    run<4, 0, 4, 64>("4 dmma + 64 imad", zero);
    run<0, 0, 3, 64>("64 lds", zero);
    run<4, 0, 3, 64>("4 dmma + 64 lds", zero);
    run<0, 0, 1, 64>("64 ffma", zero);
    run<4, 0, 1, 64>("4 dmma + 64 ffma", zero);
    run<0, 32, 2, 64>("32 dfma + 64 lop3+iadd3 pairs", zero);
    run<0, 32, 3, 64>("32 dfma + 64 lds", zero);
    run<0, 32, 0, 0>("32 dfma", zero);
    return 0;
}
