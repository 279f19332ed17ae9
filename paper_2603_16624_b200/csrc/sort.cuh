// sort.cuh -- per-cell binning and counting sort of one species (PAPER.md L149:
// "sorting the particles and employing a reduction", which the paper could not realise in OpenACC).
//
//   k_cell_hist   cell id per particle (+ its rank inside the cell) and the per-cell histogram
//   k_scan_*      exclusive scan of the histogram -> start[cells+1]
//   k_build_perm  perm[start[cell] + rank] = old index
//   k_gather_f64  out[new] = in[perm[new]]   (one SoA array at a time)
//
// Integer work only; results (cell ids, counts) are bit-exact functions of the stored positions.
#pragma once
#include "common.cuh"

// cell id = node id of the lower corner N- (L131).
__device__ __forceinline__ int cell_of(const Geom& g, double x, double y, double z)
{
    const int i = lower_node(x * g.rdx, g.nx);
    const int j = lower_node(y * g.rdy, g.ny);
    const int k = lower_node(z * g.rdz, g.nz);
    return (i * g.ny + j) * g.nz + k;
}

// One thread per particle.  Lanes of a warp that fall in the same cell are aggregated with
// match_any so that a cell-sorted input costs one atomic per (warp, cell) instead of 32.
template <bool WITH_RANK>
__global__ void __launch_bounds__(256)
k_cell_hist(Geom g, uint32_t n, const double* __restrict__ x, const double* __restrict__ y,
            const double* __restrict__ z, int32_t* __restrict__ cell_out,
            uint32_t* __restrict__ rank_out, uint32_t* __restrict__ count)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    const size_t n_round = ((size_t)n + 31) & ~(size_t)31;   // keep whole warps in the loop
    for (size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x; p < n_round; p += stride) {
        const bool active = p < n;
        int c = -1;
        if (active) c = cell_of(g, x[p], y[p], z[p]);
        const unsigned peers = __match_any_sync(0xffffffffu, c);
        if (active) {
            const int leader = __ffs(peers) - 1;
            uint32_t base = 0;
            if ((int)lane_id() == leader) base = atomicAdd(&count[c], (uint32_t)__popc(peers));
            base = __shfl_sync(peers, base, leader);
            if (cell_out) cell_out[p] = c;
            if (WITH_RANK) rank_out[p] = base + __popc(peers & ((1u << lane_id()) - 1u));
        }
    }
}

// Cell id only (ecsim_cell_index).
__global__ void __launch_bounds__(256)
k_cell_index(Geom g, uint32_t n, const double* __restrict__ x, const double* __restrict__ y,
             const double* __restrict__ z, int32_t* __restrict__ cell_out)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += stride)
        cell_out[p] = cell_of(g, x[p], y[p], z[p]);
}

// ---- exclusive scan of count[m] -> start[m+1], three small kernels (m <= a few million) ----
constexpr int SCAN_BLOCK = 1024;

__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t v, uint32_t* total)
{
    __shared__ uint32_t warp_sums[32];
    const unsigned lane = lane_id(), warp = threadIdx.x >> 5;
    uint32_t incl = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        uint32_t t = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= (unsigned)d) incl += t;
    }
    if (lane == 31) warp_sums[warp] = incl;
    __syncthreads();
    if (warp == 0) {
        uint32_t w = warp_sums[lane];
        uint32_t wi = w;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            uint32_t t = __shfl_up_sync(0xffffffffu, wi, d);
            if (lane >= (unsigned)d) wi += t;
        }
        warp_sums[lane] = wi - w;   // exclusive
        if (lane == 31) *total = wi;
    }
    __syncthreads();
    const uint32_t r = warp_sums[warp] + incl - v;
    __syncthreads();
    return r;
}

__global__ void __launch_bounds__(SCAN_BLOCK)
k_scan_blocks(const uint32_t* __restrict__ count, uint32_t* __restrict__ start,
              uint32_t* __restrict__ block_sums, uint32_t m)
{
    __shared__ uint32_t total;
    const uint32_t i = blockIdx.x * SCAN_BLOCK + threadIdx.x;
    const uint32_t v = i < m ? count[i] : 0u;
    const uint32_t e = block_exclusive_scan(v, &total);
    if (i < m) start[i] = e;
    if (threadIdx.x == 0) block_sums[blockIdx.x] = total;
}

// single block: exclusive scan of block_sums[nb] in place, chunk by chunk; total -> start[m]
__global__ void __launch_bounds__(SCAN_BLOCK)
k_scan_sums(uint32_t* __restrict__ block_sums, uint32_t nb, uint32_t* __restrict__ start, uint32_t m)
{
    __shared__ uint32_t total;
    uint32_t carry = 0;
    for (uint32_t base = 0; base < nb; base += SCAN_BLOCK) {
        const uint32_t i = base + threadIdx.x;
        const uint32_t v = i < nb ? block_sums[i] : 0u;
        const uint32_t e = block_exclusive_scan(v, &total);
        if (i < nb) block_sums[i] = carry + e;
        carry += total;
        __syncthreads();
    }
    if (threadIdx.x == 0) start[m] = carry;
}

__global__ void __launch_bounds__(SCAN_BLOCK)
k_scan_add(uint32_t* __restrict__ start, const uint32_t* __restrict__ block_sums, uint32_t m)
{
    const uint32_t i = blockIdx.x * SCAN_BLOCK + threadIdx.x;
    if (i < m) start[i] += block_sums[blockIdx.x];
}

__global__ void __launch_bounds__(256)
k_build_perm(uint32_t n, const int32_t* __restrict__ cell, const uint32_t* __restrict__ rank,
             const uint32_t* __restrict__ start, uint32_t* __restrict__ perm)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += stride)
        perm[start[cell[p]] + rank[p]] = (uint32_t)p;
}

__global__ void __launch_bounds__(256)
k_gather_f64(uint32_t n, const uint32_t* __restrict__ perm, const double* __restrict__ in,
             double* __restrict__ out)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += stride)
        out[p] = in[perm[p]];
}

__global__ void __launch_bounds__(256)
k_copy_u32_to_i32(uint32_t m, const uint32_t* __restrict__ in, int32_t* __restrict__ out)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x; p < m; p += stride)
        out[p] = (int32_t)in[p];
}
