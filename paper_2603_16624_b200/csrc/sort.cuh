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

// Histogram of the particles [p0, p1) of a cell-sorted species that must all lie in the cells [c0, c1) (one x-slab of the
// pipelined host step): particles outside the range are counted in *bad instead (the caller then falls back).
__global__ void __launch_bounds__(256)
k_cell_hist_range(Geom g, uint32_t p0, uint32_t p1, const double* __restrict__ x, const double* __restrict__ y,
                  const double* __restrict__ z, uint32_t* __restrict__ count, uint32_t c0, uint32_t c1,
                  uint32_t* __restrict__ bad)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    const size_t n = (size_t)(p1 - p0), n_round = (n + 31) & ~(size_t)31;
    for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < n_round; t += stride) {
        const bool active = t < n;
        int c = -1;
        if (active) {
            const size_t p = p0 + t;
            c = cell_of(g, x[p], y[p], z[p]);
            if ((uint32_t)c < c0 || (uint32_t)c >= c1) { atomicAdd(bad, 1u); c = -1; }
        }
        const unsigned peers = __match_any_sync(0xffffffffu, c);
        if (c >= 0 && (int)lane_id() == __ffs(peers) - 1) atomicAdd(&count[c], (uint32_t)__popc(peers));
    }
}

__global__ void __launch_bounds__(256)
k_add_u32(uint32_t* __restrict__ a, uint32_t m, uint32_t v)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < m) a[i] += v;
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

// ---------------------------------------------------------------------------------------------
// Moving the seven SoA arrays of a species given in RANDOM order (config 4) to their sorted places.
// A random 8-byte gather from HBM costs ~97 bytes of traffic on B200 (3.26 GB per 33.5 M elements,
// profiles/r01d), and scattered 8-byte stores are bound by L2 transactions, so the permutation is applied in
// two steps that are both local.  dest[p] = start[cell[p]] + rank[p] is the final place of particle p;
// places are cut into <= SORT_MAX_BUCKETS buckets of 2^shift consecutive places (every bucket is full,
// dest being a permutation).
//   step A, k_stage_to_slots: a tile of SORT_TILE particles per CTA.  slot[p] = (places of p's bucket taken by
//          earlier tiles) + (p's arrival rank in the tile).  The tile is ordered by bucket in shared memory and
//          written to tmp[] in runs of ~SORT_TILE/buckets consecutive elements: coalesced.
//   step B, k_gather_f64 with perm2[dest[p]] = slot[p]: out[d] = tmp[perm2[d]], a gather whose sources lie
//          inside one bucket's window of tmp (<= 1 MB): L2 hits; the writes are coalesced.
// slot and perm2 are computed once and serve all seven arrays; tmp is the one spare array and `out` is the
// caller's own array, so nothing is copied back.  (A species that is re-sorted after a push is nearly
// sorted: there the direct gather of ecsim_sort_particles reads almost sequentially and stays.)
constexpr int SORT_TILE = 8192;
constexpr int SORT_MAX_BUCKETS = 512;
constexpr int SORT_STAGE_THREADS = 512;
constexpr size_t SORT_STAGE_SMEM = (size_t)SORT_TILE * (sizeof(double) + sizeof(uint32_t)) + 2 * SORT_MAX_BUCKETS * sizeof(uint32_t);

// dest (in place of rank) and the per-(bucket, tile) histogram H[b * tiles + tile]
__global__ void __launch_bounds__(256)
k_dest_and_tile_hist(uint32_t n, const int32_t* __restrict__ cell, uint32_t* __restrict__ rank_to_dest,
                     const uint32_t* __restrict__ start, int shift, uint32_t tiles, uint32_t* __restrict__ H)
{
    __shared__ uint32_t cnt[SORT_MAX_BUCKETS];
    for (int t = threadIdx.x; t < SORT_MAX_BUCKETS; t += blockDim.x) cnt[t] = 0;
    __syncthreads();
    const size_t p0 = (size_t)blockIdx.x * SORT_TILE;
    for (int e = threadIdx.x; e < SORT_TILE; e += blockDim.x) {
        const size_t p = p0 + e;
        if (p < n) {
            const uint32_t d = start[cell[p]] + rank_to_dest[p];
            rank_to_dest[p] = d;
            atomicAdd(&cnt[d >> shift], 1u);
        }
    }
    __syncthreads();
    const uint32_t nb = ((n - 1) >> shift) + 1;
    for (uint32_t b = threadIdx.x; b < nb; b += blockDim.x) H[(size_t)b * tiles + blockIdx.x] = cnt[b];
}

// slot[p] (over the cell array's storage) and perm2[dest[p]] = slot[p]; Hs = exclusive scan of H
__global__ void __launch_bounds__(256)
k_assign_slots(uint32_t n, const uint32_t* __restrict__ dest, const uint32_t* __restrict__ Hs, int shift,
               uint32_t tiles, uint32_t* __restrict__ slot, uint32_t* __restrict__ perm2)
{
    __shared__ uint32_t base[SORT_MAX_BUCKETS];
    const uint32_t nb = ((n - 1) >> shift) + 1;
    for (uint32_t b = threadIdx.x; b < nb; b += blockDim.x) base[b] = Hs[(size_t)b * tiles + blockIdx.x];
    __syncthreads();
    const size_t p0 = (size_t)blockIdx.x * SORT_TILE;
    for (int e = threadIdx.x; e < SORT_TILE; e += blockDim.x) {
        const size_t p = p0 + e;
        if (p < n) {
            const uint32_t d = dest[p];
            const uint32_t s = atomicAdd(&base[d >> shift], 1u);
            slot[p] = s;
            perm2[d] = s;
        }
    }
}

// step A for one array: tmp[slot[p]] = in[p], the tile ordered by bucket in shared memory first
__global__ void __launch_bounds__(SORT_STAGE_THREADS)
k_stage_to_slots(uint32_t n, const uint32_t* __restrict__ dest, const uint32_t* __restrict__ slot,
                 const uint32_t* __restrict__ H, const uint32_t* __restrict__ Hs, int shift, uint32_t tiles,
                 const double* __restrict__ in, double* __restrict__ tmp)
{
    extern __shared__ __align__(16) unsigned char stage_smem[];
    double* vals = reinterpret_cast<double*>(stage_smem);
    uint32_t* dsts = reinterpret_cast<uint32_t*>(vals + SORT_TILE);
    uint32_t* base = dsts + SORT_TILE;          // first slot of this tile's share of bucket b
    uint32_t* toff = base + SORT_MAX_BUCKETS;   // where bucket b starts in the tile's bucket order
    __shared__ uint32_t total;
    const uint32_t nb = ((n - 1) >> shift) + 1;
    const uint32_t b = threadIdx.x;
    const uint32_t c = b < nb ? H[(size_t)b * tiles + blockIdx.x] : 0u;
    const uint32_t ex = block_exclusive_scan(c, &total);
    toff[b] = ex;
    base[b] = b < nb ? Hs[(size_t)b * tiles + blockIdx.x] : 0u;
    __syncthreads();
    const size_t p0 = (size_t)blockIdx.x * SORT_TILE;
    const uint32_t tile_n = (uint32_t)min((size_t)SORT_TILE, (size_t)n - p0);
    for (uint32_t e = threadIdx.x; e < tile_n; e += SORT_STAGE_THREADS) {
        const size_t p = p0 + e;
        const uint32_t s = slot[p], bk = dest[p] >> shift;
        const uint32_t lp = s - base[bk] + toff[bk];
        vals[lp] = in[p];
        dsts[lp] = s;
    }
    __syncthreads();
    for (uint32_t t = threadIdx.x; t < tile_n; t += SORT_STAGE_THREADS) tmp[dsts[t]] = vals[t];
}

// fixPosition on stored particles (L123): pin the masked coordinates of n slots (set-up of a reduced-dimension run)
__global__ void __launch_bounds__(256)
k_fix_position(Geom g, size_t n, double* __restrict__ x, double* __restrict__ y, double* __restrict__ z)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += stride) {
        if (g.fix_mask & 1) x[p] = g.fix_pos[0];
        if (g.fix_mask & 2) y[p] = g.fix_pos[1];
        if (g.fix_mask & 4) z[p] = g.fix_pos[2];
    }
}

// list[i] = i, *count = n ("every particle" as a list, for kernels that take one)
__global__ void __launch_bounds__(256)
k_iota_u32(uint32_t n, uint32_t* __restrict__ list, uint32_t* __restrict__ count)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += stride) list[p] = (uint32_t)p;
    if (blockIdx.x == 0 && threadIdx.x == 0) *count = n;
}

// perm[dest[p]] = p (only when the caller asks for the permutation)
__global__ void __launch_bounds__(256)
k_perm_from_dest(uint32_t n, const uint32_t* __restrict__ dest, uint32_t* __restrict__ perm)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += stride) perm[dest[p]] = (uint32_t)p;
}
