// sort.cuh -- per-cell binning and counting sort of one species (PAPER.md L149:
// "sorting the particles and employing a reduction", which the paper could not realise in OpenACC).
//
//   k_cell_hist   cell id per particle (+ its rank inside the cell) and the per-cell histogram
//   k_scan_*      exclusive scan of the histogram -> start[cells+1]
//   k_build_perm  perm[start[cell] + rank] = old index
//   k_gather7     out[new] = in[perm[new]] for the seven SoA arrays (re-sort of a nearly sorted species)
//   k_stage7_to_slots / k_scatter7  the two-step move of a species in arbitrary order
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
//   step A, k_stage7_to_slots: a tile of SORT_TILE particles per CTA.  A particle's slot = (places of its bucket taken
//          by earlier tiles, from the scanned per-(bucket, tile) histogram) + (its arrival rank in the tile, a shared-
//          memory atomic).  The tile is ordered by bucket in shared memory and written to tmp[] in runs of
//          ~SORT_TILE/buckets consecutive elements: coalesced.  ALL SEVEN arrays go through one launch -- the slot
//          bookkeeping is computed once, kept in registers, and the final place travels with the particle (tmpdest).
//   step B, k_invert_slots + k_gather7: perm2 = tmpdest^-1, then out[d] = tmp[perm2[d]] for the seven arrays: a gather
//          whose sources lie inside the windows of the ~9 buckets in flight (grid-stride; 2^shift places x 7 arrays x 8 B
//          = 3.5 MB each): L2 hits; the writes are coalesced.
// Round 1 moved one array per launch pair (14 launches, the bookkeeping re-read 7 times, a separate slot-assignment
// pass with a random 4-byte scatter): 4.35 ms per 33.5 M particles.  tmp = seven spare arrays of the workspace.
// (measured in round 2, 33.5 M particles: 4096 x 256 buckets 3.75 ms, 8192 x 256 3.80, 8192 x 512 3.81, 16384 x 512 3.80,
// 16384 x 256 3.83: the move is not sensitive to the tile / bucket geometry)
constexpr int SORT_TILE = 8192;
constexpr int SORT_MAX_BUCKETS = 512;
constexpr int SORT_STAGE_THREADS = 512;
constexpr int SORT_PER_THREAD = SORT_TILE / SORT_STAGE_THREADS;
constexpr size_t SORT_STAGE_SMEM = (size_t)SORT_TILE * (sizeof(double) + sizeof(uint32_t)) + 3 * SORT_MAX_BUCKETS * sizeof(uint32_t);

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

struct Sort7 { const double* in[7]; double* tmp[7]; };

// step A for the seven arrays of one tile.  H: per-(bucket, tile) histogram, Hs: its exclusive scan.
__global__ void __launch_bounds__(SORT_STAGE_THREADS)
k_stage7_to_slots(uint32_t n, const uint32_t* __restrict__ dest, const uint32_t* __restrict__ H,
                  const uint32_t* __restrict__ Hs, int shift, uint32_t tiles, Sort7 a, uint32_t* __restrict__ tmpdest,
                  uint32_t* __restrict__ tmpidx /* or null */)
{
    extern __shared__ __align__(16) unsigned char stage_smem[];
    double* vals = reinterpret_cast<double*>(stage_smem);
    uint32_t* dsts = reinterpret_cast<uint32_t*>(vals + SORT_TILE);   // slot of the element at tile position lp
    uint32_t* base = dsts + SORT_TILE;          // first slot of this tile's share of bucket b
    uint32_t* toff = base + SORT_MAX_BUCKETS;   // where bucket b starts in the tile's bucket order
    uint32_t* cnt = toff + SORT_MAX_BUCKETS;    // arrivals so far
    __shared__ uint32_t total;
    const uint32_t nb = ((n - 1) >> shift) + 1;
    const uint32_t b = threadIdx.x;
    const uint32_t c = b < nb ? H[(size_t)b * tiles + blockIdx.x] : 0u;
    const uint32_t ex = block_exclusive_scan(c, &total);
    static_assert(SORT_MAX_BUCKETS <= SORT_STAGE_THREADS, "one thread per bucket in the tile-local scan");
    if (b < (uint32_t)SORT_MAX_BUCKETS) {
        toff[b] = ex;
        base[b] = b < nb ? Hs[(size_t)b * tiles + blockIdx.x] : 0u;
        cnt[b] = 0u;
    }
    __syncthreads();
    const size_t p0 = (size_t)blockIdx.x * SORT_TILE;
    const uint32_t tile_n = (uint32_t)min((size_t)SORT_TILE, (size_t)n - p0);
    uint32_t lp[SORT_PER_THREAD];               // this thread's elements: their positions in the tile's bucket order
    uint32_t* dvals = reinterpret_cast<uint32_t*>(vals);
#pragma unroll
    for (int j = 0; j < SORT_PER_THREAD; ++j) {
        const uint32_t e = threadIdx.x + j * SORT_STAGE_THREADS;
        lp[j] = 0xffffffffu;
        if (e < tile_n) {
            const uint32_t d = dest[p0 + e], bk = d >> shift;
            const uint32_t r = atomicAdd(&cnt[bk], 1u);
            lp[j] = toff[bk] + r;
            dsts[lp[j]] = base[bk] + r;
            dvals[lp[j]] = d;
        }
    }
    __syncthreads();
    for (uint32_t t = threadIdx.x; t < tile_n; t += SORT_STAGE_THREADS) tmpdest[dsts[t]] = dvals[t];
    __syncthreads();
    if (tmpidx) {
#pragma unroll
        for (int j = 0; j < SORT_PER_THREAD; ++j)
            if (lp[j] != 0xffffffffu) dvals[lp[j]] = (uint32_t)(p0 + threadIdx.x + j * SORT_STAGE_THREADS);
        __syncthreads();
        for (uint32_t t = threadIdx.x; t < tile_n; t += SORT_STAGE_THREADS) tmpidx[dsts[t]] = dvals[t];
        __syncthreads();
    }
#pragma unroll 1
    for (int k = 0; k < 7; ++k) {
        const double* __restrict__ in = a.in[k];
        double* __restrict__ tmp = a.tmp[k];
#pragma unroll
        for (int j = 0; j < SORT_PER_THREAD; ++j)
            if (lp[j] != 0xffffffffu) vals[lp[j]] = in[p0 + threadIdx.x + j * SORT_STAGE_THREADS];
        __syncthreads();
        for (uint32_t t = threadIdx.x; t < tile_n; t += SORT_STAGE_THREADS) tmp[dsts[t]] = vals[t];
        __syncthreads();
    }
}

struct Move7 { const double* src[7]; double* dst[7]; };

// step B, first half: the inverse of tmpdest, perm2[tmpdest[t]] = t (a 4-byte scatter that stays inside the bucket's
// window: L2), and the permutation for the caller if asked.  (Scattering the seven payload arrays the same way was
// measured: 5.5 ms per 33.5 M particles, every 8-byte store a read-modify-write of its DRAM sector; the gather below
// reads at random from the L2-resident window instead and writes whole sectors.)
__global__ void __launch_bounds__(256)
k_invert_slots(uint32_t n, const uint32_t* __restrict__ tmpdest, uint32_t* __restrict__ perm2,
               const uint32_t* __restrict__ tmpidx, uint32_t* __restrict__ perm_out)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += stride) {
        const uint32_t d = tmpdest[t];
        perm2[d] = (uint32_t)t;
        if (perm_out) perm_out[d] = tmpidx[t];
    }
}

// re-sort of a nearly sorted species: dst[new] = src[perm[new]], seven arrays, the permutation read once
__global__ void __launch_bounds__(256)
k_gather7(uint32_t n, const uint32_t* __restrict__ perm, Move7 a)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += stride) {
        const uint32_t q = perm[p];
#pragma unroll
        for (int k = 0; k < 7; ++k) a.dst[k][p] = a.src[k][q];
    }
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

// ecsim_validate_particles: particles with a non-finite coordinate, velocity or charge, or a position outside [0, L)
__global__ void __launch_bounds__(256)
k_validate(Geom g, size_t n, const double* __restrict__ x, const double* __restrict__ y, const double* __restrict__ z,
           const double* __restrict__ u, const double* __restrict__ v, const double* __restrict__ w,
           const double* __restrict__ q, unsigned long long* __restrict__ bad)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    unsigned mine = 0;
    for (size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += stride) {
        const double a = x[p], b = y[p], c = z[p];
        const bool ok = isfinite(u[p]) && isfinite(v[p]) && isfinite(w[p]) && isfinite(q[p]) &&
                        a >= 0.0 && a < g.Lx && b >= 0.0 && b < g.Ly && c >= 0.0 && c < g.Lz;   // (NaN fails every compare)
        mine += ok ? 0u : 1u;
    }
    mine = __reduce_add_sync(0xffffffffu, mine);
    if (lane_id() == 0 && mine) atomicAdd(bad, (unsigned long long)mine);
}
