// sort.cuh -- per-cell binning and counting sort of one species (PAPER.md L149:
// "sorting the particles and employing a reduction", which the paper could not realise in OpenACC).
//
//   k_cell_hist   cell id per particle (+ its rank inside the cell) and the per-cell histogram
//   k_scan_*      exclusive scan of the histogram -> start[cells+1]
//   k_build_perm  perm[start[cell] + rank] = old index
//   k_gather7     out[new] = in[perm[new]] for the seven SoA arrays (re-sort of a nearly sorted species)
//   k_stage_records / k_gather_records  the two-step move of a species in arbitrary order
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

// One thread per particle, HIST_ILP particles per thread and loop pass.  Lanes of a warp that fall in the same cell are
// aggregated with match_any so that a cell-sorted input costs one atomic per (warp, cell) instead of 32; for an input
// in arbitrary order every particle pays its own L2 atomic, whose round trip bounds the kernel: the HIST_ILP atomics of
// a pass are issued before the first result is used (33.5 M random particles: 1 per pass 0.52 ms, 4: 0.43, 8: 0.56).
constexpr int HIST_ILP = 4;
template <bool WITH_RANK>
__global__ void __launch_bounds__(256)
k_cell_hist(Geom g, uint32_t n, const double* __restrict__ x, const double* __restrict__ y,
            const double* __restrict__ z, int32_t* __restrict__ cell_out,
            uint32_t* __restrict__ rank_out, uint32_t* __restrict__ count)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    const size_t n_round = ((size_t)n + 31) & ~(size_t)31;   // keep whole warps in the loop
    const unsigned lane = lane_id(), lt = (1u << lane) - 1u;
    for (size_t p0 = (size_t)blockIdx.x * blockDim.x + threadIdx.x; p0 < n_round; p0 += stride * HIST_ILP) {
        int c[HIST_ILP];
        unsigned peers[HIST_ILP];
        uint32_t base[HIST_ILP];
#pragma unroll
        for (int j = 0; j < HIST_ILP; ++j) {
            const size_t p = p0 + (size_t)j * stride;
            c[j] = p < n ? cell_of(g, x[p], y[p], z[p]) : -1;
        }
#pragma unroll
        for (int j = 0; j < HIST_ILP; ++j) {
            const size_t p = p0 + (size_t)j * stride;
            base[j] = 0;
            peers[j] = 0;
            if (p < n_round) {                                // warp-uniform: p - lane is the same multiple of 32 for the warp
                peers[j] = __match_any_sync(0xffffffffu, c[j]);
                if (c[j] >= 0 && (int)lane == __ffs(peers[j]) - 1) base[j] = atomicAdd(&count[c[j]], (uint32_t)__popc(peers[j]));
            }
        }
#pragma unroll
        for (int j = 0; j < HIST_ILP; ++j) {
            const size_t p = p0 + (size_t)j * stride;
            if (p < n_round) {
                const uint32_t b = __shfl_sync(0xffffffffu, base[j], __ffs(peers[j]) - 1);
                if (c[j] >= 0) {
                    if (cell_out) cell_out[p] = c[j];
                    if (WITH_RANK) rank_out[p] = b + __popc(peers[j] & lt);
                }
            }
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
// profiles/r01d), and scattered 8-byte stores are read-modify-writes of their sectors, so the permutation is
// applied in two steps that are both local.  dest[p] = start[cell[p]] + rank[p] is the final place of particle p;
// places are cut into <= NB buckets of 2^shift consecutive places (every bucket is full,
// dest being a permutation).
//   step A, k_stage_records: a tile of TILE particles per CTA.  A particle's slot = (places of its bucket taken
//          by earlier tiles, from the scanned per-(bucket, tile) histogram) + (its arrival rank in the tile, a shared-
//          memory atomic).  The seven values of a particle are read once (coalesced SoA loads, 28 in flight per
//          thread at 1024, 14 at 512), put together as ONE 64-byte record {x,y,z,u,v,w,q, (dest, original index)} at the particle's position in
//          the tile's bucket order in shared memory, and the tile is written to tmp[] in runs of ~TILE/buckets
//          whole records: one load phase, one barrier, one store phase per tile (round 2 first moved array by array:
//          seven load / store phase pairs per tile, 128-byte runs, 1.52 ms per 33.5 M particles at 2.9 TB/s).
//   step B, k_invert_slots + k_gather_records: perm2 = tmpdest^-1, then place d takes record perm2[d]: four lanes read
//          one record (two whole sectors; the 8-byte gather of the SoA version fetched seven sectors per particle and
//          ran at 83 % of the L1 tag rate, ncu), a per-warp transposition in shared memory, seven coalesced stores.
//          The sources of the places in flight lie inside the windows of a few buckets (2^shift records of 64 B).
// tmp = eight spare arrays of the workspace.  Tile size, 33.5 M particles, step A + table kernels: 1024 records (3 CTAs
// per SM) 0.89 + 0.22 ms, 512 (5 CTAs) 0.76 + 0.27, 256 (8 CTAs) 0.85 + 0.38.
// Three geometries <buckets NB = threads of a step-A CTA, TILE>, chosen by the species' size so that a bucket stays at
// <= 131,072 places (step B's windows inside L2, the inverse built in shared memory): <256, 512> (5 CTAs per SM) up to 2^25
// particles, <512, 1024> up to 2^26, <1024, 2048> above.  With the first geometry alone the sort cost 0.069 ns per particle
// at 33.5 M particles but 0.085 / 0.092 / 0.105 at 50 / 67 / 134 M; with the three it stays at 0.070 - 0.072 (134 M: 9.7 ms).
constexpr int SORT_NB_SMALL = 256, SORT_TILE_SMALL = 512;
constexpr int SORT_NB_LARGE = 512, SORT_TILE_LARGE = 1024;
constexpr int SORT_NB_HUGE = 1024, SORT_TILE_HUGE = 2048;
constexpr uint32_t SORT_SMALL_MAX_N = 1u << 25, SORT_LARGE_MAX_N = 1u << 26;
constexpr size_t sort_stage_smem(int nb, int tile) { return (size_t)tile * (8 * sizeof(double) + sizeof(uint32_t)) + 3 * (size_t)nb * sizeof(uint32_t); }
// table entries (rows of NB per tile) and chunk sums for at most n particles, whichever geometry is used
constexpr int SORT_CHUNK = 128;
constexpr size_t sort_table_entries(size_t n) { return n / 2 + 2 * SORT_NB_HUGE; }
constexpr size_t sort_chunk_entries(size_t n) { return n / 256 + 2 * SORT_NB_HUGE; }

// dest (in place of rank), the per-(tile, bucket) histogram H[tile][b] and its tile-local exclusive scan T[tile][b]
// (where bucket b starts in the tile's bucket order); rows of NB entries, one CTA of NB threads per tile
template <int NB, int TILE>
__global__ void __launch_bounds__(NB)
k_dest_and_tile_hist(uint32_t n, const int32_t* __restrict__ cell, uint32_t* __restrict__ rank_to_dest,
                     const uint32_t* __restrict__ start, int shift, uint32_t* __restrict__ H, uint32_t* __restrict__ T)
{
    __shared__ uint32_t cnt[NB];
    __shared__ uint32_t total;
    cnt[threadIdx.x] = 0;
    __syncthreads();
    const size_t p0 = (size_t)blockIdx.x * TILE;
#pragma unroll
    for (int e = threadIdx.x; e < TILE; e += NB) {
        const size_t p = p0 + e;
        if (p < n) {
            const uint32_t d = start[cell[p]] + rank_to_dest[p];
            rank_to_dest[p] = d;
            atomicAdd(&cnt[d >> shift], 1u);
        }
    }
    __syncthreads();
    const uint32_t c = cnt[threadIdx.x];
    const uint32_t ex = block_exclusive_scan(c, &total);
    const size_t row = (size_t)blockIdx.x * NB + threadIdx.x;
    H[row] = c;
    T[row] = ex;
}

// First slot of every (tile, bucket) share: Hs[tile][b] = (b << shift) + sum of H[t][b] over the tiles t < tile (every
// bucket holds exactly 2^shift places).  Column-wise running sums, thread = bucket (blockDim.x = NB = the row pitch), in
// chunks of SORT_CHUNK tiles: column sums per chunk, their running sums over the chunks, then the rows of every chunk.
__global__ void __launch_bounds__(SORT_NB_HUGE)
k_tile_colsum(uint32_t tiles, const uint32_t* __restrict__ H, uint32_t* __restrict__ S)
{
    const uint32_t nb = blockDim.x, t0 = blockIdx.x * SORT_CHUNK, t1 = min(t0 + (uint32_t)SORT_CHUNK, tiles);
    uint32_t sum = 0;
    for (uint32_t t = t0; t < t1; ++t) sum += H[(size_t)t * nb + threadIdx.x];
    S[(size_t)blockIdx.x * nb + threadIdx.x] = sum;
}

__global__ void __launch_bounds__(SORT_NB_HUGE)
k_tile_chunkscan(uint32_t chunks, uint32_t* __restrict__ S)
{
    const uint32_t nb = blockDim.x;
    uint32_t run = 0;
    for (uint32_t ch = 0; ch < chunks; ++ch) {
        const size_t i = (size_t)ch * nb + threadIdx.x;
        const uint32_t v = S[i];
        S[i] = run;
        run += v;
    }
}

__global__ void __launch_bounds__(SORT_NB_HUGE)
k_tile_colscan(uint32_t tiles, int shift, const uint32_t* __restrict__ H, const uint32_t* __restrict__ S,
               uint32_t* __restrict__ Hs)
{
    const uint32_t nb = blockDim.x, t0 = blockIdx.x * SORT_CHUNK, t1 = min(t0 + (uint32_t)SORT_CHUNK, tiles);
    uint32_t run = (threadIdx.x << shift) + S[(size_t)blockIdx.x * nb + threadIdx.x];
    for (uint32_t t = t0; t < t1; ++t) {
        const size_t i = (size_t)t * nb + threadIdx.x;
        const uint32_t v = H[i];
        Hs[i] = run;
        run += v;
    }
}

struct Sort7 { const double* in[7]; };

// step A: the records of one tile.  T: where bucket b starts in the tile's bucket order, Hs: the first slot of the tile's
// share of bucket b.
template <int NB, int TILE>
__global__ void __launch_bounds__(NB, NB == SORT_NB_SMALL ? 5 : (NB == SORT_NB_LARGE ? 2 : 1))
k_stage_records(uint32_t n, const uint32_t* __restrict__ dest, const uint32_t* __restrict__ T,
                const uint32_t* __restrict__ Hs, int shift, Sort7 a, double* __restrict__ tmp,
                uint32_t* __restrict__ tmpdest)
{
    extern __shared__ __align__(16) unsigned char stage_smem[];
    double* rec = reinterpret_cast<double*>(stage_smem);
    uint32_t* slot = reinterpret_cast<uint32_t*>(rec + (size_t)TILE * 8);   // slot of the record at tile position lp
    uint32_t* base = slot + TILE;          // first slot of this tile's share of bucket b
    uint32_t* toff = base + NB;   // where bucket b starts in the tile's bucket order
    uint32_t* cnt = toff + NB;    // arrivals so far
    constexpr int PER_THREAD = TILE / NB;
    {
        const size_t row = (size_t)blockIdx.x * NB + threadIdx.x;
        toff[threadIdx.x] = T[row];
        base[threadIdx.x] = Hs[row];
        cnt[threadIdx.x] = 0u;
    }
    const size_t p0 = (size_t)blockIdx.x * TILE;
    const uint32_t tile_n = (uint32_t)min((size_t)TILE, (size_t)n - p0);
    // load phase: all 7 x PER_THREAD values of this thread are requested before the first is used
    double v[PER_THREAD][7];
    uint32_t d[PER_THREAD];
#pragma unroll
    for (int j = 0; j < PER_THREAD; ++j) {
        const uint32_t e = threadIdx.x + j * NB;
        if (e < tile_n) {
            d[j] = dest[p0 + e];
#pragma unroll
            for (int k = 0; k < 7; ++k) v[j][k] = a.in[k][p0 + e];
        }
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < PER_THREAD; ++j) {
        const uint32_t e = threadIdx.x + j * NB;
        if (e < tile_n) {
            const uint32_t bk = d[j] >> shift;
            const uint32_t r = atomicAdd(&cnt[bk], 1u);
            const uint32_t lp = toff[bk] + r;
            slot[lp] = base[bk] + r;
            // 16-byte piece p of the record at tile position lp sits at piece p ^ ((lp >> 1) & 3): the four STS.128 of a warp
            // (one piece each, scattered lp) spread over all eight 16-byte bank groups
            double2* w = reinterpret_cast<double2*>(rec + (size_t)lp * 8);
            const uint32_t sw = (lp >> 1) & 3u;
            w[0u ^ sw] = make_double2(v[j][0], v[j][1]);
            w[1u ^ sw] = make_double2(v[j][2], v[j][3]);
            w[2u ^ sw] = make_double2(v[j][4], v[j][5]);
            // the original index (low word) and the final place (high word) travel with the record
            w[3u ^ sw] = make_double2(v[j][6], __longlong_as_double((long long)(((unsigned long long)d[j] << 32) | (unsigned long long)(p0 + e))));
        }
    }
    __syncthreads();
    // store phase: 16-byte pieces, consecutive threads = consecutive pieces of consecutive records of a run
    for (uint32_t t = threadIdx.x; t < tile_n * 4u; t += NB) {
        const uint32_t r = t >> 2, part = t & 3u;
        const double2 pr = *reinterpret_cast<const double2*>(rec + (size_t)r * 8 + 2u * (part ^ ((r >> 1) & 3u)));
        *reinterpret_cast<double2*>(tmp + (size_t)slot[r] * 8 + 2u * part) = pr;
    }
    for (uint32_t t = threadIdx.x; t < tile_n; t += NB)
        tmpdest[slot[t]] = (uint32_t)((unsigned long long)__double_as_longlong(rec[(size_t)t * 8 + 2u * (3u ^ ((t >> 1) & 3u)) + 1u]) >> 32);
}

struct Move7 { const double* src[7]; double* dst[7]; };

// step B, first half: the inverse of tmpdest, perm2[tmpdest[t]] = t (a 4-byte scatter that stays inside the bucket's
// window: L2).  (Scattering the payload the same way was measured: 5.5 ms per 33.5 M particles, every 8-byte store a
// read-modify-write of its DRAM sector; the gather below reads whole records and writes whole sectors.)
__global__ void __launch_bounds__(256)
k_invert_slots(uint32_t n, const uint32_t* __restrict__ tmpdest, uint32_t* __restrict__ perm2)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += stride) perm2[tmpdest[t]] = (uint32_t)t;
}

// The same inverse without the scattered global stores, for buckets of <= 4 x INV_SUB places: a CTA owns INV_SUB consecutive
// places of one bucket, streams the bucket's tmpdest window (coalesced; the window's other CTAs read it from L2), keeps the
// entries that point into its places in shared memory and writes its part of perm2 coalesced.  (33.5 M particles: 0.29 ms
// as a scatter -- 117 G partial L2 writes per second -- against the time below.)
constexpr int INV_SUB = 32768;
constexpr int INV_THREADS = 1024;
__global__ void __launch_bounds__(INV_THREADS)
k_invert_slots_local(uint32_t n, int shift, const uint32_t* __restrict__ tmpdest, uint32_t* __restrict__ perm2)
{
    extern __shared__ uint32_t inv_smem[];
    const uint32_t bucket_places = 1u << shift;
    const uint32_t sub = min(bucket_places, (uint32_t)INV_SUB), subs_per_bucket = bucket_places / sub;
    const uint32_t bucket = blockIdx.x / subs_per_bucket, part = blockIdx.x % subs_per_bucket;
    const size_t b0 = (size_t)bucket << shift, b1 = min(b0 + bucket_places, (size_t)n);
    const size_t lo = b0 + (size_t)part * sub;
    if (lo >= b1) return;
    const uint32_t len = (uint32_t)min((size_t)sub, b1 - lo);
    for (size_t t0 = b0 + threadIdx.x; t0 < b1; t0 += 8 * INV_THREADS) {      // eight loads in flight per thread
        uint32_t d[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const size_t t = t0 + (size_t)j * INV_THREADS;
            d[j] = t < b1 ? __ldg(tmpdest + t) : 0xffffffffu;
        }
#pragma unroll
        for (int j = 0; j < 8; ++j)
            if (d[j] >= lo && d[j] - lo < len) inv_smem[d[j] - (uint32_t)lo] = (uint32_t)(t0 + (size_t)j * INV_THREADS);
    }
    __syncthreads();
    for (uint32_t i = threadIdx.x; i < len; i += INV_THREADS) perm2[lo + i] = inv_smem[i];
}

struct Out7 { double* dst[7]; };

// L2 residency hints of the gather: the two records of a 128-byte line are wanted at unrelated moments while their
// bucket is in flight, so the record loads ask to be evicted last and everything streamed (places, outputs) first
// (without the hints the records were fetched from DRAM 1.7 times each, ncu dram__bytes_read)
__device__ __forceinline__ unsigned long long l2_policy_evict_last()
{
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ double2 ld_evict_last_f64x2(const double* p, unsigned long long pol)
{
    double2 v;
    asm volatile("ld.global.L2::cache_hint.v2.f64 {%0, %1}, [%2], %3;" : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(pol));
    return v;
}

// step B, second half: place d takes record perm2[d].  A warp owns 32 consecutive places; lanes 4j..4j+3 read the four
// 16-byte pieces of one record (8 records per load instruction), the warp transposes through shared memory (pitch 9:
// conflict-free) and writes the seven arrays (and the permutation, if asked) coalesced.
constexpr int GATHER_WARPS = 8;
__global__ void __launch_bounds__(GATHER_WARPS * 32)
k_gather_records(uint32_t n, const uint32_t* __restrict__ perm2, const double* __restrict__ tmp, Out7 a,
                 uint32_t* __restrict__ perm_out /* or null */)
{
    __shared__ double stage[GATHER_WARPS][32 * 9];
    const unsigned lane = lane_id(), warp = threadIdx.x >> 5;
    double* st = stage[warp];
    const uint32_t j = lane >> 2, part = lane & 3u;
    const size_t chunks = ((size_t)n + 31) / 32;
    const unsigned long long keep = l2_policy_evict_last();
    for (size_t ch = (size_t)blockIdx.x * GATHER_WARPS + warp; ch < chunks; ch += (size_t)gridDim.x * GATHER_WARPS) {
        const size_t dp = ch * 32 + lane;
        const uint32_t q = dp < n ? __ldcs(perm2 + dp) : 0u;
        double2 pr[4];
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const uint32_t src = __shfl_sync(0xffffffffu, q, 8 * r + (int)j);
            pr[r] = ld_evict_last_f64x2(tmp + (size_t)src * 8 + 2u * part, keep);
        }
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            double* w = st + (8 * r + j) * 9 + 2 * part;
            w[0] = pr[r].x; w[1] = pr[r].y;
        }
        __syncwarp();
        if (dp < n) {
#pragma unroll
            for (int k = 0; k < 7; ++k) __stcs(a.dst[k] + dp, st[lane * 9 + k]);
            if (perm_out) __stcs(perm_out + dp, (uint32_t)__double_as_longlong(st[lane * 9 + 7]));
        }
        __syncwarp();
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
