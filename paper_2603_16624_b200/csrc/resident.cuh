// resident.cuh -- layout kernels of a RESIDENT species (LAYOUT_GAPPED of fused_mma.cuh, the
// sort-preserving push; PAPER.md L149 is the paper's own, unrealised, "sorting the particles").
//
// A resident species lives in two library-managed buffers of seven arrays (x,y,z,u,v,w,q).  Cell c owns the slots
// [seg[c], seg[c+1]) of both: its particles plus slack.  In the buffer being read, cell c holds a front run of F[c]
// particles from seg[c] upwards and a back run of R[c] particles from seg[c+1]-1 downwards.  The kernels here build
// that layout from dense arrays (after the binning of sort.cuh), turn it back into dense cell-ordered arrays, and
// append the overflow list of a push before a fresh layout.  Integer / copy work only.
#pragma once
#include "common.cuh"

struct Soa7 { double* a[7]; };
struct Soa7c { const double* a[7]; };

// slots of cell c = its particles + max(min_slack, ceil(slack * max(particles, mean particles per cell))), rounded up to a
// multiple of 4 (32-byte sector alignment of every segment).  The mean enters because the arrivals of a step scale with
// the population of the NEIGHBOURHOOD, not of the cell itself: a depleted cell beside a dense one needs room too.
__global__ void __launch_bounds__(256)
k_gapped_caps(uint32_t cells, const uint32_t* __restrict__ count, double slack, uint32_t min_slack, double mean,
              uint32_t* __restrict__ cap)
{
    const uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= cells) return;
    const uint32_t n = count[c];
    uint32_t extra = (uint32_t)ceil(slack * fmax((double)n, mean));
    if (extra < min_slack) extra = min_slack;
    cap[c] = (n + extra + 3u) & ~3u;
}

// dense (any order, binned by k_cell_hist<true>) -> gapped front runs: dst[seg[cell[p]] + rank[p]] = src[p]
__global__ void __launch_bounds__(256)
k_scatter_gapped(uint32_t n, const int32_t* __restrict__ cell, const uint32_t* __restrict__ rank,
                 const uint32_t* __restrict__ seg, Soa7c src, Soa7 dst)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += stride) {
        const uint32_t d = seg[cell[p]] + rank[p];
#pragma unroll
        for (int k = 0; k < 7; ++k) dst.a[k][d] = src.a[k][p];
    }
}

__global__ void __launch_bounds__(256)
k_runs_from_count(uint32_t cells, const uint32_t* __restrict__ count, uint32_t* __restrict__ F, uint32_t* __restrict__ R)
{
    const uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c < cells) { F[c] = count[c]; R[c] = 0u; }
}

__global__ void __launch_bounds__(256)
k_run_totals(uint32_t cells, const uint32_t* __restrict__ F, const uint32_t* __restrict__ R, uint32_t* __restrict__ total)
{
    const uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c < cells) total[c] = F[c] + R[c];
}

// gapped -> dense, cell-major: one warp per cell (grid-stride); start = exclusive scan of F + R
__global__ void __launch_bounds__(256)
k_export_gapped(uint32_t cells, const uint32_t* __restrict__ seg, const uint32_t* __restrict__ F,
                const uint32_t* __restrict__ R, const uint32_t* __restrict__ start, Soa7c src, Soa7 dst)
{
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t warps = (gridDim.x * blockDim.x) >> 5;
    for (uint32_t c = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; c < cells; c += warps) {
        const uint32_t s0 = seg[c], s1 = seg[c + 1], nf = F[c], nt = nf + R[c], d0 = start[c];
        for (uint32_t v = lane; v < nt; v += 32u) {
            const uint32_t p = v < nf ? s0 + v : s1 - 1u - (v - nf);
#pragma unroll
            for (int k = 0; k < 7; ++k) dst.a[k][d0 + v] = src.a[k][p];
        }
    }
}

// the overflow list of the last push, appended behind the exported particles: dst[*base + i] = ovf[k][i]
__global__ void __launch_bounds__(256)
k_append_overflow(const uint32_t* __restrict__ count, uint32_t ovf_cap, const double* __restrict__ ovf,
                  const uint32_t* __restrict__ base, Soa7 dst)
{
    const uint32_t n = min(*count, ovf_cap), b = *base;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
#pragma unroll
        for (int k = 0; k < 7; ++k) dst.a[k][b + i] = ovf[(size_t)k * ovf_cap + i];
    }
}

// ---- a fresh layout straight from the gapped buffer (the particles are binned already: only the segments move) ----
// cell of every particle of an overflow list, added to the per-cell totals
__global__ void __launch_bounds__(256)
k_count_list(Geom g, const uint32_t* __restrict__ n_ptr, uint32_t cap, const double* __restrict__ list,
             uint32_t* __restrict__ count)
{
    const uint32_t n = min(*n_ptr, cap);
    const size_t stride = (size_t)gridDim.x * blockDim.x, m = cap;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const int ci = lower_node(list[i] * g.rdx, g.nx), cj = lower_node(list[m + i] * g.rdy, g.ny),
                  ck = lower_node(list[2 * m + i] * g.rdz, g.nz);
        atomicAdd(&count[(ci * g.ny + cj) * g.nz + ck], 1u);
    }
}

// old segments (front + back runs) -> front runs of the new segments in the other buffer; F_new = F + R, R_new = 0
__global__ void __launch_bounds__(256)
k_copy_gapped(uint32_t cells, const uint32_t* __restrict__ seg, const uint32_t* __restrict__ F,
              const uint32_t* __restrict__ R, const uint32_t* __restrict__ seg_new, uint32_t* __restrict__ F_new,
              uint32_t* __restrict__ R_new, Soa7c src, Soa7 dst)
{
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t warps = (gridDim.x * blockDim.x) >> 5;
    for (uint32_t c = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; c < cells; c += warps) {
        const uint32_t s0 = seg[c], s1 = seg[c + 1], nf = F[c], nt = nf + R[c], d0 = seg_new[c];
        for (uint32_t v = lane; v < nt; v += 32u) {
            const uint32_t p = v < nf ? s0 + v : s1 - 1u - (v - nf);
#pragma unroll
            for (int k = 0; k < 7; ++k) dst.a[k][d0 + v] = src.a[k][p];
        }
        if (lane == 0) { F_new[c] = nt; R_new[c] = 0u; }
    }
}

// the particles of an overflow list into the back runs of the new segments (room is certain: the new capacities
// counted them)
__global__ void __launch_bounds__(256)
k_place_list(Geom g, const uint32_t* __restrict__ n_ptr, uint32_t cap, const double* __restrict__ list,
             const uint32_t* __restrict__ seg_new, uint32_t* __restrict__ R_new, Soa7 dst)
{
    const uint32_t n = min(*n_ptr, cap);
    const size_t stride = (size_t)gridDim.x * blockDim.x, m = cap;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const int ci = lower_node(list[i] * g.rdx, g.nx), cj = lower_node(list[m + i] * g.rdy, g.ny),
                  ck = lower_node(list[2 * m + i] * g.rdz, g.nz);
        const uint32_t c = (uint32_t)((ci * g.ny + cj) * g.nz + ck);
        const uint32_t pos = seg_new[c + 1] - 1u - atomicAdd(&R_new[c], 1u);
#pragma unroll
        for (int k = 0; k < 7; ++k) dst.a[k][pos] = list[(size_t)k * m + i];
    }
}
