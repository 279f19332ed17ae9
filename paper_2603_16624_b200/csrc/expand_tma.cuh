// expand_tma.cuh -- k_expand_M_stream: the expansion of the per-cell class sums AM to the node array M
// (second half) as a streaming kernel whose loads are TMA bulk copies.
//
// A CTA of 128 threads walks one (i,j) column of nodes along z.  Node (i,j,k) needs the class sums of the
// 8 cells (i-1..i, j-1..j, k-1..k): four cell columns, two consecutive z levels.  The four cells of one z level
// are four contiguous 1952-byte blocks of AM; thread 0 requests them with cp.async.bulk into a ring of XS_RING
// stages in shared memory, each stage signalled by an mbarrier (expect_tx = 7808 bytes).  The loads in flight
// therefore cost no registers and no issue slots, and shared memory -- not the register file -- sets how many
// CTAs an SM holds (ring of 3 = 23.4 KB: 9 CTAs).  Per node every thread reads <= 8 terms per output from
// shared memory (term lists: expand.cuh) and writes its outputs with plain stores; only thread 0 polls the
// mbarrier, the others wait in the hardware barrier; a second __syncthreads orders "everybody has read the
// previous level" before its slot is refilled.
// Measured on config 2 (whole grid, profiles/r01c): 2.0 ms with 128 threads x ring 3; 2.2 ms (128 x 4),
// 2.4 ms (256 x 3), 2.8 ms (64 x 3), 3.2 ms (128 x 5); the register-staged k_expand_M it replaces: 2.95 ms.
#pragma once
#include "common.cuh"
#include "fused_mma.cuh"
#include "expand.cuh"

#ifndef XS_THREADS_N
#define XS_THREADS_N 128
#endif
#ifndef XS_RING_N
#define XS_RING_N 3
#endif
constexpr int XS_THREADS = XS_THREADS_N;
constexpr int XS_RING = XS_RING_N;
constexpr int XS_OUT = (243 + XS_THREADS - 1) / XS_THREADS;   // outputs per thread
constexpr int XS_STAGE_DOUBLES = 4 * AM_PER_CELL;                       // cells (i,j), (i,j-1), (i-1,j), (i-1,j-1)
constexpr int XS_STAGE_BYTES = XS_STAGE_DOUBLES * 8;                    // 7808
constexpr int XS_SMEM_BYTES = XS_RING * XS_STAGE_BYTES + XS_RING * 8;   // ring + mbarriers

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, 0x989680;\n"   // suspend-time hint (ns)
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

struct ExpandStreamArgs {
    Geom g;
    const double* AM;   // [cells][AM_PER_CELL]
    double* M;          // [nodes][27][3][3]
    int accumulate;
    int i0, i1;         // node planes [i0, i1) of this launch
};

// Stage G of a CTA's sequence: column item G / (nz+1), level q = G % (nz+1); q = 0 holds the cells at z = nz-1
// (the "k-1" of node 0), q >= 1 the cells at z = q-1.
__device__ __forceinline__ void xs_issue_stage(const ExpandStreamArgs& a, uint32_t G, uint32_t n_stages, int first_item,
                                               int item_stride, double* ring, uint64_t* bars)
{
    if (G >= n_stages) return;
    const Geom& g = a.g;
    const int per_col = g.nz + 1;
    const int item = first_item + (int)(G / per_col) * item_stride;
    const int q = (int)(G % per_col);
    const int i = a.i0 + item / g.ny, j = item % g.ny;
    const int im1 = i ? i - 1 : g.nx - 1, jm1 = j ? j - 1 : g.ny - 1;
    const int z = q ? q - 1 : g.nz - 1;
    const int slot = (int)(G % XS_RING);
    double* dst = ring + (size_t)slot * XS_STAGE_DOUBLES;
    uint64_t* bar = bars + slot;
    mbar_expect_tx(bar, XS_STAGE_BYTES);
    const int ci[4] = {i, i, im1, im1}, cj[4] = {j, jm1, j, jm1};
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const double* src = a.AM + (((size_t)ci[c] * g.ny + cj[c]) * g.nz + z) * AM_PER_CELL;
        bulk_g2s(dst + c * AM_PER_CELL, src, AM_PER_CELL * 8, bar);
    }
}

__global__ void __launch_bounds__(XS_THREADS, 1024 / XS_THREADS)   // <= 64 registers
k_expand_M_stream(const __grid_constant__ ExpandStreamArgs a)
{
    extern __shared__ __align__(128) unsigned char xs_smem[];
    double* ring = reinterpret_cast<double*>(xs_smem);
    uint64_t* bars = reinterpret_cast<uint64_t*>(xs_smem + (size_t)XS_RING * XS_STAGE_BYTES);
    const Geom& g = a.g;
    const int tid = threadIdx.x;
    const int n_items = (a.i1 - a.i0) * g.ny;
    const int first_item = blockIdx.x, item_stride = gridDim.x;
    if (first_item >= n_items) return;
    const int my_items = (n_items - first_item + item_stride - 1) / item_stride;
    const int per_col = g.nz + 1;
    const uint32_t n_stages = (uint32_t)my_items * (uint32_t)per_col;   // < 2^32: a CTA's columns x (nz + 1)

    if (tid == 0) {
        for (int s = 0; s < XS_RING; ++s) mbar_init(bars + s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0)
        for (int s = 0; s < XS_RING; ++s) xs_issue_stage(a, s, n_stages, first_item, item_stride, ring, bars);

    // the four outputs of this thread: elements e = tid + 64 m of the 243, in the order of EXPAND_ORDER.
    // Packed per output: offsets (in doubles, inside a stage) of its <= 4 x-y terms, and its z list.
    unsigned offs01[XS_OUT], offs23[XS_OUT], zinfo[XS_OUT];
    int mbase[XS_OUT];
#pragma unroll
    for (int m = 0; m < XS_OUT; ++m) {
        const int e = tid + XS_THREADS * m;
        const int ee = e < 243 ? e : 0;
        const int o = EXPAND_ORDER[ee / 9], ij = ee % 9;
        const int dx = o / 9 - 1, dy = (o / 3) % 3 - 1, dz = o % 3 - 1;
        const int ebase = ij < 8 ? ij : AM_A8, emul = ij < 8 ? 8 : 1;
        const int ntx = dx == 0 ? 2 : 1, nty = dy == 0 ? 2 : 1, ntz = dz == 0 ? 2 : 1;
        const int nxy = ntx * nty;
        unsigned off[4];
#pragma unroll
        for (int t = 0; t < 4; ++t) {
            const int tt = t < nxy ? t : 0;
            const int ty = tt % nty, tx = tt / nty;
            // column slot = xsel*2 + ysel, sel 0 = own (i or j), 1 = previous
            const int xsel = tx == 0 ? (dx >= 0 ? 0 : 1) : 1, cx = tx == 0 ? (dx == 0 ? 0 : 1) : 2;
            const int ysel = ty == 0 ? (dy >= 0 ? 0 : 1) : 1, cy = ty == 0 ? (dy == 0 ? 0 : 1) : 2;
            off[t] = (unsigned)((xsel * 2 + ysel) * AM_PER_CELL + ebase + emul * (9 * cx + 3 * cy));
        }
        offs01[m] = off[0] | (off[1] << 16);
        offs23[m] = off[2] | (off[3] << 16);
        // z list: dz = 0: (own level, class 0), (previous level, class 2); dz = +1: (own, 1); dz = -1: (previous, 1)
        const unsigned ezA = (unsigned)(emul * (dz == 0 ? 0 : 1)), ezB = (unsigned)(emul * 2);
        zinfo[m] = ezA | (ezB << 8) | ((unsigned)nxy << 16) | ((unsigned)(ntz == 2) << 24) | ((unsigned)(dz < 0) << 25) |
                   ((unsigned)(e < 243) << 26);
        mbase[m] = o * 9 + ij;
    }

    uint32_t G = 0;     // stage holding the "previous level" of the node being computed
#pragma unroll 1
    for (int it = 0; it < my_items; ++it) {
        const int item = first_item + it * item_stride;
        const int i = a.i0 + item / g.ny, j = item % g.ny;
        double* mcol = a.M + ((size_t)i * g.ny + j) * g.nz * 243;
        // level q = 0 of this column.  Only thread 0 polls the mbarriers; the others sit in the hardware barrier
        // and take no issue slots from the fused CTA next door.
        if (tid == 0) mbar_wait(bars + (int)(G % XS_RING), (unsigned)((G / XS_RING) & 1));
#pragma unroll 1
        for (int k = 0; k < g.nz; ++k) {
            const uint32_t Gown = G + 1;
            if (tid == 0) mbar_wait(bars + (int)(Gown % XS_RING), (unsigned)((Gown / XS_RING) & 1));
            __syncthreads();
            const double* prev = ring + (size_t)(G % XS_RING) * XS_STAGE_DOUBLES;
            const double* own = ring + (size_t)(Gown % XS_RING) * XS_STAGE_DOUBLES;
            double* mnode = mcol + (size_t)k * 243;
#pragma unroll
            for (int m = 0; m < XS_OUT; ++m) {
                const unsigned zi = zinfo[m];
                if (!((zi >> 26) & 1u)) continue;
                const int nxy = (int)((zi >> 16) & 0xffu);
                const double* zA = (((zi >> 25) & 1u) ? prev : own) + (zi & 0xffu);
                const double* zB = prev + ((zi >> 8) & 0xffu);
                const bool two = (zi >> 24) & 1u;
                double s = a.accumulate ? mnode[mbase[m]] : 0.0;
                const unsigned o4[4] = {offs01[m] & 0xffffu, offs01[m] >> 16, offs23[m] & 0xffffu, offs23[m] >> 16};
#pragma unroll
                for (int t = 0; t < 4; ++t) {
                    if (t < nxy) {
                        s += zA[o4[t]];
                        if (two) s += zB[o4[t]];
                    }
                }
                mnode[mbase[m]] = s;
            }
            __syncthreads();                                   // stage G has been read by everybody: refill its slot
            if (tid == 0) xs_issue_stage(a, G + XS_RING, n_stages, first_item, item_stride, ring, bars);
            G = Gown;
        }
        // the last level of the column is nobody's "previous" (the barrier above covers its readers): refill it too
        if (tid == 0) xs_issue_stage(a, G + XS_RING, n_stages, first_item, item_stride, ring, bars);
        G += 1;
    }
}
