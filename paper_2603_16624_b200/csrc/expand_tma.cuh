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
// previous level" before its slot is refilled.  Slots, mbarrier phases and output pointers advance incrementally
// and the term loops are shaped per warp (the first version spent 640 warp instructions per node, 90 % of them
// address arithmetic and divergence bookkeeping).
// Measured on config 2 (whole grid, profiles/r01c): 1.68 ms with 128 threads x ring 3 (128 x 4, 256 x 4 and 96 x 3
// are within 2 % of it, 256 x 3 and 64 x 3 slower); the register-staged k_expand_M it replaces: 2.95 ms.
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
// (with an L2 evict-last policy: a cell's class sums are read by the four node columns around it, at different moments)
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, uint64_t* bar, unsigned long long pol)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(pol) : "memory");
}

struct ExpandStreamArgs {
    Geom g;
    const double* AM;   // [cells][AM_PER_CELL]
    double* M;          // [nodes][NSLOT][3][3]
    int accumulate;
    int i0, i1;         // node planes [i0, i1) of this launch
};

__device__ __forceinline__ double lds_f64(uint32_t addr)
{
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
    return v;
}

// Sum of one output's terms at one node.  NXY / TWO are the warp-wide longest lists (warp-uniform: no divergence);
// a lane with a shorter list reads its term 0 again and adds nothing.  offA / offB: byte addresses (shared space) of
// the output's z-list entries in the stages that hold them; o[t]: byte offsets of its x-y terms inside a stage.
template <int NXY, bool TWO>
__device__ __forceinline__ double xs_sum(double s, uint32_t offA, uint32_t offB, const uint32_t (&o)[4], int nxy, bool two)
{
    double vA[NXY], vB[NXY];
#pragma unroll
    for (int t = 0; t < NXY; ++t) {
        vA[t] = lds_f64(offA + o[t]);
        if (TWO) vB[t] = lds_f64(offB + o[t]);
    }
#pragma unroll
    for (int t = 0; t < NXY; ++t) {
        s += t < nxy ? vA[t] : 0.0;
        if (TWO) s += (t < nxy && two) ? vB[t] : 0.0;
    }
    return s;
}

// One CTA per (i,j) column of nodes; stage q = 0 holds the cells at z = nz-1 (the "k-1" of node 0), stage q >= 1 the
// cells at z = q-1; node k reads stages k ("previous level") and k+1 ("own level"); stage q lives in slot q % XS_RING.
// NSLOT = 27: every neighbour slot (the north-star layout).  NSLOT = 14: the symmetric storage of the paper (L73, L129):
// only the slots o >= 13 (self and the 13 "upper" neighbours) are written, M14[node][o - 13][3][3]; the others follow
// from M[g][o] = M[g + off(o)][26 - o].
template <int NSLOT>
__global__ void __launch_bounds__(XS_THREADS, 1024 / XS_THREADS)   // <= 64 registers
k_expand_M_stream(const __grid_constant__ ExpandStreamArgs a)
{
    constexpr int NOUT = NSLOT * 9;
    constexpr int XS_OUT = (NOUT + XS_THREADS - 1) / XS_THREADS;   // outputs per thread
    extern __shared__ __align__(128) unsigned char xs_smem[];
    double* ring = reinterpret_cast<double*>(xs_smem);
    uint64_t* bars = reinterpret_cast<uint64_t*>(xs_smem + (size_t)XS_RING * XS_STAGE_BYTES);
    const Geom& g = a.g;
    const int tid = threadIdx.x;
    const int i = a.i0 + (int)(blockIdx.x / (unsigned)g.ny), j = (int)(blockIdx.x % (unsigned)g.ny);
    const int im1 = i ? i - 1 : g.nx - 1, jm1 = j ? j - 1 : g.ny - 1;
    const int n_stages = g.nz + 1;
    // the four cell columns of this node column: (i,j), (i,j-1), (i-1,j), (i-1,j-1)
    const double* colsrc[4] = {a.AM + ((size_t)i * g.ny + j) * g.nz * AM_PER_CELL,
                               a.AM + ((size_t)i * g.ny + jm1) * g.nz * AM_PER_CELL,
                               a.AM + ((size_t)im1 * g.ny + j) * g.nz * AM_PER_CELL,
                               a.AM + ((size_t)im1 * g.ny + jm1) * g.nz * AM_PER_CELL};
    unsigned long long keep;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(keep));
    auto issue = [&](int q) {      // thread 0 only
        if (q >= n_stages) return;
        const int z = q ? q - 1 : g.nz - 1;
        const int slot = q % XS_RING;
        uint64_t* bar = bars + slot;
        mbar_expect_tx(bar, XS_STAGE_BYTES);
#pragma unroll
        for (int c = 0; c < 4; ++c)
            bulk_g2s(ring + (size_t)slot * XS_STAGE_DOUBLES + c * AM_PER_CELL, colsrc[c] + (size_t)z * AM_PER_CELL,
                     AM_PER_CELL * 8, bar, keep);
    };

    if (tid == 0) {
        for (int s = 0; s < XS_RING; ++s) mbar_init(bars + s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0)
        for (int s = 0; s < XS_RING; ++s) issue(s);

    // the outputs of this thread: elements e = tid + XS_THREADS m of the NOUT, in the order of EXPAND_ORDER
    uint32_t off[XS_OUT][4];       // byte offsets of the <= 4 x-y terms inside a stage (term 0 repeated when fewer)
    uint32_t ezA[XS_OUT], ezB[XS_OUT];
    int nxy[XS_OUT], wxy[XS_OUT];
    bool two[XS_OUT], wtwo[XS_OUT], a_prev[XS_OUT], valid[XS_OUT];
    double* mptr[XS_OUT];
#pragma unroll
    for (int m = 0; m < XS_OUT; ++m) {
        const int e = tid + XS_THREADS * m;
        valid[m] = e < NOUT;
        const int ee = valid[m] ? e : 0;
        const int o = NSLOT == 27 ? EXPAND_ORDER[ee / 9] : EXPAND_ORDER14[ee / 9], ij = ee % 9;
        const int dx = o / 9 - 1, dy = (o / 3) % 3 - 1, dz = o % 3 - 1;
        const int ebase = ij < 8 ? ij : AM_A8, emul = ij < 8 ? 8 : 1;
        const int ntx = dx == 0 ? 2 : 1, nty = dy == 0 ? 2 : 1;
        nxy[m] = ntx * nty;
        two[m] = dz == 0;
#pragma unroll
        for (int t = 0; t < 4; ++t) {
            const int tt = t < nxy[m] ? t : 0;
            const int ty = tt % nty, tx = tt / nty;
            // column slot = xsel*2 + ysel, sel 0 = own (i or j), 1 = previous
            const int xsel = tx == 0 ? (dx >= 0 ? 0 : 1) : 1, cx = tx == 0 ? (dx == 0 ? 0 : 1) : 2;
            const int ysel = ty == 0 ? (dy >= 0 ? 0 : 1) : 1, cy = ty == 0 ? (dy == 0 ? 0 : 1) : 2;
            off[m][t] = 8u * (unsigned)((xsel * 2 + ysel) * AM_PER_CELL + ebase + emul * (9 * cx + 3 * cy));
        }
        // z list: dz = 0: (own level, class 0), (previous level, class 2); dz = +1: (own, 1); dz = -1: (previous, 1)
        ezA[m] = 8u * (unsigned)(emul * (dz == 0 ? 0 : 1));
        ezB[m] = 8u * (unsigned)(emul * 2);
        a_prev[m] = dz < 0;
        mptr[m] = a.M + ((size_t)i * g.ny + j) * g.nz * NOUT + (size_t)((NSLOT == 27 ? o : o - 13) * 9 + ij);
        // the warp's longest lists (whole warps take part: 128 threads)
        wxy[m] = __reduce_max_sync(0xffffffffu, valid[m] ? nxy[m] : 1);
        wtwo[m] = __any_sync(0xffffffffu, valid[m] && two[m]);
    }

    const uint32_t ring_s = smem_u32(ring);
    int slot_prev = 0, slot_own = 1;          // stage k in slot k % XS_RING
    uint32_t phase_bits = 0;                  // bit s: parity of the next wait on slot s
    if (tid == 0) { mbar_wait(bars + 0, 0); phase_bits ^= 1u; }
#pragma unroll 1
    for (int k = 0; k < g.nz; ++k) {
        // only thread 0 polls the mbarrier; the others wait in the hardware barrier and take no issue slots
        if (tid == 0) { mbar_wait(bars + slot_own, (phase_bits >> slot_own) & 1u); phase_bits ^= 1u << slot_own; }
        __syncthreads();
        const uint32_t prev_s = ring_s + (uint32_t)slot_prev * XS_STAGE_BYTES;
        const uint32_t own_s = ring_s + (uint32_t)slot_own * XS_STAGE_BYTES;
#pragma unroll
        for (int m = 0; m < XS_OUT; ++m) {
            if (valid[m]) {
                const uint32_t offA = (a_prev[m] ? prev_s : own_s) + ezA[m], offB = prev_s + ezB[m];
                double s = a.accumulate ? *mptr[m] : 0.0;
                if (wtwo[m]) {
                    if (wxy[m] == 4) s = xs_sum<4, true>(s, offA, offB, off[m], nxy[m], two[m]);
                    else if (wxy[m] == 2) s = xs_sum<2, true>(s, offA, offB, off[m], nxy[m], two[m]);
                    else s = xs_sum<1, true>(s, offA, offB, off[m], nxy[m], two[m]);
                } else {
                    if (wxy[m] == 4) s = xs_sum<4, false>(s, offA, offB, off[m], nxy[m], two[m]);
                    else if (wxy[m] == 2) s = xs_sum<2, false>(s, offA, offB, off[m], nxy[m], two[m]);
                    else s = xs_sum<1, false>(s, offA, offB, off[m], nxy[m], two[m]);
                }
                __stcs(mptr[m], s);                        // M is written once and not read here: streamed
            }
            mptr[m] += NOUT;
        }
        __syncthreads();                                   // the previous level has been read by everybody: refill its slot
        if (tid == 0) issue(k + XS_RING);
        slot_prev = slot_own;
        slot_own = slot_own + 1 == XS_RING ? 0 : slot_own + 1;
    }
}
