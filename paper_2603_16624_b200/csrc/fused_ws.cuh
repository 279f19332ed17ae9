// fused_ws.cuh -- warp-specialised form of k_fused_push_moments (fused_mma.cuh): the two phases run in different warps.
//
// Why: one `mma.sync.m8n8k4.f64` holds the issuing warp for 16 cycles (ptxas pads every DMMA with a stall of 15 + a NOP:
// the FP64 pipe is not interlocked), so a warp that does phase 2 cannot issue its integer / shared-memory / address
// work underneath its own DMMAs, and with 3 warps per scheduler the FP64 pipe idles a third of the time
// (profiles/r01c: pipe 66 % busy, stall "wait" 34 %).  Here a CTA is 16 warps = 8 PAIRS; the two warps of a pair sit
// on the same scheduler (warp ids p and p + 8):
//   producer (warp p, 168 registers via setmaxnreg): walks the pair's cell range exactly like k_fused_push_moments,
//       runs phase 1 (weights, gather, alpha, push, deposit factors) of a batch into one of the pair's TWO staging
//       tiles, stores the pushed particles, lists strays, prefetches the next batch, and hands the tile over
//       (mbarrier "full") with a 16-byte descriptor: groups, species, cell, end-of-species / end-of-cell flags;
//   consumer (warp p + 8, 88 registers): waits for the tile, runs phase 2 (5 DMMA + 4 DFMA per 4 particles) into the
//       accumulator fragments, releases the tile (mbarrier "empty"), and on the flags stores AJ[species][cell] /
//       AM[cell] straight from the fragments.
// The consumer's 16-cycle DMMA stalls now block nobody who has other work, the producer's dependent DFMA chains fill
// the gaps between DMMAs, and 2 + 2 warps per scheduler replace 3.
// MODE / LAYOUT as in fused_mma.cuh (MODE_PUSH has no phase 2 and is not specialised).
#pragma once
#include "fused_mma.cuh"

constexpr int WS_PAIRS = 8;
constexpr int WS_WARPS = 2 * WS_PAIRS;
constexpr int WS_TILE_DOUBLES = ST_ROWS * ST_PITCH;
constexpr int WS_PRODUCER_REGS = 168, WS_CONSUMER_REGS = 88;
// dynamic shared memory: [16 tiles][WS_TILE_DOUBLES] | [8 producers][FLD_DOUBLES] | [16 tiles] uint4 descriptors | [16] full | [16] empty
constexpr size_t WS_SMEM_BYTES = (size_t)(2 * WS_PAIRS * WS_TILE_DOUBLES + WS_PAIRS * FLD_DOUBLES) * 8 + 2 * WS_PAIRS * 16 +
                                 2 * 2 * WS_PAIRS * 8;

constexpr unsigned WS_END_SPECIES = 1u << 8, WS_END_CELL = 1u << 9, WS_LAST = 1u << 10;

__device__ __forceinline__ uint32_t ws_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void ws_bar_init(uint64_t* bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(ws_smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void ws_bar_arrive(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.release.cta.shared::cta.b64 _, [%0];" ::"r"(ws_smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void ws_bar_wait(uint64_t* bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WSW_%=:\n"
        "mbarrier.try_wait.parity.acquire.cta.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WSD_%=;\n"
        "bra WSW_%=;\n"
        "WSD_%=:\n"
        "}\n" ::"r"(ws_smem_u32(bar)), "r"(parity) : "memory");
}

template <int MODE, int LAYOUT>
__global__ void __launch_bounds__(WS_WARPS * 32, 1)
k_fused_ws(const __grid_constant__ FusedArgs a)
{
    extern __shared__ __align__(16) double smem[];
    constexpr bool PUSH = MODE == MODE_FUSED, GAPPED = LAYOUT == LAYOUT_GAPPED;
    static_assert(MODE == MODE_FUSED || MODE == MODE_MOMENTS, "specialised for the depositing modes");
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int pair = warp & (WS_PAIRS - 1);
    const bool producer = warp < WS_PAIRS;

    double* tiles = smem + (size_t)pair * 2 * WS_TILE_DOUBLES;                       // the pair's two tiles
    double* fld = smem + (size_t)2 * WS_PAIRS * WS_TILE_DOUBLES + (size_t)pair * FLD_DOUBLES;
    uint4* desc = reinterpret_cast<uint4*>(smem + (size_t)2 * WS_PAIRS * WS_TILE_DOUBLES + (size_t)WS_PAIRS * FLD_DOUBLES) + pair * 2;
    uint64_t* bars = reinterpret_cast<uint64_t*>(reinterpret_cast<uint4*>(smem + (size_t)2 * WS_PAIRS * WS_TILE_DOUBLES +
                                                                           (size_t)WS_PAIRS * FLD_DOUBLES) + 2 * WS_PAIRS);
    uint64_t* full = bars + pair * 2;
    uint64_t* empty = bars + 2 * WS_PAIRS + pair * 2;

    // zero the tiles (pad columns and the constant row), init the barriers
    for (int t = threadIdx.x; t < 2 * WS_PAIRS * WS_TILE_DOUBLES; t += WS_WARPS * 32) smem[t] = 0.0;
    if (threadIdx.x < 2 * 2 * WS_PAIRS) ws_bar_init(bars + threadIdx.x, 1);
    __syncthreads();
    if (producer)
        for (int t = lane; t < ST_PITCH; t += 32) { tiles[ROW_ONE * ST_PITCH + t] = 1.0; tiles[WS_TILE_DOUBLES + ROW_ONE * ST_PITCH + t] = 1.0; }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncthreads();

    const Geom& g = a.g;
    const int nsp = a.n_species;
    const uint32_t W = gridDim.x * WS_PAIRS, wid = blockIdx.x * WS_PAIRS + pair;
    const unsigned long long w0 = cells_weight(a, a.c_begin), wtot = cells_weight(a, a.c_end) - w0;
    const uint32_t c_lo = range_bound(a, wid, W, w0, wtot), c_hi = range_bound(a, wid + 1, W, w0, wtot);

    if (!producer) {
        // ============================== consumer: phase 2 ==============================
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(WS_CONSUMER_REGS));
        if (c_lo >= c_hi) return;
        const int fr = lane >> 2, fk = lane & 3;
        double2 accM[4], accJ = make_double2(0.0, 0.0);
        double acc8[4];
#pragma unroll
        for (int mt = 0; mt < 4; ++mt) { accM[mt] = make_double2(0.0, 0.0); acc8[mt] = 0.0; }
        uint32_t b = 0;
        while (true) {
            const int t = (int)(b & 1u);
            ws_bar_wait(full + t, (b >> 1) & 1u);
            const uint4 d = desc[t];
            const int ng = (int)(d.x & 0xffu);
            const double* frag = tiles + (size_t)t * WS_TILE_DOUBLES + fr * ST_PITCH + fk;
#pragma unroll 2
            for (int gq = 0; gq < ng; ++gq) {
                const double* f = frag + gq * 4;
                const double b0 = f[ROW_BA * ST_PITCH], a8 = f[(ROW_A8 - fr) * ST_PITCH];
                const double wq = f[ROW_WQ * ST_PITCH], bj = f[ROW_BJ * ST_PITCH];
#pragma unroll
                for (int mt = 0; mt < 4; ++mt) {
                    const double av = f[(ROW_C + 8 * mt) * ST_PITCH];
                    dmma_m8n8k4(accM[mt], av, b0);
                    acc8[mt] = fma(av, a8, acc8[mt]);
                }
                dmma_m8n8k4(accJ, wq, bj);
            }
            __syncwarp();
            if (lane == 0) ws_bar_arrive(empty + t);
            ++b;
            if (d.x & WS_END_SPECIES) {
                double* AJ = a.sp[d.y].AJ;
                if (fk >= 2) *reinterpret_cast<double2*>(AJ + (size_t)d.z * AJ_PER_CELL + fr * 4 + 2 * (fk - 2)) = accJ;
                accJ = make_double2(0.0, 0.0);
            }
            if (d.x & WS_END_CELL) {
                double* dst = a.AM + (size_t)d.z * AM_PER_CELL;
#pragma unroll
                for (int mt = 0; mt < 4; ++mt) {
                    const int cls = 8 * mt + fr;
                    double s8 = acc8[mt];
                    s8 += shfl_xor_f64(s8, 1);
                    s8 += shfl_xor_f64(s8, 2);
                    if (cls < 27) {
                        *reinterpret_cast<double2*>(dst + mt * 64 + fr * 8 + 2 * fk) = accM[mt];
                        if (fk == 0) dst[AM_A8 + cls] = s8;
                    }
                    accM[mt] = make_double2(0.0, 0.0);
                    acc8[mt] = 0.0;
                }
            }
            if (d.x & WS_LAST) break;
        }
        return;
    }

    // ============================== producer: phase 1 ==============================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(WS_PRODUCER_REGS));
    if (c_lo >= c_hi) return;
    const double dt = a.dt;
    const unsigned lt_mask = (1u << lane) - 1u;

    // field staging: lane t and t+32 (< 48) hold corner t/6, component t%6 of the next cell
    const int fc0 = lane / 6, fk0 = lane - fc0 * 6;
    const int fc1 = (lane + 32) / 6, fk1 = (lane + 32) - fc1 * 6;
    const double* fsrc0 = fk0 < 3 ? a.E + (size_t)fk0 * g.nodes : a.B + (size_t)(fk0 - 3) * g.nodes;
    const double* fsrc1 = fk1 < 3 ? a.E + (size_t)fk1 * g.nodes : a.B + (size_t)(fk1 - 3) * g.nodes;
    auto load_fields = [&](int ci, int cj, int ck, double& f0, double& f1) {
        if (MODE != MODE_MOMENTS || fk0 >= 3) {
            int ii = ci + ((fc0 >> 2) & 1); if (ii == g.nx) ii = 0;
            int jj = cj + ((fc0 >> 1) & 1); if (jj == g.ny) jj = 0;
            int kk = ck + (fc0 & 1);        if (kk == g.nz) kk = 0;
            f0 = __ldg(fsrc0 + ((long long)ii * g.ny + jj) * g.nz + kk);
        }
        if (lane < FLD_DOUBLES - 32 && (MODE != MODE_MOMENTS || fk1 >= 3)) {
            int ii = ci + ((fc1 >> 2) & 1); if (ii == g.nx) ii = 0;
            int jj = cj + ((fc1 >> 1) & 1); if (jj == g.ny) jj = 0;
            int kk = ck + (fc1 & 1);        if (kk == g.nz) kk = 0;
            f1 = __ldg(fsrc1 + ((long long)ii * g.ny + jj) * g.nz + kk);
        }
    };

    int ck = (int)(c_lo % (uint32_t)g.nz);
    int cj = (int)((c_lo / (uint32_t)g.nz) % (uint32_t)g.ny);
    int ci = (int)(c_lo / ((uint32_t)g.nz * (uint32_t)g.ny));

    uint32_t g0 = 0, g1 = 0, g2 = 0, nf0 = 0, nt0 = 0, nf1 = 0, nt1 = 0;
    const SpeciesDev& mysp = a.sp[lane < nsp ? lane : 0];
    auto load_counts = [&](uint32_t c, uint32_t lo, uint32_t hi, uint32_t& nf, uint32_t& nt) {
        if (GAPPED) { nf = __ldg(mysp.Fin + c); nt = nf + __ldg(mysp.Rin + c); }
        else { nf = nt = hi - lo; }
    };
    if (lane < nsp) {
        g0 = __ldg(mysp.seg + c_lo);
        g1 = __ldg(mysp.seg + c_lo + 1);
        load_counts(c_lo, g0, g1, nf0, nt0);
        if (c_lo + 1 < c_hi) {
            g2 = __ldg(mysp.seg + c_lo + 2);
            load_counts(c_lo + 1, g1, g2, nf1, nt1);
        }
    }
    double f0 = 0.0, f1 = 0.0;
    bool fld_ready = false;

    unsigned long long lv_acc = 0;
    int in_state = 0;
    int in_s = 0, in_nb = 0;
    uint32_t in_v0 = 0, in_base = 0, in_end = 0, in_nf = 0, in_p = 0;
    ParticleRegs in;
    in.x = in.y = in.z = in.u = in.v = in.w = in.q = 0.0;
    auto describe = [&](int s, bool next_cell) {
        in_s = s;
        in_v0 = 0;
        in_base = __shfl_sync(0xffffffffu, next_cell ? g1 : g0, s);
        const uint32_t nt = __shfl_sync(0xffffffffu, next_cell ? nt1 : nt0, s);
        in_nb = (int)min(32u, nt);
        if (GAPPED) {
            in_end = __shfl_sync(0xffffffffu, next_cell ? g2 : g1, s);
            in_nf = __shfl_sync(0xffffffffu, next_cell ? nf1 : nf0, s);
        }
    };
    auto fetch = [&]() {
        const uint32_t v = in_v0 + (uint32_t)lane;
        in_p = (GAPPED && v >= in_nf) ? in_end - 1u - (v - in_nf) : in_base + v;
        load_batch(a.sp[in_s], in_p, lane < in_nb, in);
    };
    {
        const unsigned ne = __ballot_sync(0xffffffffu, lane < nsp && nt0 > 0);
        if (ne) {
            describe(__ffs(ne) - 1, false);
            in_state = 1;
            fetch();
        }
    }

    uint32_t b = 0;              // tiles handed over so far
    auto hand_over = [&](int t, unsigned word, int s, uint32_t c) {
        __syncwarp();
        if (lane == 0) {
            desc[t] = make_uint4(word, (unsigned)s, c, 0u);
            ws_bar_arrive(full + t);
        }
        ++b;
    };

    for (uint32_t c = c_lo; c < c_hi; ++c) {
        if (!fld_ready) load_fields(ci, cj, ck, f0, f1);
        fld[lane] = f0;
        if (lane < FLD_DOUBLES - 32) fld[lane + 32] = f1;
        fld_ready = false;
        const bool has_next = c + 1 < c_hi;
        int nk = ck + 1, nj = cj, ni = ci;
        if (nk == g.nz) { nk = 0; nj = cj + 1; if (nj == g.ny) { nj = 0; ni = ci + 1; } }
        __syncwarp();
        const double dci = (double)ci, dcj = (double)cj, dck = (double)ck;
        const unsigned ne_cur = __ballot_sync(0xffffffffu, lane < nsp && nt0 > 0);
        unsigned my_leavers = 0;
        uint32_t nstay = 0;

        // species without particles in this cell still own an AJ block (zeros) and a front run (empty)
        {
            unsigned none = ~ne_cur & ((nsp >= 32) ? 0xffffffffu : ((1u << nsp) - 1u));
            while (none) {
                const int s = __ffs(none) - 1;
                none &= none - 1;
                a.sp[s].AJ[(size_t)c * AJ_PER_CELL + lane] = 0.0;
                if (PUSH && GAPPED && lane == 0) a.sp[s].Fout[c] = 0u;
            }
        }
        if (ne_cur == 0) {
            // a cell without particles: an empty hand-over so that the consumer stores the cell's (zero) class sums
            const int t = (int)(b & 1u);
            ws_bar_wait(empty + t, ((b >> 1) & 1u) ^ 1u);
            hand_over(t, WS_END_CELL | (has_next ? 0u : WS_LAST), 0, c);
        }

        while (in_state == 1) {
            const int s = in_s, nb = in_nb;
            const uint32_t p = in_p, cell_base = in_base;
            const ParticleRegs cur = in;
            const SpeciesDev& sp = a.sp[s];
            {
                const uint32_t e = __shfl_sync(0xffffffffu, nt0, s);
                const unsigned later = ne_cur & ~((2u << s) - 1u);
                if (in_v0 + 32 < e) {
                    in_v0 += 32;
                    in_nb = (int)min(32u, e - in_v0);
                } else if (later) {
                    describe(__ffs(later) - 1, false);
                } else {
                    const unsigned ne_next = __ballot_sync(0xffffffffu, has_next && lane < nsp && nt1 > 0);
                    if (ne_next) {
                        describe(__ffs(ne_next) - 1, true);
                        in_state = 2;
                    } else {
                        in_state = has_next ? 3 : 0;
                    }
                }
            }
            const bool end_species = in_state != 1 || in_s != s, end_cell = in_state != 1;
            // the next batch's particles (and the next cell's corner fields) are requested BEFORE this batch's phase 1:
            // the producer has no phase 2 to hide the loads behind
            if (in_state == 1 || in_state == 2) fetch();
            if (in_state != 1 && has_next) { load_fields(ni, nj, nk, f0, f1); fld_ready = true; }

            // ---- phase 1 into the pair's free tile ----
            const int t = (int)(b & 1u);
            ws_bar_wait(empty + t, ((b >> 1) & 1u) ^ 1u);
            double* stcol = tiles + (size_t)t * WS_TILE_DOUBLES + lane;
            PushedRegs o;
            const bool active = lane < nb;
            const bool inside = phase1<MODE, LAYOUT>(g, cur, active, sp.beta, dt, dci, dcj, dck, fld, stcol, o);
            hand_over(t, (unsigned)(nb > 28 ? 8 : (nb + 3) >> 2) | (end_species ? WS_END_SPECIES : 0u) |
                             (end_cell ? WS_END_CELL : 0u) | ((end_cell && !has_next) ? WS_LAST : 0u), s, c);
            if (PUSH) {
                if (GAPPED) {
                    const bool stay = inside && o.stays;
                    const unsigned smask = __ballot_sync(0xffffffffu, stay);
                    if (stay) {
                        const uint32_t d = cell_base + nstay + (uint32_t)__popc(smask & lt_mask);
                        sp.ox[d] = o.x; sp.oy[d] = o.y; sp.oz[d] = o.z;
                        sp.ou[d] = o.u; sp.ov[d] = o.v; sp.ow[d] = o.w; sp.oq[d] = cur.q;
                    }
                    nstay += (uint32_t)__popc(smask);
                    if (inside && !o.stays) { relocate(g, sp, o, cur.q); my_leavers += 1u; }
                } else if (inside) {
                    sp.u[p] = o.u; sp.v[p] = o.v; sp.w[p] = o.w;
                    sp.x[p] = o.x; sp.y[p] = o.y; sp.z[p] = o.z;
                    my_leavers += o.stays ? 0u : 1u;
                }
            }
            if (!GAPPED) {
                const unsigned smask = __ballot_sync(0xffffffffu, active && !inside);
                if (smask) {
                    uint32_t base = 0;
                    if (lane == 0) base = atomicAdd(sp.stray_count, (uint32_t)__popc(smask));
                    base = __shfl_sync(0xffffffffu, base, 0);
                    if (active && !inside) sp.stray_list[base + __popc(smask & lt_mask)] = p;
                }
            }
            if (end_species && PUSH) {
                if (GAPPED && lane == 0) sp.Fout[c] = nstay;
                nstay = 0;
                my_leavers = __reduce_add_sync(0xffffffffu, my_leavers);
                if (lane == s) lv_acc += my_leavers;
                my_leavers = 0;
            }
        }

        // ---- advance to the next cell ----
        if (lane < nsp) {
            g0 = g1; g1 = g2; nf0 = nf1; nt0 = nt1;
            if (c + 2 < c_hi) {
                g2 = __ldg(mysp.seg + c + 3);
                load_counts(c + 2, g1, g2, nf1, nt1);
            }
        }
        ci = ni; cj = nj; ck = nk;
        if (in_state == 2) {
            in_state = 1;
        } else if (has_next) {
            const unsigned ne = __ballot_sync(0xffffffffu, lane < nsp && nt0 > 0);
            in_state = 0;
            if (ne) {
                describe(__ffs(ne) - 1, false);
                in_state = 1;
                fetch();
            }
        }
    }
    if (PUSH && lane < nsp && lv_acc) atomicAdd(a.sp[lane].leavers, lv_acc);
}
