// apply_m.cuh -- the mass-matrix operator of the field equations, out_N = sum_N' M_NN' E_N' (Eq. 4-5:
// the term the implicit Maxwell solve applies at every Krylov iteration), as a 27-offset stencil mat-vec over the node
// array M the deposit produced.  HBM-bound streaming: M is read once.
//
// One warp per RUN of APPLY_RUN consecutive nodes along z (grid-stride over the runs).  The warp first stages the E of the
// run's neighbourhood -- 9 node columns x (run + 2) levels x 3 components, read coalesced along z -- in its block of shared
// memory; then, node by node, lane q (and q + 32, q + 64 < 81) owns the pair (neighbour slot o, column s): it reads the
// three matrix entries M[o][r][s], r = 0..2, multiplies them by E_s of that neighbour and adds to its three row sums
// (one FMA per entry, no selects).  The three sums are reduced over the warp with six 64-bit shuffles (pairs of values
// folded in the first two steps).  The next node's nine entries are requested before the current node is reduced; the
// results of the run are written coalesced at its end.  (Round 2 first had one warp per node, every node's 27 neighbour E
// vectors fetched by scattered loads before its M loads were issued, a select per row and 30 shuffles: 2.6 TB/s.)
//
// 14-slot (symmetric) storage, L73 / L129: M14[g][o - 13] holds the slots o >= 13; a slot o < 13 of node g is slot
// 26 - o of the node g' = g + off(o) it points at (M_NN' = M_N'N per component, no transpose: DESIGN.md R11), so it is
// read from g' block: 9 contiguous doubles that g' own warp reads anyway (L1 / L2).
#pragma once
#include "common.cuh"

struct ApplyMArgs {
    Geom g;
    const double* M;    // [nodes][NSLOT][3][3]
    const double* E;    // [3][nodes]
    double* out;        // [3][nodes]
    int accumulate;     // out += instead of out =
};

constexpr int APPLY_WARPS = 8;
constexpr int APPLY_RUN = 8;                       // nodes per run (<= 8: their results sit in lanes r, 8 + r, 16 + r)
constexpr int APPLY_LEVELS = APPLY_RUN + 2;
constexpr int APPLY_SE = 9 * 3 * APPLY_LEVELS;     // sE[column 0..8][component][level]

template <int NSLOT>
__global__ void __launch_bounds__(APPLY_WARPS * 32)
k_apply_M(const __grid_constant__ ApplyMArgs a)
{
    __shared__ double sE_all[APPLY_WARPS][APPLY_SE];
    __shared__ long long sC_all[APPLY_WARPS][9];       // first node of the 9 neighbour columns
    __shared__ int sK_all[APPLY_WARPS][APPLY_LEVELS];  // wrapped z index of level l = k0 - 1 + l
    const Geom& g = a.g;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double* sE = sE_all[warp];
    long long* sC = sC_all[warp];
    int* sK = sK_all[warp];
    const long long nodes = g.nodes;
    const int runs_per_col = (g.nz + APPLY_RUN - 1) / APPLY_RUN;
    const long long n_runs = (long long)g.nx * g.ny * runs_per_col;

    // this lane's (slot, column) pairs q = lane + 32 j < 81: where their E sits in sE (level of node 0 of the run) and where
    // their first-row entry sits in the node's block of M
    int eoff[3], moff[3], col9[3], dkp[3];
    bool have[3], own[3];
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        const int q = lane + 32 * j;
        have[j] = q < 81;
        const int qq = have[j] ? q : 0;
        const int o = qq / 3, s = qq % 3;
        col9[j] = o / 3;
        dkp[j] = o % 3;                                       // level of the neighbour relative to the node: dk + 1
        eoff[j] = (col9[j] * 3 + s) * APPLY_LEVELS + dkp[j];
        own[j] = NSLOT == 27 || o >= 13;
        moff[j] = NSLOT == 27 ? 9 * o + s : (o >= 13 ? 9 * (o - 13) + s : 9 * (13 - o) + s);
    }
    constexpr int PER_NODE = NSLOT * 9;

    for (long long run = (long long)blockIdx.x * APPLY_WARPS + warp; run < n_runs; run += (long long)gridDim.x * APPLY_WARPS) {
        const long long col = run / runs_per_col;
        const int k0 = (int)(run % runs_per_col) * APPLY_RUN;
        const int len = min(APPLY_RUN, g.nz - k0);
        const int i = (int)(col / g.ny), j0 = (int)(col % g.ny);
        if (lane < 9) {
            int ii = i + lane / 3 - 1; ii = ii < 0 ? ii + g.nx : (ii >= g.nx ? ii - g.nx : ii);
            int jj = j0 + lane % 3 - 1; jj = jj < 0 ? jj + g.ny : (jj >= g.ny ? jj - g.ny : jj);
            sC[lane] = ((long long)ii * g.ny + jj) * g.nz;
        }
        if (lane < APPLY_LEVELS) {
            sK[lane] = ((k0 - 1 + lane) % g.nz + g.nz) % g.nz;              // (levels past the run's end are staged but not used)
        }
        __syncwarp();
        const double* m_node = a.M + (size_t)(sC[4] + k0) * PER_NODE;      // column 4 = the nodes' own column
        // the first node's entries are requested before the E neighbourhood is staged
        double mv[3][3];
        auto load_node = [&](int r, double (&v)[3][3]) {
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                if (have[j]) {
                    const double* p = own[j] ? m_node + (size_t)r * PER_NODE + moff[j]
                                             : a.M + (size_t)(sC[col9[j]] + sK[r + dkp[j]]) * PER_NODE + moff[j];
#pragma unroll
                    for (int rr = 0; rr < 3; ++rr) v[j][rr] = __ldg(p + 3 * rr);
                }
            }
        };
        load_node(0, mv);
        for (int t = lane; t < APPLY_SE; t += 32) {
            const int cs = t / APPLY_LEVELS, l = t - cs * APPLY_LEVELS;
            sE[t] = __ldg(a.E + (size_t)(cs % 3) * nodes + sC[cs / 3] + sK[l]);
        }
        __syncwarp();

        double res = 0.0;                                   // lane 8 c + r: component c of node r of the run
        for (int r = 0; r < len; ++r) {
            double a0 = 0.0, a1 = 0.0, a2 = 0.0;
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                if (have[j]) {
                    const double e = sE[eoff[j] + r];
                    a0 = fma(mv[j][0], e, a0); a1 = fma(mv[j][1], e, a1); a2 = fma(mv[j][2], e, a2);
                }
            }
            if (r + 1 < len) load_node(r + 1, mv);          // in flight during the reduction
            // (a0, a1, a2, 0) over the warp: fold pairs at xor 16 and xor 8, then one value per lane
            const bool up16 = lane & 16, up8 = lane & 8;
            const double x = shfl_xor_f64(up16 ? a0 : a2, 16), y = shfl_xor_f64(up16 ? a1 : 0.0, 16);
            const double k0v = (up16 ? a2 : a0) + x, k1v = (up16 ? 0.0 : a1) + y;    // lanes < 16: (a0, a1); >= 16: (a2, 0)
            double v = (up8 ? k1v : k0v) + shfl_xor_f64(up8 ? k0v : k1v, 8);         // lane bits (16, 8): a0, a1, a2, 0
            v += shfl_xor_f64(v, 4);
            v += shfl_xor_f64(v, 2);
            v += shfl_xor_f64(v, 1);
            if ((lane & 7) == r) res = v;
        }
        if (lane < 24 && (lane & 7) < len) {
            double* dst = a.out + (size_t)(lane >> 3) * nodes + sC[4] + k0 + (lane & 7);
            *dst = a.accumulate ? *dst + res : res;
        }
        __syncwarp();
    }
}
