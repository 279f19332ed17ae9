// apply_m.cuh -- the mass-matrix operator of the field equations, out_N = sum_N' M_NN' E_N' (Eq. 4-5:
// the term the implicit Maxwell solve applies at every Krylov iteration), as a 27-offset stencil mat-vec over the node
// array M the deposit produced.  HBM-bound streaming: M is read once.
//
// One warp per node (grid-stride, z fastest).  Lanes 0..26 fetch the 27 neighbours' E into a per-warp block of shared
// memory; then the node's 243 (27-slot layout) or 126 + 117 (14-slot layout) matrix entries stream through the lanes,
// coalesced, each multiplied by its neighbour's E component and added to the lane's three row sums; a shuffle tree
// finishes the three sums.
//
// 14-slot (symmetric) storage, L73 / L129: M14[g][o - 13] holds the slots o >= 13; a slot o < 13 of node g is slot
// 26 - o of the node g' = g + off(o) it points at (M_NN' = M_N'N per component, no transpose: DESIGN.md R11), so it is
// read from g' block: 9 contiguous doubles that g' own warp reads anyway (L2).
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

template <int NSLOT>
__global__ void __launch_bounds__(APPLY_WARPS * 32)
k_apply_M(const __grid_constant__ ApplyMArgs a)
{
    __shared__ double sE[APPLY_WARPS][27 * 3];
    __shared__ long long sN[APPLY_WARPS][27];
    const Geom& g = a.g;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const long long nodes = g.nodes;
    const long long wstride = (long long)gridDim.x * APPLY_WARPS;
    // neighbour offset of lane o < 27
    const int o_l = lane < 27 ? lane : 13;
    const int di = o_l / 9 - 1, dj = (o_l / 3) % 3 - 1, dk = o_l % 3 - 1;
    for (long long n = (long long)blockIdx.x * APPLY_WARPS + warp; n < nodes; n += wstride) {
        const int k = (int)(n % g.nz);
        const int j = (int)((n / g.nz) % g.ny);
        const int i = (int)(n / ((long long)g.nz * g.ny));
        if (lane < 27) {
            int ii = i + di; ii = ii < 0 ? ii + g.nx : (ii >= g.nx ? ii - g.nx : ii);
            int jj = j + dj; jj = jj < 0 ? jj + g.ny : (jj >= g.ny ? jj - g.ny : jj);
            int kk = k + dk; kk = kk < 0 ? kk + g.nz : (kk >= g.nz ? kk - g.nz : kk);
            const long long nb = ((long long)ii * g.ny + jj) * g.nz + kk;
            sN[warp][lane] = nb;
            sE[warp][lane * 3 + 0] = __ldg(a.E + nb);
            sE[warp][lane * 3 + 1] = __ldg(a.E + nodes + nb);
            sE[warp][lane * 3 + 2] = __ldg(a.E + 2 * nodes + nb);
        }
        __syncwarp();
        double acc0 = 0.0, acc1 = 0.0, acc2 = 0.0;
        if (NSLOT == 27) {
            const double* m = a.M + (size_t)n * 243;
#pragma unroll
            for (int it = 0; it < 8; ++it) {
                const int e = lane + 32 * it;
                if (e < 243) {
                    const int o = e / 9, r = (e % 9) / 3, s = e % 3;
                    const double t = __ldg(m + e) * sE[warp][o * 3 + s];
                    acc0 += r == 0 ? t : 0.0; acc1 += r == 1 ? t : 0.0; acc2 += r == 2 ? t : 0.0;
                }
            }
        } else {
            // own block: slots 13..26
            const double* m = a.M + (size_t)n * 126;
#pragma unroll
            for (int it = 0; it < 4; ++it) {
                const int e = lane + 32 * it;
                if (e < 126) {
                    const int o = 13 + e / 9, r = (e % 9) / 3, s = e % 3;
                    const double t = __ldg(m + e) * sE[warp][o * 3 + s];
                    acc0 += r == 0 ? t : 0.0; acc1 += r == 1 ? t : 0.0; acc2 += r == 2 ? t : 0.0;
                }
            }
            // slots 0..12: slot 26 - o of the neighbour they point at
#pragma unroll
            for (int it = 0; it < 4; ++it) {
                const int e = lane + 32 * it;
                if (e < 117) {
                    const int o = e / 9, r = (e % 9) / 3, s = e % 3;
                    const double t = __ldg(a.M + (size_t)sN[warp][o] * 126 + (size_t)(13 - o) * 9 + (e % 9)) * sE[warp][o * 3 + s];
                    acc0 += r == 0 ? t : 0.0; acc1 += r == 1 ? t : 0.0; acc2 += r == 2 ? t : 0.0;
                }
            }
        }
#pragma unroll
        for (int d = 16; d >= 1; d >>= 1) {
            acc0 += shfl_xor_f64(acc0, d);
            acc1 += shfl_xor_f64(acc1, d);
            acc2 += shfl_xor_f64(acc2, d);
        }
        if (lane < 3) {
            const double v = lane == 0 ? acc0 : (lane == 1 ? acc1 : acc2);
            double* dst = a.out + (size_t)lane * nodes + n;
            *dst = a.accumulate ? *dst + v : v;
        }
        __syncwarp();
    }
}
