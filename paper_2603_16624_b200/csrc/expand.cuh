// expand.cuh -- expansion of the fused kernel's per-cell accumulators to the node arrays
// (the flush).  HBM-bound streaming: reads AM / AJ once, writes M / rho / Jhat once.
//
// Node N = (i,j,k) is corner a=0 of cell i and corner a=1 of cell i-1 (per axis).  For neighbour
// offset d along an axis the pairs (a, a') with a' - a = d inside one cell are
//     d =  0 : (0,0) in cell i   -> class 0 (w0^2)   and (1,1) in cell i-1 -> class 2 (w1^2)
//     d = +1 : (0,1) in cell i   -> class 1 (w0 w1)
//     d = -1 : (1,0) in cell i-1 -> class 1
// and the 3-D term list of M[N][o] is the product of the three per-axis lists: 1, 2, 4 or 8 cells
// (Eq. 3 summed over the particles of every cell that holds both N and N').
//
// k_expand_M: one CTA walks EXPAND_Z consecutive nodes of one (i,j) column; thread t < 243 owns one
// element (o, ij).  Threads are ordered by the SHAPE of their term list ((x-y terms) x (z terms)) so that
// a warp's load count is uniform and short, and every load of a node is issued before the first use
// (straight-line code per shape: the memory-level parallelism the first version lacked, profiles/r01a).
#pragma once
#include "common.cuh"
#include "fused_mma.cuh"

constexpr int EXPAND_Z = 32;

struct ExpandArgs {
    Geom g;
    const double* AM;   // [cells][AM_PER_CELL]
    double* M;          // [nodes][27][3][3]
    int accumulate;
    int i0;             // first node plane (x index) of this launch; the grid covers planes i0, i0+1, ...
};

// neighbour slots ordered by (x-y terms, z terms) = (4,2) | (4,1) | (2,2) | (2,1) | (1,2) | (1,1)
__device__ __constant__ unsigned char EXPAND_ORDER[27] = {
    13,
    12, 14,
    4, 10, 16, 22,
    3, 5, 9, 11, 15, 17, 21, 23,
    1, 7, 19, 25,
    0, 2, 6, 8, 18, 20, 24, 26};

// Offset, in doubles inside a cell's AM block, of (class, ij): 8*class + ij for ij < 8, AM_A8 + class for
// ij = 8 -- additive in the per-axis parts of class = 9 clx + 3 cly + clz.
template <int NXY, int NTZ>
__device__ __forceinline__ void expand_nodes(const ExpandArgs& a, const double* const (&col)[4], int ezA, int ezB,
                                             bool zA_is_prev, int nxy, int ntz, int k0, int k1,
                                             double* __restrict__ dst0)
{
    const int nz = a.g.nz;
#pragma unroll 2
    for (int k = k0; k < k1; ++k) {
        // z terms: A = first entry of the z list, B = second (cell k-1, class 2) when dz = 0
        const int km1 = k ? k - 1 : nz - 1;
        const int zA = (zA_is_prev ? km1 : k) * AM_PER_CELL + ezA, zB = km1 * AM_PER_CELL + ezB;
        double v[NXY][NTZ];
#pragma unroll
        for (int t = 0; t < NXY; ++t) {
            v[t][0] = __ldg(col[t] + zA);
            if (NTZ == 2) v[t][1] = __ldg(col[t] + zB);
        }
        double s = a.accumulate ? dst0[(size_t)k * 243] : 0.0;
#pragma unroll
        for (int t = 0; t < NXY; ++t) {
            s += t < nxy ? v[t][0] : 0.0;
            if (NTZ == 2) s += (t < nxy && ntz == 2) ? v[t][1] : 0.0;
        }
        dst0[(size_t)k * 243] = s;
    }
}

// <= 64 registers (it needs ~60: capped at 40 it runs 2.5x slower): one CTA fits beside a 12-warp x 128-register
// fused CTA on every SM
__global__ void __launch_bounds__(256, 4)
k_expand_M(const __grid_constant__ ExpandArgs a)
{
    const int t = threadIdx.x;
    if (t >= 243) return;
    const Geom& g = a.g;
    const int o = EXPAND_ORDER[t / 9], ij = t % 9;
    const int dx = o / 9 - 1, dy = (o / 3) % 3 - 1, dz = o % 3 - 1;
    const int zchunks = (g.nz + EXPAND_Z - 1) / EXPAND_Z;
    const int zc = (int)(blockIdx.x % (unsigned)zchunks);
    const int j = (int)((blockIdx.x / (unsigned)zchunks) % (unsigned)g.ny);
    const int i = a.i0 + (int)(blockIdx.x / ((unsigned)zchunks * (unsigned)g.ny));
    const int im1 = i ? i - 1 : g.nx - 1, jm1 = j ? j - 1 : g.ny - 1;
    const int ebase = ij < 8 ? ij : AM_A8, emul = ij < 8 ? 8 : 1;

    // x and y term lists: (cell index, class); d = 0: (own, 0), (previous, 2); d = +1: (own, 1); d = -1: (previous, 1)
    const int ntx = dx == 0 ? 2 : 1, nty = dy == 0 ? 2 : 1, ntz = dz == 0 ? 2 : 1;
    const int nxy = ntx * nty;
    const double* col[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        const int ee = e < nxy ? e : 0;                 // e >= nxy repeats term 0 (its value is not added)
        const int ty = ee % nty, tx = ee / nty;
        const int ci = tx == 0 ? (dx >= 0 ? i : im1) : im1, cx = tx == 0 ? (dx == 0 ? 0 : 1) : 2;
        const int cj = ty == 0 ? (dy >= 0 ? j : jm1) : jm1, cy = ty == 0 ? (dy == 0 ? 0 : 1) : 2;
        col[e] = a.AM + ((size_t)ci * g.ny + cj) * g.nz * AM_PER_CELL + (ebase + emul * (9 * cx + 3 * cy));
    }
    // z list: dz = 0: (cell k, class 0), (cell k-1, class 2); dz = +1: (cell k, class 1); dz = -1: (cell k-1, class 1)
    const int ezA = emul * (dz == 0 ? 0 : 1), ezB = emul * 2;
    const bool zA_is_prev = dz < 0;

    const int k0 = zc * EXPAND_Z;
    const int k1 = min(k0 + EXPAND_Z, g.nz);
    double* dst0 = a.M + ((size_t)i * g.ny + j) * g.nz * 243 + (size_t)(o * 9 + ij);
    // longest lists in the warp: warps 0..7 see (4,2), (2,2), (2,1), (2,1), (2,2), (1,2), (1,1), (1,1)
    const unsigned am = __activemask();
    const int wxy = __reduce_max_sync(am, nxy), wz = __reduce_max_sync(am, ntz);
    if (wz == 2) {
        if (wxy == 4) expand_nodes<4, 2>(a, col, ezA, ezB, zA_is_prev, nxy, ntz, k0, k1, dst0);
        else if (wxy == 2) expand_nodes<2, 2>(a, col, ezA, ezB, zA_is_prev, nxy, ntz, k0, k1, dst0);
        else expand_nodes<1, 2>(a, col, ezA, ezB, zA_is_prev, nxy, ntz, k0, k1, dst0);
    } else {
        if (wxy == 4) expand_nodes<4, 1>(a, col, ezA, ezB, zA_is_prev, nxy, ntz, k0, k1, dst0);
        else if (wxy == 2) expand_nodes<2, 1>(a, col, ezA, ezB, zA_is_prev, nxy, ntz, k0, k1, dst0);
        else expand_nodes<1, 1>(a, col, ezA, ezB, zA_is_prev, nxy, ntz, k0, k1, dst0);
    }
}

struct ExpandJArgs {
    Geom g;
    const double* AJ;   // [cells][8][4]
    double* rho;        // [nodes] or null
    double* J;          // [3][nodes] or null
    int accumulate;
    long long n0, n1;   // nodes [n0, n1) of this launch
};

__global__ void __launch_bounds__(256)
k_expand_rhoJ(ExpandJArgs a)
{
    const Geom& g = a.g;
    const long long node = a.n0 + (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (node >= a.n1) return;
    const int k = (int)(node % g.nz);
    const int j = (int)((node / g.nz) % g.ny);
    const int i = (int)(node / ((long long)g.nz * g.ny));
    double s0 = 0, s1 = 0, s2 = 0, s3 = 0;
#pragma unroll
    for (int corner = 0; corner < 8; ++corner) {
        // the node is corner (a,b,c) of cell (i-a, j-b, k-c)
        int ci = i - ((corner >> 2) & 1); if (ci < 0) ci += g.nx;
        int cj = j - ((corner >> 1) & 1); if (cj < 0) cj += g.ny;
        int ck = k - (corner & 1);        if (ck < 0) ck += g.nz;
        const long long cell = ((long long)ci * g.ny + cj) * g.nz + ck;
        const double2 v0 = *reinterpret_cast<const double2*>(a.AJ + (size_t)cell * AJ_PER_CELL + corner * 4);
        const double2 v1 = *reinterpret_cast<const double2*>(a.AJ + (size_t)cell * AJ_PER_CELL + corner * 4 + 2);
        s0 += v0.x; s1 += v0.y; s2 += v1.x; s3 += v1.y;
    }
    if (a.rho) a.rho[node] = (a.accumulate ? a.rho[node] : 0.0) + s0;
    if (a.J) {
        a.J[node] = (a.accumulate ? a.J[node] : 0.0) + s1;
        a.J[g.nodes + node] = (a.accumulate ? a.J[g.nodes + node] : 0.0) + s2;
        a.J[2 * g.nodes + node] = (a.accumulate ? a.J[2 * g.nodes + node] : 0.0) + s3;
    }
}
