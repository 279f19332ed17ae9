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
// element (o, ij).  Threads are ordered by the LENGTH of their term list (8, 4, 2, 1) so that a warp's
// loop count is uniform and short, every load of a node is issued before the first use (straight-line
// code per term count: the memory-level parallelism the first version lacked, profiles/r01a), and two
// nodes are in flight per iteration.
#pragma once
#include "common.cuh"
#include "fused_mma.cuh"

constexpr int EXPAND_Z = 16;

struct ExpandArgs {
    Geom g;
    const double* AM;   // [cells][AM_PER_CELL]
    double* M;          // [nodes][27][3][3]
    int accumulate;
};

// neighbour slots ordered by term count: o = 13 (8 terms); the 6 face slots (4); the 12 edge slots (2);
// the 8 corner slots (1)
__device__ __constant__ unsigned char EXPAND_ORDER[27] = {
    13,
    4, 10, 12, 14, 16, 22,
    1, 3, 5, 7, 9, 11, 15, 17, 19, 21, 23, 25,
    0, 2, 6, 8, 18, 20, 24, 26};

// offset, in doubles inside a cell's AM block, of (class, ij)
__device__ __forceinline__ int am_elem(int cls, int ij)
{
    return ij < 8 ? ((cls >> 3) * 64 + (cls & 7) * 8 + ij) : (AM_A8 + cls);
}

template <int NT>
__device__ __forceinline__ void expand_nodes(const ExpandArgs& a, const size_t (&off)[8], unsigned zbits, int T,
                                             int k0, int k1, double* __restrict__ dst0)
{
    const int nz = a.g.nz;
    int k = k0;
    for (; k + 1 < k1; k += 2) {
        const size_t zA0 = (size_t)k * AM_PER_CELL, zB0 = (size_t)(k ? k - 1 : nz - 1) * AM_PER_CELL;
        const size_t zA1 = (size_t)(k + 1) * AM_PER_CELL, zB1 = zA0;
        double v0[NT], v1[NT];
#pragma unroll
        for (int t = 0; t < NT; ++t) {
            v0[t] = __ldg(a.AM + off[t] + (((zbits >> t) & 1u) ? zB0 : zA0));
            v1[t] = __ldg(a.AM + off[t] + (((zbits >> t) & 1u) ? zB1 : zA1));
        }
        double s0 = 0.0, s1 = 0.0;
        if (a.accumulate) { s0 = dst0[(size_t)k * 243]; s1 = dst0[(size_t)(k + 1) * 243]; }
#pragma unroll
        for (int t = 0; t < NT; ++t) {
            s0 += t < T ? v0[t] : 0.0;
            s1 += t < T ? v1[t] : 0.0;
        }
        dst0[(size_t)k * 243] = s0;
        dst0[(size_t)(k + 1) * 243] = s1;
    }
    if (k < k1) {
        const size_t zA0 = (size_t)k * AM_PER_CELL, zB0 = (size_t)(k ? k - 1 : nz - 1) * AM_PER_CELL;
        double v0[NT];
#pragma unroll
        for (int t = 0; t < NT; ++t) v0[t] = __ldg(a.AM + off[t] + (((zbits >> t) & 1u) ? zB0 : zA0));
        double s0 = a.accumulate ? dst0[(size_t)k * 243] : 0.0;
#pragma unroll
        for (int t = 0; t < NT; ++t) s0 += t < T ? v0[t] : 0.0;
        dst0[(size_t)k * 243] = s0;
    }
}

__global__ void __launch_bounds__(256)
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
    const int i = (int)(blockIdx.x / ((unsigned)zchunks * (unsigned)g.ny));
    const int im1 = i ? i - 1 : g.nx - 1, jm1 = j ? j - 1 : g.ny - 1;

    // per-axis term lists: (cell index or z selector, class)
    const int ntx = dx == 0 ? 2 : 1, nty = dy == 0 ? 2 : 1, ntz = dz == 0 ? 2 : 1;
    const int cix[2] = {dx >= 0 ? i : im1, im1}, clx[2] = {dx == 0 ? 0 : 1, 2};
    const int cjy[2] = {dy >= 0 ? j : jm1, jm1}, cly[2] = {dy == 0 ? 0 : 1, 2};
    const int zsel[2] = {dz >= 0 ? 0 : 1, 1}, clz[2] = {dz == 0 ? 0 : 1, 2};   // zsel 1 = cell k-1
    const int T = ntx * nty * ntz;
    size_t off[8];
    unsigned zbits = 0;
#pragma unroll
    for (int e = 0; e < 8; ++e) {
        // term e < T in mixed radix (ntx, nty, ntz); e >= T repeats term 0 (its value is not added)
        const int ee = e < T ? e : 0;
        const int tz = ee % ntz, ty = (ee / ntz) % nty, tx = ee / (ntz * nty);
        off[e] = ((size_t)cix[tx] * g.ny + cjy[ty]) * g.nz * AM_PER_CELL +
                 (size_t)am_elem(clx[tx] * 9 + cly[ty] * 3 + clz[tz], ij);
        zbits |= (unsigned)zsel[tz] << e;
    }
    const int k0 = zc * EXPAND_Z;
    const int k1 = min(k0 + EXPAND_Z, g.nz);
    double* dst0 = a.M + ((size_t)i * g.ny + j) * g.nz * 243 + (size_t)(o * 9 + ij);
    // longest term list in the warp (the thread order makes it 8, 4, 2, 2, 2, 2, 1, 1 for warps 0..7)
    const int Tw = __reduce_max_sync(__activemask(), T);
    if (Tw == 8) expand_nodes<8>(a, off, zbits, T, k0, k1, dst0);
    else if (Tw == 4) expand_nodes<4>(a, off, zbits, T, k0, k1, dst0);
    else if (Tw == 2) expand_nodes<2>(a, off, zbits, T, k0, k1, dst0);
    else expand_nodes<1>(a, off, zbits, T, k0, k1, dst0);
}

struct ExpandJArgs {
    Geom g;
    const double* AJ;   // [cells][8][4]
    double* rho;        // [nodes] or null
    double* J;          // [3][nodes] or null
    int accumulate;
};

__global__ void __launch_bounds__(256)
k_expand_rhoJ(ExpandJArgs a)
{
    const Geom& g = a.g;
    const long long node = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (node >= g.nodes) return;
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
