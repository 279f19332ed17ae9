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
// k_expand_M_stream (expand_tma.cuh) builds M; the outputs of a node are taken in the order of EXPAND_ORDER,
// i.e. by the SHAPE of their term list ((x-y terms) x (z terms)), so that the threads of a warp loop equally long.
// k_expand_rhoJ (below) builds rho and Jhat: 8 corner sums per node.
#pragma once
#include "common.cuh"
#include "fused_mma.cuh"

// neighbour slots ordered by (x-y terms, z terms) = (4,2) | (4,1) | (2,2) | (2,1) | (1,2) | (1,1)
__device__ __constant__ unsigned char EXPAND_ORDER[27] = {
    13,
    12, 14,
    4, 10, 16, 22,
    3, 5, 9, 11, 15, 17, 21, 23,
    1, 7, 19, 25,
    0, 2, 6, 8, 18, 20, 24, 26};
// the 14 slots o >= 13 of the symmetric storage (L73), same ordering rule
__device__ __constant__ unsigned char EXPAND_ORDER14[14] = {
    13,
    14,
    16, 22,
    15, 17, 21, 23,
    19, 25,
    18, 20, 24, 26};

// Offset, in doubles inside a cell's AM block, of (class, ij): 8*class + ij for ij < 8, AM_A8 + class for
// ij = 8 -- additive in the per-axis parts of class = 9 clx + 3 cly + clz.

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

// MODE_DIAG (fused_mma.cuh): node sums of the per-cell corner blocks AD[cell][8][16] -> rho, J (un-rotated), P, Q
// (PAPER.md L121, L147).  Column c of a corner block: 0 rho; 1..3 J; 4..9 P (xx,xy,xz,yy,yz,zz); 10..12 Q.
struct ExpandDiagArgs {
    Geom g;
    const double* AD;   // [cells][8][16]
    double *rho, *J, *P, *Q;   // [nodes], [3][nodes], [6][nodes], [3][nodes]; any may be null
};

__global__ void __launch_bounds__(256)
k_expand_diag(ExpandDiagArgs a)
{
    const Geom& g = a.g;
    const long long node = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (node >= g.nodes) return;
    const int k = (int)(node % g.nz);
    const int j = (int)((node / g.nz) % g.ny);
    const int i = (int)(node / ((long long)g.nz * g.ny));
    double s[13];
#pragma unroll
    for (int c = 0; c < 13; ++c) s[c] = 0.0;
#pragma unroll
    for (int corner = 0; corner < 8; ++corner) {
        int ci = i - ((corner >> 2) & 1); if (ci < 0) ci += g.nx;
        int cj = j - ((corner >> 1) & 1); if (cj < 0) cj += g.ny;
        int ck = k - (corner & 1);        if (ck < 0) ck += g.nz;
        const long long cell = ((long long)ci * g.ny + cj) * g.nz + ck;
        const double* src = a.AD + (size_t)cell * AD_PER_CELL + corner * 16;
#pragma unroll
        for (int c = 0; c < 12; c += 2) {
            const double2 v = *reinterpret_cast<const double2*>(src + c);
            s[c] += v.x; s[c + 1] += v.y;
        }
        s[12] += src[12];
    }
    if (a.rho) a.rho[node] = s[0];
    if (a.J) for (int c = 0; c < 3; ++c) a.J[(size_t)c * g.nodes + node] = s[1 + c];
    if (a.P) for (int c = 0; c < 6; ++c) a.P[(size_t)c * g.nodes + node] = s[4 + c];
    if (a.Q) for (int c = 0; c < 3; ++c) a.Q[(size_t)c * g.nodes + node] = s[10 + c];
}
