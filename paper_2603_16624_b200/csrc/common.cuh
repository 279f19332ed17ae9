// common.cuh -- grid geometry, context and small device helpers shared by the libecpush kernels.
// Product code (sm_100a).  Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>

#define ECSIM_MAX_SPECIES 8

// Periodic grid: node n = (i*ny + j)*nz + k, z fastest; cells = nodes.
struct Geom {
    int nx, ny, nz;
    double dx, dy, dz;
    double rdx, rdy, rdz;   // 1/dx ... formed once on the host in IEEE double
    double Lx, Ly, Lz;      // box lengths n*d
    double invV;            // 1/(dx dy dz): V_N is the same for every node of a periodic grid (L49)
    long long nodes;
    // reduced dimensionality (fixPosition, L123): coordinates of the axes in fix_mask (bit 0 x, 1 y, 2 z) are pinned
    // to fix_pos[axis] by every push, so that all particles stay on one line / plane of the grid
    int fix_mask;
    double fix_pos[3];
};

// fixPosition (L123): "set the particle position along the same line or on the same plane" after updatePosition.
__device__ __forceinline__ void pin_axes(const Geom& g, double& x, double& y, double& z)
{
    if (g.fix_mask) {
        if (g.fix_mask & 1) x = g.fix_pos[0];
        if (g.fix_mask & 2) y = g.fix_pos[1];
        if (g.fix_mask & 4) z = g.fix_pos[2];
    }
}

// A particle's lower node N- per axis (L131): floor(x/dx) clamped into the grid.
__device__ __forceinline__ int lower_node(double s, int n)
{
    int i = __double2int_rd(s);
    return min(max(i, 0), n - 1);
}

// Periodic wrap into [0, L) (reading R13).  The fast path is exact: for x in [0,L)
// floor(x/L) = 0 and x - L*0 = x.
__device__ __forceinline__ double wrap_periodic(double x, double L)
{
    if (x >= 0.0 && x < L) return x;
    x -= L * floor(x / L);
    if (x >= L || x < 0.0) x = 0.0;
    return x;
}

__device__ __forceinline__ unsigned lane_id() { return threadIdx.x & 31u; }

__device__ __forceinline__ double shfl_down_f64(double v, int d)
{
    return __shfl_down_sync(0xffffffffu, v, d);
}
__device__ __forceinline__ double shfl_xor_f64(double v, int d)
{
    return __shfl_xor_sync(0xffffffffu, v, d);
}
