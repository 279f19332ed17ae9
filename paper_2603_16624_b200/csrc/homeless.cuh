// homeless.cuh -- resident species (LAYOUT_GAPPED): the particles a push could not place in their new cell's segment
// (it was full) wait in the species' overflow list.  They are ordinary particles without a slot: every pass handles them
// here, one warp per particle, exactly like the strays of the dense layout (k_push_strays_bulk) -- deposit with ONE
// bulk reduction onto the per-cell accumulators of the cell they are in (before the expansion reads them), push -- and
// then tries again to give them a slot (relocate(), fused_mma.cuh): most find room one step later, when their cell's own
// leavers have made space.  Only when the list keeps growing does the host lay the species out afresh (rent-or-buy, as
// for the re-sort of a dense species).
#pragma once
#include "atomic_path.cuh"
#include "fused_mma.cuh"

struct HomelessArgs {
    Geom g;
    SpeciesDev sp;              // tables, output buffer and OUTPUT overflow list of the species (as in FusedArgs)
    const double* in;           // [7][in_cap] INPUT overflow list (the one the previous push wrote)
    uint32_t in_cap;
    const uint32_t* in_count;
    const double *E, *B;
    double dt;
    double* AM;
    int do_deposit, do_push;
};

__global__ void __launch_bounds__(STRAY_WARPS * 32)
k_push_homeless(const __grid_constant__ HomelessArgs a)
{
    __shared__ __align__(128) double stage[STRAY_WARPS][STRAY_SMEM_DOUBLES];
    const Geom& g = a.g;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double* sm = stage[warp];
    const size_t count = (size_t)min(*a.in_count, a.in_cap);
    const size_t wstride = (size_t)gridDim.x * STRAY_WARPS;
    const size_t m = a.in_cap;
    const double beta = a.sp.beta;
    const int cls = lane < 27 ? lane : 0;
    const int kx = cls / 9, ky = (cls / 3) % 3, kz = cls % 3;
    const int ca = (lane >> 2) & 1, cb = (lane >> 1) & 1, cc = lane & 1;
    unsigned moved = 0;
    for (size_t t = (size_t)blockIdx.x * STRAY_WARPS + warp; t < count; t += wstride) {
        const double x = a.in[t], y = a.in[m + t], z = a.in[2 * m + t];
        const double vx = a.in[3 * m + t], vy = a.in[4 * m + t], vz = a.in[5 * m + t];
        const double q = a.in[6 * m + t];
        const double sx = x * g.rdx, sy = y * g.rdy, sz = z * g.rdz;
        const int i0 = lower_node(sx, g.nx), j0 = lower_node(sy, g.ny), k0 = lower_node(sz, g.nz);
        const int i1 = (i0 + 1 == g.nx) ? 0 : i0 + 1;
        const int j1 = (j0 + 1 == g.ny) ? 0 : j0 + 1;
        const int k1 = (k0 + 1 == g.nz) ? 0 : k0 + 1;
        const double xi = sx - i0, eta = sy - j0, zeta = sz - k0;
        const double wx[2] = {1.0 - xi, xi}, wy[2] = {1.0 - eta, eta}, wz[2] = {1.0 - zeta, zeta};
        double Ep[3] = {0, 0, 0}, Bp[3] = {0, 0, 0};
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            const int ia = (c >> 2) & 1, ib = (c >> 1) & 1, ic = c & 1;
            const double Wc = (wx[ia] * wy[ib]) * wz[ic];
            const long long node = ((long long)(ia ? i1 : i0) * g.ny + (ib ? j1 : j0)) * g.nz + (ic ? k1 : k0);
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                if (a.do_push) Ep[d] += Wc * __ldg(a.E + d * g.nodes + node);
                Bp[d] += Wc * __ldg(a.B + d * g.nodes + node);
            }
        }
        // rotation matrix, Eq. (2) as nine scalars (L53, L135); (I x B) v = B x v
        const double bx = beta * Bp[0], by = beta * Bp[1], bz = beta * Bp[2];
        const double invD = 1.0 / (1.0 + (bx * bx + by * by + bz * bz));
        double al[9];
        al[0] = invD * (1.0 + bx * bx); al[1] = invD * (bx * by + bz); al[2] = invD * (bx * bz - by);
        al[3] = invD * (bx * by - bz); al[4] = invD * (1.0 + by * by); al[5] = invD * (by * bz + bx);
        al[6] = invD * (bx * bz + by); al[7] = invD * (by * bz - bx); al[8] = invD * (1.0 + bz * bz);
        if (a.do_deposit) {
            const double vh[3] = {al[0] * vx + al[1] * vy + al[2] * vz, al[3] * vx + al[4] * vy + al[5] * vz,
                                  al[6] * vx + al[7] * vy + al[8] * vz};
            const double qV = q * g.invV, qbV = qV * beta;
            const double fx = (kx == 0 ? wx[0] * wx[0] : kx == 1 ? wx[0] * wx[1] : wx[1] * wx[1]);
            const double fy = (ky == 0 ? wy[0] * wy[0] : ky == 1 ? wy[0] * wy[1] : wy[1] * wy[1]);
            const double fz = (kz == 0 ? wz[0] * wz[0] : kz == 1 ? wz[0] * wz[1] : wz[1] * wz[1]);
            const double cf = qbV * ((fx * fy) * fz);
            if (lane < 27) {
#pragma unroll
                for (int e = 0; e < 8; e += 2)
                    *reinterpret_cast<double2*>(sm + lane * 8 + e) = make_double2(cf * al[e], cf * al[e + 1]);
                sm[AM_A8 + lane] = cf * al[8];
            } else if (lane == 27) {
                sm[243] = 0.0;
            }
            if (lane < 8) {
                const double wq = qV * ((wx[ca] * wy[cb]) * wz[cc]);
                *reinterpret_cast<double2*>(sm + 244 + lane * 4) = make_double2(wq, wq * vh[0]);
                *reinterpret_cast<double2*>(sm + 244 + lane * 4 + 2) = make_double2(wq * vh[1], wq * vh[2]);
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            __syncwarp();
            const size_t cell = ((size_t)i0 * g.ny + j0) * g.nz + k0;
            if (lane == 0) {
                bulk_reduce_add_f64(a.AM + cell * AM_PER_CELL, sm, 244 * 8);
                bulk_reduce_add_f64(a.sp.AJ + cell * AJ_PER_CELL, sm + 244, 32 * 8);
                asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            }
        }
        if (lane == 0 && a.do_push) {
            // mover, Eq. (6)-(8), then another try at a slot in the buffer being written
            const double tx = vx + beta * Ep[0], ty = vy + beta * Ep[1], tz = vz + beta * Ep[2];
            PushedRegs o;
            o.u = 2.0 * (al[0] * tx + al[1] * ty + al[2] * tz) - vx;
            o.v = 2.0 * (al[3] * tx + al[4] * ty + al[5] * tz) - vy;
            o.w = 2.0 * (al[6] * tx + al[7] * ty + al[8] * tz) - vz;
            double xn = x + a.dt * o.u, yn = y + a.dt * o.v, zn = z + a.dt * o.w;
            pin_axes(g, xn, yn, zn);
            o.x = wrap_periodic(xn, g.Lx); o.y = wrap_periodic(yn, g.Ly); o.z = wrap_periodic(zn, g.Lz);
            o.stays = false;
            relocate(g, a.sp, o, q);
            moved += 1;
        }
        if (lane == 0 && a.do_deposit) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
        __syncwarp();
    }
    if (lane == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    if (lane == 0 && moved && a.sp.leavers) atomicAdd(a.sp.leavers, (unsigned long long)moved);
}
