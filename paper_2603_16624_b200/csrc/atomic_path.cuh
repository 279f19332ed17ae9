// atomic_path.cuh -- the paper's own GPU design: one thread per particle, every deposit an atomic
// update on the global arrays ("#pragma acc atomic update"; computeMoments L131-L141
// followed by the mover Eq. 6-8).  Correct for ANY particle order.  In libecpush it serves as
//   (1) ECSIM_VARIANT_ATOMIC, the in-repo prior-art timing, and
//   (2) the stray path of the fused kernel: particles listed in `list` (those found outside the
//       cell segment they are stored in) are pushed and deposited here.
#pragma once
#include "common.cuh"

struct AtomicArgs {
    Geom g;
    uint32_t n;                 // particles (or capacity of the list)
    const uint32_t* list;       // optional: indices to process
    const uint32_t* list_count; // device count of valid list entries
    double *x, *y, *z, *u, *v, *w;
    const double* q;
    const double *E, *B;        // [3][nodes]
    double beta;                // q dt / (2 m) (L55)
    double dt;
    double *rho, *J, *M;        // any may be null (deposit skipped)
    unsigned long long* leavers; // optional: particles whose cell changed in the push
    int do_push;                // 0: deposit only, x and v untouched (ecsim_moments)
};

template <bool USE_LIST>
__global__ void __launch_bounds__(128)
k_push_moments_atomic(AtomicArgs a)
{
    const Geom& g = a.g;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    const size_t count = USE_LIST ? (size_t)*a.list_count : (size_t)a.n;
    unsigned my_leavers = 0;
    for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < count; t += stride) {
        const size_t p = USE_LIST ? a.list[t] : t;
        const double x = a.x[p], y = a.y[p], z = a.z[p];
        const double vx = a.u[p], vy = a.v[p], vz = a.w[p];
        const double q = a.q[p];

        // nodes N-, N+ and the 2x2x2 linear weights (L49, L131)
        const double sx = x * g.rdx, sy = y * g.rdy, sz = z * g.rdz;
        const int i0 = lower_node(sx, g.nx), j0 = lower_node(sy, g.ny), k0 = lower_node(sz, g.nz);
        const int i1 = (i0 + 1 == g.nx) ? 0 : i0 + 1;
        const int j1 = (j0 + 1 == g.ny) ? 0 : j0 + 1;
        const int k1 = (k0 + 1 == g.nz) ? 0 : k0 + 1;
        const double xi = sx - i0, eta = sy - j0, zeta = sz - k0;
        const double wx[2] = {1.0 - xi, xi}, wy[2] = {1.0 - eta, eta}, wz[2] = {1.0 - zeta, zeta};
        double W[8];
        long long node[8];
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            const int ia = (c >> 2) & 1, ib = (c >> 1) & 1, ic = c & 1;
            W[c] = (wx[ia] * wy[ib]) * wz[ic];
            node[c] = ((long long)(ia ? i1 : i0) * g.ny + (ib ? j1 : j0)) * g.nz + (ic ? k1 : k0);
        }

        // gather E^{n+theta}, B^n (L88, L133)
        double Ep[3] = {0, 0, 0}, Bp[3] = {0, 0, 0};
#pragma unroll
        for (int c = 0; c < 8; ++c)
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                Ep[d] += W[c] * __ldg(a.E + d * g.nodes + node[c]);
                Bp[d] += W[c] * __ldg(a.B + d * g.nodes + node[c]);
            }

        // rotation matrix, Eq. (2) as nine scalars (L53, L135); (I x B) v = B x v
        const double bx = a.beta * Bp[0], by = a.beta * Bp[1], bz = a.beta * Bp[2];
        const double invD = 1.0 / (1.0 + (bx * bx + by * by + bz * bz));
        double al[9];
        al[0] = invD * (1.0 + bx * bx);
        al[1] = invD * (bx * by + bz);
        al[2] = invD * (bx * bz - by);
        al[3] = invD * (bx * by - bz);
        al[4] = invD * (1.0 + by * by);
        al[5] = invD * (by * bz + bx);
        al[6] = invD * (bx * bz + by);
        al[7] = invD * (by * bz - bx);
        al[8] = invD * (1.0 + bz * bz);

        // deposits with the pre-push position and velocity (L49): rho (L147), Eq. (1), Eq. (3)
        const double vh[3] = {al[0] * vx + al[1] * vy + al[2] * vz,
                              al[3] * vx + al[4] * vy + al[5] * vz,
                              al[6] * vx + al[7] * vy + al[8] * vz};
        const double qV = q * g.invV;
        const double qbV = qV * a.beta;
#pragma unroll 1
        for (int c = 0; c < 8; ++c) {
            const long long gn = node[c];
            const double dr = qV * W[c];
            if (a.rho) atomicAdd(a.rho + gn, dr);
            if (a.J) {
                atomicAdd(a.J + 0 * g.nodes + gn, dr * vh[0]);
                atomicAdd(a.J + 1 * g.nodes + gn, dr * vh[1]);
                atomicAdd(a.J + 2 * g.nodes + gn, dr * vh[2]);
            }
            if (a.M) {
#pragma unroll
                for (int c2 = 0; c2 < 8; ++c2) {
                    // neighbour slot of N' relative to N: o = (di+1)*9 + (dj+1)*3 + (dk+1)
                    const int o = (((c2 >> 2) & 1) - ((c >> 2) & 1) + 1) * 9 +
                                  (((c2 >> 1) & 1) - ((c >> 1) & 1) + 1) * 3 +
                                  ((c2 & 1) - (c & 1) + 1);
                    const double cf = qbV * (W[c] * W[c2]);
                    double* m = a.M + ((size_t)gn * 27 + o) * 9;
#pragma unroll
                    for (int e = 0; e < 9; ++e) atomicAdd(m + e, cf * al[e]);
                }
            }
        }

        if (!a.do_push) continue;
        // mover, Eq. (6)-(8) with periodic wrap
        const double tx = vx + a.beta * Ep[0], ty = vy + a.beta * Ep[1], tz = vz + a.beta * Ep[2];
        const double vbx = al[0] * tx + al[1] * ty + al[2] * tz;
        const double vby = al[3] * tx + al[4] * ty + al[5] * tz;
        const double vbz = al[6] * tx + al[7] * ty + al[8] * tz;
        const double un = 2.0 * vbx - vx, vn = 2.0 * vby - vy, wn = 2.0 * vbz - vz;
        double xn = x + a.dt * un, yn = y + a.dt * vn, zn = z + a.dt * wn;
        pin_axes(g, xn, yn, zn);
        xn = wrap_periodic(xn, g.Lx); yn = wrap_periodic(yn, g.Ly); zn = wrap_periodic(zn, g.Lz);
        a.u[p] = un; a.v[p] = vn; a.w[p] = wn;
        a.x[p] = xn; a.y[p] = yn; a.z[p] = zn;
        if (USE_LIST) {
            my_leavers += 1;   // a stray stays outside the segment it is stored in
        } else if (a.leavers) {
            const int i2 = lower_node(xn * g.rdx, g.nx), j2 = lower_node(yn * g.rdy, g.ny),
                      k2 = lower_node(zn * g.rdz, g.nz);
            my_leavers += (i2 != i0) | (j2 != j0) | (k2 != k0);
        }
    }
    if (a.leavers) {
        my_leavers = __reduce_add_sync(0xffffffffu, my_leavers);
        if (lane_id() == 0 && my_leavers) atomicAdd(a.leavers, (unsigned long long)my_leavers);
    }
}

// ---------------------------------------------------------------------------------------------
// Strays of the fused variant are deposited into the PER-CELL accumulators of their true cell -- AM[cell][class][ij]
// and AJ[cell][corner][4] (layouts of fused_mma.cuh) -- after the fused kernel stored them and before the expansion
// reads them.  Cost per stray, measured on config 2 (profiles/r01d): 16 ns with 576 + 32 atomics on the node arrays
// (eight 1.9 KB node blocks of HBM read-modify-write), 7.7 ns with 243 + 32 atomics on the cell's block, 1.4-2.2 ns
// with the bulk reduction below.
struct StrayArgs {
    Geom g;
    const uint32_t* list;       // indices of the strays
    const uint32_t* list_count; // device count
    double *x, *y, *z, *u, *v, *w;
    const double* q;
    const double *E, *B;        // [3][nodes]
    double beta, dt;
    double* AM;                 // [cells][AM_PER_CELL]
    double* AJ;                 // [cells][8][4] of this species
    unsigned long long* leavers;
    int do_deposit, do_push;    // ecsim_moments: (1, 0); ecsim_push: (0, 1); ecsim_push_and_moments: (1, 1)
};

// ---------------------------------------------------------------------------------------------
// ONE bulk reduction per stray instead of 275 atomics: a warp handles a stray, builds its
// 244-double contribution to AM[cell] (and 32 doubles to AJ[cell]) in shared memory -- lane = class for the mass
// matrix, lane = corner for rho / Jhat -- and adds both blocks to global memory with cp.reduce.async.bulk
// (.add.f64: the reduction runs in L2 on whole sectors; SASS UBLKRED).  All lanes compute the particle's scalars
// redundantly; lane 0 writes the pushed particle back.
constexpr int STRAY_WARPS = 4;
constexpr int STRAY_SMEM_DOUBLES = 244 + 32;

__device__ __forceinline__ void bulk_reduce_add_f64(double* dst_global, const double* src_shared, unsigned bytes)
{
    asm volatile("cp.reduce.async.bulk.global.shared::cta.bulk_group.add.f64 [%0], [%1], %2;"
                 ::"l"(dst_global), "r"((uint32_t)__cvta_generic_to_shared(src_shared)), "r"(bytes) : "memory");
}

__global__ void __launch_bounds__(STRAY_WARPS * 32)
k_push_strays_bulk(StrayArgs a, int am_per_cell, int am_a8)
{
    __shared__ __align__(128) double stage[STRAY_WARPS][STRAY_SMEM_DOUBLES];
    const Geom& g = a.g;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double* sm = stage[warp];
    const size_t count = (size_t)*a.list_count;
    const size_t wstride = (size_t)gridDim.x * STRAY_WARPS;
    unsigned my_leavers = 0;
    // lane roles: class (kx, ky, kz) of lanes 0..26; corner (ca, cb, cc) of lanes 0..7
    const int cls = lane < 27 ? lane : 0;
    const int kx = cls / 9, ky = (cls / 3) % 3, kz = cls % 3;
    const int ca = (lane >> 2) & 1, cb = (lane >> 1) & 1, cc = lane & 1;
    for (size_t t = (size_t)blockIdx.x * STRAY_WARPS + warp; t < count; t += wstride) {
        const size_t p = a.list[t];
        const double x = a.x[p], y = a.y[p], z = a.z[p];
        const double vx = a.u[p], vy = a.v[p], vz = a.w[p];
        const double q = a.q[p];
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
                Ep[d] += Wc * __ldg(a.E + d * g.nodes + node);
                Bp[d] += Wc * __ldg(a.B + d * g.nodes + node);
            }
        }
        // rotation matrix, Eq. (2) as nine scalars (L53, L135); (I x B) v = B x v
        const double bx = a.beta * Bp[0], by = a.beta * Bp[1], bz = a.beta * Bp[2];
        const double invD = 1.0 / (1.0 + (bx * bx + by * by + bz * bz));
        double al[9];
        al[0] = invD * (1.0 + bx * bx); al[1] = invD * (bx * by + bz); al[2] = invD * (bx * bz - by);
        al[3] = invD * (bx * by - bz); al[4] = invD * (1.0 + by * by); al[5] = invD * (by * bz + bx);
        al[6] = invD * (bx * bz + by); al[7] = invD * (by * bz - bx); al[8] = invD * (1.0 + bz * bz);
        const double vh[3] = {al[0] * vx + al[1] * vy + al[2] * vz, al[3] * vx + al[4] * vy + al[5] * vz,
                              al[6] * vx + al[7] * vy + al[8] * vz};
        const double qV = q * g.invV, qbV = qV * a.beta;
        // this lane's class weight: p?[0..2] = (w0^2, w0 w1, w1^2) per axis (Eq. 3)
        const double fx = (kx == 0 ? wx[0] * wx[0] : kx == 1 ? wx[0] * wx[1] : wx[1] * wx[1]);
        const double fy = (ky == 0 ? wy[0] * wy[0] : ky == 1 ? wy[0] * wy[1] : wy[1] * wy[1]);
        const double fz = (kz == 0 ? wz[0] * wz[0] : kz == 1 ? wz[0] * wz[1] : wz[1] * wz[1]);
        const double cf = qbV * ((fx * fy) * fz);
        if (!a.do_deposit) {
            // push only
        } else if (lane < 27) {
#pragma unroll
            for (int e = 0; e < 8; e += 2)
                *reinterpret_cast<double2*>(sm + lane * 8 + e) = make_double2(cf * al[e], cf * al[e + 1]);
            sm[am_a8 + lane] = cf * al[8];
        } else if (lane == 27) {
            sm[243] = 0.0;                                   // the pad entry of the block
        }
        if (a.do_deposit && lane < 8) {
            // rho / Jhat of corner (ca, cb, cc) (L147, Eq. 1)
            const double wq = qV * ((wx[ca] * wy[cb]) * wz[cc]);
            *reinterpret_cast<double2*>(sm + 244 + lane * 4) = make_double2(wq, wq * vh[0]);
            *reinterpret_cast<double2*>(sm + 244 + lane * 4 + 2) = make_double2(wq * vh[1], wq * vh[2]);
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncwarp();
        const size_t cell = ((size_t)i0 * g.ny + j0) * g.nz + k0;
        if (lane == 0) {
            if (a.do_deposit) {
                bulk_reduce_add_f64(a.AM + cell * am_per_cell, sm, 244 * 8);
                bulk_reduce_add_f64(a.AJ + cell * 32, sm + 244, 32 * 8);
            }
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        }
        if (lane == 0 && a.do_push) {
            // mover, Eq. (6)-(8) with periodic wrap
            const double tx = vx + a.beta * Ep[0], ty = vy + a.beta * Ep[1], tz = vz + a.beta * Ep[2];
            const double un = 2.0 * (al[0] * tx + al[1] * ty + al[2] * tz) - vx;
            const double vn = 2.0 * (al[3] * tx + al[4] * ty + al[5] * tz) - vy;
            const double wn = 2.0 * (al[6] * tx + al[7] * ty + al[8] * tz) - vz;
            a.u[p] = un; a.v[p] = vn; a.w[p] = wn;
            double xn = x + a.dt * un, yn = y + a.dt * vn, zn = z + a.dt * wn;
            pin_axes(g, xn, yn, zn);
            a.x[p] = wrap_periodic(xn, g.Lx);
            a.y[p] = wrap_periodic(yn, g.Ly);
            a.z[p] = wrap_periodic(zn, g.Lz);
            my_leavers += 1;   // a stray stays outside the segment it is stored in
        }
        if (lane == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // the staging block may be rewritten
        __syncwarp();
    }
    if (lane == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");   // every reduction of this warp has landed
    if (a.leavers && lane == 0 && my_leavers) atomicAdd(a.leavers, (unsigned long long)my_leavers);
}

// Strays of the diagnostics pass (dense layout): one thread per listed particle, 8 corners x 13 atomics onto the node
// arrays, after the expansion wrote them.
struct DiagStrayArgs {
    Geom g;
    const uint32_t* list;        // indices, or null: entries 0..count-1 themselves
    const uint32_t* list_count;
    uint32_t count_cap;          // the count is clamped to this
    const double *x, *y, *z, *u, *v, *w, *q;
    double *rho, *J, *P, *Q;
};

__global__ void __launch_bounds__(128)
k_diag_strays(DiagStrayArgs a)
{
    const Geom& g = a.g;
    const size_t count = (size_t)min(*a.list_count, a.count_cap);
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < count; t += stride) {
        const size_t p = a.list ? a.list[t] : t;
        const double sx = a.x[p] * g.rdx, sy = a.y[p] * g.rdy, sz = a.z[p] * g.rdz;
        const int i0 = lower_node(sx, g.nx), j0 = lower_node(sy, g.ny), k0 = lower_node(sz, g.nz);
        const int i1 = (i0 + 1 == g.nx) ? 0 : i0 + 1, j1 = (j0 + 1 == g.ny) ? 0 : j0 + 1, k1 = (k0 + 1 == g.nz) ? 0 : k0 + 1;
        const double xi = sx - i0, eta = sy - j0, zeta = sz - k0;
        const double wx[2] = {1.0 - xi, xi}, wy[2] = {1.0 - eta, eta}, wz[2] = {1.0 - zeta, zeta};
        const double vx = a.u[p], vy = a.v[p], vz = a.w[p];
        const double h = 0.5 * ((vx * vx + vy * vy) + vz * vz);
        const double col[13] = {1.0, vx, vy, vz, vx * vx, vx * vy, vx * vz, vy * vy, vy * vz, vz * vz, h * vx, h * vy, h * vz};
        const double qV = a.q[p] * g.invV;
#pragma unroll 1
        for (int c = 0; c < 8; ++c) {
            const int ia = (c >> 2) & 1, ib = (c >> 1) & 1, ic = c & 1;
            const long long n = ((long long)(ia ? i1 : i0) * g.ny + (ib ? j1 : j0)) * g.nz + (ic ? k1 : k0);
            const double dr = qV * ((wx[ia] * wy[ib]) * wz[ic]);
            if (a.rho) atomicAdd(a.rho + n, dr);
            if (a.J) for (int r = 0; r < 3; ++r) atomicAdd(a.J + (size_t)r * g.nodes + n, dr * col[1 + r]);
            if (a.P) for (int r = 0; r < 6; ++r) atomicAdd(a.P + (size_t)r * g.nodes + n, dr * col[4 + r]);
            if (a.Q) for (int r = 0; r < 3; ++r) atomicAdd(a.Q + (size_t)r * g.nodes + n, dr * col[10 + r]);
        }
    }
}
