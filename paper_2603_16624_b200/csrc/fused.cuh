// fused.cuh -- the fused gather / push / deposit kernel for cell-sorted particles and the
// per-node expansion of its per-cell accumulators.
//
// Design:
//   * One warp owns one cell at a time.  All particles of the cell (all species of the call) are
//     streamed through it in batches of 32.
//   * Phase 1, lane = particle: CIC weights (L49, L131), gather of E^{n+theta}, B^n from the
//     cell's 8 corner nodes staged in shared memory (L88, L133), alpha_p as nine scalars (Eq. 2,
//     L53, L135), push (Eq. 6-8), and the per-particle factors of the deposits, which
//     are written to a per-warp staging tile in shared memory:
//         c[27]   = q beta/V * px[kx] py[ky] pz[kz],   p?[0..2] = (w0^2, w0 w1, w1^2)
//         alpha[9], Wq[8] = q/V * W_corner,  vhat[3] = alpha v^n.
//     Only 27 distinct products W_pN W_pN' exist per particle (three per axis), so the 8x8 = 64
//     (node, neighbour) pairs of Eq. (3) collapse onto 27 "classes" per cell.
//   * Phase 2, lane = accumulator tile: the per-cell sums  A[k][ij] = sum_p c_k(p) alpha_ij(p)
//     (243 numbers), rho/Jhat corner sums (32 numbers) are rank-1 updates with the particles as
//     the contraction index.  Each of 27 lanes keeps a 3 (classes) x 9 (alpha) register tile for
//     one of three particle slots; all 32 lanes keep rho/Jhat for (4 particle slots) x (8 corners).
//     This is the pre-reduction of same-cell particles (north-star (b)), done in registers.
//   * At the end of a cell the tiles are combined with warp shuffles and written ONCE, with plain
//     coalesced stores, to the per-cell arrays AM[cell][27][9], AJ[species][cell][8][4].
//     No atomics; the result is deterministic for a given particle order.
//   * k_expand_* then build the node arrays: M[N][o] is the sum over the 1, 2, 4 or 8 cells that
//     contain both N and N+o of the matching class; rho/Jhat are sums over the 8 cells of a node.
//   * A particle found outside the cell whose segment it is stored in (a "stray") is skipped here,
//     listed, and handled by the atomic path afterwards.
#pragma once
#include "common.cuh"

constexpr int STG_STRIDE = 50;   // doubles per particle in the staging tile (25 x 16 B: odd)
constexpr int STG_C01 = 0;       // 9 pairs (c[rg][0], c[rg][1])
constexpr int STG_C2 = 18;       // 9 x c[rg][2]
constexpr int STG_AL = 28;       // alpha row-major [9]
constexpr int STG_WQ = 38;       // q/V * W[8], corner = a*4 + b*2 + c
constexpr int STG_VH = 46;       // alpha v^n [3]
constexpr int FLD_DOUBLES = 48;  // 8 corners x (Ex,Ey,Ez,Bx,By,Bz)
constexpr int WARP_SMEM_DOUBLES = 32 * STG_STRIDE + FLD_DOUBLES;
constexpr int AM_PER_CELL = 243;
constexpr int AJ_PER_CELL = 32;

struct SpeciesDev {
    const uint32_t* start;   // [cells+1] segment table
    double *x, *y, *z, *u, *v, *w;
    const double* q;
    double beta;             // q dt/(2m) (L55)
    double* AJ;              // [cells][8][4]: rho, Jx, Jy, Jz per corner
    uint32_t* stray_list;
    uint32_t* stray_count;
    unsigned long long* leavers;
};

struct FusedArgs {
    Geom g;
    int n_species;
    const double *E, *B;
    double dt;
    double* AM;              // [cells][27][9]
    SpeciesDev sp[ECSIM_MAX_SPECIES];
};

__device__ __forceinline__ bool in_unit_interval(double t)
{
    // t in [+0, 1): sign clear and exponent below that of 1.0 (NaN and negatives fail)
    return (unsigned)__double2hiint(t) < 0x3FF00000u;
}

template <int NW>
__global__ void __launch_bounds__(NW * 32, 1)
k_fused_push_moments(const __grid_constant__ FusedArgs a)
{
    extern __shared__ __align__(16) double smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double* stg = smem + (size_t)warp * WARP_SMEM_DOUBLES;
    double* fld = stg + 32 * STG_STRIDE;
    for (int t = lane; t < WARP_SMEM_DOUBLES; t += 32) stg[t] = 0.0;
    __syncwarp();

    const Geom& g = a.g;
    const uint32_t cells = (uint32_t)g.nodes;
    const uint32_t total_warps = gridDim.x * NW;
    const int pt = lane / 9, rg = lane - pt * 9;   // M tile: particle slot, class group (lane < 27)
    const int sl = lane >> 3, cn = lane & 7;       // rho/Jhat: particle slot, corner
    const double dt = a.dt;

    for (uint32_t c = blockIdx.x * NW + warp; c < cells; c += total_warps) {
        const int ck = (int)(c % (uint32_t)g.nz);
        const int cj = (int)((c / (uint32_t)g.nz) % (uint32_t)g.ny);
        const int ci = (int)(c / ((uint32_t)g.nz * (uint32_t)g.ny));
        const double dci = (double)ci, dcj = (double)cj, dck = (double)ck;

        // stage the 8 corner nodes' E and B (48 doubles)
        for (int t = lane; t < FLD_DOUBLES; t += 32) {
            const int corner = t / 6, comp = t - corner * 6;
            int ii = ci + ((corner >> 2) & 1); if (ii == g.nx) ii = 0;
            int jj = cj + ((corner >> 1) & 1); if (jj == g.ny) jj = 0;
            int kk = ck + (corner & 1);        if (kk == g.nz) kk = 0;
            const long long node = ((long long)ii * g.ny + jj) * g.nz + kk;
            const double* src = comp < 3 ? a.E + (size_t)comp * g.nodes : a.B + (size_t)(comp - 3) * g.nodes;
            fld[t] = __ldg(src + node);
        }
        __syncwarp();

        double accM[27];
#pragma unroll
        for (int m = 0; m < 27; ++m) accM[m] = 0.0;

        for (int s = 0; s < a.n_species; ++s) {
            const SpeciesDev& sp = a.sp[s];
            const uint32_t beg = __ldg(sp.start + c), end = __ldg(sp.start + c + 1);
            const double beta = sp.beta;
            double aJ0 = 0.0, aJ1 = 0.0, aJ2 = 0.0, aJ3 = 0.0;
            unsigned my_leavers = 0;

            for (uint32_t p0 = beg; p0 < end; p0 += 32) {
                const int nb = (int)min(32u, end - p0);
                const uint32_t p = p0 + lane;
                bool stray = false;
                // ---------------- phase 1: lane = particle ----------------
                if (lane < nb) {
                    const double x = sp.x[p], y = sp.y[p], z = sp.z[p];
                    const double vx = sp.u[p], vy = sp.v[p], vz = sp.w[p];
                    const double q = __ldg(sp.q + p);
                    double* st = stg + lane * STG_STRIDE;
                    // weights relative to the warp's cell; outside [0,1) => not in this cell
                    const double xi = x * g.rdx - dci, eta = y * g.rdy - dcj, zeta = z * g.rdz - dck;
                    if (in_unit_interval(xi) && in_unit_interval(eta) && in_unit_interval(zeta)) {
                        const double wx0 = 1.0 - xi, wy0 = 1.0 - eta, wz0 = 1.0 - zeta;
                        double W[8];
                        {
                            const double w00 = wx0 * wy0, w01 = wx0 * eta, w10 = xi * wy0, w11 = xi * eta;
                            W[0] = w00 * wz0; W[1] = w00 * zeta; W[2] = w01 * wz0; W[3] = w01 * zeta;
                            W[4] = w10 * wz0; W[5] = w10 * zeta; W[6] = w11 * wz0; W[7] = w11 * zeta;
                        }
                        double Ex = 0, Ey = 0, Ez = 0, Bx = 0, By = 0, Bz = 0;
#pragma unroll
                        for (int k = 0; k < 8; ++k) {
                            const double2 f0 = *reinterpret_cast<const double2*>(fld + k * 6);
                            const double2 f1 = *reinterpret_cast<const double2*>(fld + k * 6 + 2);
                            const double2 f2 = *reinterpret_cast<const double2*>(fld + k * 6 + 4);
                            Ex = fma(W[k], f0.x, Ex); Ey = fma(W[k], f0.y, Ey); Ez = fma(W[k], f1.x, Ez);
                            Bx = fma(W[k], f1.y, Bx); By = fma(W[k], f2.x, By); Bz = fma(W[k], f2.y, Bz);
                        }
                        // alpha_p, Eq. (2): (I - [b]x ... ) with (I x B) v = B x v, b = beta B_p
                        const double bx = beta * Bx, by = beta * By, bz = beta * Bz;
                        const double invD = 1.0 / (1.0 + (bx * bx + by * by + bz * bz));
                        const double a00 = invD * (1.0 + bx * bx), a01 = invD * (bx * by + bz), a02 = invD * (bx * bz - by);
                        const double a10 = invD * (bx * by - bz), a11 = invD * (1.0 + by * by), a12 = invD * (by * bz + bx);
                        const double a20 = invD * (bx * bz + by), a21 = invD * (by * bz - bx), a22 = invD * (1.0 + bz * bz);
                        // deposit factors (pre-push x and v, L49)
                        const double vh0 = a00 * vx + a01 * vy + a02 * vz;
                        const double vh1 = a10 * vx + a11 * vy + a12 * vz;
                        const double vh2 = a20 * vx + a21 * vy + a22 * vz;
                        const double qV = q * g.invV, qbV = qV * beta;
                        *reinterpret_cast<double2*>(st + STG_AL + 0) = make_double2(a00, a01);
                        *reinterpret_cast<double2*>(st + STG_AL + 2) = make_double2(a02, a10);
                        *reinterpret_cast<double2*>(st + STG_AL + 4) = make_double2(a11, a12);
                        *reinterpret_cast<double2*>(st + STG_AL + 6) = make_double2(a20, a21);
                        st[STG_AL + 8] = a22;
                        *reinterpret_cast<double2*>(st + STG_WQ + 0) = make_double2(qV * W[0], qV * W[1]);
                        *reinterpret_cast<double2*>(st + STG_WQ + 2) = make_double2(qV * W[2], qV * W[3]);
                        *reinterpret_cast<double2*>(st + STG_WQ + 4) = make_double2(qV * W[4], qV * W[5]);
                        *reinterpret_cast<double2*>(st + STG_WQ + 6) = make_double2(qV * W[6], qV * W[7]);
                        *reinterpret_cast<double2*>(st + STG_VH + 0) = make_double2(vh0, vh1);
                        st[STG_VH + 2] = vh2;
                        {
                            // 27 classes: q beta/V * px[kx] * py[ky] * pz[kz]
                            const double qx0 = qbV * wx0, qx1 = qbV * xi;
                            const double px[3] = {qx0 * wx0, qx0 * xi, qx1 * xi};
                            const double py[3] = {wy0 * wy0, wy0 * eta, eta * eta};
                            const double pz0 = wz0 * wz0, pz1 = wz0 * zeta, pz2 = zeta * zeta;
#pragma unroll
                            for (int kx = 0; kx < 3; ++kx)
#pragma unroll
                                for (int ky = 0; ky < 3; ++ky) {
                                    const double pxy = px[kx] * py[ky];
                                    const int r = kx * 3 + ky;
                                    *reinterpret_cast<double2*>(st + STG_C01 + 2 * r) = make_double2(pxy * pz0, pxy * pz1);
                                    st[STG_C2 + r] = pxy * pz2;
                                }
                        }
                        // mover, Eq. (6)-(8)
                        const double tx = vx + beta * Ex, ty = vy + beta * Ey, tz = vz + beta * Ez;
                        const double vbx = a00 * tx + a01 * ty + a02 * tz;
                        const double vby = a10 * tx + a11 * ty + a12 * tz;
                        const double vbz = a20 * tx + a21 * ty + a22 * tz;
                        const double un = 2.0 * vbx - vx, vn = 2.0 * vby - vy, wn = 2.0 * vbz - vz;
                        const double xn = wrap_periodic(x + dt * un, g.Lx);
                        const double yn = wrap_periodic(y + dt * vn, g.Ly);
                        const double zn = wrap_periodic(z + dt * wn, g.Lz);
                        sp.u[p] = un; sp.v[p] = vn; sp.w[p] = wn;
                        sp.x[p] = xn; sp.y[p] = yn; sp.z[p] = zn;
                        const bool stays = in_unit_interval(xn * g.rdx - dci) && in_unit_interval(yn * g.rdy - dcj) &&
                                           in_unit_interval(zn * g.rdz - dck);
                        my_leavers += stays ? 0u : 1u;
                    } else {
                        stray = true;
#pragma unroll
                        for (int r = 0; r < 9; ++r) {
                            *reinterpret_cast<double2*>(st + STG_C01 + 2 * r) = make_double2(0.0, 0.0);
                            st[STG_C2 + r] = 0.0;
                        }
#pragma unroll
                        for (int k = 0; k < 8; ++k) st[STG_WQ + k] = 0.0;
                    }
                }
                const unsigned smask = __ballot_sync(0xffffffffu, stray);
                if (smask) {
                    uint32_t base = 0;
                    if (lane == 0) base = atomicAdd(sp.stray_count, (uint32_t)__popc(smask));
                    base = __shfl_sync(0xffffffffu, base, 0);
                    if (stray) sp.stray_list[base + __popc(smask & ((1u << lane) - 1u))] = p;
                }
                __syncwarp();

                // ---------------- phase 2: lane = accumulator tile ----------------
                if (lane < 27) {
                    const int nsteps = (nb + 2) / 3;
#pragma unroll 2
                    for (int s3 = 0; s3 < nsteps; ++s3) {
                        const int pp = s3 * 3 + pt;
                        if (pp < nb) {
                            const double* b = stg + pp * STG_STRIDE;
                            const double2 c01 = *reinterpret_cast<const double2*>(b + STG_C01 + 2 * rg);
                            const double c2 = b[STG_C2 + rg];
                            const double2 l0 = *reinterpret_cast<const double2*>(b + STG_AL + 0);
                            const double2 l1 = *reinterpret_cast<const double2*>(b + STG_AL + 2);
                            const double2 l2 = *reinterpret_cast<const double2*>(b + STG_AL + 4);
                            const double2 l3 = *reinterpret_cast<const double2*>(b + STG_AL + 6);
                            const double l8 = b[STG_AL + 8];
                            const double al[9] = {l0.x, l0.y, l1.x, l1.y, l2.x, l2.y, l3.x, l3.y, l8};
#pragma unroll
                            for (int j = 0; j < 9; ++j) {
                                accM[j] = fma(c01.x, al[j], accM[j]);
                                accM[9 + j] = fma(c01.y, al[j], accM[9 + j]);
                                accM[18 + j] = fma(c2, al[j], accM[18 + j]);
                            }
                        }
                    }
                }
                {
                    const int nsteps = (nb + 3) / 4;
#pragma unroll 2
                    for (int s4 = 0; s4 < nsteps; ++s4) {
                        const int pp = s4 * 4 + sl;
                        if (pp < nb) {
                            const double* b = stg + pp * STG_STRIDE;
                            const double wq = b[STG_WQ + cn];
                            const double2 vh01 = *reinterpret_cast<const double2*>(b + STG_VH);
                            const double vh2 = b[STG_VH + 2];
                            aJ0 += wq;
                            aJ1 = fma(wq, vh01.x, aJ1);
                            aJ2 = fma(wq, vh01.y, aJ2);
                            aJ3 = fma(wq, vh2, aJ3);
                        }
                    }
                }
                __syncwarp();
            }

            // rho/Jhat of this species for this cell: combine the 4 particle slots, one store
            aJ0 += shfl_xor_f64(aJ0, 8);  aJ1 += shfl_xor_f64(aJ1, 8);
            aJ2 += shfl_xor_f64(aJ2, 8);  aJ3 += shfl_xor_f64(aJ3, 8);
            aJ0 += shfl_xor_f64(aJ0, 16); aJ1 += shfl_xor_f64(aJ1, 16);
            aJ2 += shfl_xor_f64(aJ2, 16); aJ3 += shfl_xor_f64(aJ3, 16);
            if (lane < 8) {
                double* dst = sp.AJ + (size_t)c * AJ_PER_CELL + lane * 4;
                *reinterpret_cast<double2*>(dst) = make_double2(aJ0, aJ1);
                *reinterpret_cast<double2*>(dst + 2) = make_double2(aJ2, aJ3);
            }
            my_leavers = __reduce_add_sync(0xffffffffu, my_leavers);
            if (lane == 0 && my_leavers) atomicAdd(sp.leavers, (unsigned long long)my_leavers);
        }

        // mass-matrix classes of this cell: combine the 3 particle slots, write 243 doubles once
#pragma unroll
        for (int m = 0; m < 27; ++m) {
            double v = accM[m];
            v += shfl_down_f64(accM[m], 9);
            v += shfl_down_f64(accM[m], 18);
            if (lane < 9) stg[rg * 27 + m] = v;
        }
        __syncwarp();
        {
            double* dst = a.AM + (size_t)c * AM_PER_CELL;
            for (int t = lane; t < AM_PER_CELL; t += 32) dst[t] = stg[t];
        }
        __syncwarp();
    }
}

// ---------------------------------------------------------------------------------------------
// Expansion of the per-cell classes to the node arrays.
//
// Node N = (i,j,k) is corner a=0 of cell i and corner a=1 of cell i-1 (per axis).  For neighbour
// offset d along an axis the pairs (a, a') with a' - a = d inside one cell are
//     d =  0 : (0,0) in cell i   -> class 0 (w0^2)   and (1,1) in cell i-1 -> class 2 (w1^2)
//     d = +1 : (0,1) in cell i   -> class 1 (w0 w1)
//     d = -1 : (1,0) in cell i-1 -> class 1
// and the 3-D term list is the product of the three per-axis lists (1, 2, 4 or 8 cells).
// One CTA walks EXPAND_NODES consecutive nodes; thread r < 243 owns element (o, ij) = (r/9, r%9).
constexpr int EXPAND_NODES = 16;

struct ExpandArgs {
    Geom g;
    const double* AM;
    double* M;
    int accumulate;
};

__global__ void __launch_bounds__(256)
k_expand_M(ExpandArgs a)
{
    const int r = threadIdx.x;
    if (r >= 243) return;
    const Geom& g = a.g;
    const int o = r / 9, ij = r - o * 9;
    const int d[3] = {o / 9 - 1, (o / 3) % 3 - 1, o % 3 - 1};
    // per axis: number of terms, cell shift (0 or -1) and class of each term
    int nt[3], sh[3][2], cl[3][2];
#pragma unroll
    for (int ax = 0; ax < 3; ++ax) {
        if (d[ax] == 0)      { nt[ax] = 2; sh[ax][0] = 0;  cl[ax][0] = 0; sh[ax][1] = -1; cl[ax][1] = 2; }
        else if (d[ax] > 0)  { nt[ax] = 1; sh[ax][0] = 0;  cl[ax][0] = 1; sh[ax][1] = 0;  cl[ax][1] = 0; }
        else                 { nt[ax] = 1; sh[ax][0] = -1; cl[ax][0] = 1; sh[ax][1] = 0;  cl[ax][1] = 0; }
    }
    const long long n0 = (long long)blockIdx.x * EXPAND_NODES;
    for (int t = 0; t < EXPAND_NODES; ++t) {
        const long long node = n0 + t;
        if (node >= g.nodes) break;
        const int k = (int)(node % g.nz);
        const int j = (int)((node / g.nz) % g.ny);
        const int i = (int)(node / ((long long)g.nz * g.ny));
        double sum = 0.0;
        for (int tx = 0; tx < nt[0]; ++tx) {
            int ci = i + sh[0][tx]; if (ci < 0) ci += g.nx;
            for (int ty = 0; ty < nt[1]; ++ty) {
                int cj = j + sh[1][ty]; if (cj < 0) cj += g.ny;
                for (int tz = 0; tz < nt[2]; ++tz) {
                    int ck = k + sh[2][tz]; if (ck < 0) ck += g.nz;
                    const long long cell = ((long long)ci * g.ny + cj) * g.nz + ck;
                    const int cls = cl[0][tx] * 9 + cl[1][ty] * 3 + cl[2][tz];
                    sum += a.AM[(size_t)cell * AM_PER_CELL + cls * 9 + ij];
                }
            }
        }
        double* dst = a.M + (size_t)node * 243 + r;
        if (a.accumulate) sum += *dst;
        *dst = sum;
    }
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
