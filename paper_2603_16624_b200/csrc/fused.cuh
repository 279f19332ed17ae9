// fused.cuh -- the fused gather / push / deposit kernel for cell-sorted particles and the
// per-node expansion of its per-cell accumulators.
//
// Design:
//   * The FP64 pipe bounds this path (DMMA shares that pipe on sm_100a, so
//     tensor cores give nothing).  Everything below is about keeping the DFMA pipe fed: few
//     non-FP64 instructions per DFMA, no divergent branches, global loads issued a batch ahead.
//   * One warp owns a contiguous range of cells, chosen from the segment tables so that every warp
//     of the grid gets the same number of particles (+ a per-cell weight): a particle-balanced
//     schedule that also serves non-uniform loads (Harris sheet).
//   * Per cell, all particles of all species of the call stream through the warp in batches of 32.
//   * Phase 1, lane = particle, branch-free: CIC weights (L49, L131), gather of E^{n+theta}, B^n
//     from the cell's 8 corner nodes staged in shared memory (L88, L133), alpha_p as nine scalars
//     (Eq. 2), push (Eq. 6-8), and the per-particle factors of the deposits,
//     written to a per-warp staging tile in shared memory:
//         c[27]   = q beta/V * px[kx] py[ky] pz[kz],   p?[0..2] = (w0^2, w0 w1, w1^2)
//         alpha[9], Wq[8] = q/V * W_corner,  vhat[3] = alpha v^n.
//     Only 27 distinct products W_pN W_pN' exist per particle (three per axis), so the 8x8 = 64
//     (node, neighbour) pairs of Eq. (3) collapse onto 27 "classes" per cell.  Lanes without a
//     particle (ragged tail, strays) run the same code with q = 0, so their rows hold zeros.
//   * Phase 2, lane = accumulator tile: A[k][ij] = sum_p c_k(p) alpha_ij(p) (243 numbers) and the
//     rho/Jhat corner sums (32 numbers) are rank-1 updates with the particles as the contraction
//     index.  Lane (pt, rg) of the first 27 keeps a 3 (classes) x 9 (alpha) register tile for
//     particle slot pt; all 32 lanes keep rho/Jhat for (4 particle slots) x (8 corners).  A full
//     batch is 11 + 8 fully unrolled steps of LDS + DFMA with constant offsets.
//     This is the pre-reduction of same-cell particles (north-star (b)), done in registers.
//   * At the end of a cell the slot tiles are summed through shared memory and written ONCE, with
//     plain coalesced stores, to AM[cell][27][9], AJ[species][cell][8][4].  No atomics; the result
//     is deterministic for a given particle order.
//   * k_expand_* then build the node arrays: M[N][o] is the sum over the 1, 2, 4 or 8 cells that
//     contain both N and N+o of the matching class; rho/Jhat are sums over the 8 cells of a node.
//   * A particle found outside the cell whose segment it is stored in (a "stray") is skipped here,
//     listed, and handled by the atomic path afterwards.
#pragma once
#include "common.cuh"

constexpr int STG_STRIDE = 50;   // doubles per particle row of the staging tile (25 x 16 B: odd)
constexpr int STG_C01 = 0;       // 9 pairs (c[rg][0], c[rg][1])
constexpr int STG_C2 = 18;       // 9 x c[rg][2]
constexpr int STG_AL = 28;       // alpha row-major [9]
constexpr int STG_WQ = 38;       // q/V * W[8], corner = a*4 + b*2 + c
constexpr int STG_VH = 46;       // alpha v^n [3]
constexpr int STG_ROWS = 33;     // 32 particles + one row that stays zero (11 steps x 3 slots)
constexpr int FLD_DOUBLES = 48;  // 8 corners x (Ex,Ey,Ez,Bx,By,Bz)
constexpr int WARP_SMEM_DOUBLES = STG_ROWS * STG_STRIDE + FLD_DOUBLES;
constexpr int AM_PER_CELL = 243;
constexpr int AJ_PER_CELL = 32;
constexpr int FLUSH_RG_STRIDE = 28;             // 27 accumulators of a lane, padded to 16 B
constexpr int FLUSH_SLOT_STRIDE = 9 * FLUSH_RG_STRIDE;
constexpr unsigned CELL_WEIGHT = 8;             // schedule weight of a cell, in particles

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
    double* AM;                      // [cells][27][9]
    unsigned long long weight_total; // sum of particles of the listed species + CELL_WEIGHT * cells
    SpeciesDev sp[ECSIM_MAX_SPECIES];
};

__device__ __forceinline__ bool in_unit_interval(double t)
{
    // t in [+0, 1): sign clear and exponent below that of 1.0 (NaN and negatives fail)
    return (unsigned)__double2hiint(t) < 0x3FF00000u;
}

// Periodic wrap with an integer fast-path test: for x >= +0 the order of doubles is the order of
// their bit patterns, so "0 <= x < L" is one unsigned 64-bit compare (negatives and NaN fail it).
__device__ __forceinline__ double wrap_fast(double x, double L)
{
    if ((unsigned long long)__double_as_longlong(x) < (unsigned long long)__double_as_longlong(L)) return x;
    return wrap_periodic(x, L);
}

// First cell of warp w's range: smallest c with  CELL_WEIGHT*c + sum_s start_s[c] >= w/W of the total.
__device__ __forceinline__ uint32_t range_bound(const FusedArgs& a, uint32_t w, uint32_t W)
{
    const uint32_t cells = (uint32_t)a.g.nodes;
    if (w == 0) return 0;
    if (w >= W) return cells;
    const unsigned long long target = a.weight_total / W * w + (a.weight_total % W) * w / W;
    uint32_t lo = 0, hi = cells;
    while (lo < hi) {
        const uint32_t mid = lo + (hi - lo) / 2;
        unsigned long long f = (unsigned long long)CELL_WEIGHT * mid;
        for (int s = 0; s < a.n_species; ++s) f += __ldg(a.sp[s].start + mid);
        if (f >= target) hi = mid; else lo = mid + 1;
    }
    return lo;
}

struct ParticleRegs { double x, y, z, u, v, w, q; };

__device__ __forceinline__ void load_batch(const SpeciesDev& sp, uint32_t p0, int nb, int lane, ParticleRegs& r)
{
    if (lane < nb) {
        const uint32_t p = p0 + lane;
        r.x = sp.x[p]; r.y = sp.y[p]; r.z = sp.z[p];
        r.u = sp.u[p]; r.v = sp.v[p]; r.w = sp.w[p];
        r.q = __ldg(sp.q + p);
    }
}

// Phase 1 for one lane: returns true if the lane holds a stray.  `st` = the lane's staging row,
// `fld` = the cell's corner fields, (dci,dcj,dck) = the cell's integer coordinates as doubles.
__device__ __forceinline__ bool phase1(const Geom& g, const SpeciesDev& sp, const ParticleRegs& r, bool active,
                                       uint32_t p, double beta, double dt, double dci, double dcj, double dck,
                                       const double* __restrict__ fld, double* __restrict__ st, unsigned& leavers)
{
    // weights relative to the warp's cell; outside [0,1) => not in this cell
    double xi = r.x * g.rdx - dci, eta = r.y * g.rdy - dcj, zeta = r.z * g.rdz - dck;
    const bool inside = active && in_unit_interval(xi) && in_unit_interval(eta) && in_unit_interval(zeta);
    // lanes without a particle of this cell compute on harmless numbers with zero charge
    if (!inside) { xi = 0.5; eta = 0.5; zeta = 0.5; }
    const double vx = inside ? r.u : 0.0, vy = inside ? r.v : 0.0, vz = inside ? r.w : 0.0;
    const double q = inside ? r.q : 0.0;
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
    // alpha_p, Eq. (2): (I x B) v = B x v, b = beta B_p;  alpha = (I + [b]x)^-1
    const double bx = beta * Bx, by = beta * By, bz = beta * Bz;
    const double invD = 1.0 / (1.0 + (bx * bx + by * by + bz * bz));
    const double sx = invD * bx, sy = invD * by, sz = invD * bz;
    const double a00 = fma(bx, sx, invD), a01 = fma(bx, sy, sz), a02 = fma(bx, sz, -sy);
    const double a10 = fma(by, sx, -sz), a11 = fma(by, sy, invD), a12 = fma(by, sz, sx);
    const double a20 = fma(bz, sx, sy), a21 = fma(bz, sy, -sx), a22 = fma(bz, sz, invD);
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
                const int rr = kx * 3 + ky;
                *reinterpret_cast<double2*>(st + STG_C01 + 2 * rr) = make_double2(pxy * pz0, pxy * pz1);
                st[STG_C2 + rr] = pxy * pz2;
            }
    }
    // mover, Eq. (6)-(8)
    const double tx = fma(beta, Ex, vx), ty = fma(beta, Ey, vy), tz = fma(beta, Ez, vz);
    const double vbx = a00 * tx + a01 * ty + a02 * tz;
    const double vby = a10 * tx + a11 * ty + a12 * tz;
    const double vbz = a20 * tx + a21 * ty + a22 * tz;
    const double un = 2.0 * vbx - vx, vn = 2.0 * vby - vy, wn = 2.0 * vbz - vz;
    if (inside) {
        const double xn = wrap_fast(fma(dt, un, r.x), g.Lx);
        const double yn = wrap_fast(fma(dt, vn, r.y), g.Ly);
        const double zn = wrap_fast(fma(dt, wn, r.z), g.Lz);
        sp.u[p] = un; sp.v[p] = vn; sp.w[p] = wn;
        sp.x[p] = xn; sp.y[p] = yn; sp.z[p] = zn;
        const bool stays = in_unit_interval(xn * g.rdx - dci) && in_unit_interval(yn * g.rdy - dcj) &&
                           in_unit_interval(zn * g.rdz - dck);
        leavers += stays ? 0u : 1u;
    }
    return active && !inside;
}

// Phase 2, mass-matrix part: one step = three particle rows (row0 + slot), lane tile 3 classes x 9 alpha.
// `bc01`, `bc2`, `bal` are the lane's base pointers (slot row, class group folded in).
__device__ __forceinline__ void m_step(const double* __restrict__ bc01, const double* __restrict__ bc2,
                                       const double* __restrict__ bal, int off, double (&accM)[27])
{
    const double2 c01 = *reinterpret_cast<const double2*>(bc01 + off);
    const double c2 = bc2[off];
    const double2 l0 = *reinterpret_cast<const double2*>(bal + off + 0);
    const double2 l1 = *reinterpret_cast<const double2*>(bal + off + 2);
    const double2 l2 = *reinterpret_cast<const double2*>(bal + off + 4);
    const double2 l3 = *reinterpret_cast<const double2*>(bal + off + 6);
    const double l8 = bal[off + 8];
    const double al[9] = {l0.x, l0.y, l1.x, l1.y, l2.x, l2.y, l3.x, l3.y, l8};
#pragma unroll
    for (int j = 0; j < 9; ++j) {
        accM[j] = fma(c01.x, al[j], accM[j]);
        accM[9 + j] = fma(c01.y, al[j], accM[9 + j]);
        accM[18 + j] = fma(c2, al[j], accM[18 + j]);
    }
}

// Phase 2, rho/Jhat part: one step = four particle rows, lane = (slot, corner).
__device__ __forceinline__ void j_step(const double* __restrict__ bwq, const double* __restrict__ bvh, int off,
                                       double& aJ0, double& aJ1, double& aJ2, double& aJ3)
{
    const double wq = bwq[off];
    const double2 vh01 = *reinterpret_cast<const double2*>(bvh + off);
    const double vh2 = bvh[off + 2];
    aJ0 += wq;
    aJ1 = fma(wq, vh01.x, aJ1);
    aJ2 = fma(wq, vh01.y, aJ2);
    aJ3 = fma(wq, vh2, aJ3);
}

template <int NW>
__global__ void __launch_bounds__(NW * 32, 1)
k_fused_push_moments(const __grid_constant__ FusedArgs a)
{
    extern __shared__ __align__(16) double smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double* stg = smem + (size_t)warp * WARP_SMEM_DOUBLES;
    double* fld = stg + STG_ROWS * STG_STRIDE;
    for (int t = lane; t < WARP_SMEM_DOUBLES; t += 32) stg[t] = 0.0;
    __syncwarp();

    const Geom& g = a.g;
    const int nsp = a.n_species;
    const double dt = a.dt;
    const uint32_t W = gridDim.x * NW, wid = blockIdx.x * NW + warp;
    const uint32_t c_lo = range_bound(a, wid, W), c_hi = range_bound(a, wid + 1, W);
    if (c_lo >= c_hi) return;

    // lane roles of phase 2.  Lanes 27..31 shadow lanes 0..4 in the M part (results unused).
    const int ml = lane < 27 ? lane : lane - 27;
    const int pt = ml / 9, rg = ml - pt * 9;       // particle slot, class group
    const int sl = lane >> 3, cn = lane & 7;       // rho/Jhat: particle slot, corner
    const double* bc01 = stg + pt * STG_STRIDE + STG_C01 + 2 * rg;
    const double* bc2 = stg + pt * STG_STRIDE + STG_C2 + rg;
    const double* bal = stg + pt * STG_STRIDE + STG_AL;
    const double* bwq = stg + sl * STG_STRIDE + STG_WQ + cn;
    const double* bvh = stg + sl * STG_STRIDE + STG_VH;
    double* strow = stg + lane * STG_STRIDE;

    // field staging: lane t and t+32 (< 48) hold corner t/6, component t%6 of the next cell
    const int fc0 = lane / 6, fk0 = lane - fc0 * 6;
    const int fc1 = (lane + 32) / 6, fk1 = (lane + 32) - fc1 * 6;
    const double* fsrc0 = fk0 < 3 ? a.E + (size_t)fk0 * g.nodes : a.B + (size_t)(fk0 - 3) * g.nodes;
    const double* fsrc1 = fk1 < 3 ? a.E + (size_t)fk1 * g.nodes : a.B + (size_t)(fk1 - 3) * g.nodes;
    auto load_fields = [&](int ci, int cj, int ck, double& f0, double& f1) {
        {
            int ii = ci + ((fc0 >> 2) & 1); if (ii == g.nx) ii = 0;
            int jj = cj + ((fc0 >> 1) & 1); if (jj == g.ny) jj = 0;
            int kk = ck + (fc0 & 1);        if (kk == g.nz) kk = 0;
            f0 = __ldg(fsrc0 + ((long long)ii * g.ny + jj) * g.nz + kk);
        }
        if (lane < FLD_DOUBLES - 32) {
            int ii = ci + ((fc1 >> 2) & 1); if (ii == g.nx) ii = 0;
            int jj = cj + ((fc1 >> 1) & 1); if (jj == g.ny) jj = 0;
            int kk = ck + (fc1 & 1);        if (kk == g.nz) kk = 0;
            f1 = __ldg(fsrc1 + ((long long)ii * g.ny + jj) * g.nz + kk);
        }
    };

    // cell coordinates of the first cell (one division per warp; then incremented)
    int ck = (int)(c_lo % (uint32_t)g.nz);
    int cj = (int)((c_lo / (uint32_t)g.nz) % (uint32_t)g.ny);
    int ci = (int)(c_lo / ((uint32_t)g.nz * (uint32_t)g.ny));

    // segment registers of lane s < nsp: start_s[c], start_s[c+1], start_s[c+2]
    uint32_t sb = 0, se = 0, sn = 0;
    const uint32_t* my_start = a.sp[lane < nsp ? lane : 0].start;
    if (lane < nsp) {
        sb = __ldg(my_start + c_lo);
        se = __ldg(my_start + c_lo + 1);
        if (c_lo + 1 < c_hi) sn = __ldg(my_start + c_lo + 2);
    }
    double f0 = 0.0, f1 = 0.0;
    load_fields(ci, cj, ck, f0, f1);

    // incoming batch descriptor (warp-uniform) and its particle registers
    unsigned long long lv_acc = 0;
    int in_state = 0;            // 0 none, 1 belongs to the current cell, 2 to the next cell, 3 next cell looked empty
    int in_s = 0, in_nb = 0;
    uint32_t in_p0 = 0;
    ParticleRegs in;
    in.x = in.y = in.z = in.u = in.v = in.w = in.q = 0.0;
    {
        const unsigned ne = __ballot_sync(0xffffffffu, lane < nsp && sb < se);
        if (ne) {
            in_s = __ffs(ne) - 1;
            in_p0 = __shfl_sync(0xffffffffu, sb, in_s);
            in_nb = (int)min(32u, __shfl_sync(0xffffffffu, se, in_s) - in_p0);
            in_state = 1;
            load_batch(a.sp[in_s], in_p0, in_nb, lane, in);
        }
    }

    for (uint32_t c = c_lo; c < c_hi; ++c) {
        // ---- cell prologue: publish this cell's corner fields, prefetch the next cell's ----
        fld[lane] = f0;
        if (lane < FLD_DOUBLES - 32) fld[lane + 32] = f1;
        const bool has_next = c + 1 < c_hi;
        int nk = ck + 1, nj = cj, ni = ci;
        if (nk == g.nz) { nk = 0; nj = cj + 1; if (nj == g.ny) { nj = 0; ni = ci + 1; } }
        if (has_next) load_fields(ni, nj, nk, f0, f1);
        __syncwarp();
        const double dci = (double)ci, dcj = (double)cj, dck = (double)ck;
        const unsigned ne_cur = __ballot_sync(0xffffffffu, lane < nsp && sb < se);

        double accM[27];
#pragma unroll
        for (int m = 0; m < 27; ++m) accM[m] = 0.0;
        double aJ0 = 0.0, aJ1 = 0.0, aJ2 = 0.0, aJ3 = 0.0;
        unsigned my_leavers = 0;

        while (in_state == 1) {
            // ---- take the incoming batch ----
            const int s = in_s, nb = in_nb;
            const uint32_t p0 = in_p0;
            const ParticleRegs cur = in;
            const SpeciesDev& sp = a.sp[s];

            // ---- descriptor of the batch after this one ----
            {
                const uint32_t e = __shfl_sync(0xffffffffu, se, s);
                const unsigned later = ne_cur & ~((2u << s) - 1u);
                if (p0 + 32 < e) {
                    in_p0 = p0 + 32;
                    in_nb = (int)min(32u, e - in_p0);
                } else if (later) {
                    in_s = __ffs(later) - 1;
                    in_p0 = __shfl_sync(0xffffffffu, sb, in_s);
                    in_nb = (int)min(32u, __shfl_sync(0xffffffffu, se, in_s) - in_p0);
                } else {
                    const unsigned ne_next = __ballot_sync(0xffffffffu, has_next && lane < nsp && se < sn);
                    if (ne_next) {
                        in_s = __ffs(ne_next) - 1;
                        in_p0 = __shfl_sync(0xffffffffu, se, in_s);
                        in_nb = (int)min(32u, __shfl_sync(0xffffffffu, sn, in_s) - in_p0);
                        in_state = 2;
                    } else {
                        in_state = has_next ? 3 : 0;   // 3: the next cell is empty, look again there
                    }
                }
            }

            // ---- phase 1: lane = particle ----
            const bool stray = phase1(g, sp, cur, lane < nb, p0 + lane, sp.beta, dt, dci, dcj, dck, fld, strow, my_leavers);
            // global loads of the next batch fly during phase 2
            if (in_state == 1 || in_state == 2) load_batch(a.sp[in_s], in_p0, in_nb, lane, in);
            const unsigned smask = __ballot_sync(0xffffffffu, stray);
            if (smask) {
                uint32_t base = 0;
                if (lane == 0) base = atomicAdd(sp.stray_count, (uint32_t)__popc(smask));
                base = __shfl_sync(0xffffffffu, base, 0);
                if (stray) sp.stray_list[base + __popc(smask & ((1u << lane) - 1u))] = p0 + lane;
            }
            __syncwarp();

            // ---- phase 2: lane = accumulator tile (rows >= nb hold zeros) ----
            if (nb > 30) {
#pragma unroll
                for (int s3 = 0; s3 < 11; ++s3) m_step(bc01, bc2, bal, s3 * 3 * STG_STRIDE, accM);
#pragma unroll
                for (int s4 = 0; s4 < 8; ++s4) j_step(bwq, bvh, s4 * 4 * STG_STRIDE, aJ0, aJ1, aJ2, aJ3);
            } else {
                const int n3 = (nb + 2) / 3, n4 = (nb + 3) / 4;
#pragma unroll 1
                for (int s3 = 0; s3 < n3; ++s3) m_step(bc01, bc2, bal, s3 * 3 * STG_STRIDE, accM);
#pragma unroll 1
                for (int s4 = 0; s4 < n4; ++s4) j_step(bwq, bvh, s4 * 4 * STG_STRIDE, aJ0, aJ1, aJ2, aJ3);
            }
            __syncwarp();

            // ---- end of a species in this cell: rho/Jhat of the species, one store ----
            if (in_state != 1 || in_s != s) {
                aJ0 += shfl_xor_f64(aJ0, 8);  aJ1 += shfl_xor_f64(aJ1, 8);
                aJ2 += shfl_xor_f64(aJ2, 8);  aJ3 += shfl_xor_f64(aJ3, 8);
                aJ0 += shfl_xor_f64(aJ0, 16); aJ1 += shfl_xor_f64(aJ1, 16);
                aJ2 += shfl_xor_f64(aJ2, 16); aJ3 += shfl_xor_f64(aJ3, 16);
                if (lane < 8) {
                    double* dst = sp.AJ + (size_t)c * AJ_PER_CELL + lane * 4;
                    *reinterpret_cast<double2*>(dst) = make_double2(aJ0, aJ1);
                    *reinterpret_cast<double2*>(dst + 2) = make_double2(aJ2, aJ3);
                }
                aJ0 = aJ1 = aJ2 = aJ3 = 0.0;
                my_leavers = __reduce_add_sync(0xffffffffu, my_leavers);
                if (lane == s) lv_acc += my_leavers;     // lane s keeps the warp's count for species s
                my_leavers = 0;
            }
        }

        // species without particles in this cell still own an AJ block: zeros
        {
            unsigned empty = ~ne_cur & ((nsp >= 32) ? 0xffffffffu : ((1u << nsp) - 1u));
            while (empty) {
                const int s = __ffs(empty) - 1;
                empty &= empty - 1;
                if (lane < 8) {
                    double* dst = a.sp[s].AJ + (size_t)c * AJ_PER_CELL + lane * 4;
                    *reinterpret_cast<double2*>(dst) = make_double2(0.0, 0.0);
                    *reinterpret_cast<double2*>(dst + 2) = make_double2(0.0, 0.0);
                }
            }
        }

        // ---- mass-matrix classes of this cell: sum the 3 particle slots through shared memory ----
        if (lane < 27) {
            double* d = stg + pt * FLUSH_SLOT_STRIDE + rg * FLUSH_RG_STRIDE;
#pragma unroll
            for (int m = 0; m < 26; m += 2) *reinterpret_cast<double2*>(d + m) = make_double2(accM[m], accM[m + 1]);
            d[26] = accM[26];
        }
        __syncwarp();
        {
            double* dst = a.AM + (size_t)c * AM_PER_CELL;
#pragma unroll
            for (int r8 = 0; r8 < 8; ++r8) {
                const int t = r8 * 32 + lane;
                if (t < AM_PER_CELL) {
                    const int grp = t / 27, m = t - grp * 27;
                    const double* q0 = stg + grp * FLUSH_RG_STRIDE + m;
                    dst[t] = (q0[0] + q0[FLUSH_SLOT_STRIDE]) + q0[2 * FLUSH_SLOT_STRIDE];
                }
            }
        }
        __syncwarp();
        // the flush overwrote staging rows 0..15; row 32 (the zero row) is beyond 3*252 = 756 < 1600

        // ---- advance to the next cell ----
        if (lane < nsp) {
            sb = se; se = sn;
            if (c + 2 < c_hi) sn = __ldg(my_start + c + 3);
        }
        ci = ni; cj = nj; ck = nk;
        if (in_state == 2) {
            in_state = 1;
        } else if (has_next) {
            // nothing was prefetched for the cell just entered (it looked empty, or the previous cell had
            // no batch to prefetch from): look for its first batch now
            const unsigned ne = __ballot_sync(0xffffffffu, lane < nsp && sb < se);
            in_state = 0;
            if (ne) {
                in_s = __ffs(ne) - 1;
                in_p0 = __shfl_sync(0xffffffffu, sb, in_s);
                in_nb = (int)min(32u, __shfl_sync(0xffffffffu, se, in_s) - in_p0);
                in_state = 1;
                load_batch(a.sp[in_s], in_p0, in_nb, lane, in);
            }
        }
    }
    if (lane < nsp && lv_acc) atomicAdd(a.sp[lane].leavers, lv_acc);
}

// ---------------------------------------------------------------------------------------------
// Expansion of the per-cell classes to the node arrays (HBM-bound: reads AM once, writes M once).
//
// Node N = (i,j,k) is corner a=0 of cell i and corner a=1 of cell i-1 (per axis).  For neighbour
// offset d along an axis the pairs (a, a') with a' - a = d inside one cell are
//     d =  0 : (0,0) in cell i   -> class 0 (w0^2)   and (1,1) in cell i-1 -> class 2 (w1^2)
//     d = +1 : (0,1) in cell i   -> class 1 (w0 w1)
//     d = -1 : (1,0) in cell i-1 -> class 1
// and the 3-D term list is the product of the three per-axis lists (1, 2, 4 or 8 cells).
// One CTA walks EXPAND_Z consecutive nodes of one (i,j) column; thread r < 243 owns element
// (o, ij) = (r/9, r%9) and keeps its x-y term list (<= 4 column offsets) in registers, so the
// per-node work is <= 8 loads, the adds and one coalesced store.
constexpr int EXPAND_Z = 16;

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
    const int dx = o / 9 - 1, dy = (o / 3) % 3 - 1, dz = o % 3 - 1;
    const int zchunks = (g.nz + EXPAND_Z - 1) / EXPAND_Z;
    const int zc = (int)(blockIdx.x % (unsigned)zchunks);
    const int j = (int)((blockIdx.x / (unsigned)zchunks) % (unsigned)g.ny);
    const int i = (int)(blockIdx.x / ((unsigned)zchunks * (unsigned)g.ny));
    const int im1 = i ? i - 1 : g.nx - 1, jm1 = j ? j - 1 : g.ny - 1;

    // per-axis term lists: cell index and class
    int ntx, cix[2], clx[2], nty, cjy[2], cly[2];
    if (dx == 0)     { ntx = 2; cix[0] = i;   clx[0] = 0; cix[1] = im1; clx[1] = 2; }
    else if (dx > 0) { ntx = 1; cix[0] = i;   clx[0] = 1; cix[1] = i;   clx[1] = 1; }
    else             { ntx = 1; cix[0] = im1; clx[0] = 1; cix[1] = im1; clx[1] = 1; }
    if (dy == 0)     { nty = 2; cjy[0] = j;   cly[0] = 0; cjy[1] = jm1; cly[1] = 2; }
    else if (dy > 0) { nty = 1; cjy[0] = j;   cly[0] = 1; cjy[1] = j;   cly[1] = 1; }
    else             { nty = 1; cjy[0] = jm1; cly[0] = 1; cjy[1] = jm1; cly[1] = 1; }
    // up to four x-y terms: offset of (column, class_x, class_y, ij) in AM, in doubles
    const int nxy = ntx * nty;
    size_t col[4];
#pragma unroll
    for (int t = 0; t < 4; ++t) {
        const int tx = min(t / nty, 1), ty = t % nty;   // t = tx * nty + ty for t < nxy
        col[t] = ((size_t)cix[tx] * g.ny + cjy[ty]) * g.nz * AM_PER_CELL + (size_t)((clx[tx] * 9 + cly[ty] * 3) * 9 + ij);
    }
    // z terms: A = own cell k (class 0 for dz = 0, class 1 for dz = +1), B = cell k-1 (class 2 / class 1)
    const bool useA = dz >= 0, useB = dz <= 0;
    const int offA = (dz == 0 ? 0 : 1) * 9, offB = (dz == 0 ? 2 : 1) * 9;

    const int k0 = zc * EXPAND_Z;
    const int k1 = min(k0 + EXPAND_Z, g.nz);
    const size_t node0 = ((size_t)i * g.ny + j) * g.nz;
#pragma unroll 4
    for (int k = k0; k < k1; ++k) {
        const int km1 = k ? k - 1 : g.nz - 1;
        const size_t zA = (size_t)k * AM_PER_CELL + offA, zB = (size_t)km1 * AM_PER_CELL + offB;
        double sum = 0.0;
#pragma unroll
        for (int t = 0; t < 4; ++t) {
            if (t < nxy) {
                if (useA) sum += __ldg(a.AM + col[t] + zA);
                if (useB) sum += __ldg(a.AM + col[t] + zB);
            }
        }
        double* dst = a.M + (node0 + k) * 243 + r;
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
