// fused_mma.cuh -- the gather / push / deposit kernel for cell-ordered particles.
//
// One kernel template, four MODEs and two particle LAYOUTs:
//   MODE_FUSED    deposit (rho, Jhat, M at the pre-push x, v) and push in one pass: E^{n+theta} is an input (north-star)
//   MODE_MOMENTS  deposit only: x, v untouched (the "moment gathering" block of a real ECsim step)
//   MODE_PUSH     push only, Eq. 6-8 with the E^{n+theta} the field solve returned (L86-L96)
//   MODE_DIAG     the diagnostic moments written with the I/O (L121, L147: computeCharge / computeCurrent): charge
//                 density, un-rotated current, pressure tensor, heat flux -- 13 sums per corner, same tile machinery
//   LAYOUT_DENSE  the caller's arrays, cell c = [start[c], start[c+1]), pushed in place; a particle found outside
//                 the cell whose segment it is stored in (a "stray") is skipped here, listed, and handled by
//                 k_push_strays_bulk (atomic_path.cuh)
//   LAYOUT_GAPPED library-managed ("resident") double buffers: cell c owns the slots [seg[c], seg[c+1]) of both
//                 buffers, more than it holds.  In the buffer that is read its particles are a FRONT run of F[c]
//                 and a BACK run of R[c] growing down from the segment's end (the arrivals of the previous push).
//                 A push writes the other buffer: particles that stay go, compacted, to the front of the cell's
//                 segment, a particle that leaves goes straight to the back of its NEW cell's segment (slot from an
//                 atomic counter).  Every step starts cell-sorted: no strays, no re-sort (the sort-preserving push
//                 of SURVEY §8(f)1; the paper's own attempt at "sorting the particles", L149).
//
// Design:
//   * One FP64 pipe bounds this path.  DFMA and DMMA share it (measured: 34.1 / 37.1 / 32-33
//     TFLOP/s alone / alone / mixed), but one `mma.sync.m8n8k4.f64` carries 256 FMAs in one instruction with two
//     operand registers per lane, where 256 DFMA-FMAs as rank-1 updates need ~100 operand doubles from shared memory.
//   * One warp owns a contiguous range of cells, chosen from the segment tables so that every warp of the launch
//     gets the same number of particles (+ a per-cell weight): a particle-balanced schedule that also serves
//     non-uniform loads (Harris sheet).
//   * Per cell, all particles of all species of the call stream through the warp in batches of 32.
//   * Phase 1, lane = particle, branch-free: CIC weights (L49, L131), gather of E^{n+theta}, B^n from the cell's 8
//     corner nodes staged in shared memory (L88, L133), alpha_p as nine scalars (Eq. 2), push (Eq. 6-8,
//     L88-L96), and the per-particle factors of the deposits, written TRANSPOSED ([value][particle]) to a per-warp
//     staging tile in shared memory:
//         c[27]  = q beta/V * px[kx] py[ky] pz[kz],   p?[0..2] = (w0^2, w0 w1, w1^2)
//         Wq[8]  = q/V * W[corner];   alpha[9];   1;   vhat[3] = alpha v^n
//     Only 27 distinct products W_pN W_pN' exist per particle (three per axis), so the 8x8 = 64 (node, neighbour)
//     pairs of Eq. (3) collapse onto 27 "classes" per cell.  Lanes without a particle of the cell (ragged tail,
//     strays) run the same code with q = 0: zero columns.
//   * Phase 2, the pre-reduction of same-cell particles (north-star (b)) as tall-skinny contractions over the
//     particle index, four particles per step:
//         accM[mt] (4 DMMA)  += c[8 mt + r]  x  alpha[0..7]       32 padded classes x 8
//         acc8[mt] (4 DFMA)  += c[8 mt + r]  *  alpha[8]          on the A fragment already in registers
//         accJ     (1 DMMA)  += Wq[8 corners] x (.., 1, vhat)     rho and Jhat per corner (Eq. 1)
//     Lane (r = lane/4, k = lane%4) reads row X + r, particle 4g + k: conflict-free LDS.64.
//   * End of a species in a cell: accJ goes straight from the fragment to AJ[species][cell][8][4].
//     End of a cell: accM / acc8 go straight from the fragments, 16-byte coalesced, to AM[cell][244].
//     No atomics; the result is deterministic for a given particle order.
//   * k_expand_* (expand.cuh, expand_tma.cuh) then build the node arrays.
#pragma once
#include "common.cuh"

constexpr int MODE_FUSED = 0, MODE_MOMENTS = 1, MODE_PUSH = 2, MODE_DIAG = 3;
constexpr int LAYOUT_DENSE = 0, LAYOUT_GAPPED = 1;

constexpr int ST_PITCH = 36;     // doubles per staging row: 32 particles + 4 (pitch = 4 mod 16: LDS.64 conflict-free)
constexpr int ROW_C = 0;         // rows 0..26: the 27 classes, class = kx*9 + ky*3 + kz
constexpr int ROW_WQ = 27;       // rows 27..34: q/V * W[8], corner = a*4 + b*2 + c (also the junk rows 27..31 of A tile 3)
constexpr int ROW_BA = 35;       // rows 35..42: alpha[0..7]
constexpr int ROW_A8 = 43;       // row 43: alpha[8]
constexpr int ROW_ONE = 44;      // row 44: 1 (constant);  rows 45..47: alpha v^n
constexpr int ROW_VH = 45;
constexpr int ROW_BJ = 40;       // B tile of the rho/Jhat contraction: rows 40..47, useful columns 4..7 = (1, vhat)
constexpr int ST_ROWS = 48;
constexpr int FLD_DOUBLES = 48;  // 8 corners x (Ex,Ey,Ez,Bx,By,Bz)
constexpr int WARP_SMEM_DOUBLES = ST_ROWS * ST_PITCH + FLD_DOUBLES;
constexpr int AM_PER_CELL = 244; // [27 classes][8 alpha entries] + [27 classes] alpha[8] + 1 pad: 1952 B, a 16-byte multiple
constexpr int AM_A8 = 216;
constexpr int AJ_PER_CELL = 32;
constexpr int AD_PER_CELL = 128; // MODE_DIAG: [8 corners][16]: rho, J[3], P[6] (xx,xy,xz,yy,yz,zz), Q[3], 3 pad
constexpr int ROW_D = 0;         // MODE_DIAG: rows 0..15 = the 16 columns (1, v, v v^T, |v|^2/2 v, 0, 0, 0) of the two B tiles
constexpr unsigned CELL_WEIGHT = 8;   // schedule weight of a cell, in particles
constexpr int LQ_CAP = 64;            // GAPPED push: leavers waiting in a warp's shared-memory queue (flushed 32 at a time)
constexpr int LQ_DOUBLES = 8 * LQ_CAP;   // [x,y,z,u,v,w,q,species][LQ_CAP]
// shared memory of one warp of k_fused_push_moments<.., MODE, LAYOUT>, in doubles
__host__ __device__ constexpr int fused_warp_doubles(int mode, int layout)
{
    return (mode == MODE_PUSH ? FLD_DOUBLES : WARP_SMEM_DOUBLES) +
           ((layout == LAYOUT_GAPPED && (mode == MODE_FUSED || mode == MODE_PUSH)) ? LQ_DOUBLES : 0);
}

struct SpeciesDev {
    const uint32_t* seg;     // [cells+1]: DENSE start table; GAPPED first slot of every cell's segment
    const uint32_t* Fin;     // GAPPED: [cells] front run of the buffer read
    const uint32_t* Rin;     // GAPPED: [cells] back run of the buffer read (arrivals of the previous push)
    uint32_t* Fout;          // GAPPED push: [cells] front run of the buffer written (stored by the cell's warp)
    uint32_t* Rout;          // GAPPED push: [cells] arrival counters of the buffer written (zeroed before the launch)
    double *x, *y, *z, *u, *v, *w;      // arrays read (DENSE: pushed in place)
    const double* q;
    double *ox, *oy, *oz, *ou, *ov, *ow, *oq;   // GAPPED push: arrays written
    double* ovf;             // GAPPED push: [7][ovf_cap] particles that found their new cell's segment full
    uint32_t ovf_cap;
    uint32_t* ovf_count;
    double beta;             // q dt/(2m) (L55)
    uint32_t n;              // particles of the species
    double* AJ;              // [cells][8][4]: rho, Jx, Jy, Jz per corner  (MODE_DIAG: [cells][8][16])
    uint32_t* stray_list;    // DENSE
    uint32_t* stray_count;
    unsigned long long* leavers;
};

struct FusedArgs {
    Geom g;
    int n_species;
    const double *E, *B;
    double dt;
    double* AM;                      // [cells][AM_PER_CELL]
    uint32_t c_begin, c_end;         // cells [c_begin, c_end) of this launch
    SpeciesDev sp[ECSIM_MAX_SPECIES];
};

__device__ __forceinline__ bool in_unit_interval(double t)
{
    // t in [+0, 1): sign clear and exponent below that of 1.0 (NaN and negatives fail)
    return (unsigned)__double2hiint(t) < 0x3FF00000u;
}

// D(8x8) += A(8x4) * B(4x8) in FP64.  Lane l holds A[l/4][l%4], B[l%4][l/4], D[l/4][2(l%4) + {0,1}].
__device__ __forceinline__ void dmma_m8n8k4(double2& d, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(d.x), "+d"(d.y) : "d"(a), "d"(b));
}

// 1/d for finite d >= 1 (D = 1 + |b|^2 of Eq. 2): hardware seed (~20 bits) and two Newton steps; no
// subnormal / infinity / zero path is needed for this range.  Error <= 1 ulp.
__device__ __forceinline__ double rcp_ge1(double d)
{
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(d));
    double e = fma(-d, r, 1.0);
    r = fma(r, e, r);
    e = fma(-d, r, 1.0);
    return fma(r, e, r);
}

// Schedule weight of the cells [0, c): CELL_WEIGHT per cell + its particles (DENSE) or slots (GAPPED) of every species.
__device__ __forceinline__ unsigned long long cells_weight(const FusedArgs& a, uint32_t c)
{
    unsigned long long f = (unsigned long long)CELL_WEIGHT * c;
    for (int s = 0; s < a.n_species; ++s) f += __ldg(a.sp[s].seg + c);
    return f;
}

// First cell of warp w's range: smallest c in [c_begin, c_end] whose weight from c_begin reaches w/W of the launch's.
__device__ __forceinline__ uint32_t range_bound(const FusedArgs& a, uint32_t w, uint32_t W, unsigned long long w0,
                                                unsigned long long total)
{
    if (w == 0) return a.c_begin;
    if (w >= W) return a.c_end;
    const unsigned long long target = w0 + total / W * w + (total % W) * w / W;
    uint32_t lo = a.c_begin, hi = a.c_end;
    while (lo < hi) {
        const uint32_t mid = lo + (hi - lo) / 2;
        if (cells_weight(a, mid) >= target) hi = mid; else lo = mid + 1;
    }
    return lo;
}

struct ParticleRegs { double x, y, z, u, v, w, q; };
struct PushedRegs { double x, y, z, u, v, w; bool stays; };

__device__ __forceinline__ void load_batch(const SpeciesDev& sp, uint32_t p, bool active, ParticleRegs& r)
{
    if (active) {
        r.x = sp.x[p]; r.y = sp.y[p]; r.z = sp.z[p];
        r.u = sp.u[p]; r.v = sp.v[p]; r.w = sp.w[p];
        r.q = __ldg(sp.q + p);
    }
}

// Phase 1 for one lane.  `st` = staging tile + lane (the lane's column), `fld` = the cell's corner fields,
// (dci,dcj,dck) = the cell's integer coordinates.  Returns `inside`: the lane holds a particle of this cell
// (DENSE: tested; GAPPED: every stored particle is, by construction of the layout).
template <int MODE, int LAYOUT>
__device__ __forceinline__ bool phase1(const Geom& g, const ParticleRegs& r, bool active, double beta, double dt,
                                       double dci, double dcj, double dck, const double* __restrict__ fld,
                                       double* __restrict__ st, PushedRegs& out)
{
    // weights relative to the warp's cell; outside [0,1) => not in this cell
    const double xi = r.x * g.rdx - dci, eta = r.y * g.rdy - dcj, zeta = r.z * g.rdz - dck;
    const bool inside = LAYOUT == LAYOUT_GAPPED
                            ? active
                            : (active && in_unit_interval(xi) && in_unit_interval(eta) && in_unit_interval(zeta));
    // Lanes without a particle of this cell (ragged tail, strays) run the same code on whatever finite
    // particle their registers hold, with zero charge: their class weights and corner weights are exact zeros.
    const double vx = r.u, vy = r.v, vz = r.w;
    const double q = inside ? r.q : 0.0;
    const double wx0 = 1.0 - xi, wy0 = 1.0 - eta, wz0 = 1.0 - zeta;
    double Ex = 0, Ey = 0, Ez = 0, Bx = 0, By = 0, Bz = 0;
    double W[8];
    {
        const double w00 = wx0 * wy0, w01 = wx0 * eta, w10 = xi * wy0, w11 = xi * eta;
        W[0] = w00 * wz0; W[1] = w00 * zeta; W[2] = w01 * wz0; W[3] = w01 * zeta;
        W[4] = w10 * wz0; W[5] = w10 * zeta; W[6] = w11 * wz0; W[7] = w11 * zeta;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const double2 f1 = *reinterpret_cast<const double2*>(fld + k * 6 + 2);
            const double2 f2 = *reinterpret_cast<const double2*>(fld + k * 6 + 4);
            if (MODE != MODE_MOMENTS) {
                const double2 f0 = *reinterpret_cast<const double2*>(fld + k * 6);
                Ex = fma(W[k], f0.x, Ex); Ey = fma(W[k], f0.y, Ey); Ez = fma(W[k], f1.x, Ez);
            }
            Bx = fma(W[k], f1.y, Bx); By = fma(W[k], f2.x, By); Bz = fma(W[k], f2.y, Bz);
        }
    }
    // alpha_p, Eq. (2): (I x B) v = B x v, b = beta B_p;  alpha = (I + [b]x)^-1
    const double bx = beta * Bx, by = beta * By, bz = beta * Bz;
    const double invD = rcp_ge1(1.0 + (bx * bx + by * by + bz * bz));
    const double sx = invD * bx, sy = invD * by, sz = invD * bz;
    const double a00 = fma(bx, sx, invD), a01 = fma(bx, sy, sz), a02 = fma(bx, sz, -sy);
    const double a10 = fma(by, sx, -sz), a11 = fma(by, sy, invD), a12 = fma(by, sz, sx);
    const double a20 = fma(bz, sx, sy), a21 = fma(bz, sy, -sx), a22 = fma(bz, sz, invD);
    if (MODE != MODE_PUSH) {
        // deposit factors (pre-push x and v, L49): operands of the contractions, one column per particle
        {
            double* sb = st + ROW_BA * ST_PITCH;
            sb[0 * ST_PITCH] = a00; sb[1 * ST_PITCH] = a01; sb[2 * ST_PITCH] = a02;
            sb[3 * ST_PITCH] = a10; sb[4 * ST_PITCH] = a11; sb[5 * ST_PITCH] = a12;
            sb[6 * ST_PITCH] = a20; sb[7 * ST_PITCH] = a21; sb[8 * ST_PITCH] = a22;
            double* sv = st + ROW_VH * ST_PITCH;
            sv[0 * ST_PITCH] = a00 * vx + a01 * vy + a02 * vz;
            sv[1 * ST_PITCH] = a10 * vx + a11 * vy + a12 * vz;
            sv[2 * ST_PITCH] = a20 * vx + a21 * vy + a22 * vz;
        }
        {
            const double qV = q * g.invV;
            double* sw = st + ROW_WQ * ST_PITCH;
#pragma unroll
            for (int k = 0; k < 8; ++k) sw[k * ST_PITCH] = qV * W[k];
            // 27 classes: q beta/V * px[kx] * py[ky] * pz[kz]  (beta rides on the class weights, alpha stays unscaled)
            const double qbV = qV * beta;
            const double qx0 = qbV * wx0, qx1 = qbV * xi;
            const double px[3] = {qx0 * wx0, qx0 * xi, qx1 * xi};
            const double py[3] = {wy0 * wy0, wy0 * eta, eta * eta};
            const double pz0 = wz0 * wz0, pz1 = wz0 * zeta, pz2 = zeta * zeta;
#pragma unroll
            for (int kx = 0; kx < 3; ++kx)
#pragma unroll
                for (int ky = 0; ky < 3; ++ky) {
                    const double pxy = px[kx] * py[ky];
                    double* sc = st + (ROW_C + (kx * 3 + ky) * 3) * ST_PITCH;
                    sc[0] = pxy * pz0; sc[ST_PITCH] = pxy * pz1; sc[2 * ST_PITCH] = pxy * pz2;
                }
        }
    }
    if (MODE != MODE_MOMENTS) {
        // mover, Eq. (6)-(8)
        const double tx = fma(beta, Ex, vx), ty = fma(beta, Ey, vy), tz = fma(beta, Ez, vz);
        const double vbx = a00 * tx + a01 * ty + a02 * tz;
        const double vby = a10 * tx + a11 * ty + a12 * tz;
        const double vbz = a20 * tx + a21 * ty + a22 * tz;
        out.u = 2.0 * vbx - vx; out.v = 2.0 * vby - vy; out.w = 2.0 * vbz - vz;
        double xn = fma(dt, out.u, r.x), yn = fma(dt, out.v, r.y), zn = fma(dt, out.w, r.z);
        pin_axes(g, xn, yn, zn);        // reduced dimensionality (L123 fixPosition); a warp-uniform no-op in 3-D
        // for x >= +0 the order of doubles is the order of their bit patterns: "0 <= x < L" is one unsigned compare
        const bool in_box = (unsigned long long)__double_as_longlong(xn) < (unsigned long long)__double_as_longlong(g.Lx) &&
                            (unsigned long long)__double_as_longlong(yn) < (unsigned long long)__double_as_longlong(g.Ly) &&
                            (unsigned long long)__double_as_longlong(zn) < (unsigned long long)__double_as_longlong(g.Lz);
        if (inside && !in_box) { xn = wrap_periodic(xn, g.Lx); yn = wrap_periodic(yn, g.Ly); zn = wrap_periodic(zn, g.Lz); }
        out.x = xn; out.y = yn; out.z = zn;
        out.stays = in_unit_interval(xn * g.rdx - dci) && in_unit_interval(yn * g.rdy - dcj) &&
                    in_unit_interval(zn * g.rdz - dck);
    }
    return inside;
}

// Phase 1 of MODE_DIAG for one lane (L147; readings R22-R24 of DESIGN.md): corner weights q/V W[8] (the A tile) and the
// 13 per-particle factors 1, v, v v^T (xx,xy,xz,yy,yz,zz), |v|^2/2 v (two B tiles; rows 13..15 stay zero).
template <int LAYOUT>
__device__ __forceinline__ bool phase1_diag(const Geom& g, const ParticleRegs& r, bool active, double dci, double dcj,
                                            double dck, double* __restrict__ st)
{
    const double xi = r.x * g.rdx - dci, eta = r.y * g.rdy - dcj, zeta = r.z * g.rdz - dck;
    const bool inside = LAYOUT == LAYOUT_GAPPED
                            ? active
                            : (active && in_unit_interval(xi) && in_unit_interval(eta) && in_unit_interval(zeta));
    const double qV = (inside ? r.q : 0.0) * g.invV;
    const double wx0 = 1.0 - xi, wy0 = 1.0 - eta, wz0 = 1.0 - zeta;
    const double w00 = wx0 * wy0, w01 = wx0 * eta, w10 = xi * wy0, w11 = xi * eta;
    double* sw = st + ROW_WQ * ST_PITCH;
    sw[0 * ST_PITCH] = qV * (w00 * wz0); sw[1 * ST_PITCH] = qV * (w00 * zeta);
    sw[2 * ST_PITCH] = qV * (w01 * wz0); sw[3 * ST_PITCH] = qV * (w01 * zeta);
    sw[4 * ST_PITCH] = qV * (w10 * wz0); sw[5 * ST_PITCH] = qV * (w10 * zeta);
    sw[6 * ST_PITCH] = qV * (w11 * wz0); sw[7 * ST_PITCH] = qV * (w11 * zeta);
    const double vx = r.u, vy = r.v, vz = r.w;
    const double h = 0.5 * ((vx * vx + vy * vy) + vz * vz);
    double* sd = st + ROW_D * ST_PITCH;
    sd[0 * ST_PITCH] = 1.0;
    sd[1 * ST_PITCH] = vx; sd[2 * ST_PITCH] = vy; sd[3 * ST_PITCH] = vz;
    sd[4 * ST_PITCH] = vx * vx; sd[5 * ST_PITCH] = vx * vy; sd[6 * ST_PITCH] = vx * vz;
    sd[7 * ST_PITCH] = vy * vy; sd[8 * ST_PITCH] = vy * vz; sd[9 * ST_PITCH] = vz * vz;
    sd[10 * ST_PITCH] = h * vx; sd[11 * ST_PITCH] = h * vy; sd[12 * ST_PITCH] = h * vz;
    return inside;
}

// Cell coordinate of a pushed position along one axis, consistent with the weights phase 1 will form there next step
// (xi = fma(x, rd, -i) must land in [0, 1)): floor of the rounded product, corrected by one where the rounding of the
// product and the single rounding of the fused form disagree.
__device__ __forceinline__ int dest_coord(double x, double rd, int n)
{
    int i = min(max(__double2int_rd(x * rd), 0), n - 1);
    const double t = fma(x, rd, -(double)i);
    if (t < 0.0 && i > 0) --i;
    else if (t >= 1.0 && i < n - 1) ++i;
    return i;
}

// GAPPED push: a particle that leaves its cell goes to the back run of its new cell's segment in the buffer being
// written.  The slot comes from the cell's arrival counter; the segment has room for it if the slots the cell may still
// need for its own particles (all it holds now) plus the arrivals so far stay inside the segment -- a bound that needs
// no coordination with the warp that owns the cell.  Otherwise the particle goes to the species' overflow list and the
// next call lays the species out afresh.
struct Relocation { uint32_t d, a, room, s1; };

// first half: the new cell and a ticket from its arrival counter.  (Requesting the ticket before phase 2 and using it
// after -- to hide the atomic's latency -- was measured: no gain, 0.2-0.5 ms slower per step at configs[2]; the 14 extra
// live registers cost more than the few stalled warps.)
__device__ __forceinline__ Relocation relocate_begin(const Geom& g, const SpeciesDev& sp, const PushedRegs& o)
{
    const int di = dest_coord(o.x, g.rdx, g.nx), dj = dest_coord(o.y, g.rdy, g.ny), dk = dest_coord(o.z, g.rdz, g.nz);
    Relocation r;
    r.d = (uint32_t)((di * g.ny + dj) * g.nz + dk);
    const uint32_t s0 = __ldg(sp.seg + r.d);
    r.s1 = __ldg(sp.seg + r.d + 1);
    const uint32_t held = __ldg(sp.Fin + r.d) + __ldg(sp.Rin + r.d);
    r.room = r.s1 - s0 > held ? r.s1 - s0 - held : 0u;
    r.a = atomicAdd(sp.Rout + r.d, 1u);
    return r;
}

// second half: the slot, or the overflow list
__device__ __forceinline__ void relocate_end(const SpeciesDev& sp, const Relocation& r, const PushedRegs& o, double q)
{
    if (r.a < r.room) {
        const uint32_t pos = r.s1 - 1u - r.a;
        sp.ox[pos] = o.x; sp.oy[pos] = o.y; sp.oz[pos] = o.z;
        sp.ou[pos] = o.u; sp.ov[pos] = o.v; sp.ow[pos] = o.w; sp.oq[pos] = q;
    } else {
        atomicSub(sp.Rout + r.d, 1u);        // slots >= the bound are never handed out: the counter ends at min(arrivals, room)
        const uint32_t k = atomicAdd(sp.ovf_count, 1u);
        if (k < sp.ovf_cap) {
            double* v = sp.ovf + k;
            const size_t m = sp.ovf_cap;
            v[0] = o.x; v[m] = o.y; v[2 * m] = o.z; v[3 * m] = o.u; v[4 * m] = o.v; v[5 * m] = o.w; v[6 * m] = q;
        }
    }
}

__device__ __forceinline__ void relocate(const Geom& g, const SpeciesDev& sp, const PushedRegs& o, double q)
{
    const Relocation r = relocate_begin(g, sp, o);
    relocate_end(sp, r, o, q);
}

// REGS: register cap.  Measured on config 2 (whole grid, ms): 12 warps x 168 regs 11.89, 12 x 144 12.23, 16 x 128
// 12.15, 12 x 128 12.88, 8 x 200 13.63; warp counts that are not a multiple of the 4 schedulers lose (14 x 128 13.58).
template <int NW, int REGS, int MODE, int LAYOUT>
__global__ void __maxnreg__(REGS)
k_fused_push_moments(const __grid_constant__ FusedArgs a)
{
    extern __shared__ __align__(16) double smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    constexpr bool DIAG = MODE == MODE_DIAG;
    constexpr bool DEPOSIT = MODE == MODE_FUSED || MODE == MODE_MOMENTS, PUSH = MODE == MODE_FUSED || MODE == MODE_PUSH;
    constexpr bool GAPPED = LAYOUT == LAYOUT_GAPPED, TILE = DEPOSIT || DIAG;
    constexpr int WSM = fused_warp_doubles(MODE, LAYOUT);
    constexpr bool QUEUE = GAPPED && PUSH;

    double* stg = smem + (size_t)warp * WSM;
    double* fld = TILE ? stg + ST_ROWS * ST_PITCH : stg;
    if (TILE) {
        for (int t = lane; t < WARP_SMEM_DOUBLES; t += 32) stg[t] = 0.0;
        __syncwarp();
        if (DEPOSIT)
            for (int t = lane; t < ST_PITCH; t += 32) stg[ROW_ONE * ST_PITCH + t] = 1.0;   // the rho column of the rho/Jhat B tile
        __syncwarp();
    }

    const Geom& g = a.g;
    const int nsp = a.n_species;
    const double dt = a.dt;
    const uint32_t W = gridDim.x * NW, wid = blockIdx.x * NW + warp;
    const unsigned long long w0 = cells_weight(a, a.c_begin), wtot = cells_weight(a, a.c_end) - w0;
    const uint32_t c_lo = range_bound(a, wid, W, w0, wtot), c_hi = range_bound(a, wid + 1, W, w0, wtot);
    if (c_lo >= c_hi) return;

    // lane roles of phase 2: row r of the A / B tiles, particle k of a group of four
    const int fr = lane >> 2, fk = lane & 3;
    const double* frag = stg + fr * ST_PITCH + fk;
    double* stcol = stg + lane;
    const unsigned lt_mask = (1u << lane) - 1u;

    // GAPPED push: particles that leave their cell wait in a per-warp queue and are placed 32 at a time -- the four table
    // reads, the arrival ticket and the seven scattered stores of a relocation are two dependent L2 round trips, paid once
    // per 32 leavers instead of once per batch that holds one (31 % of the batches at 1.2 % leavers, 70 % at 3.7 %)
    double* lq = stg + (TILE ? WARP_SMEM_DOUBLES : FLD_DOUBLES);
    uint32_t qn = 0;
    auto flush_leavers = [&](uint32_t first, uint32_t count) {
        const bool mine = (uint32_t)lane < count;
        const uint32_t e = first + (uint32_t)lane;
        PushedRegs o;
        double q = 0.0;
        int sidx = -1;
        if (mine) {
            o.x = lq[e]; o.y = lq[LQ_CAP + e]; o.z = lq[2 * LQ_CAP + e];
            o.u = lq[3 * LQ_CAP + e]; o.v = lq[4 * LQ_CAP + e]; o.w = lq[5 * LQ_CAP + e];
            q = lq[6 * LQ_CAP + e];
            sidx = (int)lq[7 * LQ_CAP + e];
        }
        o.stays = false;
        for (int t = 0; t < nsp; ++t)
            if (mine && sidx == t) relocate(g, a.sp[t], o, q);
        __syncwarp();
    };

    // field staging: lane t and t+32 (< 48) hold corner t/6, component t%6 of the next cell
    const int fc0 = lane / 6, fk0 = lane - fc0 * 6;
    const int fc1 = (lane + 32) / 6, fk1 = (lane + 32) - fc1 * 6;
    const double* fsrc0 = fk0 < 3 ? a.E + (size_t)fk0 * g.nodes : a.B + (size_t)(fk0 - 3) * g.nodes;
    const double* fsrc1 = fk1 < 3 ? a.E + (size_t)fk1 * g.nodes : a.B + (size_t)(fk1 - 3) * g.nodes;
    auto load_fields = [&](int ci, int cj, int ck, double& f0, double& f1) {
        if (DIAG) return;                            // the diagnostics gather no field
        if (MODE != MODE_MOMENTS || fk0 >= 3) {      // moments need B only (E may be absent)
            int ii = ci + ((fc0 >> 2) & 1); if (ii == g.nx) ii = 0;
            int jj = cj + ((fc0 >> 1) & 1); if (jj == g.ny) jj = 0;
            int kk = ck + (fc0 & 1);        if (kk == g.nz) kk = 0;
            f0 = __ldg(fsrc0 + ((long long)ii * g.ny + jj) * g.nz + kk);
        }
        if (lane < FLD_DOUBLES - 32 && (MODE != MODE_MOMENTS || fk1 >= 3)) {
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

    // segment registers of lane s < nsp.  g0, g1, g2 = seg[c], seg[c+1], seg[c+2]; (f0, t0) / (f1, t1) = front run and
    // total particles of cells c / c+1 (DENSE: the whole segment is the front run)
    uint32_t g0 = 0, g1 = 0, g2 = 0, nf0 = 0, nt0 = 0, nf1 = 0, nt1 = 0;
    const SpeciesDev& mysp = a.sp[lane < nsp ? lane : 0];
    auto load_counts = [&](uint32_t c, uint32_t lo, uint32_t hi, uint32_t& nf, uint32_t& nt) {
        if (GAPPED) { nf = __ldg(mysp.Fin + c); nt = nf + __ldg(mysp.Rin + c); }
        else { nf = nt = hi - lo; }
    };
    if (lane < nsp) {
        g0 = __ldg(mysp.seg + c_lo);
        g1 = __ldg(mysp.seg + c_lo + 1);
        load_counts(c_lo, g0, g1, nf0, nt0);
        if (c_lo + 1 < c_hi) {
            g2 = __ldg(mysp.seg + c_lo + 2);
            load_counts(c_lo + 1, g1, g2, nf1, nt1);
        }
    }
    // corner fields of the NEXT cell are requested while the last batch of a cell is in phase 2, so that
    // their registers are not live across a phase 1 (fld_ready: warp-uniform)
    double f0 = 0.0, f1 = 0.0;
    bool fld_ready = false;

    // incoming batch descriptor (warp-uniform) and its particle registers.  A batch = up to 32 consecutive particles of
    // one species' run in a cell, counted in "virtual" order: front run first, then the back run downwards from the end
    // of the segment.
    unsigned long long lv_acc = 0;
    int in_state = 0;            // 0 none, 1 belongs to the current cell, 2 to the next cell, 3 next cell looked empty
    int in_s = 0, in_nb = 0;
    uint32_t in_v0 = 0, in_base = 0, in_end = 0, in_nf = 0, in_p = 0;
    ParticleRegs in;
    in.x = in.y = in.z = in.u = in.v = in.w = in.q = 0.0;
    auto describe = [&](int s, bool next_cell) {       // first batch of species s in the current / next cell
        in_s = s;
        in_v0 = 0;
        in_base = __shfl_sync(0xffffffffu, next_cell ? g1 : g0, s);
        const uint32_t nt = __shfl_sync(0xffffffffu, next_cell ? nt1 : nt0, s);
        in_nb = (int)min(32u, nt);
        if (GAPPED) {
            in_end = __shfl_sync(0xffffffffu, next_cell ? g2 : g1, s);
            in_nf = __shfl_sync(0xffffffffu, next_cell ? nf1 : nf0, s);
        }
    };
    auto fetch = [&]() {                               // address of this lane's particle of the incoming batch; load it
        const uint32_t v = in_v0 + (uint32_t)lane;
        in_p = (GAPPED && v >= in_nf) ? in_end - 1u - (v - in_nf) : in_base + v;
        load_batch(a.sp[in_s], in_p, lane < in_nb, in);
    };
    {
        const unsigned ne = __ballot_sync(0xffffffffu, lane < nsp && nt0 > 0);
        if (ne) {
            describe(__ffs(ne) - 1, false);
            in_state = 1;
            fetch();
        }
    }

    // accumulators (lane = row fr of a tile, particle fk of a group of four):
    //   accM[mt]  C tile of sum_p c[8 mt + fr] * beta alpha[2 fk + {0,1}]            (DMMA)
    //   acc8[mt]  this lane's share (particles = fk mod 4) of sum_p c[8 mt + fr] * beta alpha[8]   (DFMA on the A fragment)
    //   accJ      C tile of sum_p q/V W[fr] * (.., .., .., .., 1, vhat): fk = 2 holds (rho, Jx), fk = 3 (Jy, Jz)
    //   MODE_DIAG: accJ / accD = C tiles of sum_p q/V W[fr] * (columns 0..7 / 8..15 of ROW_D)
    double2 accM[4], accJ = make_double2(0.0, 0.0), accD = make_double2(0.0, 0.0);
    double acc8[4];
#pragma unroll
    for (int mt = 0; mt < 4; ++mt) { accM[mt] = make_double2(0.0, 0.0); acc8[mt] = 0.0; }

    for (uint32_t c = c_lo; c < c_hi; ++c) {
        // ---- cell prologue: publish this cell's corner fields ----
        if (!fld_ready) load_fields(ci, cj, ck, f0, f1);     // first cell of the range, or after an empty cell
        fld[lane] = f0;
        if (lane < FLD_DOUBLES - 32) fld[lane + 32] = f1;
        fld_ready = false;
        const bool has_next = c + 1 < c_hi;
        int nk = ck + 1, nj = cj, ni = ci;
        if (nk == g.nz) { nk = 0; nj = cj + 1; if (nj == g.ny) { nj = 0; ni = ci + 1; } }
        __syncwarp();
        const double dci = (double)ci, dcj = (double)cj, dck = (double)ck;
        const unsigned ne_cur = __ballot_sync(0xffffffffu, lane < nsp && nt0 > 0);
        unsigned my_leavers = 0;
        uint32_t nstay = 0;          // GAPPED push: particles of the current species written to the front run so far

        while (in_state == 1) {
            // ---- take the incoming batch ----
            const int s = in_s, nb = in_nb;
            const uint32_t p = in_p, cell_base = in_base;
            const ParticleRegs cur = in;
            const SpeciesDev& sp = a.sp[s];

            // ---- descriptor of the batch after this one ----
            {
                const uint32_t e = __shfl_sync(0xffffffffu, nt0, s);
                const unsigned later = ne_cur & ~((2u << s) - 1u);
                if (in_v0 + 32 < e) {
                    in_v0 += 32;
                    in_nb = (int)min(32u, e - in_v0);
                } else if (later) {
                    describe(__ffs(later) - 1, false);
                } else {
                    const unsigned ne_next = __ballot_sync(0xffffffffu, has_next && lane < nsp && nt1 > 0);
                    if (ne_next) {
                        describe(__ffs(ne_next) - 1, true);
                        in_state = 2;
                    } else {
                        in_state = has_next ? 3 : 0;   // 3: the next cell is empty, look again there
                    }
                }
            }

            // push only: there is no phase 2 for the next batch's loads to fly under, and registers to spare, so they are
            // requested before phase 1 (config 2, ecsim_push_all: 16 warps x 128 registers 6.0 ms; with the early loads 5.64; 20 x 96
            // with them 5.33 = 5.2 TB/s; 24 x 80 and 32 x 64 spill: 6.2 / 6.5; no gain for the diagnostics)
            constexpr bool EARLY_FETCH = MODE == MODE_PUSH;
            if (EARLY_FETCH && (in_state == 1 || in_state == 2)) fetch();

            // ---- phase 1: lane = particle ----
            PushedRegs o;
            const bool active = lane < nb;
            const bool inside = DIAG ? phase1_diag<LAYOUT>(g, cur, active, dci, dcj, dck, stcol)
                                     : phase1<MODE, LAYOUT>(g, cur, active, sp.beta, dt, dci, dcj, dck, fld, stcol, o);
            if (PUSH) {
                if (GAPPED) {
                    // stayers go, compacted, to the front run of the cell's segment in the other buffer
                    const bool stay = inside && o.stays;
                    const unsigned smask = __ballot_sync(0xffffffffu, stay);
                    if (stay) {
                        const uint32_t d = cell_base + nstay + (uint32_t)__popc(smask & lt_mask);
                        sp.ox[d] = o.x; sp.oy[d] = o.y; sp.oz[d] = o.z;
                        sp.ou[d] = o.u; sp.ov[d] = o.v; sp.ow[d] = o.w; sp.oq[d] = cur.q;
                    }
                    nstay += (uint32_t)__popc(smask);
                    const bool leave = inside && !o.stays;
                    const unsigned lmask = __ballot_sync(0xffffffffu, leave);
                    if (lmask) {
                        if (leave) {
                            const uint32_t e = qn + (uint32_t)__popc(lmask & lt_mask);
                            lq[e] = o.x; lq[LQ_CAP + e] = o.y; lq[2 * LQ_CAP + e] = o.z;
                            lq[3 * LQ_CAP + e] = o.u; lq[4 * LQ_CAP + e] = o.v; lq[5 * LQ_CAP + e] = o.w;
                            lq[6 * LQ_CAP + e] = cur.q; lq[7 * LQ_CAP + e] = (double)s;
                            my_leavers += 1u;
                        }
                        qn += (uint32_t)__popc(lmask);
                        __syncwarp();
                        if (qn >= 32u) { flush_leavers(qn - 32u, 32u); qn -= 32u; }
                    }
                } else if (inside) {
                    sp.u[p] = o.u; sp.v[p] = o.v; sp.w[p] = o.w;
                    sp.x[p] = o.x; sp.y[p] = o.y; sp.z[p] = o.z;
                    my_leavers += o.stays ? 0u : 1u;
                }
            }
            // global loads of the next batch fly during phase 2 (requesting them before phase 1 was measured: 11.90 vs
            // 11.65 ms, the 14 extra live registers cost more than the longer flight time gains)
            if (!EARLY_FETCH && (in_state == 1 || in_state == 2)) fetch();
            if (in_state != 1 && has_next) { load_fields(ni, nj, nk, f0, f1); fld_ready = true; }
            if (!GAPPED) {
                const unsigned smask = __ballot_sync(0xffffffffu, active && !inside);
                if (smask) {
                    uint32_t base = 0;
                    if (lane == 0) base = atomicAdd(sp.stray_count, (uint32_t)__popc(smask));
                    base = __shfl_sync(0xffffffffu, base, 0);
                    if (active && !inside) sp.stray_list[base + __popc(smask & lt_mask)] = p;
                }
            }

            if (DEPOSIT) {
                __syncwarp();
                // ---- phase 2: contractions over the batch, four particles per step (columns >= nb hold c = 0, Wq = 0) ----
                auto group = [&](int gq) {
                    const double* f = frag + gq * 4;
                    const double b0 = f[ROW_BA * ST_PITCH], a8 = f[(ROW_A8 - fr) * ST_PITCH];
                    const double wq = f[ROW_WQ * ST_PITCH], bj = f[ROW_BJ * ST_PITCH];
#pragma unroll
                    for (int mt = 0; mt < 4; ++mt) {
                        const double av = f[(ROW_C + 8 * mt) * ST_PITCH];
                        dmma_m8n8k4(accM[mt], av, b0);
                        acc8[mt] = fma(av, a8, acc8[mt]);
                    }
                    dmma_m8n8k4(accJ, wq, bj);
                };
                // groups in pairs, two pairs per iteration; ng odd: the extra group reads valid columns whose c and Wq
                // are zero.  (Measured: 4 groups per iteration 11.7 ms, 2 groups 11.75, fully unrolled 11.9.)
                const int ng = nb > 28 ? 8 : (nb + 3) >> 2;
#pragma unroll 1
                for (int gq = 0; gq < ng; gq += 4) {
                    group(gq); group(gq + 1);
                    if (gq + 2 < ng) { group(gq + 2); group(gq + 3); }
                }
                __syncwarp();
            }

            if (DIAG) {
                __syncwarp();
                const int ng = nb > 28 ? 8 : (nb + 3) >> 2;
#pragma unroll 2
                for (int gq = 0; gq < ng; ++gq) {
                    const double* f = frag + gq * 4;
                    const double wq = f[ROW_WQ * ST_PITCH];
                    dmma_m8n8k4(accJ, wq, f[ROW_D * ST_PITCH]);
                    dmma_m8n8k4(accD, wq, f[(ROW_D + 8) * ST_PITCH]);
                }
                __syncwarp();
            }

            // ---- end of a species in this cell ----
            if (in_state != 1 || in_s != s) {
                if (DIAG) {
                    double* dst = sp.AJ + (size_t)c * AD_PER_CELL + fr * 16 + 2 * fk;
                    *reinterpret_cast<double2*>(dst) = accJ;
                    *reinterpret_cast<double2*>(dst + 8) = accD;
                    accJ = make_double2(0.0, 0.0);
                    accD = make_double2(0.0, 0.0);
                }
                if (DEPOSIT) {
                    // its rho/Jhat corner sums, straight from the fragment
                    if (fk >= 2) *reinterpret_cast<double2*>(sp.AJ + (size_t)c * AJ_PER_CELL + fr * 4 + 2 * (fk - 2)) = accJ;
                    accJ = make_double2(0.0, 0.0);
                }
                if (PUSH) {
                    if (GAPPED && lane == 0) sp.Fout[c] = nstay;
                    nstay = 0;
                    my_leavers = __reduce_add_sync(0xffffffffu, my_leavers);
                    if (lane == s) lv_acc += my_leavers;     // lane s keeps the warp's count for species s
                    my_leavers = 0;
                }
            }
        }

        // species without particles in this cell still own an AJ block (zeros) and a front run (empty)
        {
            unsigned empty = ~ne_cur & ((nsp >= 32) ? 0xffffffffu : ((1u << nsp) - 1u));
            while (empty) {
                const int s = __ffs(empty) - 1;
                empty &= empty - 1;
                if (DEPOSIT) a.sp[s].AJ[(size_t)c * AJ_PER_CELL + lane] = 0.0;
                if (DIAG) {
                    double* dst = a.sp[s].AJ + (size_t)c * AD_PER_CELL + 4 * lane;
                    *reinterpret_cast<double2*>(dst) = make_double2(0.0, 0.0);
                    *reinterpret_cast<double2*>(dst + 2) = make_double2(0.0, 0.0);
                }
                if (PUSH && GAPPED && lane == 0) a.sp[s].Fout[c] = 0u;
            }
        }

        // ---- mass-matrix classes of this cell: straight from the fragments, 16-byte coalesced stores ----
        if (DEPOSIT) {
            double* dst = a.AM + (size_t)c * AM_PER_CELL;
#pragma unroll
            for (int mt = 0; mt < 4; ++mt) {
                const int cls = 8 * mt + fr;
                double s8 = acc8[mt];
                s8 += shfl_xor_f64(s8, 1);
                s8 += shfl_xor_f64(s8, 2);
                if (cls < 27) {
                    *reinterpret_cast<double2*>(dst + mt * 64 + fr * 8 + 2 * fk) = accM[mt];
                    if (fk == 0) dst[AM_A8 + cls] = s8;
                }
                accM[mt] = make_double2(0.0, 0.0);
                acc8[mt] = 0.0;
            }
        }

        // ---- advance to the next cell ----
        if (lane < nsp) {
            g0 = g1; g1 = g2; nf0 = nf1; nt0 = nt1;
            if (c + 2 < c_hi) {
                g2 = __ldg(mysp.seg + c + 3);
                load_counts(c + 2, g1, g2, nf1, nt1);
            }
        }
        ci = ni; cj = nj; ck = nk;
        if (in_state == 2) {
            in_state = 1;
        } else if (has_next) {
            // nothing was prefetched for the cell just entered (it looked empty, or the previous cell had
            // no batch to prefetch from): look for its first batch now
            const unsigned ne = __ballot_sync(0xffffffffu, lane < nsp && nt0 > 0);
            in_state = 0;
            if (ne) {
                describe(__ffs(ne) - 1, false);
                in_state = 1;
                fetch();
            }
        }
    }
    if (QUEUE && qn) flush_leavers(0u, qn);
    if (PUSH && lane < nsp && lv_acc) atomicAdd(a.sp[lane].leavers, lv_acc);
}
