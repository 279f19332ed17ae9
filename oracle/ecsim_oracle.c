/*
 * ecsim_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, single-threaded, double-precision CPU restatement of the particle hot path of
 * ECsim as the paper defines it (arxiv 2603.16624, PAPER.md):
 *     Eq. (1)  L47   hatted current      J_sN   = (1/V_N) sum_p q_p (alpha_p v_p) W_pN
 *     Eq. (2)  L53   rotation matrix     alpha_p = (I - beta I x B_p + beta^2 B_p B_p) / (1 + (beta B_p)^2)
 *     Eq. (3)  L59   mass matrices       M^{ij}_{NN'} = sum_p (beta_p/V_N) q_p alpha_p^{ij} W_pN' W_pN
 *     Eq. (6,7) L88-L92  velocity        vbar = alpha (v + beta E_p),  v' = 2 vbar - v
 *     Eq. (8)  L96   position            x' = x + dt v'
 * plus the diagnostic charge density rho_N = (1/V_N) sum_p q_p W_pN (L147, computeCharge).
 * Readings of everything the paper leaves open are those of DESIGN.md "Readings" (R1..R21).
 *
 * It follows the paper's computeMoments loop particle by particle, in input order (L131-L141):
 * lower node N- and upper node N+ = N- + 1 per axis, a 2x2x2 weight array, 8-term gathers,
 * nine scalars for alpha, then the deposits.  No blocking, fusion, reordering or threading.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call this file.  It shares no code, header, table or helper with the CUDA path
 * (paper_2603_16624_b200/csrc), and the CUDA path never calls it.
 *
 * Pins (tests/test_oracle_pins.py): alpha (I + [b]x) = I; Lorentz implicit-midpoint residual;
 * B=0 kick and E=0 Cayley rotation closed forms; |v| preserved at E=0; per-particle and global
 * (ECsim) energy identities; charge/current/mass-matrix sums; single particle on a node;
 * mirror symmetry; dense hat-function brute force (oracle/dense.py) on tiny anisotropic grids;
 * exact-rational worked example (tests/golden); translation invariance.
 * Absolute values: the paper prints no numeric example, so no paper-printed value pins them.
 *
 * Build: gcc -O2 -ffp-contract=off -shared -fPIC (oracle/build.py).
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>

/* Layout: node n = (i*ny + j)*nz + k (z fastest, the paper's Nx x Ny x Nz
 * flattening, L127); fields F[c*nodes + n]; J[c*nodes + n]; neighbour slot
 * o = (di+1)*9 + (dj+1)*3 + (dk+1), self = 13; M[((n*27 + o)*3 + i)*3 + j].                    */

static int lower_node(double s, int n)
{
    /* L131: the paper finds the highest node N+ first and N- = N+ - 1; here N- = floor(x/dx). */
    int i = (int)floor(s);
    if (i < 0) i = 0;
    if (i > n - 1) i = n - 1;
    return i;
}

/* cell id of every particle (= node id of its N- corner) and the per-cell histogram */
int ecsim_oracle_cells(int nx, int ny, int nz, double dx, double dy, double dz, int64_t n,
                       const double *x, const double *y, const double *z,
                       int32_t *cell /* [n] */, int32_t *count /* [cells], zeroed here, or NULL */)
{
    const double rdx = 1.0 / dx, rdy = 1.0 / dy, rdz = 1.0 / dz;
    if (count)
        for (int64_t c = 0; c < (int64_t)nx * ny * nz; ++c) count[c] = 0;
    for (int64_t p = 0; p < n; ++p) {
        int i = lower_node(x[p] * rdx, nx);
        int j = lower_node(y[p] * rdy, ny);
        int k = lower_node(z[p] * rdz, nz);
        int32_t c = (int32_t)(((int64_t)i * ny + j) * nz + k);
        cell[p] = c;
        if (count) count[c] += 1;
    }
    return 0;
}

static double wrap(double x, double L)
{
    /* Reading R13: periodic wrap into [0, L); several box lengths allowed; x' == L folds to 0 */
    x -= L * floor(x / L);
    if (x >= L || x < 0.0) x = 0.0;
    return x;
}

/*
 * One push + moment-gathering step for one species, particles in input order.
 *   x..w      in/out: positions and velocities, updated in place (Eq. 6-8)
 *   q         per-particle charge q_p; qom = q_p/m_p of the species, beta_p = qom*dt/2 (L55)
 *   E, B      node fields [3][nodes]: E^{n+theta}, B^n
 *   rho, J, M accumulated into (+=); caller zeroes
 *   *_abs     optional (NULL): sum of |addend| per output scalar, the tolerance normaliser
 *   vbar      optional (NULL): [3][n] vbar_p, for the energy identities
 *   do_push   0: deposit only (x, v untouched)
 */
int ecsim_oracle_step(int nx, int ny, int nz, double dx, double dy, double dz,
                      int64_t n, double qom, double dt,
                      double *x, double *y, double *z, double *u, double *v, double *w,
                      const double *q, const double *E, const double *B,
                      double *rho, double *J, double *M,
                      double *rho_abs, double *J_abs, double *M_abs,
                      double *vbar, int do_push)
{
    const int64_t nodes = (int64_t)nx * ny * nz;
    const double rdx = 1.0 / dx, rdy = 1.0 / dy, rdz = 1.0 / dz;
    const double Lx = nx * dx, Ly = ny * dy, Lz = nz * dz;
    const double invV = 1.0 / (dx * dy * dz);  /* R7: V_N = dx dy dz for every node (periodic) */
    const double beta = qom * dt / 2.0;        /* L55 */

    for (int64_t p = 0; p < n; ++p) {
        /* 1. nodes N-, N+ per axis (L131) */
        const double sx = x[p] * rdx, sy = y[p] * rdy, sz = z[p] * rdz;
        const int i0 = lower_node(sx, nx), j0 = lower_node(sy, ny), k0 = lower_node(sz, nz);
        const int in[2] = {i0, (i0 + 1) % nx};
        const int jn[2] = {j0, (j0 + 1) % ny};
        const int kn[2] = {k0, (k0 + 1) % nz};

        /* 2. linear interpolation weights, 2x2x2 array (L49, L131) */
        const double xi = sx - i0, eta = sy - j0, zeta = sz - k0;
        const double wx[2] = {1.0 - xi, xi}, wy[2] = {1.0 - eta, eta}, wz[2] = {1.0 - zeta, zeta};
        double W[2][2][2];
        int64_t node[2][2][2];
        for (int a = 0; a < 2; ++a)
            for (int b = 0; b < 2; ++b)
                for (int c = 0; c < 2; ++c) {
                    W[a][b][c] = (wx[a] * wy[b]) * wz[c];
                    node[a][b][c] = ((int64_t)in[a] * ny + jn[b]) * nz + kn[c];
                }

        /* 3. gather E^{n+theta} and B^n at the particle (L88, L133), a-major order */
        double Ep[3] = {0, 0, 0}, Bp[3] = {0, 0, 0};
        for (int a = 0; a < 2; ++a)
            for (int b = 0; b < 2; ++b)
                for (int c = 0; c < 2; ++c)
                    for (int d = 0; d < 3; ++d) {
                        Ep[d] += W[a][b][c] * E[d * nodes + node[a][b][c]];
                        Bp[d] += W[a][b][c] * B[d * nodes + node[a][b][c]];
                    }

        /* 4. rotation matrix, Eq. (2), nine scalars (L135).  R1: (I x B) v = B x v, so
         *    alpha = (I + [b]x)^-1 with b = beta B_p;  R4: (beta B)^2 = |b|^2.                 */
        const double bx = beta * Bp[0], by = beta * Bp[1], bz = beta * Bp[2];
        const double invD = 1.0 / (1.0 + (bx * bx + by * by + bz * bz));
        double al[3][3];
        al[0][0] = invD * (1.0 + bx * bx);
        al[0][1] = invD * (bx * by + bz);
        al[0][2] = invD * (bx * bz - by);
        al[1][0] = invD * (bx * by - bz);
        al[1][1] = invD * (1.0 + by * by);
        al[1][2] = invD * (by * bz + bx);
        al[2][0] = invD * (bx * bz + by);
        al[2][1] = invD * (by * bz - bx);
        al[2][2] = invD * (1.0 + bz * bz);

        /* 5. deposits with the pre-push position and velocity (L49 "both evaluated at time n") */
        const double vn[3] = {u[p], v[p], w[p]};
        double vhat[3];
        for (int r = 0; r < 3; ++r)
            vhat[r] = al[r][0] * vn[0] + al[r][1] * vn[1] + al[r][2] * vn[2];
        const double qV = q[p] * invV;
        const double qbV = qV * beta;
        for (int a = 0; a < 2; ++a)
            for (int b = 0; b < 2; ++b)
                for (int c = 0; c < 2; ++c) {
                    const int64_t g = node[a][b][c];
                    const double Wg = W[a][b][c];
                    const double dr = qV * Wg;
                    rho[g] += dr;                                   /* rho_N (L147) */
                    if (rho_abs) rho_abs[g] += fabs(dr);
                    for (int r = 0; r < 3; ++r) {                   /* Eq. (1) */
                        const double dj = dr * vhat[r];
                        J[r * nodes + g] += dj;
                        if (J_abs) J_abs[r * nodes + g] += fabs(dj);
                    }
                    for (int a2 = 0; a2 < 2; ++a2)                  /* Eq. (3), all 8 N' */
                        for (int b2 = 0; b2 < 2; ++b2)
                            for (int c2 = 0; c2 < 2; ++c2) {
                                const int o = (a2 - a + 1) * 9 + (b2 - b + 1) * 3 + (c2 - c + 1);
                                /* W_pN W_pN' formed first: M[g][o] and M[g'][26-o] then get
                                 * bit-identical addends (M_NN' = M_N'N, L73)                   */
                                const double ww = Wg * W[a2][b2][c2];
                                const double cf = qbV * ww;
                                double *m = M + ((size_t)g * 27 + o) * 9;
                                for (int r = 0; r < 3; ++r)
                                    for (int s = 0; s < 3; ++s) {
                                        const double dm = cf * al[r][s];
                                        m[r * 3 + s] += dm;
                                        if (M_abs) M_abs[((size_t)g * 27 + o) * 9 + r * 3 + s] += fabs(dm);
                                    }
                            }
                }

        /* 6. mover, Eq. (6)-(8) */
        double vt[3], vb[3];
        for (int r = 0; r < 3; ++r) vt[r] = vn[r] + beta * Ep[r];
        for (int r = 0; r < 3; ++r)
            vb[r] = al[r][0] * vt[0] + al[r][1] * vt[1] + al[r][2] * vt[2];
        if (vbar) {
            vbar[0 * n + p] = vb[0];
            vbar[1 * n + p] = vb[1];
            vbar[2 * n + p] = vb[2];
        }
        if (do_push) {
            const double un = 2.0 * vb[0] - vn[0];
            const double vnw = 2.0 * vb[1] - vn[1];
            const double wn = 2.0 * vb[2] - vn[2];
            u[p] = un;
            v[p] = vnw;
            w[p] = wn;
            x[p] = wrap(x[p] + dt * un, Lx);
            y[p] = wrap(y[p] + dt * vnw, Ly);
            z[p] = wrap(z[p] + dt * wn, Lz);
        }
    }
    return 0;
}

/* sum_N' M_NN' E_N' at every node (the operator of Eq. 4-5): out[c][n].
 * Used only by the global energy-identity pin.                                                 */
int ecsim_oracle_apply_M(int nx, int ny, int nz, const double *M, const double *E, double *out)
{
    const int64_t nodes = (int64_t)nx * ny * nz;
    for (int i = 0; i < nx; ++i)
        for (int j = 0; j < ny; ++j)
            for (int k = 0; k < nz; ++k) {
                const int64_t g = ((int64_t)i * ny + j) * nz + k;
                double acc[3] = {0, 0, 0};
                for (int di = -1; di <= 1; ++di)
                    for (int dj = -1; dj <= 1; ++dj)
                        for (int dk = -1; dk <= 1; ++dk) {
                            const int o = (di + 1) * 9 + (dj + 1) * 3 + (dk + 1);
                            const int64_t g2 = ((int64_t)((i + di + nx) % nx) * ny + (j + dj + ny) % ny) * nz
                                               + (k + dk + nz) % nz;
                            const double *m = M + ((size_t)g * 27 + o) * 9;
                            for (int r = 0; r < 3; ++r)
                                for (int s = 0; s < 3; ++s)
                                    acc[r] += m[r * 3 + s] * E[s * nodes + g2];
                        }
                for (int r = 0; r < 3; ++r) out[r * nodes + g] = acc[r];
            }
    return 0;
}

/*
 * Diagnostic moments for I/O ("plasma density, current, pressure, and heat flux ... interpolating
 * particle to the grid"; L147 computeCharge / computeCurrent: "charge density, charge current, and pressure tensor.
 * The diagnostic charge current differs from J-hat, as it excludes the effect of velocity rotation").  The paper
 * prints no formula for them; the readings are DESIGN.md R22-R24: with the same 2x2x2 weights W_pN as Eq. (1),
 *     rho_N  = (1/V_N) sum_p q_p W_pN                               (the same rho as ecsim_oracle_step)
 *     J_N    = (1/V_N) sum_p q_p W_pN v_p                           (no alpha_p: un-rotated)
 *     P_N^ij = (1/V_N) sum_p q_p W_pN v_p^i v_p^j                   6 components xx, xy, xz, yy, yz, zz
 *     Q_N^i  = (1/V_N) sum_p q_p W_pN (|v_p|^2 / 2) v_p^i           heat (energy) flux
 * Per particle, in input order; outputs accumulated into (+=), caller zeroes; *_abs optional |addend| sums.
 * Layout: rho[n]; J[c*nodes + n]; P[c*nodes + n], c = 0..5; Q[c*nodes + n].
 */
int ecsim_oracle_diagnostics(int nx, int ny, int nz, double dx, double dy, double dz, int64_t n,
                             const double *x, const double *y, const double *z,
                             const double *u, const double *v, const double *w, const double *q,
                             double *rho, double *J, double *P, double *Q,
                             double *rho_abs, double *J_abs, double *P_abs, double *Q_abs)
{
    const int64_t nodes = (int64_t)nx * ny * nz;
    const double rdx = 1.0 / dx, rdy = 1.0 / dy, rdz = 1.0 / dz;
    const double invV = 1.0 / (dx * dy * dz);
    for (int64_t p = 0; p < n; ++p) {
        const double sx = x[p] * rdx, sy = y[p] * rdy, sz = z[p] * rdz;
        const int i0 = lower_node(sx, nx), j0 = lower_node(sy, ny), k0 = lower_node(sz, nz);
        const int in[2] = {i0, (i0 + 1) % nx};
        const int jn[2] = {j0, (j0 + 1) % ny};
        const int kn[2] = {k0, (k0 + 1) % nz};
        const double xi = sx - i0, eta = sy - j0, zeta = sz - k0;
        const double wx[2] = {1.0 - xi, xi}, wy[2] = {1.0 - eta, eta}, wz[2] = {1.0 - zeta, zeta};
        const double vv[3] = {u[p], v[p], w[p]};
        const double pp[6] = {vv[0] * vv[0], vv[0] * vv[1], vv[0] * vv[2], vv[1] * vv[1], vv[1] * vv[2], vv[2] * vv[2]};
        const double half_v2 = 0.5 * ((vv[0] * vv[0] + vv[1] * vv[1]) + vv[2] * vv[2]);
        const double qV = q[p] * invV;
        for (int a = 0; a < 2; ++a)
            for (int b = 0; b < 2; ++b)
                for (int c = 0; c < 2; ++c) {
                    const int64_t g = ((int64_t)in[a] * ny + jn[b]) * nz + kn[c];
                    const double dr = qV * ((wx[a] * wy[b]) * wz[c]);
                    rho[g] += dr;
                    if (rho_abs) rho_abs[g] += fabs(dr);
                    for (int r = 0; r < 3; ++r) {
                        const double dj = dr * vv[r];
                        J[r * nodes + g] += dj;
                        if (J_abs) J_abs[r * nodes + g] += fabs(dj);
                        const double dq = dr * (half_v2 * vv[r]);
                        Q[r * nodes + g] += dq;
                        if (Q_abs) Q_abs[r * nodes + g] += fabs(dq);
                    }
                    for (int r = 0; r < 6; ++r) {
                        const double dp = dr * pp[r];
                        P[r * nodes + g] += dp;
                        if (P_abs) P_abs[r * nodes + g] += fabs(dp);
                    }
                }
    }
    return 0;
}

/*
 * TIMING VARIANT of ecsim_oracle_step on all host cores (SURVEY §8(d) "oracle_omp"; reported beside the GPU number,
 * never the parity reference).  No arithmetic of its own: it calls ecsim_oracle_step on the particles of one x-plane
 * of cells at a time.  The particles must be ordered by x-plane of cells: plane i = [plane_start[i], plane_start[i+1]).
 * A plane of cells deposits only on the node planes i and i+1, so planes of the same parity never touch the same node
 * (nx even, or nx odd and the last plane taken alone): even planes run in parallel, then odd planes.  Per-node summation
 * order differs from the sequential loop, results agree to rounding (tests: <= 1e-12 of the |addend| sums).
 * Returns -1 if a particle is not in the plane its range claims.
 */
#ifdef _OPENMP
#include <omp.h>
#endif
int ecsim_oracle_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

int ecsim_oracle_step_planes(int nx, int ny, int nz, double dx, double dy, double dz,
                             const int64_t *plane_start /* [nx+1] */, double qom, double dt,
                             double *x, double *y, double *z, double *u, double *v, double *w,
                             const double *q, const double *E, const double *B,
                             double *rho, double *J, double *M, int do_push)
{
    const double rdx = 1.0 / dx;
    int bad = 0;
    for (int i = 0; i < nx && !bad; ++i)
        for (int64_t p = plane_start[i]; p < plane_start[i + 1]; ++p)
            if (lower_node(x[p] * rdx, nx) != i) { bad = 1; break; }
    if (bad) return -1;
    const int last_alone = (nx % 2) != 0;        /* odd nx: plane nx-1 and plane 0 are both even and share node plane 0 */
    for (int colour = 0; colour < 2; ++colour) {
#pragma omp parallel for schedule(dynamic, 1)
        for (int i = colour; i < nx - last_alone; i += 2) {
            const int64_t o = plane_start[i], n = plane_start[i + 1] - o;
            ecsim_oracle_step(nx, ny, nz, dx, dy, dz, n, qom, dt, x + o, y + o, z + o, u + o, v + o, w + o, q + o, E, B,
                              rho, J, M, NULL, NULL, NULL, NULL, do_push);
        }
    }
    if (last_alone) {
        const int64_t o = plane_start[nx - 1], n = plane_start[nx] - o;
        ecsim_oracle_step(nx, ny, nz, dx, dy, dz, n, qom, dt, x + o, y + o, z + o, u + o, v + o, w + o, q + o, E, B,
                          rho, J, M, NULL, NULL, NULL, NULL, do_push);
    }
    return 0;
}

/*
 * fixPosition: "only called if the simulation is one or two-dimensional and set the particle position
 * along the same line or on the same plane.  This step is necessary to ensure the correctness of the mass matrix
 * calculations in case of reduced simulation dimensions."  Reading R25: after updatePosition the coordinates
 * of the inactive axes (axis_mask bit 0 x, 1 y, 2 z) are overwritten with fixed values; velocities keep three components.
 */
int ecsim_oracle_fix_position(int64_t n, double *x, double *y, double *z, int axis_mask, double px, double py, double pz)
{
    for (int64_t p = 0; p < n; ++p) {
        if (axis_mask & 1) x[p] = px;
        if (axis_mask & 2) y[p] = py;
        if (axis_mask & 4) z[p] = pz;
    }
    return 0;
}
