/*
 * ecpush.h -- C ABI of libecpush: the particle hot path of the energy-conserving semi-implicit
 * PIC scheme ECsim (arxiv 2603.16624; citations are PAPER.md lines) on one NVIDIA B200 (sm_100a).
 *
 * Per species the path is:
 *   gather  E^{n+theta}, B^n at the particle with linear (CIC) weights W_pN        (L49, L88, L131-L133)
 *   beta_p = q_p dt / (2 m_p);  alpha_p = (I - beta I x B_p + beta^2 B_p B_p)/(1+(beta B_p)^2)   (Eq. 2)
 *   vbar = alpha_p (v^n + beta_p E_p);  v^{n+1} = 2 vbar - v^n;  x += dt v^{n+1}, periodic wrap (Eq. 6-8)
 *   rho_N  += q_p W_pN / V_N                                                          (L147)
 *   Jhat_N += q_p W_pN (alpha_p v_p^n) / V_N                                          (Eq. 1)
 *   M^{ij}_{NN'} += beta_p q_p alpha_p^{ij} W_pN W_pN' / V_N,  27 neighbours N' of N  (Eq. 3)
 * with the deposits taken at the pre-push position and velocity (L49).
 *
 * Conventions
 *   - Every function returns 0 (ECSIM_OK) or a negative ecsim_status; nothing throws, aborts or exits.
 *   - "device" pointers are CUDA device memory of the context's device, allocated and owned by the
 *     caller (PyTorch in the harness).  The library BORROWS them: particle arrays from
 *     ecsim_load_particles until the next load of that species / ecsim_destroy; the workspace from
 *     ecsim_set_workspace until replaced / destroy; field and moment arrays only during the call
 *     (stream-ordered).  The library owns only its small host context and a few CUDA events.
 *   - All work is enqueued on the context's stream; no call synchronises with the host unless
 *     its comment says so.
 *   - Grid: periodic, nx*ny*nz cells = nodes; node n = (i*ny + j)*nz + k (z fastest, L127).
 *     A particle's cell is the node id of its lower corner N- = floor(x/dx) per axis (L131).
 *   - Fields:   F[c*nodes + n], c = 0,1,2 (x,y,z), double.
 *   - Moments:  rho[n];  Jhat[c*nodes + n];  M[((n*27 + o)*3 + i)*3 + j] with neighbour slot
 *     o = (di+1)*9 + (dj+1)*3 + (dk+1), di,dj,dk in {-1,0,1} (self = 13, mirror slot = 26-o),
 *     i = row, j = column of alpha^{ij}.  All 27 slots are produced (L73 stores 14 by symmetry).
 *   - Particles: structure of arrays of double: x,y,z (position, in [0,L)), u,v,w (velocity),
 *     q (charge of the macro-particle); q_p/m_p is one number per species.
 */
#ifndef ECPUSH_H
#define ECPUSH_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ecsim_ctx ecsim_ctx;

enum ecsim_status {
    ECSIM_OK = 0,
    ECSIM_ERR_INVALID_ARG = -1, /* null pointer, n < 0, dims < 2, spacing <= 0, dt <= 0, theta outside [0.5,1], bad species */
    ECSIM_ERR_NOT_LOADED = -2,  /* species has no particles loaded */
    ECSIM_ERR_WORKSPACE = -3,   /* workspace missing or smaller than ecsim_workspace_bytes() */
    ECSIM_ERR_CUDA = -4,        /* a CUDA call failed; text via ecsim_last_error() */
    ECSIM_ERR_NOMEM = -5,       /* host allocation failed */
    ECSIM_ERR_OVERFLOW = -6     /* resident species: its last push found segments AND the overflow list full; that push was
                                   undone, no particle is lost (see ecsim_make_resident) */
};

/* `accumulate` argument of the push_and_moments calls. */
enum ecsim_accumulate {
    ECSIM_ACC_NONE = 0,  /* every output is overwritten */
    ECSIM_ACC_ALL = 1,   /* contributions are added to rho, Jhat and M (sum over species, L84) */
    ECSIM_ACC_M_ONLY = 2 /* added to M (mass matrices are summed over species, L59); rho and Jhat of this
                            species are overwritten (Jhat is kept per species, L129) */
};

/* Storage of the mass matrices (ecsim_set_m_layout). */
enum ecsim_m_layout {
    ECSIM_M_27 = 0, /* default: M[node][27][3][3], every neighbour slot (the north-star layout) */
    ECSIM_M_14 = 1  /* the paper's symmetric storage (L73, L129): M14[node][14][3][3] = the slots o = 13..26 (self and the 13
                       "upper" neighbours); slot o < 13 of node g is slot 26-o of node g + off(o) (M_NN' = M_N'N per component) */
};

/* Kernel variants of ecsim_push_and_moments (ecsim_set_variant). */
enum ecsim_variant {
    ECSIM_VARIANT_ATOMIC = 0, /* the paper's design (L143): one thread per particle, one global atomic per
                                 scalar contribution; correct for any particle order                    */
    ECSIM_VARIANT_FUSED = 1   /* default: cell-ordered particles, a warp per contiguous range of cells, per-cell register
                                 accumulators (27 weight-product classes x 9 + Jhat + rho, pre-reduced on the FP64 matrix
                                 path) written once per cell with plain stores and expanded to the node arrays; strays
                                 are added to the per-cell accumulators of their true cell */
};

/* Create a context for a periodic grid of nx*ny*nz cells (each >= 2) with spacing dx,dy,dz (> 0).
 * cuda_stream is a cudaStream_t (NULL = legacy default stream) on the CURRENT device.  *ctx receives the context. */
int ecsim_init_grid(ecsim_ctx **ctx, int nx, int ny, int nz, double dx, double dy, double dz,
                    int n_species, void *cuda_stream);

/* Scratch bytes needed for species holding at most n_particles_max particles each: per-species cell segment
 * tables, sort keys / ranks / permutation, eight spare arrays for the out-of-place permutation (seven arrays of a
 * re-sort, or the 64-byte records of a sort of arbitrary order), stray lists,
 * and the per-cell accumulator arrays AM[cells][244], AJ[n_species][cells][8][4] of the fused kernel. */
size_t ecsim_workspace_bytes(const ecsim_ctx *ctx, int64_t n_particles_max);

/* Lend device scratch (256-byte aligned).  Host-only call. */
int ecsim_set_workspace(ecsim_ctx *ctx, void *dev_ptr, size_t bytes);

/* Register the device SoA of one species (n >= 0 particles, q_over_m = q_p/m_p).  x..w are updated in
 * place by push and by sort; q is permuted by sort.  `sorted` != 0 declares the arrays cell-sorted
 * (a performance hint only: particles found outside their cell's segment are still deposited correctly).
 * Host-only call: no device work is enqueued. */
int ecsim_load_particles(ecsim_ctx *ctx, int species, int64_t n, double q_over_m,
                         double *x, double *y, double *z, double *u, double *v, double *w, double *q,
                         int sorted);

/* Number of particles of a (non-resident) species that the hot path cannot take: a non-finite position, velocity or
 * charge, or a position outside [0, L) (ecsim_load_particles does not look at the data; positions are expected
 * wrapped).  Synchronises the stream.  Returns the count (0 = all fine) or a negative ecsim_status. */
int64_t ecsim_validate_particles(ecsim_ctx *ctx, int species);

/* Counting sort of the species by cell id (L149: the sort the paper could not realise with OpenACC).
 * On return (stream-ordered) the caller's arrays hold the particles grouped by cell, cells ascending;
 * order within a cell is unspecified.  cell_count_out: device int32[cells] per-cell counts, or NULL.
 * perm_out: device uint32[n], perm_out[new] = old index, or NULL. */
int ecsim_sort_particles(ecsim_ctx *ctx, int species, int32_t *cell_count_out, uint32_t *perm_out);

/* (A resident species -- ecsim_make_resident -- keeps itself sorted: ecsim_sort_particles and ecsim_cell_index
 * return ECSIM_ERR_INVALID_ARG for it.) */

/* Build the per-cell segment table (start[cells+1]) of a species whose arrays are ALREADY cell-sorted
 * (histogram + exclusive scan, no particle moves).  ecsim_push_and_moments does this by itself for a
 * species loaded with sorted != 0; calling it first keeps that set-up out of a timed step. */
int ecsim_build_segments(ecsim_ctx *ctx, int species);

/* Cell id of every particle as stored now: device int32[n].  (Parity of the integer binning.) */
int ecsim_cell_index(ecsim_ctx *ctx, int species, int32_t *cell_out);

/* One hot-path step for one species: gather, alpha, push, deposit (header of this file).
 *   E_theta, B : device [3][nodes], E^{n+theta} and B^n at nodes
 *   dt > 0; theta in [0.5, 1] is validated and stored, no formula of this path uses it (L84)
 *   rho [nodes], Jhat [3][nodes], M [nodes][27][3][3]: device outputs; any may be NULL (skipped)
 *   accumulate : enum ecsim_accumulate
 * With variant FUSED an unsorted species is sorted first (same effect as ecsim_sort_particles).  After the
 * call the species keeps its segment table; the kernel counts the particles that left their cell, and the
 * next call re-sorts first when that count, plus the strays handled since the last sort, exceeds
 * ecsim_set_resort_fraction() * n (default 4 %: the measured cost of a re-sort in strays), otherwise
 * the leavers are handled as strays (pushed one warp per particle, added with one bulk reduction to the per-cell
 * accumulators of their true cell before the expansion).  (The count is read through pinned memory: the next
 * call waits for this call's kernels to finish before it decides.) */
int ecsim_push_and_moments(ecsim_ctx *ctx, int species, const double *E_theta, const double *B,
                           double dt, double theta, double *rho, double *Jhat, double *M, int accumulate);

/* The same step for ALL species of the context in one pass (the mass matrices are summed over species, L59;
 * Jhat is kept per species, L129): each cell's particles of every species go through the same per-cell
 * accumulators, so M is flushed once.  rho [n_species][nodes], Jhat [n_species][3][nodes], M as above. */
int ecsim_push_and_moments_all(ecsim_ctx *ctx, const double *E_theta, const double *B, double dt, double theta,
                               double *rho, double *Jhat, double *M, int accumulate);

/* The two halves of the step as separate calls (moment gathering -> field solve -> particle mover; in a
 * real time loop E^{n+theta} comes out of the solve that the moments feed, L86).  Same kernels, same layouts, same
 * conventions as ecsim_push_and_moments:
 *   ecsim_moments  deposits rho, Jhat, M from the stored x, v (L49: "both evaluated at time n"); particles untouched;
 *                  needs B^n only (alpha_p, Eq. 2).  Arguments as above.
 *   ecsim_push     Eq. 6-8 with E^{n+theta} and the same B^n: v^{n+1}, x advanced and wrapped; no deposit.
 * ecsim_moments followed by ecsim_push with the same B equals ecsim_push_and_moments (up to rounding order: none, the
 * per-particle arithmetic is the same code).  The *_all forms take every species of the context in one pass. */
int ecsim_moments(ecsim_ctx *ctx, int species, const double *B, double dt, double *rho, double *Jhat, double *M,
                  int accumulate);
int ecsim_moments_all(ecsim_ctx *ctx, const double *B, double dt, double *rho, double *Jhat, double *M, int accumulate);
int ecsim_push(ecsim_ctx *ctx, int species, const double *E_theta, const double *B, double dt, double theta);
int ecsim_push_all(ecsim_ctx *ctx, const double *E_theta, const double *B, double dt, double theta);

/* RESIDENT species: the sort-preserving push (L149: the sort the paper could not realise).
 * ecsim_make_resident bins a loaded species and copies it into two library-managed buffers inside dev_buf (device
 * memory lent by the caller until ecsim_destroy / the next ecsim_load_particles of that species; 256-byte aligned,
 * ecsim_resident_bytes(ctx, n, slack) large).  Each cell owns a segment of slots in both buffers: its particles plus
 * max(8, slack * max(particles, mean particles per cell)) spare slots.  From then on every push of that species (ecsim_push, ecsim_push_and_moments,
 * *_all) reads one buffer and writes the other: particles that stay in their cell are written, compacted, to the front
 * of the cell's segment, a particle that moves to another cell is written straight to the back of THAT cell's segment.
 * Every step therefore starts from cell-sorted particles: no strays, no re-sort.  A particle whose new cell has no free
 * slot goes to an overflow list (n/8 entries) and is handled, one warp per particle, by every later pass until a slot
 * is free; when the list has cost more than a fresh layout (ecsim_set_resort_fraction, as for the re-sort of a dense
 * species) the species is laid out afresh (counted by ecsim_relayout_count).  The arrays given to ecsim_load_particles are not referenced after ecsim_make_resident returns
 * and are NOT updated by pushes: read the species back with ecsim_export_particles (device arrays of n doubles each;
 * cell-major order; also works, as a plain copy, for a species that is not resident).
 * (A species loaded with sorted = 0 is sorted in place first -- its arrays are permuted -- so that the copy is sequential.)
 * ecsim_make_resident synchronises the stream once (it checks the data-dependent slot count against the buffer);
 * slack in [0, 4], typically 0.25.  All species of one *_all call must be of one kind (all resident or none).
 * When a push finds a cell's segment AND the overflow list full, no particle is lost: the push writes the idle buffer and
 * never its input, so the NEXT call that touches the species (any call: they all look at the list's counter first) undoes
 * that push by swapping the buffers back, lays the pre-push state out afresh, enqueues nothing of its own and returns
 * ECSIM_ERR_OVERFLOW; ecsim_last_error() names the species.  The moments of a fused call were deposited from the pre-push
 * state and stay valid: repeat the push of THAT species alone (ecsim_push, same E, B, dt), or make it resident again with
 * more slack.  ecsim_set_overflow_capacity lowers the list's capacity (1 .. n/8, at least 65536 by default) -- for
 * tests of this path and for callers that want the error earlier. */
size_t ecsim_resident_bytes(const ecsim_ctx *ctx, int64_t n_particles, double slack);
int ecsim_make_resident(ecsim_ctx *ctx, int species, void *dev_buf, size_t bytes, double slack);
int ecsim_export_particles(ecsim_ctx *ctx, int species, double *x, double *y, double *z, double *u, double *v,
                           double *w, double *q);
int64_t ecsim_relayout_count(const ecsim_ctx *ctx);
int ecsim_set_overflow_capacity(ecsim_ctx *ctx, int species, int64_t entries);

/* Reduced dimensionality (L123: "fixPosition ... is only called if the simulation is one or two-dimensional and set the
 * particle position along the same line or on the same plane.  This step is necessary to ensure the correctness of the
 * mass matrix calculations").  axis_mask: bit 0 x, bit 1 y, bit 2 z; from this call on every push (all variants, all
 * layouts) overwrites the masked coordinates of the pushed position with px / py / pz (each in [0, L)) before the
 * periodic wrap; velocities keep all three components.  Species already loaded are pinned by the call (and re-binned
 * before their next step); ecsim_load_particles pins on load while a mask is set (the one case where a load enqueues
 * device work).  A 2-D run in the x-y plane: any nz >= 2, axis_mask = 4, pz = a node plane k0*dz: every z weight is
 * (1, 0), all moments land on node plane k0.  axis_mask = 0 switches the pinning off. */
int ecsim_set_fixed_axes(ecsim_ctx *ctx, int axis_mask, double px, double py, double pz);

/* Diagnostic moments of one species, the quantities ECsim writes with its I/O (L121 "plasma density, current, pressure,
 * and heat flux"; L147 computeCharge / computeCurrent: "The diagnostic charge current differs from J-hat, as it excludes
 * the effect of velocity rotation").  With the same weights W_pN as Eq. (1) (the paper prints no formulas; readings
 * R22-R24 of DESIGN.md):
 *   rho [nodes]     = sum_p q_p W_pN / V_N
 *   J   [3][nodes]  = sum_p q_p W_pN v_p / V_N                      (no alpha_p)
 *   P   [6][nodes]  = sum_p q_p W_pN v_p^i v_p^j / V_N              components xx, xy, xz, yy, yz, zz
 *   Q   [3][nodes]  = sum_p q_p W_pN (|v_p|^2 / 2) v_p^i / V_N
 * Device outputs, overwritten; any may be NULL.  Particles untouched.  Works for dense and resident species. */
int ecsim_diagnostics(ecsim_ctx *ctx, int species, double *rho, double *J, double *P, double *Q);

/* Mass-matrix storage for all later deposit calls and for ecsim_apply_M: enum ecsim_m_layout.  With ECSIM_M_14 the M
 * argument of the deposit calls is M14[nodes][14][3][3] (half the bytes; VARIANT_ATOMIC supports ECSIM_M_27 only). */
int ecsim_set_m_layout(ecsim_ctx *ctx, int layout);

/* out_N = sum_N' M_NN' E_N' over the 27 neighbours of every node (Eq. 4-5: the mass-matrix term of the
 * field equations, applied once per Krylov iteration of the implicit solve).  M in the context's current layout;
 * E, out: device [3][nodes], E != out; accumulate != 0: out += . */
int ecsim_apply_M(ecsim_ctx *ctx, const double *M, const double *E, double *out, int accumulate);

/* Same step with HOST buffers: copies particles and fields to device staging (carved from the
 * workspace, which must be ecsim_host_step_workspace_bytes() large), runs the step, copies particles
 * and moments back, and synchronises the stream.  Host arrays: x..w in/out [n], q in [n], E/B in,
 * rho/Jhat/M out (with accumulate != 0 the accumulated arrays are copied in first).  Pinned host memory makes the copies asynchronous. */
/* When the arrays are declared cell-sorted (sorted != 0, accumulate = 0, variant FUSED) the step runs as a pipeline over
 * slabs of x-planes on three streams -- upload slab k+1 | bin, deposit + push, expand slab k | download slab k-1 -- so
 * that the two directions of the PCIe link overlap (one cudaMemcpyAsync per array per slab; pinned host memory is
 * needed for the overlap, pageable memory still gives the right result).  For these two host entries `sorted` != 0 is
 * therefore a CONTRACT, not a hint: if a particle is found outside the slab / cell its place in the arrays implies, the
 * call returns ECSIM_ERR_INVALID_ARG (text in ecsim_last_error) and the particle arrays are left partially advanced.
 * Pass sorted = 0 when unsure (serial path, the library sorts).  ecsim_set_host_pipeline(0) forces the serial path, (2)
 * pipelines even tiny inputs (default 1: only when a slab carries >= 32 MB); ecsim_host_pipelined_count = calls that
 * completed through the pipeline.  While ecsim_set_fixed_axes is active the serial path is always taken (the particles
 * are pinned after their upload).  On any error return no copy of the call is still in flight. */
int ecsim_set_host_pipeline(ecsim_ctx *ctx, int on);
int64_t ecsim_host_pipelined_count(const ecsim_ctx *ctx);
size_t ecsim_host_step_workspace_bytes(const ecsim_ctx *ctx, int64_t n_particles);
int ecsim_push_and_moments_host(ecsim_ctx *ctx, int64_t n, double q_over_m, int sorted,
                                double *x, double *y, double *z, double *u, double *v, double *w,
                                const double *q, const double *E_theta, const double *B,
                                double dt, double theta, double *rho, double *Jhat, double *M, int accumulate);

/* The same for ALL species of the context in one call (M crosses the bus once): n, q_over_m and the array-of-pointer
 * arguments have n_species entries; rho [n_species][nodes], Jhat [n_species][3][nodes], M shared.  The workspace must
 * be ecsim_host_step_all_workspace_bytes(ctx, max n, sum of n) large. */
size_t ecsim_host_step_all_workspace_bytes(const ecsim_ctx *ctx, int64_t n_max, int64_t n_total);
int ecsim_push_and_moments_host_all(ecsim_ctx *ctx, const int64_t *n, const double *q_over_m, int sorted,
                                    double *const *x, double *const *y, double *const *z,
                                    double *const *u, double *const *v, double *const *w, const double *const *q,
                                    const double *E_theta, const double *B, double dt, double theta,
                                    double *rho, double *Jhat, double *M, int accumulate);

/* Select the kernel variant (default ECSIM_VARIANT_FUSED). */
int ecsim_set_variant(ecsim_ctx *ctx, int variant);

/* Tuning knobs: fraction of a species that may sit outside its cell segment before the next step re-sorts
 * (default 0.04); warps per CTA of the fused kernel (8, 12 or 16, with 224, 168 or 128 registers per thread;
 * default 12). */
int ecsim_set_resort_fraction(ecsim_ctx *ctx, double fraction);
int ecsim_set_fused_warps(ecsim_ctx *ctx, int warps);
/* Instrumentation.  ecsim_enable_timing(1) records CUDA events around the deposit/push kernel of every
 * ecsim_push_and_moments call; ecsim_kernel_ms() SYNCHRONISES on the last pair and returns its time.
 * ecsim_launch_count() = kernels + memsets this context has enqueued so far;
 * ecsim_stray_count() = particles the last FUSED step found outside their segment (synchronises the stream). */
int ecsim_enable_timing(ecsim_ctx *ctx, int on);
int ecsim_kernel_ms(ecsim_ctx *ctx, float *ms_out);
int64_t ecsim_launch_count(const ecsim_ctx *ctx);
int64_t ecsim_stray_count(ecsim_ctx *ctx);
int64_t ecsim_leaver_count(ecsim_ctx *ctx);       /* particles whose cell changed in the last push (synchronises the stream) */
int64_t ecsim_resort_count(const ecsim_ctx *ctx); /* re-sorts ecsim_push_and_moments triggered so far */

/* FP64 FMA throughput of the device (dependent-chain DFMA kernel, `iters` x 128 FMAs per thread), the
 * denominator of the ALU roofline.  Synchronises.  tflops_out: 2 flops per FMA; ms_out may be NULL. */
int ecsim_probe_fp64(ecsim_ctx *ctx, int iters, double *tflops_out, float *ms_out);

int ecsim_destroy(ecsim_ctx *ctx);

/* Per-cell segment table of a species WITHOUT a context, a workspace or any allocation: the binning of L131 and the
 * histogram + exclusive scan that open the counting sort (L149), i.e. what ecsim_sort_particles / ecsim_build_segments
 * compute into the lent workspace.
 *
 * Who this is for.  Everything else in this header needs a context (ecsim_init_grid creates events and pinned host
 * buffers) and scratch that the caller obtained from cudaMalloc and lent with ecsim_set_workspace.  Some callers cannot do
 * that: a plug-in called from inside a host code whose device memory is handed out once at start-up (ECsim's own OpenACC
 * data regions, or a framework whose pool already holds the whole HBM, so that a fresh cudaMalloc fails or evicts);
 * code on a latency-critical path of a time loop, where cudaMalloc / cudaFree serialise the whole device; code running
 * under a memory budget fixed by a scheduler.  This call lets them bin a species with nothing but their own input and
 * output arrays.  Its scratch (the cell histogram and the partial sums of the scan) lives in an array compiled into the
 * library, ECSIM_STATIC_MAX_CELLS + 4096 32-bit words = 8.02 MB, which every GPU that loads libecpush holds from the
 * load of the library's device code until the process exits, whether or not this call is ever made.
 *
 *   cuda_stream    cudaStream_t (NULL = legacy default stream) of the CURRENT device; all work is enqueued on it
 *   nx, ny, nz     cells per axis, each >= 2, with nx*ny*nz <= ECSIM_STATIC_MAX_CELLS (128^3, the largest BASELINE.json
 *                  grid); a larger grid is refused with ECSIM_ERR_INVALID_ARG and a text in ecsim_last_error() that
 *                  names the limit -- nothing is enqueued
 *   dx, dy, dz     spacing > 0 (cell of a particle as in the conventions above: floor(x * (1/dx)) per axis, clamped)
 *   n, x, y, z     n >= 0 particles (n < 2^32), device arrays of n doubles, read only, any order
 *   cell_count_out device int32[cells]: particles per cell (what ecsim_sort_particles returns); or NULL
 *   start_out      device uint32[cells+1]: exclusive running sum of the counts, start_out[cells] = n; or NULL
 *                  (at least one of the two outputs must be given)
 *
 * The call makes no cudaMalloc / cudaFree / cudaMallocHost, creates no stream or event and calls no library routine that
 * allocates; it does not synchronise.  The FIRST call on each device looks up that device's address of the built-in
 * array (cudaGetSymbolAddress, which may load the library's device code): make that first call outside any stream
 * capture.  All calls on one device share the one array: the call clears the histogram itself before counting, but two
 * calls whose work can overlap on the GPU (different streams without an ordering between them, or two host threads
 * on different streams) race on it and both results are undefined -- order them on one stream or with events. */
#define ECSIM_STATIC_MAX_CELLS 2097152
int ecsim_cell_segments_static(void *cuda_stream, int nx, int ny, int nz, double dx, double dy, double dz,
                               int64_t n, const double *x, const double *y, const double *z,
                               int32_t *cell_count_out, uint32_t *start_out);

/* Static text for a status; ecsim_last_error: text of the last CUDA failure in this process. */
const char *ecsim_strerror(int status);
const char *ecsim_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* ECPUSH_H */
