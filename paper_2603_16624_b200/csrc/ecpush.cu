// ecpush.cu -- C ABI of libecpush (include/ecpush.h): context, workspace, orchestration of the sm_100a kernels in
// sort.cuh / fused_mma.cuh / resident.cuh / atomic_path.cuh / expand*.cuh / apply_m.cuh.  Product code: no CPU
// fallback, no code shared with oracle/.  Every entry point returns an ecsim_status and never throws.
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <algorithm>
#include <mutex>
#include <new>

#include "../../include/ecpush.h"
#include "common.cuh"
#include "sort.cuh"
#include "atomic_path.cuh"
#include "fused_mma.cuh"
#include "expand.cuh"
#include "expand_tma.cuh"
#include "resident.cuh"
#include "homeless.cuh"
#include "apply_m.cuh"
#include "probe.cuh"

// --------------------------------------------------------------------------------------------
static thread_local char g_last_error[512] = "";

static int cuda_fail(cudaError_t e, const char* what, int line)
{
    snprintf(g_last_error, sizeof(g_last_error), "%s failed at ecpush.cu:%d: %s (%s)", what, line,
             cudaGetErrorString(e), cudaGetErrorName(e));
    return ECSIM_ERR_CUDA;
}
#define CK(call)                                                        \
    do {                                                                \
        cudaError_t e__ = (call);                                       \
        if (e__ != cudaSuccess) return cuda_fail(e__, #call, __LINE__); \
    } while (0)
#define CK_LAUNCH() CK(cudaGetLastError())

enum SortState { ST_UNSORTED = 0, ST_DECLARED = 1, ST_SEGMENTED = 2 };
#define ECSIM_HOST_SLABS_MAX 32

// A RESIDENT species (ecsim_make_resident): library-managed gapped double buffers in memory the caller lent
// (resident.cuh; LAYOUT_GAPPED of fused_mma.cuh).
struct Resident {
    bool on = false;
    uint32_t cap_bound = 0;         // slots per array the lent buffer can hold
    double slack = 0.25;
    double* buf[2][7] = {};         // two buffers of x,y,z,u,v,w,q
    uint32_t* seg = nullptr;        // [cells+1] first slot of every cell's segment (both buffers)
    uint32_t* seg_alt = nullptr;    // [cells+1] the table a fresh layout is written to (then the two swap)
    uint32_t* F[2] = {};            // [cells] front runs
    uint32_t* R[2] = {};            // [cells] back runs (arrivals of the last push)
    int cur = 0;                    // buffer that holds the species now
    double* ovf[2] = {};            // two overflow lists [7][ovf_cap]: particles without a slot ("homeless")
    uint32_t ovf_cap = 0;
    uint32_t* ovf_count[2] = {};    // device counters
    int ovf_cur = 0;                // list that holds the homeless particles now (a push reads it and fills the other)
};

struct SpeciesHost {
    bool loaded = false;
    int64_t n = 0;
    double qom = 0.0;
    double *x = nullptr, *y = nullptr, *z = nullptr, *u = nullptr, *v = nullptr, *w = nullptr, *q = nullptr;
    int state = ST_UNSORTED;
    double stray_debt = 0.0;        // strays processed since the last sort, summed over the steps
    bool nearly_sorted = false;     // the arrays were cell-sorted before the last pushes (a re-sort, not a first sort)
    bool leavers_pending = false;   // an async copy of the leaver / overflow counters is in flight
    cudaEvent_t leavers_event = nullptr;
    Resident res;
};

struct Workspace {
    void* base = nullptr;
    size_t bytes = 0;
    int64_t n_max = 0;
    // carved regions
    uint32_t* start = nullptr;       // [n_species][cells+1]
    uint32_t* count = nullptr;       // [cells]
    uint32_t* block_sums = nullptr;  // [ceil(cells/1024)]
    int32_t* cell = nullptr;         // [n_max]
    uint32_t* rank = nullptr;        // [n_max]
    uint32_t* perm = nullptr;        // [n_max]
    double* spare = nullptr;         // [8][n_max]: the seven arrays of a species on their way through a re-sort, or its
                                     // n_max 64-byte records on their way through a sort of arbitrary order
    uint32_t* tile_hist = nullptr;   // [tiles][NB] of the two-step move of a random-order sort
    uint32_t* tile_off = nullptr;    // its tile-local exclusive scans over the buckets
    uint32_t* tile_scan = nullptr;   // first slot of every (tile, bucket) share
    uint32_t* tile_sums = nullptr;   // [chunks of tiles][NB] column sums
    uint32_t* stray_list = nullptr;  // [n_species][n_max]
    double* AM = nullptr;            // [cells][AM_PER_CELL = 244]
    double* AJ = nullptr;            // [n_species][cells][32]
    uint32_t* stray_count = nullptr; // [n_species]
    unsigned long long* leavers = nullptr; // [n_species]
    char* extra = nullptr;           // what is left (host-step staging)
    size_t extra_bytes = 0;
};

struct ecsim_ctx {
    Geom g;
    int n_species = 0;
    cudaStream_t stream = nullptr;
    SpeciesHost* sp = nullptr;
    Workspace ws;
    int variant = ECSIM_VARIANT_FUSED;
    double resort_fraction = 0.04;
    int timing = 0;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    bool ev_valid = false;
    int64_t launches = 0;
    int sm_count = 0;
    int fused_warps = 12;
    unsigned long long* h_leavers = nullptr;  // pinned [n_species]
    uint32_t* h_strays = nullptr;             // pinned [n_species]
    uint32_t* h_ovf = nullptr;                // pinned [n_species]: overflow count of the last resident push
    int last_call_species[ECSIM_MAX_SPECIES];
    int last_call_n = 0;
    int64_t resorts = 0;
    int64_t relayouts = 0;
    int m_layout = ECSIM_M_27;
    // pipelined host step: upload / download streams beside the caller's stream, one event pair per slab
    cudaStream_t s_up = nullptr, s_down = nullptr;
    cudaEvent_t ev_up[ECSIM_HOST_SLABS_MAX] = {}, ev_comp[ECSIM_HOST_SLABS_MAX] = {}, ev_exp[ECSIM_HOST_SLABS_MAX] = {};
    cudaEvent_t ev_start = nullptr, ev_fields = nullptr, ev_down = nullptr;
    int host_pipeline = 1;
    int64_t host_pipelined_calls = 0;
};

static inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

struct Carver {
    char* p;
    size_t off = 0;
    template <class T> T* take(size_t count)
    {
        T* r = p ? reinterpret_cast<T*>(p + off) : nullptr;
        off = align_up(off + count * sizeof(T), 256);
        return r;
    }
};

static size_t carve(const ecsim_ctx* c, int64_t n_max, void* base, Workspace* out)
{
    const size_t cells = (size_t)c->g.nodes;
    const size_t nsp = (size_t)c->n_species;
    const size_t n = (size_t)(n_max > 0 ? n_max : 0);
    Carver k{reinterpret_cast<char*>(base)};
    Workspace w;
    w.start = k.take<uint32_t>(nsp * (cells + 1));
    w.count = k.take<uint32_t>(cells);
    w.block_sums = k.take<uint32_t>((cells + SCAN_BLOCK - 1) / SCAN_BLOCK + 1);
    w.cell = k.take<int32_t>(n);
    w.rank = k.take<uint32_t>(n);
    w.perm = k.take<uint32_t>(n);
    w.spare = k.take<double>(8 * n);
    {
        const size_t m = sort_table_entries(n);
        w.tile_hist = k.take<uint32_t>(m);
        w.tile_off = k.take<uint32_t>(m);
        w.tile_scan = k.take<uint32_t>(m + 1);
        w.tile_sums = k.take<uint32_t>(sort_chunk_entries(n));
    }
    w.stray_list = k.take<uint32_t>(nsp * n);
    w.AM = k.take<double>(cells * AM_PER_CELL);
    w.AJ = k.take<double>(nsp * cells * AJ_PER_CELL);
    w.stray_count = k.take<uint32_t>(nsp);
    w.leavers = k.take<unsigned long long>(nsp);
    if (out) {
        w.base = base;
        w.n_max = n_max;
        *out = w;
    }
    return k.off;
}

static int grid_for(const ecsim_ctx* c, size_t work, int block, int per_sm)
{
    size_t blocks = (work + block - 1) / block;
    size_t cap = (size_t)c->sm_count * per_sm;
    if (blocks > cap) blocks = cap;
    if (blocks < 1) blocks = 1;
    return (int)blocks;
}

// --------------------------------------------------------------------------------------------
extern "C" const char* ecsim_strerror(int status)
{
    switch (status) {
    case ECSIM_OK: return "ok";
    case ECSIM_ERR_INVALID_ARG: return "invalid argument";
    case ECSIM_ERR_NOT_LOADED: return "species has no particles loaded";
    case ECSIM_ERR_WORKSPACE: return "workspace missing or too small";
    case ECSIM_ERR_CUDA: return "CUDA call failed (see ecsim_last_error)";
    case ECSIM_ERR_NOMEM: return "host allocation failed";
    case ECSIM_ERR_OVERFLOW: return "resident species: segments and overflow list full, the last push of that species was undone (see ecsim_last_error)";
    default: return "unknown status";
    }
}

extern "C" const char* ecsim_last_error(void) { return g_last_error; }

extern "C" int ecsim_init_grid(ecsim_ctx** ctx, int nx, int ny, int nz, double dx, double dy, double dz,
                               int n_species, void* cuda_stream)
{
    if (!ctx) return ECSIM_ERR_INVALID_ARG;
    *ctx = nullptr;
    if (nx < 2 || ny < 2 || nz < 2 || !(dx > 0) || !(dy > 0) || !(dz > 0) || n_species < 1 ||
        n_species > ECSIM_MAX_SPECIES || (int64_t)nx * ny * nz > 0x7fffffffLL)
        return ECSIM_ERR_INVALID_ARG;
    int dev = 0;
    CK(cudaGetDevice(&dev));
    cudaDeviceProp prop;
    CK(cudaGetDeviceProperties(&prop, dev));
    ecsim_ctx* c = new (std::nothrow) ecsim_ctx();
    if (!c) return ECSIM_ERR_NOMEM;
    c->sp = new (std::nothrow) SpeciesHost[n_species];
    if (!c->sp) { delete c; return ECSIM_ERR_NOMEM; }
    Geom& g = c->g;
    g.nx = nx; g.ny = ny; g.nz = nz;
    g.dx = dx; g.dy = dy; g.dz = dz;
    g.rdx = 1.0 / dx; g.rdy = 1.0 / dy; g.rdz = 1.0 / dz;
    g.Lx = nx * dx; g.Ly = ny * dy; g.Lz = nz * dz;
    g.invV = 1.0 / (dx * dy * dz);
    g.nodes = (long long)nx * ny * nz;
    g.fix_mask = 0;
    g.fix_pos[0] = g.fix_pos[1] = g.fix_pos[2] = 0.0;
    c->n_species = n_species;
    c->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    c->sm_count = prop.multiProcessorCount;
    cudaError_t e = cudaEventCreate(&c->ev0);
    if (e == cudaSuccess) e = cudaEventCreate(&c->ev1);
    for (int s = 0; s < n_species && e == cudaSuccess; ++s)
        e = cudaEventCreateWithFlags(&c->sp[s].leavers_event, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaMallocHost(&c->h_leavers, sizeof(unsigned long long) * n_species);
    if (e == cudaSuccess) e = cudaMallocHost(&c->h_strays, sizeof(uint32_t) * n_species);
    if (e == cudaSuccess) e = cudaMallocHost(&c->h_ovf, sizeof(uint32_t) * n_species);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&c->s_up, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&c->s_down, cudaStreamNonBlocking);
    for (int k = 0; k < ECSIM_HOST_SLABS_MAX && e == cudaSuccess; ++k) {
        e = cudaEventCreateWithFlags(&c->ev_up[k], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_comp[k], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_exp[k], cudaEventDisableTiming);
    }
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_start, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_fields, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_down, cudaEventDisableTiming);
    if (e != cudaSuccess) {
        int rc = cuda_fail(e, "context set-up", __LINE__);
        ecsim_destroy(c);
        return rc;
    }
    for (int s = 0; s < n_species; ++s) { c->h_leavers[s] = 0; c->h_strays[s] = 0; c->h_ovf[s] = 0; }
    *ctx = c;
    return ECSIM_OK;
}

extern "C" int ecsim_destroy(ecsim_ctx* c)
{
    if (!c) return ECSIM_OK;
    if (c->sp) {
        for (int s = 0; s < c->n_species; ++s)
            if (c->sp[s].leavers_event) cudaEventDestroy(c->sp[s].leavers_event);
        delete[] c->sp;
    }
    if (c->ev0) cudaEventDestroy(c->ev0);
    if (c->ev1) cudaEventDestroy(c->ev1);
    if (c->h_leavers) cudaFreeHost(c->h_leavers);
    if (c->h_strays) cudaFreeHost(c->h_strays);
    if (c->h_ovf) cudaFreeHost(c->h_ovf);
    for (int k = 0; k < ECSIM_HOST_SLABS_MAX; ++k) {
        if (c->ev_up[k]) cudaEventDestroy(c->ev_up[k]);
        if (c->ev_comp[k]) cudaEventDestroy(c->ev_comp[k]);
        if (c->ev_exp[k]) cudaEventDestroy(c->ev_exp[k]);
    }
    if (c->ev_start) cudaEventDestroy(c->ev_start);
    if (c->ev_fields) cudaEventDestroy(c->ev_fields);
    if (c->ev_down) cudaEventDestroy(c->ev_down);
    if (c->s_up) cudaStreamDestroy(c->s_up);
    if (c->s_down) cudaStreamDestroy(c->s_down);
    delete c;
    return ECSIM_OK;
}

extern "C" size_t ecsim_workspace_bytes(const ecsim_ctx* c, int64_t n_particles_max)
{
    if (!c || n_particles_max < 0) return 0;
    return carve(c, n_particles_max, nullptr, nullptr);
}

extern "C" int ecsim_set_workspace(ecsim_ctx* c, void* dev_ptr, size_t bytes)
{
    if (!c || !dev_ptr || (reinterpret_cast<uintptr_t>(dev_ptr) & 255u)) return ECSIM_ERR_INVALID_ARG;
    // n_max = the largest particle count the buffer can serve
    const size_t fixed = carve(c, 0, nullptr, nullptr);
    if (bytes < fixed) return ECSIM_ERR_WORKSPACE;
    const size_t per_particle = sizeof(int32_t) + 2 * sizeof(uint32_t) + 7 * sizeof(double) +
                                (size_t)c->n_species * sizeof(uint32_t);
    // carve() is monotone in n: bisect for the largest n that fits (the per-array 256-byte rounding
    // makes a closed form off by a few particles either way)
    int64_t lo = 0, hi = (int64_t)((bytes - fixed) / per_particle) + 1;
    if (hi > 0xffffffffLL) hi = 0xffffffffLL;
    while (lo < hi) {
        const int64_t mid = lo + (hi - lo + 1) / 2;
        if (carve(c, mid, nullptr, nullptr) <= bytes) lo = mid; else hi = mid - 1;
    }
    int64_t n_max = lo;
    const size_t used = carve(c, n_max, dev_ptr, &c->ws);
    c->ws.bytes = bytes;
    c->ws.extra = reinterpret_cast<char*>(dev_ptr) + used;
    c->ws.extra_bytes = bytes - used;
    for (int s = 0; s < c->n_species; ++s)
        if (c->sp[s].state == ST_SEGMENTED) c->sp[s].state = ST_DECLARED;  // tables lived in the old buffer
    return ECSIM_OK;
}

static int check_species(const ecsim_ctx* c, int s)
{
    if (!c || s < 0 || s >= c->n_species) return ECSIM_ERR_INVALID_ARG;
    if (!c->sp[s].loaded) return ECSIM_ERR_NOT_LOADED;
    return ECSIM_OK;
}

static int need_workspace(const ecsim_ctx* c, int64_t n)
{
    if (!c->ws.base || c->ws.n_max < n) return ECSIM_ERR_WORKSPACE;
    return ECSIM_OK;
}

extern "C" int ecsim_load_particles(ecsim_ctx* c, int s, int64_t n, double q_over_m,
                                    double* x, double* y, double* z, double* u, double* v, double* w,
                                    double* q, int sorted)
{
    if (!c || s < 0 || s >= c->n_species || n < 0 || n > 0xffffffffLL || !isfinite(q_over_m))
        return ECSIM_ERR_INVALID_ARG;
    if (n > 0 && (!x || !y || !z || !u || !v || !w || !q)) return ECSIM_ERR_INVALID_ARG;
    SpeciesHost& sp = c->sp[s];
    sp.loaded = true;
    sp.n = n;
    sp.qom = q_over_m;
    sp.x = x; sp.y = y; sp.z = z; sp.u = u; sp.v = v; sp.w = w; sp.q = q;
    sp.state = sorted ? ST_DECLARED : ST_UNSORTED;
    sp.nearly_sorted = sorted != 0;
    sp.stray_debt = 0.0;
    sp.leavers_pending = false;
    sp.res.on = false;              // a fresh load is a borrowed (dense) species again
    if (c->g.fix_mask && n > 0) {
        // reduced dimensionality: the species starts on the line / plane (the one load that enqueues device work)
        k_fix_position<<<grid_for(c, (size_t)n, 256, 16), 256, 0, c->stream>>>(c->g, (size_t)n, x, y, z);
        CK_LAUNCH();
        c->launches++;
    }
    return ECSIM_OK;
}

static int resident_settle(ecsim_ctx* c, int s);
static int resident_relayout(ecsim_ctx* c, int s, bool binned);

// Reduced dimensionality (L123 fixPosition): from now on every push pins the coordinates of the axes in axis_mask
// (bit 0 x, 1 y, 2 z) to the given values; species already loaded are pinned now.
extern "C" int ecsim_set_fixed_axes(ecsim_ctx* c, int axis_mask, double px, double py, double pz)
{
    if (!c || axis_mask < 0 || axis_mask > 7) return ECSIM_ERR_INVALID_ARG;
    const double pos[3] = {px, py, pz};
    const double L[3] = {c->g.Lx, c->g.Ly, c->g.Lz};
    for (int a = 0; a < 3; ++a)
        if ((axis_mask >> a) & 1)
            if (!(pos[a] >= 0.0 && pos[a] < L[a])) return ECSIM_ERR_INVALID_ARG;
    c->g.fix_mask = axis_mask;
    for (int a = 0; a < 3; ++a) c->g.fix_pos[a] = pos[a];
    if (!axis_mask) return ECSIM_OK;
    for (int s = 0; s < c->n_species; ++s) {
        SpeciesHost& sp = c->sp[s];
        if (!sp.loaded || sp.n == 0) continue;
        if (sp.res.on) {
            // every slot of both buffers (unused slots hold nothing that matters); cells along a pinned axis do not change
            int rc = resident_settle(c, s);
            if (rc) return rc;
            for (int b = 0; b < 2; ++b) {
                k_fix_position<<<c->sm_count * 8, 256, 0, c->stream>>>(c->g, (size_t)sp.res.cap_bound, sp.res.buf[b][0],
                                                                         sp.res.buf[b][1], sp.res.buf[b][2]);
                CK_LAUNCH();
                c->launches++;
            }
            // ... and the particles without a slot (the overflow list the next pass reads; unused entries do not matter)
            if (sp.res.ovf_cap > 0) {
                double* l = sp.res.ovf[sp.res.ovf_cur];
                const size_t cap = sp.res.ovf_cap;
                k_fix_position<<<grid_for(c, cap, 256, 16), 256, 0, c->stream>>>(c->g, cap, l, l + cap, l + 2 * cap);
                CK_LAUNCH();
                c->launches++;
            }
            // the pinned particles may now sit in other cells than their segments say: bin and lay out afresh
            rc = resident_relayout(c, s, false);
            if (rc) return rc;
        } else {
            k_fix_position<<<grid_for(c, (size_t)sp.n, 256, 16), 256, 0, c->stream>>>(c->g, (size_t)sp.n, sp.x, sp.y, sp.z);
            CK_LAUNCH();
            c->launches++;
            sp.state = ST_UNSORTED;
            sp.nearly_sorted = false;
        }
    }
    return ECSIM_OK;
}

static int scan_u32(ecsim_ctx* c, const uint32_t* in, uint32_t* out /* [m+1] */, uint32_t m)
{
    Workspace& w = c->ws;
    const uint32_t nb = (m + SCAN_BLOCK - 1) / SCAN_BLOCK;
    k_scan_blocks<<<nb, SCAN_BLOCK, 0, c->stream>>>(in, out, w.block_sums, m);
    CK_LAUNCH();
    k_scan_sums<<<1, SCAN_BLOCK, 0, c->stream>>>(w.block_sums, nb, out, m);
    CK_LAUNCH();
    k_scan_add<<<nb, SCAN_BLOCK, 0, c->stream>>>(out, w.block_sums, m);
    CK_LAUNCH();
    c->launches += 3;
    return ECSIM_OK;
}

// histogram of n particles at (x,y,z) -> ws.count (+ ws.cell / ws.rank)
static int histogram(ecsim_ctx* c, uint32_t n, const double* x, const double* y, const double* z, bool with_rank)
{
    Workspace& w = c->ws;
    const uint32_t cells = (uint32_t)c->g.nodes;
    CK(cudaMemsetAsync(w.count, 0, sizeof(uint32_t) * cells, c->stream));
    c->launches++;
    if (n > 0) {
        const int grid = grid_for(c, (size_t)n, 256, 16);
        if (with_rank)
            k_cell_hist<true><<<grid, 256, 0, c->stream>>>(c->g, n, x, y, z, w.cell, w.rank, w.count);
        else
            k_cell_hist<false><<<grid, 256, 0, c->stream>>>(c->g, n, x, y, z, nullptr, nullptr, w.count);
        CK_LAUNCH();
        c->launches++;
    }
    return ECSIM_OK;
}

// histogram of the species as stored + exclusive scan -> start table of the species
static int histogram_and_scan(ecsim_ctx* c, int s, bool with_rank)
{
    SpeciesHost& sp = c->sp[s];
    const uint32_t cells = (uint32_t)c->g.nodes;
    int rc = histogram(c, (uint32_t)sp.n, sp.x, sp.y, sp.z, with_rank);
    if (rc) return rc;
    return scan_u32(c, c->ws.count, c->ws.start + (size_t)s * (cells + 1), cells);
}

extern "C" int ecsim_build_segments(ecsim_ctx* c, int s)
{
    int rc = check_species(c, s);
    if (rc) return rc;
    if (c->sp[s].res.on) return ECSIM_OK;          // a resident species is always segmented
    rc = need_workspace(c, c->sp[s].n);
    if (rc) return rc;
    rc = histogram_and_scan(c, s, false);
    if (rc) return rc;
    c->sp[s].state = ST_SEGMENTED;
    c->sp[s].leavers_pending = false;
    return ECSIM_OK;
}

static int resident_layout_from_dense(ecsim_ctx* c, int s, const double* const src[7], int dst_buf);

// Step A of the sort of a species in arbitrary order (sort.cuh) in one of its two geometries: final places, per-tile bucket
// tables, first slots, then the records of every tile into ws.spare.  *shift_out: log2 of the bucket size chosen.
template <int NB, int TILE>
static int stage_records(ecsim_ctx* c, uint32_t n, const uint32_t* start, uint32_t* dest, double* const arrays[7],
                         uint32_t* tmpdest, int* shift_out)
{
    Workspace& w = c->ws;
    const size_t smem = sort_stage_smem(NB, TILE);
    CK(cudaFuncSetAttribute(k_stage_records<NB, TILE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int shift = 13;
    while ((((n - 1) >> shift) + 1) > (uint32_t)NB) ++shift;
    const uint32_t tiles = (n + TILE - 1) / TILE;
    const uint32_t chunks = (tiles + SORT_CHUNK - 1) / SORT_CHUNK;
    k_dest_and_tile_hist<NB, TILE><<<tiles, NB, 0, c->stream>>>(n, w.cell, dest, start, shift, w.tile_hist, w.tile_off);
    CK_LAUNCH();
    k_tile_colsum<<<chunks, NB, 0, c->stream>>>(tiles, w.tile_hist, w.tile_sums);
    CK_LAUNCH();
    k_tile_chunkscan<<<1, NB, 0, c->stream>>>(chunks, w.tile_sums);
    CK_LAUNCH();
    k_tile_colscan<<<chunks, NB, 0, c->stream>>>(tiles, shift, w.tile_hist, w.tile_sums, w.tile_scan);
    CK_LAUNCH();
    Sort7 s7;
    for (int a = 0; a < 7; ++a) s7.in[a] = arrays[a];
    k_stage_records<NB, TILE><<<tiles, NB, smem, c->stream>>>(n, dest, w.tile_off, w.tile_scan, shift, s7, w.spare, tmpdest);
    CK_LAUNCH();
    c->launches += 5;
    *shift_out = shift;
    return ECSIM_OK;
}

extern "C" int ecsim_sort_particles(ecsim_ctx* c, int s, int32_t* cell_count_out, uint32_t* perm_out)
{
    int rc = check_species(c, s);
    if (rc) return rc;
    SpeciesHost& sp = c->sp[s];
    if (sp.res.on) return ECSIM_ERR_INVALID_ARG;   // resident species keep themselves sorted
    rc = need_workspace(c, sp.n);
    if (rc) return rc;
    Workspace& w = c->ws;
    const uint32_t cells = (uint32_t)c->g.nodes;
    const uint32_t* start = w.start + (size_t)s * (cells + 1);
    rc = histogram_and_scan(c, s, true);
    if (rc) return rc;
    if (sp.n > 0) {
        const uint32_t n = (uint32_t)sp.n;
        const int grid = grid_for(c, (size_t)sp.n, 256, 16);
        double* arrays[7] = {sp.x, sp.y, sp.z, sp.u, sp.v, sp.w, sp.q};
        const size_t nmax = (size_t)w.n_max;
        if (sp.nearly_sorted) {
            // a re-sort after pushes: perm is close to the identity, the gather reads almost sequentially; the seven
            // arrays in one launch (the permutation is read once), then back into the caller's arrays
            k_build_perm<<<grid, 256, 0, c->stream>>>(n, w.cell, w.rank, start, w.perm);
            CK_LAUNCH();
            Move7 mv;
            for (int a = 0; a < 7; ++a) { mv.src[a] = arrays[a]; mv.dst[a] = w.spare + a * nmax; }
            k_gather7<<<grid, 256, 0, c->stream>>>(n, w.perm, mv);
            CK_LAUNCH();
            c->launches += 2;
            for (int a = 0; a < 7; ++a) {
                CK(cudaMemcpyAsync(arrays[a], w.spare + a * nmax, sizeof(double) * (size_t)n, cudaMemcpyDeviceToDevice, c->stream));
                c->launches++;
            }
            if (perm_out)
                CK(cudaMemcpyAsync(perm_out, w.perm, sizeof(uint32_t) * (size_t)n, cudaMemcpyDeviceToDevice, c->stream));
        } else {
            // arbitrary order: the bucketed two-step move of sort.cuh through 64-byte records
            uint32_t* dest = w.rank;                                   // rank -> dest in place
            uint32_t* tmpdest = w.perm;
            int shift = 13;
            rc = n <= SORT_SMALL_MAX_N   ? stage_records<SORT_NB_SMALL, SORT_TILE_SMALL>(c, n, start, dest, arrays, tmpdest, &shift)
                 : n <= SORT_LARGE_MAX_N ? stage_records<SORT_NB_LARGE, SORT_TILE_LARGE>(c, n, start, dest, arrays, tmpdest, &shift)
                                         : stage_records<SORT_NB_HUGE, SORT_TILE_HUGE>(c, n, start, dest, arrays, tmpdest, &shift);
            if (rc) return rc;
            uint32_t* perm2 = w.stray_list + (size_t)s * (size_t)w.n_max;      // (the stray lists are idle during a sort)
            Out7 o7;
            for (int a = 0; a < 7; ++a) o7.dst[a] = arrays[a];
            if (((uint32_t)1 << shift) <= 4u * (uint32_t)INV_SUB) {
                const uint32_t sub = std::min<uint32_t>((uint32_t)1 << shift, (uint32_t)INV_SUB), per_bucket = ((uint32_t)1 << shift) / sub;
                const uint32_t nbk = ((n - 1) >> shift) + 1;
                CK(cudaFuncSetAttribute(k_invert_slots_local, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(INV_SUB * sizeof(uint32_t))));
                k_invert_slots_local<<<nbk * per_bucket, INV_THREADS, sub * sizeof(uint32_t), c->stream>>>(n, shift, tmpdest, perm2);
            } else {
                k_invert_slots<<<grid, 256, 0, c->stream>>>(n, tmpdest, perm2);
            }
            CK_LAUNCH();
            // The two records of a 128-byte line are wanted at unrelated moments while their bucket is in flight: the bytes
            // that pass through L2 in between -- (places of a bucket + places in flight, one per thread) x 120 B -- must stay
            // well inside L2, or the line is fetched twice.  Measured at 33.5 M particles (buckets of 131,072 places): 3 CTAs
            // per SM 0.69 ms and 2.28 GB read, 2 per SM 0.84 ms (too few loads in flight), 4 per SM 0.94 ms and 3.08 GB, 8 per
            // SM 0.84 ms and 3.24 GB; whole multiples of the SM count keep the CTAs abreast.  Buckets too large for that
            // rule (species above ~130 M particles in arbitrary order) run with full occupancy and pay the second fetch.
            int per_sm = 8;
            {
                const size_t budget = ((size_t)32 << 20) / 120, bucket = (size_t)1 << shift;
                const size_t fit = budget > bucket ? (budget - bucket) / (GATHER_WARPS * 32) / (size_t)c->sm_count : 0;
                if (fit >= 2) per_sm = (int)std::min<size_t>(8, fit);
            }
            k_gather_records<<<grid_for(c, ((size_t)n + 31) / 32, GATHER_WARPS, per_sm), GATHER_WARPS * 32, 0, c->stream>>>(
                n, perm2, w.spare, o7, perm_out);
            CK_LAUNCH();
            c->launches += 2;
        }
    }
    if (cell_count_out) {
        k_copy_u32_to_i32<<<grid_for(c, cells, 256, 8), 256, 0, c->stream>>>(cells, w.count, cell_count_out);
        CK_LAUNCH();
        c->launches++;
    }
    sp.state = ST_SEGMENTED;
    sp.nearly_sorted = true;
    sp.stray_debt = 0.0;
    sp.leavers_pending = false;
    return ECSIM_OK;
}

extern "C" int ecsim_cell_index(ecsim_ctx* c, int s, int32_t* cell_out)
{
    int rc = check_species(c, s);
    if (rc) return rc;
    if (!cell_out || c->sp[s].res.on) return ECSIM_ERR_INVALID_ARG;
    SpeciesHost& sp = c->sp[s];
    if (sp.n == 0) return ECSIM_OK;
    k_cell_index<<<grid_for(c, (size_t)sp.n, 256, 16), 256, 0, c->stream>>>(c->g, (uint32_t)sp.n, sp.x, sp.y, sp.z, cell_out);
    CK_LAUNCH();
    c->launches++;
    return ECSIM_OK;
}

// --------------------------------------------------------------------------------------------
// Resident species: library-managed gapped double buffers, sort-preserving push.
static size_t resident_tables_bytes(const ecsim_ctx* c, uint32_t ovf_cap)
{
    const size_t cells = (size_t)c->g.nodes;
    return 2 * align_up(sizeof(uint32_t) * (cells + 1), 256) + 4 * align_up(sizeof(uint32_t) * cells, 256) + 2 * 256 +
           2 * align_up(sizeof(double) * 7 * (size_t)ovf_cap, 256);
}

static uint32_t resident_ovf_cap(int64_t n)
{
    int64_t v = n / 8;
    if (v < 65536) v = 65536;
    return (uint32_t)v;
}

static const uint32_t RESIDENT_MIN_SLACK = 8;

extern "C" size_t ecsim_resident_bytes(const ecsim_ctx* c, int64_t n, double slack)
{
    if (!c || n < 0 || !(slack >= 0.0) || slack > 4.0) return 0;
    const size_t cells = (size_t)c->g.nodes;
    // slots: n + ceil(slack max(n_c, mean)) per cell (<= slack n + slack n) + the minimum slack and the rounding to 4 per cell
    const size_t slots = (size_t)n + 2 * (size_t)ceil(slack * (double)n) + (RESIDENT_MIN_SLACK + 4) * cells + 64;
    return resident_tables_bytes(c, resident_ovf_cap(n)) + 14 * align_up(sizeof(double) * slots, 256);
}

// Bin the dense arrays src (n = sp.n particles, any order) and lay them out, gapped, in buffer dst_buf.
// Synchronises the stream once (the number of slots the layout needs is data dependent and is checked on the host).
static int resident_layout_from_dense(ecsim_ctx* c, int s, const double* const src[7], int dst_buf)
{
    SpeciesHost& sp = c->sp[s];
    Resident& r = sp.res;
    Workspace& w = c->ws;
    const uint32_t cells = (uint32_t)c->g.nodes;
    const uint32_t n = (uint32_t)sp.n;
    int rc = histogram(c, n, src[0], src[1], src[2], true);
    if (rc) return rc;
    const int cgrid = (int)((cells + 255) / 256);
    uint32_t* cap = r.R[dst_buf];              // scratch until the runs are written
    k_gapped_caps<<<cgrid, 256, 0, c->stream>>>(cells, w.count, r.slack, RESIDENT_MIN_SLACK, (double)n / (double)cells, cap);
    CK_LAUNCH();
    c->launches++;
    rc = scan_u32(c, cap, r.seg, cells);
    if (rc) return rc;
    uint32_t total = 0;
    CK(cudaMemcpyAsync(&total, r.seg + cells, sizeof(uint32_t), cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    if (total > r.cap_bound) return ECSIM_ERR_WORKSPACE;
    if (n > 0) {
        Soa7c in; Soa7 out;
        for (int k = 0; k < 7; ++k) { in.a[k] = src[k]; out.a[k] = r.buf[dst_buf][k]; }
        k_scatter_gapped<<<grid_for(c, (size_t)n, 256, 16), 256, 0, c->stream>>>(n, w.cell, w.rank, r.seg, in, out);
        CK_LAUNCH();
        c->launches++;
    }
    k_runs_from_count<<<cgrid, 256, 0, c->stream>>>(cells, w.count, r.F[dst_buf], r.R[dst_buf]);
    CK_LAUNCH();
    c->launches++;
    r.cur = dst_buf;
    return ECSIM_OK;
}

// gapped buffer `cur` -> dense cell-ordered arrays dst[7] (+ the overflow list of the last push behind them)
static int resident_export(ecsim_ctx* c, int s, double* const dst[7], bool with_overflow)
{
    SpeciesHost& sp = c->sp[s];
    Resident& r = sp.res;
    Workspace& w = c->ws;
    const uint32_t cells = (uint32_t)c->g.nodes;
    const int cgrid = (int)((cells + 255) / 256);
    uint32_t* start = w.start + (size_t)s * (cells + 1);   // dense start tables are not used by a resident species
    k_run_totals<<<cgrid, 256, 0, c->stream>>>(cells, r.F[r.cur], r.R[r.cur], w.count);
    CK_LAUNCH();
    c->launches++;
    int rc = scan_u32(c, w.count, start, cells);
    if (rc) return rc;
    Soa7c in; Soa7 out;
    for (int k = 0; k < 7; ++k) { in.a[k] = r.buf[r.cur][k]; out.a[k] = dst[k]; }
    k_export_gapped<<<c->sm_count * 8, 256, 0, c->stream>>>(cells, r.seg, r.F[r.cur], r.R[r.cur], start, in, out);
    CK_LAUNCH();
    c->launches++;
    if (with_overflow) {
        k_append_overflow<<<c->sm_count, 256, 0, c->stream>>>(r.ovf_count[r.ovf_cur], r.ovf_cap, r.ovf[r.ovf_cur], start + cells, out);
        CK_LAUNCH();
        c->launches++;
    }
    return ECSIM_OK;
}

// A fresh layout of a resident species (its overflow list has cost more than this does; or fixPosition moved everybody).
// binned = true: every stored particle is in the cell whose segment holds it (the normal case): only the segments move --
// new capacities from the cells' totals (+ the homeless particles), a new segment table, one cell-by-cell copy into the
// idle buffer (15 GB of traffic at configs[2], ~3 ms) and the homeless particles into their cells' back runs.
// binned = false: export to the idle buffer as dense arrays, bin again, scatter back (three passes).
static int resident_relayout(ecsim_ctx* c, int s, bool binned = true)
{
    SpeciesHost& sp = c->sp[s];
    Resident& r = sp.res;
    Workspace& w = c->ws;
    const int other = 1 - r.cur;
    const uint32_t cells = (uint32_t)c->g.nodes;
    const int cgrid = (int)((cells + 255) / 256);
    int rc;
    if (!binned) {
        rc = resident_export(c, s, r.buf[other], true);
        if (rc) return rc;
        const double* src[7];
        for (int k = 0; k < 7; ++k) src[k] = r.buf[other][k];
        rc = resident_layout_from_dense(c, s, src, r.cur);
        if (rc) return rc;
    } else {
        const double* list = r.ovf[r.ovf_cur];
        const uint32_t* list_n = r.ovf_count[r.ovf_cur];
        k_run_totals<<<cgrid, 256, 0, c->stream>>>(cells, r.F[r.cur], r.R[r.cur], w.count);
        CK_LAUNCH();
        k_count_list<<<c->sm_count * 2, 256, 0, c->stream>>>(c->g, list_n, r.ovf_cap, list, w.count);
        CK_LAUNCH();
        uint32_t* cap = r.R[other];              // scratch until the runs are written
        k_gapped_caps<<<cgrid, 256, 0, c->stream>>>(cells, w.count, r.slack, RESIDENT_MIN_SLACK, (double)sp.n / (double)cells, cap);
        CK_LAUNCH();
        c->launches += 3;
        rc = scan_u32(c, cap, r.seg_alt, cells);
        if (rc) return rc;
        uint32_t total = 0;
        CK(cudaMemcpyAsync(&total, r.seg_alt + cells, sizeof(uint32_t), cudaMemcpyDeviceToHost, c->stream));
        CK(cudaStreamSynchronize(c->stream));
        if (total > r.cap_bound) return ECSIM_ERR_WORKSPACE;
        Soa7c in; Soa7 out;
        for (int k = 0; k < 7; ++k) { in.a[k] = r.buf[r.cur][k]; out.a[k] = r.buf[other][k]; }
        k_copy_gapped<<<c->sm_count * 8, 256, 0, c->stream>>>(cells, r.seg, r.F[r.cur], r.R[r.cur], r.seg_alt, r.F[other], r.R[other], in, out);
        CK_LAUNCH();
        k_place_list<<<c->sm_count * 2, 256, 0, c->stream>>>(c->g, list_n, r.ovf_cap, list, r.seg_alt, r.R[other], out);
        CK_LAUNCH();
        c->launches += 2;
        uint32_t* t = r.seg; r.seg = r.seg_alt; r.seg_alt = t;
        r.cur = other;
    }
    CK(cudaMemsetAsync(r.ovf_count[0], 0, sizeof(uint32_t), c->stream));
    CK(cudaMemsetAsync(r.ovf_count[1], 0, sizeof(uint32_t), c->stream));
    sp.stray_debt = 0.0;
    c->h_ovf[s] = 0;
    c->relayouts++;
    return ECSIM_OK;
}

extern "C" int ecsim_make_resident(ecsim_ctx* c, int s, void* dev_buf, size_t bytes, double slack)
{
    int rc = check_species(c, s);
    if (rc) return rc;
    if (!dev_buf || (reinterpret_cast<uintptr_t>(dev_buf) & 255u) || !(slack >= 0.0) || slack > 4.0)
        return ECSIM_ERR_INVALID_ARG;
    SpeciesHost& sp = c->sp[s];
    rc = need_workspace(c, sp.n);
    if (rc) return rc;
    const size_t cells = (size_t)c->g.nodes;
    Resident r;
    r.slack = slack;
    r.ovf_cap = resident_ovf_cap(sp.n);
    const size_t tables = resident_tables_bytes(c, r.ovf_cap);
    if (bytes < tables + 14 * 256) return ECSIM_ERR_WORKSPACE;
    Carver k{reinterpret_cast<char*>(dev_buf)};
    r.seg = k.take<uint32_t>(cells + 1);
    r.seg_alt = k.take<uint32_t>(cells + 1);
    r.F[0] = k.take<uint32_t>(cells); r.F[1] = k.take<uint32_t>(cells);
    r.R[0] = k.take<uint32_t>(cells); r.R[1] = k.take<uint32_t>(cells);
    r.ovf_count[0] = k.take<uint32_t>(1);
    r.ovf_count[1] = k.take<uint32_t>(1);
    r.ovf[0] = k.take<double>(7 * (size_t)r.ovf_cap);
    r.ovf[1] = k.take<double>(7 * (size_t)r.ovf_cap);
    const size_t per_array = ((bytes - k.off) / 14) & ~(size_t)255;
    size_t slots = per_array / sizeof(double);
    if (slots > 0xfffffff0u) slots = 0xfffffff0u;
    r.cap_bound = (uint32_t)slots;
    for (int b = 0; b < 2; ++b)
        for (int a = 0; a < 7; ++a) r.buf[b][a] = reinterpret_cast<double*>(k.p + k.off + ((size_t)b * 7 + a) * per_array);
    if (sp.state == ST_UNSORTED && !sp.nearly_sorted && sp.n > 0) {
        // arbitrary order: the bucketed sort first, so that the scatter into the gapped layout is sequential
        rc = ecsim_sort_particles(c, s, nullptr, nullptr);
        if (rc) return rc;
    }
    sp.res = r;
    const double* src[7] = {sp.x, sp.y, sp.z, sp.u, sp.v, sp.w, sp.q};
    rc = resident_layout_from_dense(c, s, src, 0);
    if (rc) return rc;
    CK(cudaMemsetAsync(sp.res.ovf_count[0], 0, sizeof(uint32_t), c->stream));
    CK(cudaMemsetAsync(sp.res.ovf_count[1], 0, sizeof(uint32_t), c->stream));
    sp.res.on = true;
    sp.state = ST_SEGMENTED;
    sp.leavers_pending = false;
    sp.stray_debt = 0.0;
    c->h_ovf[s] = 0;
    return ECSIM_OK;
}

// Before a call touches a resident species: the size of its overflow list after its last push (host-visible once that
// push has finished).  Homeless particles cost a stray-kernel warp each per step (homeless.cuh); a fresh layout costs
// about as much as a re-sort: rent or buy, with the same knob as the dense layout (ecsim_set_resort_fraction).
static int resident_settle(ecsim_ctx* c, int s)
{
    SpeciesHost& sp = c->sp[s];
    if (!sp.res.on || !sp.leavers_pending) return ECSIM_OK;
    CK(cudaEventSynchronize(sp.leavers_event));
    sp.leavers_pending = false;
    if (c->h_ovf[s] > sp.res.ovf_cap) {
        // The last push found a cell's segment AND the overflow list full: the particles beyond the list's capacity
        // were not written anywhere in the buffer it filled.  The buffer it READ -- with its run tables and its own
        // overflow list -- is untouched (a gapped push never writes its input), so the push is undone by swapping back:
        // nothing is lost.  A fresh layout of that state gives every cell its slack again, so that the repeated push
        // has room where this one had none.
        const uint32_t wanted = c->h_ovf[s];
        sp.res.cur = 1 - sp.res.cur;
        sp.res.ovf_cur = 1 - sp.res.ovf_cur;
        c->h_ovf[s] = 0;
        const int rrc = resident_relayout(c, s, true);
        if (rrc) return rrc;
        snprintf(g_last_error, sizeof(g_last_error),
                 "resident species %d: its last push needed %u overflow entries, the list holds %u; that push has been "
                 "undone (no particle lost, the species is at its pre-push state, laid out afresh): repeat ecsim_push for "
                 "this species, or make it resident again with more slack", s, wanted, sp.res.ovf_cap);
        return ECSIM_ERR_OVERFLOW;
    }
    sp.stray_debt += (double)c->h_ovf[s];
    if (c->h_ovf[s] > 0 && sp.stray_debt > 0.25 * c->resort_fraction * (double)sp.n) return resident_relayout(c, s, true);   // (a homeless particle costs ~4x a stray)
    return ECSIM_OK;
}

// Lower the capacity of a resident species' overflow list (never above what ecsim_make_resident carved).  The list is
// [7][capacity]: the capacity is also its stride, so it can only change while the list is empty.
extern "C" int ecsim_set_overflow_capacity(ecsim_ctx* c, int s, int64_t entries)
{
    int rc = check_species(c, s);
    if (rc) return rc;
    SpeciesHost& sp = c->sp[s];
    if (!sp.res.on || entries < 1 || entries > (int64_t)resident_ovf_cap(sp.n)) return ECSIM_ERR_INVALID_ARG;
    rc = resident_settle(c, s);
    if (rc) return rc;
    if (c->h_ovf[s] != 0) {
        rc = resident_relayout(c, s, true);            // empties the list into fresh segments
        if (rc) return rc;
    }
    sp.res.ovf_cap = (uint32_t)entries;
    return ECSIM_OK;
}

extern "C" int ecsim_export_particles(ecsim_ctx* c, int s, double* x, double* y, double* z, double* u, double* v,
                                      double* w, double* q)
{
    int rc = check_species(c, s);
    if (rc) return rc;
    SpeciesHost& sp = c->sp[s];
    if (sp.n > 0 && (!x || !y || !z || !u || !v || !w || !q)) return ECSIM_ERR_INVALID_ARG;
    double* dst[7] = {x, y, z, u, v, w, q};
    if (!sp.res.on) {
        double* src[7] = {sp.x, sp.y, sp.z, sp.u, sp.v, sp.w, sp.q};
        for (int k = 0; k < 7; ++k)
            if (dst[k] != src[k])
                CK(cudaMemcpyAsync(dst[k], src[k], sizeof(double) * (size_t)sp.n, cudaMemcpyDeviceToDevice, c->stream));
        return ECSIM_OK;
    }
    rc = resident_settle(c, s);
    if (rc) return rc;
    return resident_export(c, s, dst, true);      // the particles without a slot follow the cell-ordered ones
}

// Number of particles of a dense species the hot path cannot take: non-finite x, v or q, or a position outside [0, L).
// Synchronises the stream.  < 0: an ecsim_status.
extern "C" int64_t ecsim_validate_particles(ecsim_ctx* c, int s)
{
    int rc = check_species(c, s);
    if (rc) return rc;
    SpeciesHost& sp = c->sp[s];
    if (sp.res.on) return ECSIM_ERR_INVALID_ARG;
    rc = need_workspace(c, 0);
    if (rc) return rc;
    if (sp.n == 0) return 0;
    unsigned long long* bad = c->ws.leavers + s;          // (a counter of the workspace that is idle between steps)
    if (cudaMemsetAsync(bad, 0, sizeof(unsigned long long), c->stream) != cudaSuccess) return ECSIM_ERR_CUDA;
    k_validate<<<grid_for(c, (size_t)sp.n, 256, 16), 256, 0, c->stream>>>(c->g, (size_t)sp.n, sp.x, sp.y, sp.z, sp.u, sp.v, sp.w, sp.q, bad);
    if (cudaGetLastError() != cudaSuccess) return ECSIM_ERR_CUDA;
    c->launches += 2;
    unsigned long long h = 0;
    if (cudaMemcpyAsync(&h, bad, sizeof(h), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess) return ECSIM_ERR_CUDA;
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return ECSIM_ERR_CUDA;
    return (int64_t)h;
}

extern "C" int64_t ecsim_relayout_count(const ecsim_ctx* c) { return c ? c->relayouts : 0; }
extern "C" int64_t ecsim_host_pipelined_count(const ecsim_ctx* c) { return c ? c->host_pipelined_calls : 0; }
extern "C" int ecsim_set_host_pipeline(ecsim_ctx* c, int on)
{
    if (!c) return ECSIM_ERR_INVALID_ARG;
    c->host_pipeline = on < 0 ? 0 : (on > 2 ? 2 : on);
    return ECSIM_OK;
}

// --------------------------------------------------------------------------------------------
extern "C" int ecsim_set_variant(ecsim_ctx* c, int variant)
{
    if (!c || (variant != ECSIM_VARIANT_ATOMIC && variant != ECSIM_VARIANT_FUSED)) return ECSIM_ERR_INVALID_ARG;
    c->variant = variant;
    return ECSIM_OK;
}

extern "C" int ecsim_set_resort_fraction(ecsim_ctx* c, double fraction)
{
    if (!c || !(fraction >= 0.0)) return ECSIM_ERR_INVALID_ARG;
    c->resort_fraction = fraction;
    return ECSIM_OK;
}

extern "C" int ecsim_set_fused_warps(ecsim_ctx* c, int warps)
{
    if (!c || (warps != 8 && warps != 12 && warps != 16)) return ECSIM_ERR_INVALID_ARG;
    c->fused_warps = warps;
    return ECSIM_OK;
}

extern "C" int ecsim_set_m_layout(ecsim_ctx* c, int layout)
{
    if (!c || (layout != ECSIM_M_27 && layout != ECSIM_M_14)) return ECSIM_ERR_INVALID_ARG;
    c->m_layout = layout;
    return ECSIM_OK;
}

extern "C" int ecsim_enable_timing(ecsim_ctx* c, int on)
{
    if (!c) return ECSIM_ERR_INVALID_ARG;
    c->timing = on ? 1 : 0;
    c->ev_valid = false;
    return ECSIM_OK;
}

extern "C" int ecsim_kernel_ms(ecsim_ctx* c, float* ms_out)
{
    if (!c || !ms_out) return ECSIM_ERR_INVALID_ARG;
    if (!c->ev_valid) return ECSIM_ERR_NOT_LOADED;
    CK(cudaEventSynchronize(c->ev1));
    CK(cudaEventElapsedTime(ms_out, c->ev0, c->ev1));
    return ECSIM_OK;
}

extern "C" int64_t ecsim_launch_count(const ecsim_ctx* c) { return c ? c->launches : 0; }
extern "C" int64_t ecsim_resort_count(const ecsim_ctx* c) { return c ? c->resorts : 0; }

extern "C" int64_t ecsim_stray_count(ecsim_ctx* c)
{
    if (!c || !c->ws.base || c->last_call_n == 0) return 0;
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return -1;
    int64_t total = 0;
    for (int i = 0; i < c->last_call_n; ++i) total += c->h_strays[c->last_call_species[i]];
    return total;
}

extern "C" int64_t ecsim_leaver_count(ecsim_ctx* c)
{
    if (!c || !c->ws.base || c->last_call_n == 0) return 0;
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return -1;
    int64_t total = 0;
    for (int i = 0; i < c->last_call_n; ++i) total += (int64_t)c->h_leavers[c->last_call_species[i]];
    return total;
}

template <int NW, int REGS, int MODE, int LAYOUT>
static cudaError_t launch_fused(const ecsim_ctx* c, const FusedArgs& fa)
{
    const size_t smem = (size_t)NW * fused_warp_doubles(MODE, LAYOUT) * sizeof(double);
    // per launch, not per process: a second device of the same process needs its own opt-in
    cudaError_t e = cudaFuncSetAttribute(k_fused_push_moments<NW, REGS, MODE, LAYOUT>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const size_t cells = (size_t)(fa.c_end - fa.c_begin);
    size_t grid = (cells + NW - 1) / NW;
    if (grid > (size_t)c->sm_count) grid = (size_t)c->sm_count;
    k_fused_push_moments<NW, REGS, MODE, LAYOUT><<<(int)grid, NW * 32, smem, c->stream>>>(fa);
    return cudaGetLastError();
}

static cudaError_t launch_fused_any(const ecsim_ctx* c, const FusedArgs& fa, int mode, bool gapped)
{
    if (mode == MODE_DIAG)
        return gapped ? launch_fused<16, 128, MODE_DIAG, LAYOUT_GAPPED>(c, fa) : launch_fused<16, 128, MODE_DIAG, LAYOUT_DENSE>(c, fa);
    if (mode == MODE_PUSH)
        return gapped ? launch_fused<16, 128, MODE_PUSH, LAYOUT_GAPPED>(c, fa) : launch_fused<20, 96, MODE_PUSH, LAYOUT_DENSE>(c, fa);
    if (mode == MODE_MOMENTS)
        return gapped ? launch_fused<12, 168, MODE_MOMENTS, LAYOUT_GAPPED>(c, fa) : launch_fused<12, 168, MODE_MOMENTS, LAYOUT_DENSE>(c, fa);
    if (gapped) return launch_fused<12, 168, MODE_FUSED, LAYOUT_GAPPED>(c, fa);
    if (c->fused_warps == 8) return launch_fused<8, 224, MODE_FUSED, LAYOUT_DENSE>(c, fa);
    if (c->fused_warps == 16) return launch_fused<16, 128, MODE_FUSED, LAYOUT_DENSE>(c, fa);
    return launch_fused<12, 168, MODE_FUSED, LAYOUT_DENSE>(c, fa);
}

// Before a pass over the listed species: segment tables (build, or re-sort when too many particles left their cell in
// the last push); resident species: a fresh layout if the last push overflowed.
static int prepare_species(ecsim_ctx* c, int n_list, const int* list, bool gapped)
{
    int rc = ECSIM_OK;
    for (int i = 0; i < n_list; ++i) {
        const int s = list[i];
        SpeciesHost& sp = c->sp[s];
        if (gapped) {
            rc = resident_settle(c, s);
            if (rc) return rc;
            continue;
        }
        if (sp.state == ST_SEGMENTED && sp.leavers_pending) {
            CK(cudaEventSynchronize(sp.leavers_event));
            sp.leavers_pending = false;
            // Rent or buy: a stray costs ~1.4-2.2 ns per step it stays a stray, a re-sort ~54 ps per particle (DESIGN.md
            // §6.2).  Re-sort when the strays handled since the last sort plus those waiting now would have paid for it.
            if (sp.stray_debt + (double)c->h_leavers[s] > c->resort_fraction * (double)sp.n) sp.state = ST_UNSORTED;
            else sp.stray_debt += (double)c->h_leavers[s];
        }
        if (sp.state == ST_UNSORTED) {
            rc = ecsim_sort_particles(c, s, nullptr, nullptr);
            c->resorts++;
        } else if (sp.state == ST_DECLARED) {
            rc = ecsim_build_segments(c, s);
        }
        if (rc) return rc;
    }
    Workspace& w = c->ws;
    CK(cudaMemsetAsync(w.stray_count, 0, sizeof(uint32_t) * c->n_species, c->stream));
    CK(cudaMemsetAsync(w.leavers, 0, sizeof(unsigned long long) * c->n_species, c->stream));
    c->launches += 2;
    return ECSIM_OK;
}

static int fill_fused_args(ecsim_ctx* c, FusedArgs& fa, int n_list, const int* list, const double* E, const double* B,
                           double dt, bool gapped, bool push)
{
    Workspace& w = c->ws;
    const uint32_t cells = (uint32_t)c->g.nodes;
    memset(&fa, 0, sizeof(fa));
    fa.g = c->g; fa.n_species = n_list; fa.E = E; fa.B = B; fa.dt = dt; fa.AM = w.AM;
    fa.c_begin = 0; fa.c_end = cells;
    for (int i = 0; i < n_list; ++i) {
        const int s = list[i];
        SpeciesHost& sp = c->sp[s];
        SpeciesDev& d = fa.sp[i];
        d.beta = sp.qom * dt / 2.0;
        d.n = (uint32_t)sp.n;
        d.AJ = w.AJ + (size_t)s * cells * AJ_PER_CELL;
        d.stray_list = w.stray_list + (size_t)s * (size_t)w.n_max;
        d.stray_count = w.stray_count + s;
        d.leavers = w.leavers + s;
        if (gapped) {
            Resident& r = sp.res;
            double* const* in = r.buf[r.cur];
            double* const* out = r.buf[1 - r.cur];
            d.seg = r.seg; d.Fin = r.F[r.cur]; d.Rin = r.R[r.cur]; d.Fout = r.F[1 - r.cur]; d.Rout = r.R[1 - r.cur];
            d.x = in[0]; d.y = in[1]; d.z = in[2]; d.u = in[3]; d.v = in[4]; d.w = in[5]; d.q = in[6];
            d.ox = out[0]; d.oy = out[1]; d.oz = out[2]; d.ou = out[3]; d.ov = out[4]; d.ow = out[5]; d.oq = out[6];
            d.ovf = r.ovf[1 - r.ovf_cur]; d.ovf_cap = r.ovf_cap; d.ovf_count = r.ovf_count[1 - r.ovf_cur];
            if (push) {
                CK(cudaMemsetAsync(d.Rout, 0, sizeof(uint32_t) * cells, c->stream));
                CK(cudaMemsetAsync(d.ovf_count, 0, sizeof(uint32_t), c->stream));
                c->launches += 2;
            }
        } else {
            d.seg = w.start + (size_t)s * (cells + 1);
            d.x = sp.x; d.y = sp.y; d.z = sp.z; d.u = sp.u; d.v = sp.v; d.w = sp.w; d.q = sp.q;
        }
    }
    return ECSIM_OK;
}

// One pass of the hot path for the listed species.  mode: MODE_FUSED (deposit + push), MODE_MOMENTS (deposit only),
// MODE_PUSH (push only).  rho/J: per listed species (stride given), M shared.
static int step_impl(ecsim_ctx* c, int mode, int n_list, const int* list, const double* E, const double* B,
                     double dt, double theta, double* rho, size_t rho_stride, double* J, size_t J_stride, double* M,
                     int accumulate)
{
    const bool deposit = mode != MODE_PUSH, push = mode != MODE_MOMENTS;
    if (!c || !B || (push && !E) || !(dt > 0.0) || !(theta >= 0.5 && theta <= 1.0)) return ECSIM_ERR_INVALID_ARG;
    for (int i = 0; i < n_list; ++i) {
        int rc = check_species(c, list[i]);
        if (rc) return rc;
    }
    if (accumulate < 0 || accumulate > 2) return ECSIM_ERR_INVALID_ARG;
    const int acc_M = accumulate != ECSIM_ACC_NONE;      // M: summed over species (L59)
    const int acc_J = accumulate == ECSIM_ACC_ALL;       // rho/Jhat: per species unless asked (L129)
    const Geom& g = c->g;
    const size_t nodes = (size_t)g.nodes;
    c->last_call_n = 0;
    int n_resident = 0;
    for (int i = 0; i < n_list; ++i) n_resident += c->sp[list[i]].res.on ? 1 : 0;
    if (n_resident != 0 && n_resident != n_list) return ECSIM_ERR_INVALID_ARG;   // one layout per call
    const bool gapped = n_resident > 0;

    if (c->variant == ECSIM_VARIANT_ATOMIC) {
        // the paper's design: zero the outputs, then one global atomic per scalar contribution
        if (gapped || c->m_layout != ECSIM_M_27) return ECSIM_ERR_INVALID_ARG;
        if (deposit) {
            if (M && !acc_M) { CK(cudaMemsetAsync(M, 0, sizeof(double) * nodes * 243, c->stream)); c->launches++; }
            if (!acc_J) {
                for (int i = 0; i < n_list; ++i) {
                    if (rho) { CK(cudaMemsetAsync(rho + i * rho_stride, 0, sizeof(double) * nodes, c->stream)); c->launches++; }
                    if (J) { CK(cudaMemsetAsync(J + i * J_stride, 0, sizeof(double) * 3 * nodes, c->stream)); c->launches++; }
                }
            }
        }
        if (c->timing) CK(cudaEventRecord(c->ev0, c->stream));
        for (int i = 0; i < n_list; ++i) {
            SpeciesHost& sp = c->sp[list[i]];
            if (sp.n == 0) continue;
            AtomicArgs a;
            a.g = g; a.n = (uint32_t)sp.n; a.list = nullptr; a.list_count = nullptr;
            a.x = sp.x; a.y = sp.y; a.z = sp.z; a.u = sp.u; a.v = sp.v; a.w = sp.w; a.q = sp.q;
            a.E = push ? E : B;            // moments only: E is not used by the deposit (any valid pointer)
            a.B = B; a.beta = sp.qom * dt / 2.0; a.dt = dt;
            a.rho = (deposit && rho) ? rho + i * rho_stride : nullptr;
            a.J = (deposit && J) ? J + i * J_stride : nullptr;
            a.M = deposit ? M : nullptr; a.leavers = nullptr;
            a.do_push = push ? 1 : 0;
            k_push_moments_atomic<false><<<grid_for(c, (size_t)sp.n, 128, 16), 128, 0, c->stream>>>(a);
            CK_LAUNCH();
            c->launches++;
            if (push) sp.state = ST_UNSORTED;
        }
        if (c->timing) { CK(cudaEventRecord(c->ev1, c->stream)); c->ev_valid = true; }
        return ECSIM_OK;
    }

    // ---- fused variant ----
    int64_t n_need = 0;
    for (int i = 0; i < n_list; ++i) n_need = c->sp[list[i]].n > n_need ? c->sp[list[i]].n : n_need;
    int rc = need_workspace(c, n_need);
    if (rc) return rc;
    Workspace& w = c->ws;

    rc = prepare_species(c, n_list, list, gapped);
    if (rc) return rc;
    FusedArgs fa;
    rc = fill_fused_args(c, fa, n_list, list, push ? E : B, B, dt, gapped, push);
    if (rc) return rc;

    if (c->timing) CK(cudaEventRecord(c->ev0, c->stream));
    {
        cudaError_t e = launch_fused_any(c, fa, mode, gapped);
        if (e != cudaSuccess) return cuda_fail(e, "k_fused_push_moments launch", __LINE__);
        c->launches++;
    }
    if (c->timing) { CK(cudaEventRecord(c->ev1, c->stream)); c->ev_valid = true; }

    // resident species: the particles without a slot (overflow list of the last push) -- deposit, push, try again for a slot
    if (gapped) {
        for (int i = 0; i < n_list; ++i) {
            SpeciesHost& sp = c->sp[list[i]];
            Resident& r = sp.res;
            HomelessArgs a;
            a.g = g; a.sp = fa.sp[i]; a.in = r.ovf[r.ovf_cur]; a.in_cap = r.ovf_cap; a.in_count = r.ovf_count[r.ovf_cur];
            a.E = fa.E; a.B = B; a.dt = dt; a.AM = w.AM;
            a.do_deposit = deposit ? 1 : 0; a.do_push = push ? 1 : 0;
            k_push_homeless<<<c->sm_count * 4, STRAY_WARPS * 32, 0, c->stream>>>(a);
            CK_LAUNCH();
            c->launches++;
        }
    }
    // strays (dense layout only): each is added to the per-cell accumulators of its true cell with one bulk reduction
    // (a 2.2 KB block instead of atomics on eight node blocks), then one expansion serves everybody
    if (!gapped) {
        for (int i = 0; i < n_list; ++i) {
            const SpeciesHost& sp = c->sp[list[i]];
            if (sp.n == 0) continue;
            StrayArgs a;
            a.g = g; a.list = fa.sp[i].stray_list; a.list_count = fa.sp[i].stray_count;
            a.x = sp.x; a.y = sp.y; a.z = sp.z; a.u = sp.u; a.v = sp.v; a.w = sp.w; a.q = sp.q;
            a.E = fa.E; a.B = B; a.beta = fa.sp[i].beta; a.dt = dt;
            a.AM = w.AM; a.AJ = fa.sp[i].AJ; a.leavers = fa.sp[i].leavers;
            a.do_deposit = deposit ? 1 : 0; a.do_push = push ? 1 : 0;
            k_push_strays_bulk<<<c->sm_count * 8, STRAY_WARPS * 32, 0, c->stream>>>(a, AM_PER_CELL, AM_A8);
            CK_LAUNCH();
            c->launches++;
        }
    }
    if (deposit) {
        if (M) {
            // one short-lived CTA per (i,j) column of nodes
            ExpandStreamArgs ea{g, w.AM, M, acc_M, 0, g.nx};
            if (c->m_layout == ECSIM_M_14) k_expand_M_stream<14><<<g.nx * g.ny, XS_THREADS, XS_SMEM_BYTES, c->stream>>>(ea);
            else k_expand_M_stream<27><<<g.nx * g.ny, XS_THREADS, XS_SMEM_BYTES, c->stream>>>(ea);
            CK_LAUNCH();
            c->launches++;
        }
        for (int i = 0; i < n_list && (rho || J); ++i) {
            ExpandJArgs ja{g, fa.sp[i].AJ, rho ? rho + i * rho_stride : nullptr, J ? J + i * J_stride : nullptr, acc_J,
                           0, (long long)nodes};
            k_expand_rhoJ<<<(unsigned)((nodes + 255) / 256), 256, 0, c->stream>>>(ja);
            CK_LAUNCH();
            c->launches++;
        }
    }
    for (int i = 0; i < n_list; ++i) {
        const int s = list[i];
        SpeciesHost& sp = c->sp[s];
        CK(cudaMemcpyAsync(c->h_strays + s, w.stray_count + s, sizeof(uint32_t), cudaMemcpyDeviceToHost, c->stream));
        if (push) {
            CK(cudaMemcpyAsync(c->h_leavers + s, w.leavers + s, sizeof(unsigned long long), cudaMemcpyDeviceToHost, c->stream));
            if (gapped) {
                sp.res.cur = 1 - sp.res.cur;            // the species now lives in the buffer just written,
                sp.res.ovf_cur = 1 - sp.res.ovf_cur;    // its homeless particles in the list just written
                CK(cudaMemcpyAsync(c->h_ovf + s, sp.res.ovf_count[sp.res.ovf_cur], sizeof(uint32_t), cudaMemcpyDeviceToHost, c->stream));
            }
            CK(cudaEventRecord(sp.leavers_event, c->stream));
            sp.leavers_pending = true;
        }
        c->last_call_species[c->last_call_n++] = s;
    }
    return ECSIM_OK;
}

static int all_species(const ecsim_ctx* c, int* list)
{
    for (int s = 0; s < c->n_species; ++s) list[s] = s;
    return c->n_species;
}

extern "C" int ecsim_push_and_moments(ecsim_ctx* c, int species, const double* E_theta, const double* B,
                                      double dt, double theta, double* rho, double* Jhat, double* M, int accumulate)
{
    return step_impl(c, MODE_FUSED, 1, &species, E_theta, B, dt, theta, rho, 0, Jhat, 0, M, accumulate);
}

extern "C" int ecsim_push_and_moments_all(ecsim_ctx* c, const double* E_theta, const double* B, double dt,
                                          double theta, double* rho, double* Jhat, double* M, int accumulate)
{
    if (!c) return ECSIM_ERR_INVALID_ARG;
    int list[ECSIM_MAX_SPECIES];
    const int n = all_species(c, list);
    const size_t nodes = (size_t)c->g.nodes;
    return step_impl(c, MODE_FUSED, n, list, E_theta, B, dt, theta, rho, nodes, Jhat, 3 * nodes, M, accumulate);
}

extern "C" int ecsim_moments(ecsim_ctx* c, int species, const double* B, double dt, double* rho, double* Jhat,
                             double* M, int accumulate)
{
    return step_impl(c, MODE_MOMENTS, 1, &species, nullptr, B, dt, 0.5, rho, 0, Jhat, 0, M, accumulate);
}

extern "C" int ecsim_moments_all(ecsim_ctx* c, const double* B, double dt, double* rho, double* Jhat, double* M,
                                 int accumulate)
{
    if (!c) return ECSIM_ERR_INVALID_ARG;
    int list[ECSIM_MAX_SPECIES];
    const int n = all_species(c, list);
    const size_t nodes = (size_t)c->g.nodes;
    return step_impl(c, MODE_MOMENTS, n, list, nullptr, B, dt, 0.5, rho, nodes, Jhat, 3 * nodes, M, accumulate);
}

extern "C" int ecsim_push(ecsim_ctx* c, int species, const double* E_theta, const double* B, double dt, double theta)
{
    return step_impl(c, MODE_PUSH, 1, &species, E_theta, B, dt, theta, nullptr, 0, nullptr, 0, nullptr, ECSIM_ACC_NONE);
}

extern "C" int ecsim_push_all(ecsim_ctx* c, const double* E_theta, const double* B, double dt, double theta)
{
    if (!c) return ECSIM_ERR_INVALID_ARG;
    int list[ECSIM_MAX_SPECIES];
    const int n = all_species(c, list);
    return step_impl(c, MODE_PUSH, n, list, E_theta, B, dt, theta, nullptr, 0, nullptr, 0, nullptr, ECSIM_ACC_NONE);
}

// Diagnostic moments of one species: rho [nodes], un-rotated J [3][nodes], pressure tensor
// P [6][nodes] (xx,xy,xz,yy,yz,zz), heat flux Q [3][nodes]; any may be NULL.  Overwrites.
extern "C" int ecsim_diagnostics(ecsim_ctx* c, int species, double* rho, double* J, double* P, double* Q)
{
    int rc = check_species(c, species);
    if (rc) return rc;
    SpeciesHost& sp = c->sp[species];
    rc = need_workspace(c, sp.n);
    if (rc) return rc;
    const Geom& g = c->g;
    const size_t nodes = (size_t)g.nodes;
    Workspace& w = c->ws;
    c->last_call_n = 0;
    if (c->variant == ECSIM_VARIANT_ATOMIC && !sp.res.on) {
        // the paper's design for these routines too (L147 "#pragma acc atomic update"): every particle through the atomic kernel
        if (rho) CK(cudaMemsetAsync(rho, 0, sizeof(double) * nodes, c->stream));
        if (J) CK(cudaMemsetAsync(J, 0, sizeof(double) * 3 * nodes, c->stream));
        if (P) CK(cudaMemsetAsync(P, 0, sizeof(double) * 6 * nodes, c->stream));
        if (Q) CK(cudaMemsetAsync(Q, 0, sizeof(double) * 3 * nodes, c->stream));
        if (sp.n > 0) {
            k_iota_u32<<<grid_for(c, (size_t)sp.n, 256, 16), 256, 0, c->stream>>>((uint32_t)sp.n, w.perm, w.stray_count + species);
            CK_LAUNCH();
            DiagStrayArgs a{g, w.perm, w.stray_count + species, 0xffffffffu, sp.x, sp.y, sp.z, sp.u, sp.v, sp.w, sp.q, rho, J, P, Q};
            k_diag_strays<<<grid_for(c, (size_t)sp.n, 128, 16), 128, 0, c->stream>>>(a);
            CK_LAUNCH();
            c->launches += 2;
        }
        return ECSIM_OK;
    }
    const bool gapped = sp.res.on;
    rc = prepare_species(c, 1, &species, gapped);
    if (rc) return rc;
    FusedArgs fa;
    rc = fill_fused_args(c, fa, 1, &species, nullptr, nullptr, 1.0, gapped, false);
    if (rc) return rc;
    fa.sp[0].AJ = w.AM;                 // the per-cell corner blocks [cells][8][16] live in the class-sum array (128 <= 244 doubles per cell)
    cudaError_t e = launch_fused_any(c, fa, MODE_DIAG, gapped);
    if (e != cudaSuccess) return cuda_fail(e, "k_fused_push_moments<MODE_DIAG> launch", __LINE__);
    c->launches++;
    ExpandDiagArgs ea{g, w.AM, rho, J, P, Q};
    k_expand_diag<<<(unsigned)((nodes + 255) / 256), 256, 0, c->stream>>>(ea);
    CK_LAUNCH();
    c->launches++;
    if (!gapped && sp.n > 0) {
        DiagStrayArgs a{g, fa.sp[0].stray_list, fa.sp[0].stray_count, 0xffffffffu, sp.x, sp.y, sp.z, sp.u, sp.v, sp.w, sp.q, rho, J, P, Q};
        k_diag_strays<<<c->sm_count * 2, 128, 0, c->stream>>>(a);
        CK_LAUNCH();
        c->launches++;
    }
    if (gapped) {
        // the particles without a slot: straight from the overflow list (list = identity)
        const Resident& r = sp.res;
        const double* o = r.ovf[r.ovf_cur];
        const size_t m = r.ovf_cap;
        DiagStrayArgs a{g, nullptr, r.ovf_count[r.ovf_cur], r.ovf_cap, o, o + m, o + 2 * m, o + 3 * m, o + 4 * m, o + 5 * m, o + 6 * m, rho, J, P, Q};
        k_diag_strays<<<c->sm_count * 2, 128, 0, c->stream>>>(a);
        CK_LAUNCH();
        c->launches++;
    }
    CK(cudaMemcpyAsync(c->h_strays + species, w.stray_count + species, sizeof(uint32_t), cudaMemcpyDeviceToHost, c->stream));
    c->last_call_species[c->last_call_n++] = species;
    return ECSIM_OK;
}

// sum_N' M_NN' E_N' (Eq. 4-5): the operator a field solve applies; M in the context's current layout (27 or 14 slots)
extern "C" int ecsim_apply_M(ecsim_ctx* c, const double* M, const double* E, double* out, int accumulate)
{
    if (!c || !M || !E || !out || E == out) return ECSIM_ERR_INVALID_ARG;
    ApplyMArgs a{c->g, M, E, out, accumulate ? 1 : 0};
    const size_t runs = (size_t)c->g.nx * c->g.ny * (size_t)((c->g.nz + APPLY_RUN - 1) / APPLY_RUN);
    const size_t blocks_needed = (runs + APPLY_WARPS - 1) / APPLY_WARPS;
    size_t grid = (size_t)c->sm_count * 8;
    if (grid > blocks_needed) grid = blocks_needed;
    if (c->m_layout == ECSIM_M_14) k_apply_M<14><<<(int)grid, APPLY_WARPS * 32, 0, c->stream>>>(a);
    else k_apply_M<27><<<(int)grid, APPLY_WARPS * 32, 0, c->stream>>>(a);
    CK_LAUNCH();
    c->launches++;
    return ECSIM_OK;
}

// --------------------------------------------------------------------------------------------
// Host-buffer steps (the end-to-end path): stage in the workspace tail, run, copy back, synchronise.
static size_t m_doubles_per_node(const ecsim_ctx* c) { return c->m_layout == ECSIM_M_14 ? 126 : 243; }

static size_t host_step_extra(const ecsim_ctx* c, int64_t n_total, int n_species_out)
{
    const size_t nodes = (size_t)c->g.nodes;
    return align_up(sizeof(double) * 7 * (size_t)n_total, 256) + align_up(sizeof(double) * 6 * nodes, 256) +
           align_up(sizeof(double) * 4 * nodes * n_species_out, 256) + align_up(sizeof(double) * 243 * nodes, 256);
}

extern "C" size_t ecsim_host_step_workspace_bytes(const ecsim_ctx* c, int64_t n_particles)
{
    if (!c || n_particles < 0) return 0;
    return ecsim_workspace_bytes(c, n_particles) + host_step_extra(c, n_particles, 1);
}

extern "C" size_t ecsim_host_step_all_workspace_bytes(const ecsim_ctx* c, int64_t n_max, int64_t n_total)
{
    if (!c || n_max < 0 || n_total < n_max) return 0;
    return ecsim_workspace_bytes(c, n_max) + host_step_extra(c, n_total, c->n_species);
}


// ---- the pipelined form of the host step ----
// Cell-sorted input: the particles of x-planes [i0, i1) of cells are one contiguous run of every SoA array, so the step
// can be cut into slabs of x-planes and run as a three-stage pipeline on three streams: upload slab k+1 (H2D) | bin + fused
// kernel + expansion of slab k (the caller's stream) | download the pushed particles and the finished node planes of
// slab k-1 (D2H).  PCIe is full duplex, so the two copy directions overlap and the step costs about
// max(bytes in, bytes out) / link instead of their sum.  Node plane i needs cell planes i-1 and i: slab k expands the
// planes (i0, i1) and plane i0 (whose lower cells came with slab k-1); plane 0 waits for the last slab.  One
// cudaMemcpyAsync per array per slab.  Returns 1 ("not applicable: take the serial path", nothing touched yet), 0 on
// success, < 0 on errors -- among them ECSIM_ERR_INVALID_ARG when the arrays are not cell-sorted as declared.
static uint32_t host_lower_bound_plane(const double* hx, uint32_t n, double rdx, int nx, int plane)
{
    uint32_t lo = 0, hi = n;
    while (lo < hi) {
        const uint32_t mid = lo + (hi - lo) / 2;
        int i = (int)floor(hx[mid] * rdx);
        i = i < 0 ? 0 : (i > nx - 1 ? nx - 1 : i);
        if (i >= plane) hi = mid; else lo = mid + 1;
    }
    return lo;
}

static int host_step_pipelined(ecsim_ctx* c, int nsp, const int64_t* n, const double* qom,
                               double* const* hp /* [nsp][7] host arrays */, const double* E_theta, const double* B,
                               double dt, double theta, double* rho, double* Jhat, double* M, bool all_species_call,
                               double* dpart, double* dE, double* dB, double* drho, double* dJ, double* dM)
{
    const Geom& g = c->g;
    const size_t nodes = (size_t)g.nodes, plane = (size_t)g.ny * g.nz;
    int64_t n_total = 0;
    for (int s = 0; s < nsp; ++s) { if (n[s] <= 0) return 1; n_total += n[s]; }
    int slabs = g.nx / 2;
    if (slabs > ECSIM_HOST_SLABS_MAX) slabs = ECSIM_HOST_SLABS_MAX;
    if (c->host_pipeline != 2)                                                    // (2: pipeline whatever the size -- tests)
        while (slabs > 1 && (double)n_total * 56.0 / slabs < 32e6) --slabs;       // slabs of >= 32 MB, else one copy is as good
    if (slabs < 2) return 1;
    Workspace& w = c->ws;
    const uint32_t cells = (uint32_t)nodes;
    const size_t mper = c->m_layout == ECSIM_M_14 ? 126 : 243;
    cudaStream_t st = c->stream, up = c->s_up, down = c->s_down;
    // slab boundaries in every species' arrays (host binary search on the sorted x)
    static thread_local uint32_t P[ECSIM_MAX_SPECIES][ECSIM_HOST_SLABS_MAX + 1];
    int i_lo[ECSIM_HOST_SLABS_MAX + 1];
    for (int k = 0; k <= slabs; ++k) i_lo[k] = (int)((long long)g.nx * k / slabs);
    for (int s = 0; s < nsp; ++s) {
        for (int k = 0; k < slabs; ++k) P[s][k] = host_lower_bound_plane(hp[s * 7], (uint32_t)n[s], g.rdx, g.nx, i_lo[k]);
        P[s][slabs] = (uint32_t)n[s];
        if (P[s][0] != 0) return 1;
    }
    uint32_t* bad = w.stray_count;              // (reused: the dense stray counters are reset below before they matter)
    // device staging layout: species s at dpart + 7 * (particles before it), array a at + a * n[s]
    size_t sp_off[ECSIM_MAX_SPECIES];
    { size_t o = 0; for (int s = 0; s < nsp; ++s) { sp_off[s] = o; o += 7 * (size_t)n[s]; } }
    CK(cudaEventRecord(c->ev_start, st));
    CK(cudaStreamWaitEvent(up, c->ev_start, 0));
    CK(cudaStreamWaitEvent(down, c->ev_start, 0));
    CK(cudaMemcpyAsync(dE, E_theta, sizeof(double) * 3 * nodes, cudaMemcpyHostToDevice, up));
    CK(cudaMemcpyAsync(dB, B, sizeof(double) * 3 * nodes, cudaMemcpyHostToDevice, up));
    CK(cudaEventRecord(c->ev_fields, up));
    CK(cudaStreamWaitEvent(st, c->ev_fields, 0));
    CK(cudaMemsetAsync(w.count, 0, sizeof(uint32_t) * cells, st));
    CK(cudaMemsetAsync(w.stray_count, 0, sizeof(uint32_t) * c->n_species, st));
    CK(cudaMemsetAsync(w.leavers, 0, sizeof(unsigned long long) * c->n_species, st));
    int list[ECSIM_MAX_SPECIES];
    for (int s = 0; s < nsp; ++s) {
        list[s] = s;
        double* d = dpart + sp_off[s];
        const size_t pn = (size_t)n[s];
        int rc = ecsim_load_particles(c, s, n[s], qom[s], d, d + pn, d + 2 * pn, d + 3 * pn, d + 4 * pn, d + 5 * pn, d + 6 * pn, 1);
        if (rc) return rc;
        c->sp[s].state = ST_SEGMENTED;          // the tables are built slab by slab below
    }
    FusedArgs fa;
    int rc = fill_fused_args(c, fa, nsp, list, dE, dB, dt, false, true);
    if (rc) return rc;
    for (int k = 0; k < slabs; ++k) {
        const int i0 = i_lo[k], i1 = i_lo[k + 1];
        const uint32_t c0 = (uint32_t)(i0 * plane), c1 = (uint32_t)(i1 * plane);
        // ---- upload ----
        for (int s = 0; s < nsp; ++s) {
            const size_t p0 = P[s][k], cnt = (size_t)P[s][k + 1] - p0, pn = (size_t)n[s];
            if (!cnt) continue;
            for (int a = 0; a < 7; ++a)
                CK(cudaMemcpyAsync(dpart + sp_off[s] + a * pn + p0, hp[s * 7 + a] + p0, sizeof(double) * cnt, cudaMemcpyHostToDevice, up));
        }
        CK(cudaEventRecord(c->ev_up[k], up));
        // ---- bin, deposit + push, expand ----
        CK(cudaStreamWaitEvent(st, c->ev_up[k], 0));
        for (int s = 0; s < nsp; ++s) {
            const uint32_t p0 = P[s][k], p1 = P[s][k + 1];
            uint32_t* start = w.start + (size_t)s * (cells + 1);
            const double* d = dpart + sp_off[s];
            const size_t pn = (size_t)n[s];
            if (s > 0) CK(cudaMemsetAsync(w.count + c0, 0, sizeof(uint32_t) * (c1 - c0), st));
            if (p1 > p0) {
                k_cell_hist_range<<<grid_for(c, (size_t)(p1 - p0), 256, 16), 256, 0, st>>>(g, p0, p1, d, d + pn, d + 2 * pn, w.count, c0, c1, bad + s);
                CK_LAUNCH();
            }
            rc = scan_u32(c, w.count + c0, start + c0, c1 - c0);
            if (rc) return rc;
            k_add_u32<<<(c1 - c0 + 1 + 255) / 256, 256, 0, st>>>(start + c0, c1 - c0 + 1, p0);
            CK_LAUNCH();
            c->launches += 2;
        }
        fa.c_begin = c0; fa.c_end = c1;
        cudaError_t e = launch_fused_any(c, fa, MODE_FUSED, false);
        if (e != cudaSuccess) return cuda_fail(e, "k_fused_push_moments launch (host pipeline)", __LINE__);
        c->launches++;
        CK(cudaEventRecord(c->ev_comp[k], st));
        const int e0 = k == 0 ? 1 : i0;             // node plane 0 needs the last slab's cells
        if (i1 > e0) {
            if (M) {
                ExpandStreamArgs ea{g, w.AM, dM, 0, e0, i1};
                if (c->m_layout == ECSIM_M_14) k_expand_M_stream<14><<<(i1 - e0) * g.ny, XS_THREADS, XS_SMEM_BYTES, st>>>(ea);
                else k_expand_M_stream<27><<<(i1 - e0) * g.ny, XS_THREADS, XS_SMEM_BYTES, st>>>(ea);
                CK_LAUNCH();
                c->launches++;
            }
            for (int s = 0; s < nsp && (rho || Jhat); ++s) {
                ExpandJArgs ja{g, fa.sp[s].AJ, rho ? drho + (all_species_call ? s * nodes : 0) : nullptr,
                               Jhat ? dJ + (all_species_call ? s * 3 * nodes : 0) : nullptr, 0, (long long)(e0 * plane), (long long)(i1 * plane)};
                k_expand_rhoJ<<<(unsigned)(((size_t)(i1 - e0) * plane + 255) / 256), 256, 0, st>>>(ja);
                CK_LAUNCH();
                c->launches++;
            }
        }
        CK(cudaEventRecord(c->ev_exp[k], st));
        // ---- download ----
        CK(cudaStreamWaitEvent(down, c->ev_comp[k], 0));
        for (int s = 0; s < nsp; ++s) {
            const size_t p0 = P[s][k], cnt = (size_t)P[s][k + 1] - p0, pn = (size_t)n[s];
            if (!cnt) continue;
            for (int a = 0; a < 6; ++a)
                CK(cudaMemcpyAsync(hp[s * 7 + a] + p0, dpart + sp_off[s] + a * pn + p0, sizeof(double) * cnt, cudaMemcpyDeviceToHost, down));
        }
        CK(cudaStreamWaitEvent(down, c->ev_exp[k], 0));
        if (M && i1 > e0)
            CK(cudaMemcpyAsync(M + (size_t)e0 * plane * mper, dM + (size_t)e0 * plane * mper, sizeof(double) * (size_t)(i1 - e0) * plane * mper,
                               cudaMemcpyDeviceToHost, down));
    }
    // node plane 0 (cells of the last and the first plane), then rho / Jhat in one piece
    if (M) {
        ExpandStreamArgs ea{g, w.AM, dM, 0, 0, 1};
        if (c->m_layout == ECSIM_M_14) k_expand_M_stream<14><<<g.ny, XS_THREADS, XS_SMEM_BYTES, st>>>(ea);
        else k_expand_M_stream<27><<<g.ny, XS_THREADS, XS_SMEM_BYTES, st>>>(ea);
        CK_LAUNCH();
        c->launches++;
    }
    for (int s = 0; s < nsp && (rho || Jhat); ++s) {
        ExpandJArgs ja{g, fa.sp[s].AJ, rho ? drho + (all_species_call ? s * nodes : 0) : nullptr,
                       Jhat ? dJ + (all_species_call ? s * 3 * nodes : 0) : nullptr, 0, 0, (long long)plane};
        k_expand_rhoJ<<<(unsigned)((plane + 255) / 256), 256, 0, st>>>(ja);
        CK_LAUNCH();
        c->launches++;
    }
    uint32_t h_bad[ECSIM_MAX_SPECIES] = {};
    CK(cudaMemcpyAsync(h_bad, bad, sizeof(uint32_t) * nsp, cudaMemcpyDeviceToHost, st));
    if (M) CK(cudaMemcpyAsync(M, dM, sizeof(double) * plane * mper, cudaMemcpyDeviceToHost, st));
    const int nout = all_species_call ? nsp : 1;
    if (rho) CK(cudaMemcpyAsync(rho, drho, sizeof(double) * nodes * nout, cudaMemcpyDeviceToHost, st));
    if (Jhat) CK(cudaMemcpyAsync(Jhat, dJ, sizeof(double) * 3 * nodes * nout, cudaMemcpyDeviceToHost, st));
    CK(cudaEventRecord(c->ev_down, down));
    CK(cudaStreamWaitEvent(st, c->ev_down, 0));
    CK(cudaStreamSynchronize(st));
    for (int s = 0; s < nsp; ++s)
        if (h_bad[s]) {
            // (bad and the stray counters share storage: a particle outside the slab its place in the arrays implies, or
            // outside its cell's segment.)  The pushed particles of earlier slabs are already in the caller's arrays:
            // there is no way back to the serial path.
            snprintf(g_last_error, sizeof(g_last_error), "host step: species %d was declared cell-sorted but %u particle(s) "
                     "are out of order; particle arrays are partially advanced", s, h_bad[s]);
            return ECSIM_ERR_INVALID_ARG;
        }
    c->host_pipelined_calls++;
    return ECSIM_OK;
}

// nsp species (slots 0..nsp-1 of the context) from host arrays; rho [nsp][nodes], Jhat [nsp][3][nodes], M shared.
static int host_step_impl(ecsim_ctx* c, int nsp, const int64_t* n, const double* qom, int sorted,
                          double* const* hx, double* const* hy, double* const* hz, double* const* hu,
                          double* const* hv, double* const* hw, const double* const* hq,
                          const double* E_theta, const double* B, double dt, double theta,
                          double* rho, double* Jhat, double* M, int accumulate, bool all_species_call)
{
    int64_t n_max = 0, n_total = 0;
    for (int s = 0; s < nsp; ++s) {
        if (n[s] < 0 || !hx[s] || !hy[s] || !hz[s] || !hu[s] || !hv[s] || !hw[s] || !hq[s]) return ECSIM_ERR_INVALID_ARG;
        n_max = n[s] > n_max ? n[s] : n_max;
        n_total += n[s];
    }
    if (!c->ws.base || c->ws.bytes < ecsim_workspace_bytes(c, n_max) + host_step_extra(c, n_total, nsp))
        return ECSIM_ERR_WORKSPACE;
    // re-carve so that exactly n_max particles are served and the tail is free for staging
    const Workspace keep = c->ws;
    const size_t used = carve(c, n_max, keep.base, &c->ws);
    c->ws.bytes = keep.bytes;
    char* tail = reinterpret_cast<char*>(keep.base) + used;
    const size_t nodes = (size_t)c->g.nodes;
    const size_t mdoubles = m_doubles_per_node(c) * nodes;
    double* dpart = reinterpret_cast<double*>(tail);
    tail += align_up(sizeof(double) * 7 * (size_t)n_total, 256);
    double* dE = reinterpret_cast<double*>(tail);
    double* dB = dE + 3 * nodes;
    tail += align_up(sizeof(double) * 6 * nodes, 256);
    double* drho = reinterpret_cast<double*>(tail);          // [nsp][nodes]
    double* dJ = drho + (size_t)nsp * nodes;                 // [nsp][3][nodes]
    tail += align_up(sizeof(double) * 4 * nodes * nsp, 256);
    double* dM = reinterpret_cast<double*>(tail);
    cudaStream_t st = c->stream;
    // a resident species parked in one of the slots: settle its last push first (restore() below forgets the pending
    // counters, and with them an ECSIM_ERR_OVERFLOW that has not been reported yet)
    for (int s = 0; s < nsp; ++s) {
        const int src = resident_settle(c, s);
        if (src) return src;
    }
    SpeciesHost saved[ECSIM_MAX_SPECIES];
    for (int s = 0; s < nsp; ++s) saved[s] = c->sp[s];

    // every exit goes through `restore`: the caller's species and the full carve come back whatever happened
    auto restore = [&]() {
        for (int s = 0; s < nsp; ++s) {
            cudaEvent_t ev = c->sp[s].leavers_event;
            c->sp[s] = saved[s];
            c->sp[s].leavers_event = ev;
            c->sp[s].leavers_pending = false;
        }
        const size_t used2 = carve(c, keep.n_max, keep.base, &c->ws);
        c->ws.bytes = keep.bytes;
        c->ws.extra = reinterpret_cast<char*>(keep.base) + used2;
        c->ws.extra_bytes = keep.bytes - used2;
        for (int s = 0; s < c->n_species; ++s)
            if (c->sp[s].state == ST_SEGMENTED && !c->sp[s].res.on) c->sp[s].state = ST_DECLARED;   // the tables lived in the re-carved buffer
    };
    auto body = [&]() -> int {
        // (with ecsim_set_fixed_axes active the serial path is taken: its load pins the particles AFTER the upload; the
        // pipeline's load would pin the still empty staging area while slab 0 is on its way)
        if (c->host_pipeline && sorted && accumulate == ECSIM_ACC_NONE && c->variant == ECSIM_VARIANT_FUSED &&
            c->g.fix_mask == 0) {
            double* hp[ECSIM_MAX_SPECIES * 7];
            for (int s = 0; s < nsp; ++s) {
                double* a7[7] = {hx[s], hy[s], hz[s], hu[s], hv[s], hw[s], const_cast<double*>(hq[s])};
                for (int a = 0; a < 7; ++a) hp[s * 7 + a] = a7[a];
            }
            const int prc = host_step_pipelined(c, nsp, n, qom, hp, E_theta, B, dt, theta, rho, Jhat, M, all_species_call,
                                                dpart, dE, dB, drho, dJ, dM);
            if (prc <= 0) return prc;          // done, or failed
            // 1: not applicable (too small, an empty species, plane 0 not first): nothing was touched, go on serially
        }
        double* d = dpart;
        for (int s = 0; s < nsp; ++s) {
            const size_t pn = (size_t)n[s];
            double* hp[7] = {hx[s], hy[s], hz[s], hu[s], hv[s], hw[s], const_cast<double*>(hq[s])};
            for (int a = 0; a < 7; ++a)
                CK(cudaMemcpyAsync(d + a * pn, hp[a], sizeof(double) * pn, cudaMemcpyHostToDevice, st));
            int rc = ecsim_load_particles(c, s, n[s], qom[s], d, d + pn, d + 2 * pn, d + 3 * pn, d + 4 * pn, d + 5 * pn,
                                          d + 6 * pn, sorted);
            if (rc) return rc;
            d += 7 * pn;
        }
        CK(cudaMemcpyAsync(dE, E_theta, sizeof(double) * 3 * nodes, cudaMemcpyHostToDevice, st));
        CK(cudaMemcpyAsync(dB, B, sizeof(double) * 3 * nodes, cudaMemcpyHostToDevice, st));
        if (accumulate == ECSIM_ACC_ALL) {
            if (rho) CK(cudaMemcpyAsync(drho, rho, sizeof(double) * nodes * nsp, cudaMemcpyHostToDevice, st));
            if (Jhat) CK(cudaMemcpyAsync(dJ, Jhat, sizeof(double) * 3 * nodes * nsp, cudaMemcpyHostToDevice, st));
        }
        if (accumulate != ECSIM_ACC_NONE && M)
            CK(cudaMemcpyAsync(dM, M, sizeof(double) * mdoubles, cudaMemcpyHostToDevice, st));
        int list[ECSIM_MAX_SPECIES];
        for (int s = 0; s < nsp; ++s) list[s] = s;
        int rc = step_impl(c, MODE_FUSED, nsp, list, dE, dB, dt, theta, rho ? drho : nullptr, all_species_call ? nodes : 0,
                           Jhat ? dJ : nullptr, all_species_call ? 3 * nodes : 0, M ? dM : nullptr, accumulate);
        if (rc) return rc;
        d = dpart;
        for (int s = 0; s < nsp; ++s) {
            const size_t pn = (size_t)n[s];
            double* hp[6] = {hx[s], hy[s], hz[s], hu[s], hv[s], hw[s]};
            for (int a = 0; a < 6; ++a)
                CK(cudaMemcpyAsync(hp[a], d + a * pn, sizeof(double) * pn, cudaMemcpyDeviceToHost, st));
            d += 7 * pn;
        }
        if (rho) CK(cudaMemcpyAsync(rho, drho, sizeof(double) * nodes * nsp, cudaMemcpyDeviceToHost, st));
        if (Jhat) CK(cudaMemcpyAsync(Jhat, dJ, sizeof(double) * 3 * nodes * nsp, cudaMemcpyDeviceToHost, st));
        if (M) CK(cudaMemcpyAsync(M, dM, sizeof(double) * mdoubles, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        return ECSIM_OK;
    };
    const int rc = body();
    if (rc != ECSIM_OK) {
        // nothing of the failed call may still use the staging area or the caller's host arrays: the pipeline's
        // uploads and downloads run on streams of their own
        cudaStreamSynchronize(st);
        cudaStreamSynchronize(c->s_up);
        cudaStreamSynchronize(c->s_down);
    }
    restore();
    return rc;
}

extern "C" int ecsim_push_and_moments_host(ecsim_ctx* c, int64_t n, double q_over_m, int sorted,
                                           double* x, double* y, double* z, double* u, double* v, double* w,
                                           const double* q, const double* E_theta, const double* B,
                                           double dt, double theta, double* rho, double* Jhat, double* M, int accumulate)
{
    if (!c || !E_theta || !B) return ECSIM_ERR_INVALID_ARG;
    return host_step_impl(c, 1, &n, &q_over_m, sorted, &x, &y, &z, &u, &v, &w, &q, E_theta, B, dt, theta, rho, Jhat, M,
                          accumulate, false);
}

extern "C" int ecsim_push_and_moments_host_all(ecsim_ctx* c, const int64_t* n, const double* q_over_m, int sorted,
                                               double* const* x, double* const* y, double* const* z,
                                               double* const* u, double* const* v, double* const* w,
                                               const double* const* q, const double* E_theta, const double* B,
                                               double dt, double theta, double* rho, double* Jhat, double* M,
                                               int accumulate)
{
    if (!c || !n || !q_over_m || !x || !y || !z || !u || !v || !w || !q || !E_theta || !B) return ECSIM_ERR_INVALID_ARG;
    return host_step_impl(c, c->n_species, n, q_over_m, sorted, x, y, z, u, v, w, q, E_theta, B, dt, theta, rho, Jhat,
                          M, accumulate, true);
}

// --------------------------------------------------------------------------------------------
// Device probes used by bench.py for the roofline denominators (not part of the hot path).
extern "C" int ecsim_probe_fp64(ecsim_ctx* c, int iters, double* tflops_out, float* ms_out)
{
    if (!c || iters < 1 || !tflops_out) return ECSIM_ERR_INVALID_ARG;
    double* sink = nullptr;
    CK(cudaMalloc(&sink, sizeof(double) * 1024));
    const int blocks = c->sm_count * 8, threads = 256;
    k_probe_dfma<<<blocks, threads, 0, c->stream>>>(sink, 16, 1.0);   // warm-up
    CK_LAUNCH();
    CK(cudaEventRecord(c->ev0, c->stream));
    k_probe_dfma<<<blocks, threads, 0, c->stream>>>(sink, iters, 1.0);
    CK_LAUNCH();
    CK(cudaEventRecord(c->ev1, c->stream));
    CK(cudaEventSynchronize(c->ev1));
    float ms = 0.f;
    CK(cudaEventElapsedTime(&ms, c->ev0, c->ev1));
    CK(cudaFree(sink));
    c->ev_valid = false;
    const double flops = 2.0 * PROBE_CHAINS * PROBE_UNROLL * (double)iters * blocks * threads;
    *tflops_out = flops / (ms * 1e-3) * 1e-12;
    if (ms_out) *ms_out = ms;
    return ECSIM_OK;
}

// --------------------------------------------------------------------------------------------
// ecsim_cell_segments_static (ecpush.h): the histogram + exclusive scan of the counting sort for callers that cannot
// obtain device memory -- a plug-in inside a host code whose HBM is handed out once at start-up (OpenACC data regions, a
// framework pool that holds the whole card), or a time loop that must not take the device-wide stall of cudaMalloc /
// cudaFree.  Nothing is allocated here, on either side of the bus: the scratch that the context-based path carves from
// the lent workspace (Workspace::count, Workspace::block_sums) is this file-scope array, part of the library's device
// image, 8.02 MB on every GPU that loads it, until the process exits.
//
// g_static_scratch is a DEVICE symbol.  In the host code below the name is only the host-side handle the runtime
// registers for it; handing `g_static_scratch` itself to a kernel would give the kernel a host address.  The address
// a kernel can use comes from cudaGetSymbolAddress, taken once per device with that device current (each device has
// its own copy of the array at its own address), and that is the only pointer passed on.
constexpr size_t STATIC_SUMS_WORDS = 4096;    // block sums of the scan: ECSIM_STATIC_MAX_CELLS / SCAN_BLOCK + 1 = 2049 used
constexpr size_t STATIC_SCRATCH_WORDS = (size_t)ECSIM_STATIC_MAX_CELLS + STATIC_SUMS_WORDS;
static_assert(ECSIM_STATIC_MAX_CELLS / SCAN_BLOCK + 1 <= STATIC_SUMS_WORDS, "block sums of the largest grid must fit");
static_assert(((size_t)ECSIM_STATIC_MAX_CELLS * sizeof(uint32_t)) % 256 == 0, "block sums start 256-byte aligned");
static __device__ __align__(256) uint32_t g_static_scratch[STATIC_SCRATCH_WORDS];

constexpr int STATIC_MAX_DEVICES = 64;
struct StaticScratchOfDevice {
    uint32_t* dev_ptr = nullptr;   // device address of this device's copy of g_static_scratch
    int sm_count = 0;
};
static StaticScratchOfDevice g_static_of_device[STATIC_MAX_DEVICES];
static std::mutex g_static_mutex;

// Set-up, once per device, with that device current: the device address of the array and the SM count (grid sizing).
// cudaGetSymbolAddress allocates nothing (the array came with the device image); it may load that image, which is why
// the first call on a device belongs outside a stream capture.
static int static_scratch_of_current_device(uint32_t** ptr_out, int* sm_count_out)
{
    int dev = -1;
    CK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) {
        snprintf(g_last_error, sizeof(g_last_error),
                 "ecsim_cell_segments_static: device ordinal %d outside the %d devices this build keeps an address for",
                 dev, STATIC_MAX_DEVICES);
        return ECSIM_ERR_INVALID_ARG;
    }
    std::lock_guard<std::mutex> lock(g_static_mutex);
    StaticScratchOfDevice& d = g_static_of_device[dev];
    if (!d.dev_ptr) {
        int sms = 0;
        CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        uint32_t* p = nullptr;
        CK(cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_static_scratch));
        if (!p || sms < 1) {
            snprintf(g_last_error, sizeof(g_last_error),
                     "ecsim_cell_segments_static: no device address for the built-in scratch on device %d", dev);
            return ECSIM_ERR_CUDA;
        }
        d.sm_count = sms;
        d.dev_ptr = p;             // last: a non-null pointer marks the device as set up
    }
    *ptr_out = d.dev_ptr;
    *sm_count_out = d.sm_count;
    return ECSIM_OK;
}

extern "C" int ecsim_cell_segments_static(void* cuda_stream, int nx, int ny, int nz, double dx, double dy, double dz,
                                          int64_t n, const double* x, const double* y, const double* z,
                                          int32_t* cell_count_out, uint32_t* start_out)
{
    if (nx < 2 || ny < 2 || nz < 2 || !(dx > 0) || !(dy > 0) || !(dz > 0) || n < 0 || n >= 0xffffffffLL)
        return ECSIM_ERR_INVALID_ARG;
    if (n > 0 && (!x || !y || !z)) return ECSIM_ERR_INVALID_ARG;
    if (!cell_count_out && !start_out) return ECSIM_ERR_INVALID_ARG;
    const long long cells_ll = (long long)nx * ny * nz;
    if (cells_ll > (long long)ECSIM_STATIC_MAX_CELLS) {
        // refused before anything is enqueued: the built-in scratch cannot grow
        snprintf(g_last_error, sizeof(g_last_error),
                 "ecsim_cell_segments_static: grid %d x %d x %d = %lld cells exceeds the built-in scratch of "
                 "ECSIM_STATIC_MAX_CELLS = %d cells; use a context with a lent workspace (ecsim_sort_particles) for "
                 "larger grids", nx, ny, nz, cells_ll, (int)ECSIM_STATIC_MAX_CELLS);
        return ECSIM_ERR_INVALID_ARG;
    }
    uint32_t* scratch = nullptr;
    int sm_count = 0;
    int rc = static_scratch_of_current_device(&scratch, &sm_count);
    if (rc) return rc;

    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    const uint32_t cells = (uint32_t)cells_ll;
    uint32_t* count = scratch;                                  // [cells]   histogram
    uint32_t* block_sums = scratch + ECSIM_STATIC_MAX_CELLS;    // [nb + 1]  partial sums of the scan
    Geom g;                                                     // as ecsim_init_grid forms it: same binning, bit for bit
    g.nx = nx; g.ny = ny; g.nz = nz;
    g.dx = dx; g.dy = dy; g.dz = dz;
    g.rdx = 1.0 / dx; g.rdy = 1.0 / dy; g.rdz = 1.0 / dz;
    g.Lx = nx * dx; g.Ly = ny * dy; g.Lz = nz * dz;
    g.invV = 1.0 / (dx * dy * dz);
    g.nodes = cells_ll;
    g.fix_mask = 0;
    g.fix_pos[0] = g.fix_pos[1] = g.fix_pos[2] = 0.0;

    // The array keeps whatever the previous call left in it: the histogram is accumulated with atomics and must start at
    // zero; the block sums are overwritten by k_scan_blocks before they are read and need no clearing.
    CK(cudaMemsetAsync(count, 0, sizeof(uint32_t) * cells, st));
    if (n > 0) {
        size_t blocks = ((size_t)n + 255) / 256;
        const size_t cap = (size_t)sm_count * 16;
        if (blocks > cap) blocks = cap;
        k_cell_hist<false><<<(int)blocks, 256, 0, st>>>(g, (uint32_t)n, x, y, z, nullptr, nullptr, count);
        CK_LAUNCH();
    }
    if (cell_count_out) {
        size_t blocks = ((size_t)cells + 255) / 256;
        const size_t cap = (size_t)sm_count * 16;
        if (blocks > cap) blocks = cap;
        k_copy_u32_to_i32<<<(int)blocks, 256, 0, st>>>(cells, count, cell_count_out);
        CK_LAUNCH();
    }
    if (start_out) {
        const uint32_t nb = (cells + SCAN_BLOCK - 1) / SCAN_BLOCK;
        k_scan_blocks<<<nb, SCAN_BLOCK, 0, st>>>(count, start_out, block_sums, cells);
        CK_LAUNCH();
        k_scan_sums<<<1, SCAN_BLOCK, 0, st>>>(block_sums, nb, start_out, cells);
        CK_LAUNCH();
        k_scan_add<<<nb, SCAN_BLOCK, 0, st>>>(start_out, block_sums, cells);
        CK_LAUNCH();
    }
    return ECSIM_OK;
}
