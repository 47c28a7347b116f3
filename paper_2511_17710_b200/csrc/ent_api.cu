// ent_api.cu -- the C ABI of include/ent.h: context, validation, kernel dispatch.  No torch types anywhere.
#include <cuda_runtime.h>
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>
#include <new>
#include <mutex>

#include "ent_kernels.cuh"
#include "ent_tiled_axisym.cuh"
#include "ent_sorted.cuh"
#include "ent_fields.cuh"

using namespace ent;

struct ent_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    char err[512] = {0};
    bool have_grid = false;
    ent_grid grid{};
    GridDev g{};
    int tile_opt[3] = {0, 0, 0};          // 0 = default
    int step_impl = 0;
    int curv_f64 = 0;                     // ENT_OPT_CURV_FP64
    int pusher = 0;                       // ENT_OPT_PUSHER
    double gca_rho = 0.0, gca_eovb = 0.0; // ent_set_gca
    int sort_mode = 0;                    // 0 auto (re-bin when the input is a sorted block), 1 always the full cell-level sort
    int last_sort_rebin = 0;
    int rebin_ordered = 1;                // re-bin keeps the particles that stay in a tile ordered by cell (Cartesian grids)
    bool ord_attr_set = false;
    long long launches = 0;
    // ---- scratch pool: ONE device allocation carved by reserve_pool(); hot calls never allocate once it is large enough (ent_reserve)
    void *pool = nullptr; size_t pool_bytes = 0;
    long long pool_n = -1;                    // particle count the pool was carved for (-1: none)
    unsigned long long *counters = nullptr;   // [0] bad moves, [1] strays, [2] stray-list length, [3] slot errors, [4] carries, [5] direct global adds
    int32_t *keys = nullptr, *count = nullptr, *offsets = nullptr, *cursor = nullptr, *chunk = nullptr, *class_count = nullptr;
    // side buffers of the non-hot paths (two-kernel step, host-buffer step): allocated on first use
    void *oldbuf = nullptr; size_t oldbuf_cap = 0;
    void *hbuf = nullptr; size_t hbuf_cap = 0;
    void *fbuf = nullptr; size_t fbuf_cap = 0;          // second set of current arrays for the filter passes
    void *cbuf = nullptr; size_t cbuf_cap = 0;          // flags and positions of ent_compact
    cudaStream_t up_stream = nullptr, down_stream = nullptr;   // copy streams of ent_step_host_pair
    cudaEvent_t ev[33] = {};                                    // 2 per sub-block of ent_step_host_pair + 1
    void *sbuf = nullptr; size_t sbuf_cap = 0;          // array-of-structures staging of the full sort (ENT_OPT_SORT_STAGING)
    int sort_staging = 0;
    size_t side_bytes = 0;
    // the blocks ent_sort / ent_step_sorted produced: each keeps its own layout so that several species stay sorted at a time
    struct SortedBlock { const int32_t *cell = nullptr; long long n = -1; int32_t *tile_off = nullptr; float *tile_wmax = nullptr;
                         int32_t *chunk_off = nullptr;      // work list of the tiled kernels (tile_chunk_for(n) particles per CTA)
                         int32_t *next_count = nullptr;     // particles per tile by their CURRENT cell (layout of the next ent_step_sorted output)
                         bool wmax_valid = false, counts_valid = false; unsigned long long stamp = 0; };
    SortedBlock sorted[8];
    unsigned long long sort_stamp = 0;
    int last_step_tiled = 0;
    TiledState tiled{};
};

static int fail(ent_ctx *c, int code, const char *fmt, ...) {
    if (c) {
        va_list ap; va_start(ap, fmt);
        vsnprintf(c->err, sizeof(c->err), fmt, ap);
        va_end(ap);
    }
    return code;
}
#define CK(call)                                                                                         \
    do { cudaError_t e_ = (call);                                                                        \
         if (e_ != cudaSuccess) return fail(ctx, ENT_ECUDA, "%s failed: %s", #call, cudaGetErrorString(e_)); } while (0)

static int launch_check(ent_ctx *ctx, const char *what) {
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(ctx, ENT_ECUDA, "launch of %s failed: %s", what, cudaGetErrorString(e));
    ctx->launches += 1;
    return ENT_OK;
}

// side buffers (non-hot paths): grown on demand; may synchronise the stream
static int ensure(ent_ctx *ctx, void **ptr, size_t *cap_bytes, size_t need) {
    if (*cap_bytes >= need && *ptr) return ENT_OK;
    if (*ptr) { CK(cudaStreamSynchronize(ctx->stream)); CK(cudaFree(*ptr)); ctx->side_bytes -= *cap_bytes; *ptr = nullptr; *cap_bytes = 0; }
    cudaError_t e = cudaMalloc(ptr, need ? need : 16);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(ctx, ENT_ENOMEM, "cudaMalloc of %zu scratch bytes failed: %s", need, cudaGetErrorString(e)); }
    *cap_bytes = need; ctx->side_bytes += need;
    return ENT_OK;
}

// ---- scratch pool --------------------------------------------------------------------------------------------
// Everything ent_sort / ent_step / ent_step_sorted need for blocks of up to n particles on the current grid, in ONE allocation.
struct PoolLayout {
    size_t keys, count, offsets, cursor, chunk, class_count, stray, slots, slot_stride, total;
    long long nkeys, ntiles, stray_cap;
};
static size_t al256(size_t b) { return (b + 255) & ~(size_t)255; }
static PoolLayout pool_layout(const GridDev &g, long long n) {
    PoolLayout L{};
    L.ntiles = (long long)g.nt[0] * g.nt[1] * g.nt[2];
    L.nkeys = L.ntiles * g.tcells;
    L.stray_cap = n / 16 + 4096;
    const size_t nchunks = (size_t)((L.nkeys + 1 + SCAN_CHUNK - 1) / SCAN_CHUNK) + 1;
    size_t off = 0;
    L.keys = off;        off += al256((size_t)(n > 0 ? n : 1) * 4);
    L.count = off;       off += al256((size_t)(L.nkeys + 1) * 4);
    L.offsets = off;     off += al256((size_t)(L.nkeys + 1) * 4);
    L.cursor = off;      off += al256((size_t)(L.nkeys + 1) * 4);
    L.chunk = off;       off += al256(nchunks * 4);
    L.class_count = off; off += al256((size_t)L.ntiles * REBIN_CLASSES * 4);
    L.stray = off;       off += al256((size_t)L.stray_cap * 4);
    L.slots = off;
    L.slot_stride = 4 * al256((size_t)(L.ntiles + 1) * 4);       // tile_off, tile_wmax, chunk_off, next_count
    off += 8 * L.slot_stride;
    L.total = off;
    return L;
}
static void forget_all(ent_ctx *ctx) { for (auto &b : ctx->sorted) { b.cell = nullptr; b.n = -1; } }

// makes the pool large enough for blocks of n particles.  Growing it synchronises the stream, frees and re-allocates (the
// sorted-block registry is lost): call ent_reserve once with the largest block to keep that out of the hot calls.
static int reserve_pool(ent_ctx *ctx, long long n) {
    if (ctx->pool && ctx->pool_n >= n) return ENT_OK;
    const PoolLayout L = pool_layout(ctx->g, n);
    if (ctx->pool) { CK(cudaStreamSynchronize(ctx->stream)); CK(cudaFree(ctx->pool)); ctx->pool = nullptr; ctx->pool_bytes = 0; ctx->pool_n = -1; }
    forget_all(ctx);
    cudaError_t e = cudaMalloc(&ctx->pool, L.total);
    if (e != cudaSuccess) { cudaGetLastError(); ctx->pool = nullptr; return fail(ctx, ENT_ENOMEM, "cudaMalloc of the %zu-byte scratch pool failed: %s", L.total, cudaGetErrorString(e)); }
    ctx->pool_bytes = L.total; ctx->pool_n = n;
    char *b = (char *)ctx->pool;
    ctx->keys = (int32_t *)(b + L.keys); ctx->count = (int32_t *)(b + L.count); ctx->offsets = (int32_t *)(b + L.offsets);
    ctx->cursor = (int32_t *)(b + L.cursor); ctx->chunk = (int32_t *)(b + L.chunk); ctx->class_count = (int32_t *)(b + L.class_count);
    ctx->tiled.stray_list = (int32_t *)(b + L.stray); ctx->tiled.stray_cap = L.stray_cap;
    const size_t part = L.slot_stride / 4;
    for (int k = 0; k < 8; ++k) {
        char *sb = b + L.slots + (size_t)k * L.slot_stride;
        auto &S = ctx->sorted[k];
        S.tile_off = (int32_t *)sb; S.tile_wmax = (float *)(sb + part); S.chunk_off = (int32_t *)(sb + 2 * part);
        S.next_count = (int32_t *)(sb + 3 * part);
    }
    return ENT_OK;
}

extern "C" const char *ent_version(void) { return "0.2"; }

extern "C" const char *ent_last_error(const ent_ctx *ctx) { return ctx ? ctx->err : "null ctx"; }

// ---- scratch of ent_compact_static: lives in the module image, no allocation call ever made for it ------------------------
// Layout = the one ent_compact carves out of its heap buffer: flags, positions, cursor copy ((n + 1) int32 each, 256-byte slots)
// and the chunk sums of the scan.  Every GPU that loads the library holds these bytes until the process exits.
constexpr long long COMPACT_STATIC_MAX_N = ENT_COMPACT_STATIC_MAX_N;
constexpr size_t COMPACT_STATIC_SLOT = ((size_t)(COMPACT_STATIC_MAX_N + 1) * 4 + 255) & ~(size_t)255;
constexpr size_t COMPACT_STATIC_CHUNKS = ((size_t)((COMPACT_STATIC_MAX_N + SCAN_CHUNK - 1) / SCAN_CHUNK) * 4 + 255) & ~(size_t)255;
constexpr size_t COMPACT_STATIC_BYTES = 3 * COMPACT_STATIC_SLOT + COMPACT_STATIC_CHUNKS;       // 12.6 MB for 2^20 particles
static __device__ __align__(256) unsigned char compact_static_scratch[COMPACT_STATIC_BYTES];

// In host code `compact_static_scratch` is a host-side stand-in, NOT a device address: the address the kernels get is looked up
// once per device (that device current) with cudaGetSymbolAddress and kept here.
constexpr int STATIC_MAX_DEVICES = 64;
constexpr long long PAIR_MIN_TILES = 148 * 3;      // ent_step_pair: one CTA per tile needs at least one full wave of tiles
static std::mutex static_scratch_mutex;
static void *static_scratch_addr[STATIC_MAX_DEVICES] = {};
static cudaError_t static_scratch_lookup(int device, void **ptr) {           // the caller has made `device` current
    *ptr = nullptr;
    if (device < 0 || device >= STATIC_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(static_scratch_mutex);
    if (!static_scratch_addr[device]) {
        void *a = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&a, compact_static_scratch);
        if (e != cudaSuccess) { cudaGetLastError(); return e; }
        static_scratch_addr[device] = a;
    }
    *ptr = static_scratch_addr[device];
    return cudaSuccess;
}

extern "C" int ent_create(ent_ctx **out, int device, void *cuda_stream) {
    if (!out) return ENT_EINVAL;
    *out = nullptr;
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev <= 0 || device < 0 || device >= ndev) { cudaGetLastError(); return ENT_ECUDA; }   // no CPU fallback
    if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return ENT_ECUDA; }
    ent_ctx *ctx = new (std::nothrow) ent_ctx();
    if (!ctx) return ENT_ENOMEM;
    ctx->device = device;
    ctx->stream = (cudaStream_t)cuda_stream;
    if (cudaMalloc((void **)&ctx->counters, 8 * sizeof(unsigned long long)) != cudaSuccess ||
        cudaMemsetAsync(ctx->counters, 0, 8 * sizeof(unsigned long long), ctx->stream) != cudaSuccess) {
        cudaGetLastError(); delete ctx; return ENT_ECUDA;
    }
    { void *unused; (void)static_scratch_lookup(device, &unused); }   // set-up of ent_compact_static; a failure is reported by that call
    *out = ctx;
    return ENT_OK;
}

extern "C" int ent_destroy(ent_ctx *ctx) {
    if (!ctx) return ENT_EINVAL;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    cudaFree(ctx->counters); cudaFree(ctx->pool); cudaFree(ctx->oldbuf); cudaFree(ctx->hbuf); cudaFree(ctx->fbuf); cudaFree(ctx->cbuf); cudaFree(ctx->sbuf);
    if (ctx->up_stream) { cudaStreamDestroy(ctx->up_stream); cudaStreamDestroy(ctx->down_stream); for (auto &e : ctx->ev) cudaEventDestroy(e); }
    cudaGetLastError();
    delete ctx;
    return ENT_OK;
}

// ---- grid --------------------------------------------------------------------------------------------------
extern "C" int ent_set_grid(ent_ctx *ctx, const ent_grid *gr) {
    if (!ctx) return ENT_EINVAL;
    if (!gr) return fail(ctx, ENT_EINVAL, "grid is NULL");
    if (gr->D != 2 && gr->D != 3) return fail(ctx, ENT_EINVAL, "D = %d, must be 2 or 3", gr->D);
    if (gr->kind != ENT_CART && gr->kind != ENT_SPH && gr->kind != ENT_QSPH) return fail(ctx, ENT_EINVAL, "unknown metric kind %d", gr->kind);
    const int D = gr->D;
    long long ncell = 1;
    for (int a = 0; a < D; ++a) {
        if (gr->N[a] < 1) return fail(ctx, ENT_EINVAL, "N[%d] = %d", a, gr->N[a]);
        if (gr->bc[a] != ENT_PERIODIC && gr->bc[a] != ENT_ABSORB && gr->bc[a] != ENT_AXIS) return fail(ctx, ENT_EINVAL, "bc[%d] = %d", a, gr->bc[a]);
        if (gr->bc[a] == ENT_PERIODIC && gr->N[a] < 3) return fail(ctx, ENT_EINVAL, "periodic dimension %d needs N >= 3 (|delta i| <= 1 would be ambiguous)", a);
        if (!(gr->xmax[a] > gr->xmin[a])) return fail(ctx, ENT_EINVAL, "xmax[%d] <= xmin[%d]", a, a);
        ncell *= gr->N[a];
        if (ncell >= (1LL << 31)) return fail(ctx, ENT_EINVAL, "more than 2^31 - 1 cells: the packed int32 cell index would overflow");
    }
    if (gr->kind != ENT_CART) {
        if (D != 2) return fail(ctx, ENT_EUNSUPPORTED, "SPH/QSPH metrics are axisymmetric: D must be 2");
        if (gr->bc[0] != ENT_ABSORB || gr->bc[1] != ENT_AXIS) return fail(ctx, ENT_EUNSUPPORTED, "SPH/QSPH need bc = {ABSORB, AXIS}");
        if (gr->kind == ENT_QSPH) {
            if (!(gr->xmin[0] > gr->r0)) return fail(ctx, ENT_EINVAL, "QSPH needs xmin[0] > r0");
            if (!(gr->vartheta >= 0.0 && gr->vartheta < 1.0)) return fail(ctx, ENT_EINVAL, "QSPH needs 0 <= vartheta < 1");
        } else if (!(gr->xmin[0] >= 0.0)) return fail(ctx, ENT_EINVAL, "SPH needs rmin >= 0");
    } else {
        for (int a = 0; a < D; ++a) if (gr->bc[a] == ENT_AXIS) return fail(ctx, ENT_EUNSUPPORTED, "AXIS boundary on a Cartesian grid");
    }
    GridDev g{};
    g.D = D; g.kind = gr->kind;
    const int deft[2][3] = { {16, 16, 1}, {8, 8, 8} };
    long long pad = 1;
    for (int a = 0; a < 3; ++a) {
        bool on = a < D;
        g.N[a] = on ? gr->N[a] : 1;
        g.P[a] = on ? gr->N[a] + 2 * NG : 1;
        g.bc[a] = on ? gr->bc[a] : ENT_PERIODIC;
        int T = on ? (ctx->tile_opt[a] > 0 ? ctx->tile_opt[a] : deft[D - 2][a]) : 1;
        if (T > g.N[a]) T = g.N[a];
        g.T[a] = T;
        g.nt[a] = (g.N[a] + T - 1) / T;
        double dx = on ? (gr->xmax[a] - gr->xmin[a]) / (double)gr->N[a] : 1.0;
        g.dx[a] = (float)dx; g.inv_dx[a] = (float)(1.0 / dx);
        pad *= g.P[a];
    }
    if (pad >= (1LL << 31)) return fail(ctx, ENT_EINVAL, "padded array has more than 2^31 - 1 elements");
    g.tcells = g.T[0] * g.T[1] * g.T[2];
    long long nkeys = (long long)g.nt[0] * g.nt[1] * g.nt[2] * g.tcells;
    if (nkeys >= (1LL << 31)) return fail(ctx, ENT_EINVAL, "sort key space exceeds int32");
    if (gr->kind == ENT_SPH) {
        g.rmin = gr->xmin[0]; g.dr = (gr->xmax[0] - gr->xmin[0]) / gr->N[0]; g.dth = PI_D / gr->N[1];
    } else if (gr->kind == ENT_QSPH) {
        g.r0 = gr->r0; g.vt = gr->vartheta;
        g.Rmin = log(gr->xmin[0] - gr->r0);
        g.dR = (log(gr->xmax[0] - gr->r0) - g.Rmin) / gr->N[0];
        g.dT = PI_D / gr->N[1];
    }
    g.rminf = (float)g.rmin; g.drf = (float)g.dr; g.dthf = (float)g.dth; g.Rminf = (float)g.Rmin; g.dRf = (float)g.dR; g.dTf = (float)g.dT;
    g.r0f = (float)g.r0; g.vtf = (float)g.vt; g.curv_f64 = ctx->curv_f64; g.pusher = ctx->pusher; g.gca_c = 0.f; g.gca_eovb2 = (float)(ctx->gca_eovb * ctx->gca_eovb);
    ctx->grid = *gr; ctx->g = g; ctx->have_grid = true;
    forget_all(ctx);
    if (ctx->pool) {                                            // the pool was carved for the previous grid
        CK(cudaStreamSynchronize(ctx->stream)); CK(cudaFree(ctx->pool));
        ctx->pool = nullptr; ctx->pool_bytes = 0; ctx->pool_n = -1; ctx->tiled.stray_list = nullptr; ctx->tiled.stray_cap = 0;
    }
    return tiled_set_grid(ctx->tiled, g, ctx->err, sizeof(ctx->err));
}

// ---- argument checks ---------------------------------------------------------------------------------------
static bool al16(const void *p) { return (((uintptr_t)p) & 15u) == 0; }

static int check_particles(ent_ctx *ctx, const ent_particles *p, const char *name, bool need_tag_if_absorb) {
    if (!p) return fail(ctx, ENT_EINVAL, "%s is NULL", name);
    if (p->n < 0) return fail(ctx, ENT_EINVAL, "%s->n < 0", name);
    if (p->n >= (1LL << 31)) return fail(ctx, ENT_EINVAL, "%s->n >= 2^31 (sort offsets are int32)", name);
    if (p->n == 0) return ENT_OK;                         // an empty block needs no arrays
    const GridDev &g = ctx->g;
    if (!p->cell || !al16(p->cell)) return fail(ctx, ENT_EINVAL, "%s->cell NULL or not 16-byte aligned", name);
    for (int a = 0; a < g.D; ++a) if (!p->d[a] || !al16(p->d[a])) return fail(ctx, ENT_EINVAL, "%s->d[%d] NULL or misaligned", name, a);
    for (int a = 0; a < 3; ++a) if (!p->u[a] || !al16(p->u[a])) return fail(ctx, ENT_EINVAL, "%s->u[%d] NULL or misaligned", name, a);
    if (!p->w || !al16(p->w)) return fail(ctx, ENT_EINVAL, "%s->w NULL or misaligned", name);
    if (g.kind != ENT_CART && (!p->phi || !al16(p->phi))) return fail(ctx, ENT_EINVAL, "%s->phi NULL or misaligned on an axisymmetric grid", name);
    if (p->tag && !al16(p->tag)) return fail(ctx, ENT_EINVAL, "%s->tag misaligned", name);
    if (need_tag_if_absorb && !p->tag)
        for (int a = 0; a < g.D; ++a) if (g.bc[a] == ENT_ABSORB) return fail(ctx, ENT_EINVAL, "%s->tag is NULL but dimension %d is ABSORB", name, a);
    return ENT_OK;
}
static int check_fields(ent_ctx *ctx, const ent_fields *F) {
    if (!F) return fail(ctx, ENT_EINVAL, "fields struct is NULL");
    for (int c = 0; c < 6; ++c) if (!F->comp[c] || !al16(F->comp[c])) return fail(ctx, ENT_EINVAL, "field component %d NULL or misaligned", c);
    return ENT_OK;
}
static int check_current(ent_ctx *ctx, const ent_current *J) {
    if (!J) return fail(ctx, ENT_EINVAL, "current struct is NULL");
    for (int c = 0; c < 3; ++c) if (!J->comp[c] || !al16(J->comp[c])) return fail(ctx, ENT_EINVAL, "current component %d NULL or misaligned", c);
    return ENT_OK;
}
static void forget_block(ent_ctx *ctx, const int32_t *cell) { for (auto &b : ctx->sorted) if (b.cell == cell) { b.cell = nullptr; b.n = -1; } }
static ent_ctx::SortedBlock *find_block(ent_ctx *ctx, const ent_particles *p) {
    if (!p->cell || p->n <= 0) return nullptr;
    for (auto &b : ctx->sorted) if (b.cell == p->cell && b.n == p->n) return &b;
    return nullptr;
}
static PartPtrs pp(const ent_particles *p) {
    PartPtrs r;
    r.cell = p->cell; for (int a = 0; a < 3; ++a) { r.d[a] = p->d[a]; r.u[a] = p->u[a]; }
    r.phi = p->phi; r.w = p->w; r.tag = p->tag;
    return r;
}
static FieldPtrs fp(const ent_fields *F) { FieldPtrs r; for (int c = 0; c < 6; ++c) r.c[c] = F->comp[c]; return r; }
static CurrentPtrs cp(const ent_current *J) { CurrentPtrs r; for (int c = 0; c < 3; ++c) r.c[c] = J->comp[c]; return r; }
static unsigned nblk(long long n) { return (unsigned)((n + TPB - 1) / TPB); }

#define ENTER()                                                                              \
    if (!ctx) return ENT_EINVAL;                                                             \
    if (!ctx->have_grid) return fail(ctx, ENT_EINVAL, "ent_set_grid has not been called");   \
    CK(cudaSetDevice(ctx->device))

// dispatch on (D, kind): the four supported combinations
#define DISPATCH(KERNEL, GRID, ...)                                                                          \
    do {                                                                                                     \
        const GridDev &g_ = ctx->g;                                                                          \
        if (g_.kind == ENT_CART && g_.D == 2) KERNEL<2, ENT_CART><<<GRID, TPB, 0, ctx->stream>>>(__VA_ARGS__); \
        else if (g_.kind == ENT_CART) KERNEL<3, ENT_CART><<<GRID, TPB, 0, ctx->stream>>>(__VA_ARGS__);        \
        else if (g_.kind == ENT_SPH) KERNEL<2, ENT_SPH><<<GRID, TPB, 0, ctx->stream>>>(__VA_ARGS__);          \
        else KERNEL<2, ENT_QSPH><<<GRID, TPB, 0, ctx->stream>>>(__VA_ARGS__);                                 \
    } while (0)

// ---- the calls ---------------------------------------------------------------------------------------------
extern "C" int ent_gather_push(ent_ctx *ctx, const ent_fields *EB, const ent_particles *in, ent_particles *out, float dt) {
    ENTER();
    int rc;
    if ((rc = check_fields(ctx, EB)) || (rc = check_particles(ctx, in, "in", false)) || (rc = check_particles(ctx, out, "out", true))) return rc;
    if (in->n != out->n) return fail(ctx, ENT_EINVAL, "in->n != out->n");
    if (!(in->m != 0.f)) return fail(ctx, ENT_EINVAL, "mass is zero");
    if (in->n == 0) return ENT_OK;
    forget_block(ctx, out->cell);                             // `out` is overwritten: it is no longer a sorted block
    ctx->g.gca_c = (float)(2.0 * ctx->gca_rho / (double)dt);      // hybrid pusher: rho_crit q/m = gca_c * eps
    float eps = 0.5f * (in->q / in->m) * dt;
    DISPATCH(gather_push_kernel, nblk(in->n), ctx->g, fp(EB), pp(in), pp(out), (long long)in->n, eps, dt);
    return launch_check(ctx, "gather_push_kernel");
}

extern "C" int ent_deposit(ent_ctx *ctx, const ent_particles *po, const ent_particles *pn, ent_current *J, float dt) {
    ENTER();
    int rc;
    if ((rc = check_current(ctx, J)) || (rc = check_particles(ctx, po, "old", false)) || (rc = check_particles(ctx, pn, "new", false))) return rc;
    if (po->n != pn->n) return fail(ctx, ENT_EINVAL, "old->n != new->n");
    if (!(dt > 0.f)) return fail(ctx, ENT_EINVAL, "dt must be positive");
    ctx->g.gca_c = (float)(2.0 * ctx->gca_rho / (double)dt);      // hybrid pusher: rho_crit q/m = gca_c * eps
    if (po->n == 0) return ENT_OK;
    DISPATCH(deposit_kernel, nblk(po->n), ctx->g, pp(po), pp(pn), cp(J), (long long)po->n, po->q, 1.0f / dt, ctx->counters + 0);
    return launch_check(ctx, "deposit_kernel");
}

extern "C" int ent_zero_current(ent_ctx *ctx, ent_current *J) {
    ENTER();
    int rc;
    if ((rc = check_current(ctx, J))) return rc;
    size_t bytes = (size_t)padded_size(ctx->g) * sizeof(float);
    for (int c = 0; c < 3; ++c) CK(cudaMemsetAsync(J->comp[c], 0, bytes, ctx->stream));
    return ENT_OK;
}

extern "C" int ent_fold_current(ent_ctx *ctx, ent_current *J) {
    ENTER();
    int rc;
    if ((rc = check_current(ctx, J))) return rc;
    const GridDev &g = ctx->g;
    // all ghost layers are added onto the active cells (dimension after dimension, so that edges and corners arrive), then
    // all ghost layers are refilled; the three components are independent and share a launch
    for (int pass = 0; pass < 2; ++pass)
        for (int d = 0; d < g.D; ++d) {
            if (g.bc[d] != ENT_PERIODIC) continue;
            long long nthreads = (long long)g.P[(d + 1) % 3] * g.P[(d + 2) % 3] * NG;
            fold_kernel<<<dim3(nblk(nthreads), 3), TPB, 0, ctx->stream>>>(g, cp(J), d, pass);
            if ((rc = launch_check(ctx, "fold_kernel"))) return rc;
        }
    return ENT_OK;
}

// step 9: npasses digital filter passes (Eqs. 9-11) + optional J = conformal J / sqrt(h)
extern "C" int ent_filter_current(ent_ctx *ctx, ent_current *J, int npasses, int divide_by_sqrt_h) {
    ENTER();
    int rc;
    if ((rc = check_current(ctx, J))) return rc;
    if (npasses < 0 || npasses > 1024) return fail(ctx, ENT_EINVAL, "npasses out of range");
    if (npasses == 0 && !divide_by_sqrt_h) return ENT_OK;
    const GridDev &g = ctx->g;
    const size_t slot = ((size_t)padded_size(g) * 4 + 255) & ~(size_t)255;
    if ((rc = ensure(ctx, &ctx->fbuf, &ctx->fbuf_cap, 3 * slot))) return rc;
    FilterGeom L;
    int nmax[3] = { 1, 1, 1 };
    for (int d = 0; d < 3; ++d) L.rule[d] = d < g.D ? g.bc[d] : ENT_PERIODIC;
    for (int c = 0; c < 3; ++c)
        for (int d = 0; d < 3; ++d) {
            int n = 1;
            if (d < g.D) n = g.bc[d] == ENT_PERIODIC ? g.N[d] : (c == d ? g.N[d] : g.N[d] + 1);       // half-integer / integer lattice
            L.n[c][d] = n;
            if (n > nmax[d]) nmax[d] = n;
        }
    CurrentPtrs a = cp(J), b;
    for (int c = 0; c < 3; ++c) b.c[c] = (float *)((char *)ctx->fbuf + slot * c);
    const int nkc = (nmax[2] + FT_K - 1) / FT_K;
    const dim3 fgrid((nmax[0] + FT_W - 1) / FT_W, (nmax[1] + FT_ROWS - 1) / FT_ROWS, 3 * nkc);
    if (fgrid.y > 65535u || fgrid.z > 65535u) return fail(ctx, ENT_EUNSUPPORTED, "grid too large for the filter kernel");
    const int total = npasses ? npasses : 1;
    for (int pass = 0; pass < total; ++pass) {
        const bool last = pass == total - 1;
        filter_pass_kernel<<<fgrid, FT_TPB, 0, ctx->stream>>>(g, L, (pass & 1) ? b : a, (pass & 1) ? a : b, npasses == 0 ? 1 : 0, last && divide_by_sqrt_h, nkc);
        if ((rc = launch_check(ctx, "filter_pass_kernel"))) return rc;
    }
    if (total & 1) {                                         // the result sits in the scratch arrays: copy the lattice points back
        filter_pass_kernel<<<fgrid, FT_TPB, 0, ctx->stream>>>(g, L, b, a, 2, 0, nkc);
        if ((rc = launch_check(ctx, "filter_pass_kernel"))) return rc;
    }
    return ENT_OK;
}

// ---- N2: field solver (sub-steps 2, 10, 11; Eqs. A1, A2, 12, 13) and the ghost fill of the field arrays ----
static int check_fields_rw(ent_ctx *ctx, const ent_fields_rw *F) {
    if (!F) return fail(ctx, ENT_EINVAL, "fields struct is NULL");
    for (int c = 0; c < 6; ++c) if (!F->comp[c] || !al16(F->comp[c])) return fail(ctx, ENT_EINVAL, "field component %d NULL or misaligned", c);
    return ENT_OK;
}
static SolverGeom solver_geom(const GridDev &g) {
    SolverGeom L;
    L.axis = -1;
    for (int d = 0; d < 3; ++d) { L.nmax[d] = 1; if (d < g.D && g.bc[d] == ENT_AXIS) L.axis = d; }
    for (int c6 = 0; c6 < 6; ++c6)
        for (int d = 0; d < 3; ++d) {
            int n = 1;
            if (d < g.D) n = g.bc[d] == ENT_PERIODIC ? g.N[d] : (fld_stag(c6, d) ? g.N[d] : g.N[d] + 1);
            L.n[c6][d] = n;
            if (n > L.nmax[d]) L.nmax[d] = n;
        }
    const double sh = (double)g.dx[0] * g.dx[1] * g.dx[2];
    for (int c = 0; c < 3; ++c) L.cov[c] = g.dx[c] * g.dx[c];
    L.inv_sqrt_h = (float)(1.0 / sh);
    return L;
}
static bool all_periodic_cart(const GridDev &g) {
    if (g.kind != ENT_CART) return false;
    for (int d = 0; d < g.D; ++d) if (g.bc[d] != ENT_PERIODIC) return false;
    return true;
}
static FieldRW frw(const ent_fields_rw *F) { FieldRW r; for (int c = 0; c < 6; ++c) r.c[c] = F->comp[c]; return r; }
static int solver_grid(ent_ctx *ctx, const SolverGeom &L, dim3 *grid) {
    *grid = dim3((unsigned)((L.nmax[0] + TPB - 1) / TPB), (unsigned)L.nmax[1], (unsigned)(3 * L.nmax[2]));
    if (grid->y > 65535u || grid->z > 65535u) return fail(ctx, ENT_EUNSUPPORTED, "grid too large for the field-solver kernels");
    return ENT_OK;
}

extern "C" int ent_faraday(ent_ctx *ctx, ent_fields_rw *EB, float dt) {
    ENTER();
    int rc;
    if ((rc = check_fields_rw(ctx, EB))) return rc;
    const GridDev &g = ctx->g;
    const SolverGeom L = solver_geom(g);
    dim3 grid;
    if ((rc = solver_grid(ctx, L, &grid))) return rc;
    if (all_periodic_cart(g)) faraday_cart_kernel<<<dim3(grid.x, (unsigned)g.N[1], (unsigned)g.N[2]), TPB, 0, ctx->stream>>>(g, L, frw(EB), dt);
    else if (g.kind == ENT_CART) faraday_kernel<true><<<grid, TPB, 0, ctx->stream>>>(g, L, frw(EB), dt);
    else faraday_kernel<false><<<grid, TPB, 0, ctx->stream>>>(g, L, frw(EB), dt);
    return launch_check(ctx, "faraday_kernel");
}

extern "C" int ent_ampere(ent_ctx *ctx, ent_fields_rw *EB, const ent_current *J, float dt, float j_coeff) {
    ENTER();
    int rc;
    if ((rc = check_fields_rw(ctx, EB))) return rc;
    if (J && (rc = check_current(ctx, J))) return rc;
    const GridDev &g = ctx->g;
    const SolverGeom L = solver_geom(g);
    dim3 grid;
    if ((rc = solver_grid(ctx, L, &grid))) return rc;
    CurrentPtrs j; for (int c = 0; c < 3; ++c) j.c[c] = J ? J->comp[c] : nullptr;
    if (all_periodic_cart(g)) ampere_cart_kernel<<<dim3(grid.x, (unsigned)g.N[1], (unsigned)g.N[2]), TPB, 0, ctx->stream>>>(g, L, frw(EB), j, J != nullptr, dt, j_coeff);
    else if (g.kind == ENT_CART) ampere_kernel<true><<<grid, TPB, 0, ctx->stream>>>(g, L, frw(EB), j, J != nullptr, dt, j_coeff);
    else ampere_kernel<false><<<grid, TPB, 0, ctx->stream>>>(g, L, frw(EB), j, J != nullptr, dt, j_coeff);
    return launch_check(ctx, "ampere_kernel");
}

extern "C" int ent_fill_field_ghosts(ent_ctx *ctx, ent_fields_rw *EB) {
    ENTER();
    int rc;
    if ((rc = check_fields_rw(ctx, EB))) return rc;
    const GridDev &g = ctx->g;
    const SolverGeom L = solver_geom(g);
    for (int d = 0; d < g.D; ++d) {
        if (g.bc[d] == ENT_ABSORB) continue;
        const long long nthreads = (long long)g.P[(d + 1) % 3] * g.P[(d + 2) % 3] * 2 * NG;
        field_ghost_kernel<<<dim3(nblk(nthreads), 6), TPB, 0, ctx->stream>>>(g, L, frw(EB), d);
        if ((rc = launch_check(ctx, "field_ghost_kernel"))) return rc;
    }
    return ENT_OK;
}

static int step_two_kernel(ent_ctx *ctx, const ent_fields *EB, ent_particles *p, ent_current *J, float dt) {
    // the paper's structure: keep a copy of the old position, push, then deposit old -> new
    const GridDev &g = ctx->g;
    const size_t n = (size_t)p->n, slot = (n * 4 + 255) & ~(size_t)255;
    int rc;
    if ((rc = ensure(ctx, &ctx->oldbuf, &ctx->oldbuf_cap, slot * 6))) return rc;
    char *b = (char *)ctx->oldbuf;
    ent_particles old = *p;
    old.cell = (int32_t *)b;
    CK(cudaMemcpyAsync(old.cell, p->cell, n * 4, cudaMemcpyDeviceToDevice, ctx->stream));
    for (int a = 0; a < g.D; ++a) {
        old.d[a] = (float *)(b + slot * (1 + a));
        CK(cudaMemcpyAsync(old.d[a], p->d[a], n * 4, cudaMemcpyDeviceToDevice, ctx->stream));
    }
    if (g.kind != ENT_CART) {
        old.phi = (float *)(b + slot * 4);
        CK(cudaMemcpyAsync(old.phi, p->phi, n * 4, cudaMemcpyDeviceToDevice, ctx->stream));
    }
    if (p->tag) {
        old.tag = (uint8_t *)(b + slot * 5);
        CK(cudaMemcpyAsync(old.tag, p->tag, n, cudaMemcpyDeviceToDevice, ctx->stream));
    }
    if ((rc = ent_gather_push(ctx, EB, p, p, dt))) return rc;
    return ent_deposit(ctx, &old, p, J, dt);
}

extern "C" int ent_workspace_bytes(ent_ctx *ctx, int64_t npart, size_t *bytes) {
    if (!ctx) return ENT_EINVAL;
    if (!ctx->have_grid) return fail(ctx, ENT_EINVAL, "ent_set_grid has not been called");
    if (!bytes || npart < 0) return fail(ctx, ENT_EINVAL, "bad argument");
    *bytes = pool_layout(ctx->g, npart).total;
    return ENT_OK;
}

extern "C" int ent_reserve(ent_ctx *ctx, int64_t npart) {
    ENTER();
    if (npart < 0 || npart >= (1LL << 31)) return fail(ctx, ENT_EINVAL, "npart out of range");
    return reserve_pool(ctx, npart);
}

extern "C" int ent_forget(ent_ctx *ctx, const ent_particles *block) {
    if (!ctx) return ENT_EINVAL;
    if (!block) return fail(ctx, ENT_EINVAL, "block is NULL");
    forget_block(ctx, block->cell);
    return ENT_OK;
}

extern "C" int ent_step(ent_ctx *ctx, const ent_fields *EB, ent_particles *p, ent_current *J, float dt) {
    ENTER();
    int rc;
    if ((rc = check_fields(ctx, EB)) || (rc = check_current(ctx, J)) || (rc = check_particles(ctx, p, "p", true))) return rc;
    if (!(dt > 0.f)) return fail(ctx, ENT_EINVAL, "dt must be positive");
    ctx->g.gca_c = (float)(2.0 * ctx->gca_rho / (double)dt);      // hybrid pusher: rho_crit q/m = gca_c * eps
    if (!(p->m != 0.f)) return fail(ctx, ENT_EINVAL, "mass is zero");
    ctx->last_step_tiled = 0;
    if (p->n == 0) return ENT_OK;
    if (ctx->step_impl == 2) return step_two_kernel(ctx, EB, p, J, dt);
    float eps = 0.5f * (p->q / p->m) * dt;
    ent_ctx::SortedBlock *sb = find_block(ctx, p);
    if ((ctx->step_impl == 0 || ctx->step_impl == 3) && sb && tiled_supported(ctx->tiled, ctx->g)) {
        if (!sb->wmax_valid) {                                   // a block ent_step_sorted produced: its per-tile max |w| was never needed
            tile_wmax_kernel<<<(unsigned)((long long)ctx->g.nt[0] * ctx->g.nt[1] * ctx->g.nt[2]), 128, 0, ctx->stream>>>(sb->tile_off, p->w, sb->tile_wmax);
            if ((rc = launch_check(ctx, "tile_wmax_kernel"))) return rc;
            sb->wmax_valid = true;
        }
        CK(cudaMemsetAsync(ctx->counters + 1, 0, 2 * sizeof(unsigned long long), ctx->stream));  // strays of THIS step, stray-list length
        rc = tiled_step(ctx->tiled, ctx->g, ctx->stream, fp(EB), pp(p), cp(J), (long long)p->n, sb->tile_off, sb->tile_wmax, sb->chunk_off, eps, dt, p->q,
                        1.0f / dt, ctx->counters, &ctx->launches, ctx->err, sizeof(ctx->err));
        if (rc == ENT_OK) ctx->last_step_tiled = 1;
        sb->counts_valid = false;          // the particles moved inside their ranges: next_count no longer describes their current tiles
        return rc;
    }
    DISPATCH(step_untiled_kernel, nblk(p->n), ctx->g, fp(EB), pp(p), cp(J), (long long)p->n, eps, dt, p->q, 1.0f / dt, ctx->counters + 0);
    return launch_check(ctx, "step_untiled_kernel");
}

// thresholds of the hybrid pusher
extern "C" int ent_set_gca(ent_ctx *ctx, double rho_crit, double e_over_b_max) {
    if (!ctx) return ENT_EINVAL;
    if (!(rho_crit >= 0.0) || !(e_over_b_max >= 0.0)) return fail(ctx, ENT_EINVAL, "ent_set_gca: thresholds must be >= 0");
    ctx->gca_rho = rho_crit; ctx->gca_eovb = e_over_b_max;
    ctx->g.gca_eovb2 = (float)(e_over_b_max * e_over_b_max);
    return ENT_OK;
}

// two species through ONE launch of the tiled kernel (one E,B box, one J tile and one flush per tile for both)
extern "C" int ent_step_pair(ent_ctx *ctx, const ent_fields *EB, ent_particles *p1, ent_particles *p2, ent_current *J, float dt) {
    ENTER();
    int rc;
    if ((rc = check_fields(ctx, EB)) || (rc = check_current(ctx, J)) || (rc = check_particles(ctx, p1, "p1", true)) || (rc = check_particles(ctx, p2, "p2", true))) return rc;
    if (!(dt > 0.f)) return fail(ctx, ENT_EINVAL, "dt must be positive");
    ctx->g.gca_c = (float)(2.0 * ctx->gca_rho / (double)dt);      // hybrid pusher: rho_crit q/m = gca_c * eps
    if (!(p1->m != 0.f) || !(p2->m != 0.f)) return fail(ctx, ENT_EINVAL, "mass is zero");
    if (p1->n > 0 && p1->cell == p2->cell) return fail(ctx, ENT_EINVAL, "ent_step_pair: the two blocks are the same");
    ent_ctx::SortedBlock *s1 = find_block(ctx, p1), *s2 = find_block(ctx, p2);
    // one CTA per tile: worth it only when the tiles fill the GPU (148 SMs x 3 CTAs); smaller grids go through the work lists of two
    // launches (tile_chunk_for), unless ENT_OPT_STEP_IMPL = 3 asks for the pair launch
    const long long ntiles_pair = (long long)ctx->g.nt[0] * ctx->g.nt[1] * ctx->g.nt[2];
    const bool pairable = (ctx->step_impl == 3 || (ctx->step_impl == 0 && ntiles_pair >= PAIR_MIN_TILES)) && s1 && s2 && p1->n > 0 && p2->n > 0 &&
                          ctx->g.kind == ENT_CART && tiled_supported(ctx->tiled, ctx->g) && (p1->tag != nullptr) == (p2->tag != nullptr);
    if (!pairable) {                                             // the same result through two launches
        if ((rc = ent_step(ctx, EB, p1, J, dt))) return rc;
        return ent_step(ctx, EB, p2, J, dt);
    }
    ent_ctx::SortedBlock *sb[2] = { s1, s2 };
    const ent_particles *pp2[2] = { p1, p2 };
    for (int k = 0; k < 2; ++k)
        if (!sb[k]->wmax_valid) {
            tile_wmax_kernel<<<(unsigned)((long long)ctx->g.nt[0] * ctx->g.nt[1] * ctx->g.nt[2]), 128, 0, ctx->stream>>>(sb[k]->tile_off, pp2[k]->w, sb[k]->tile_wmax);
            if ((rc = launch_check(ctx, "tile_wmax_kernel"))) return rc;
            sb[k]->wmax_valid = true;
        }
    CK(cudaMemsetAsync(ctx->counters + 1, 0, 2 * sizeof(unsigned long long), ctx->stream));
    PairSpecies second{ pp(p2), s2->tile_off, s2->tile_wmax, 0.5f * (p2->q / p2->m) * dt, p2->q };
    rc = tiled_step(ctx->tiled, ctx->g, ctx->stream, fp(EB), pp(p1), cp(J), (long long)p1->n, s1->tile_off, s1->tile_wmax, s1->chunk_off,
                    0.5f * (p1->q / p1->m) * dt, dt, p1->q, 1.0f / dt, ctx->counters, &ctx->launches, ctx->err, sizeof(ctx->err), &second);
    if (rc == ENT_OK) ctx->last_step_tiled = 1;
    s1->counts_valid = false; s2->counts_valid = false;
    return rc;
}

// claims a SortedBlock slot for `out` (never the one in `keep`)
static ent_ctx::SortedBlock *claim_slot(ent_ctx *ctx, const ent_ctx::SortedBlock *keep, const int32_t *out_cell) {
    forget_block(ctx, out_cell);
    ent_ctx::SortedBlock *slot = nullptr;
    for (auto &b : ctx->sorted) { if (&b == keep) continue; if (!b.cell) { slot = &b; break; } if (!slot || b.stamp < slot->stamp) slot = &b; }
    slot->cell = nullptr; slot->n = -1; slot->wmax_valid = false; slot->counts_valid = false;
    return slot;
}

static int exclusive_scan(ent_ctx *ctx, const int32_t *in, long long m, int32_t *out, int32_t *copy) {
    const int nchunks = (int)((m + SCAN_CHUNK - 1) / SCAN_CHUNK);
    int rc;
    scan_reduce_kernel<<<nchunks, TPB, 0, ctx->stream>>>(in, m, ctx->chunk);
    if ((rc = launch_check(ctx, "scan_reduce_kernel"))) return rc;
    scan_chunks_kernel<<<1, TPB, 0, ctx->stream>>>(ctx->chunk, nchunks);
    if ((rc = launch_check(ctx, "scan_chunks_kernel"))) return rc;
    scan_apply_kernel<<<nchunks, TPB, 0, ctx->stream>>>(in, m, ctx->chunk, out, copy);
    return launch_check(ctx, "scan_apply_kernel");
}

// work list of a sorted block: exclusive scan of ceil(tile population / tile_chunk_for(n)), n = particles of the block.  Scratch: ctx->count, ctx->offsets (second
// copy of the scan, unused), both idle between the phases of ent_sort / ent_step_sorted.
static int build_work_lists(ent_ctx *ctx, ent_ctx::SortedBlock *slot, long long ntiles, long long n) {
    int rc;
    tile_chunks_kernel<<<nblk(ntiles), TPB, 0, ctx->stream>>>(slot->tile_off, ntiles, tile_chunk_for(n), ctx->count);
    if ((rc = launch_check(ctx, "tile_chunks_kernel"))) return rc;
    return exclusive_scan(ctx, ctx->count, ntiles, slot->chunk_off, ctx->offsets);
}

static RebinGeom rebin_geom(const GridDev &g) {
    RebinGeom G;
    G.D = g.D;
    for (int a = 0; a < 3; ++a) { G.N[a] = g.N[a]; G.T[a] = g.T[a]; G.nt[a] = g.nt[a]; G.per[a] = g.bc[a] == ENT_PERIODIC; G.dT[a] = make_magicdiv((uint32_t)g.T[a]); }
    G.dN0 = make_magicdiv((uint32_t)g.N[0]); G.dN01 = make_magicdiv((uint32_t)(g.N[0] * g.N[1]));
    G.dnt0 = make_magicdiv((uint32_t)g.nt[0]); G.dnt01 = make_magicdiv((uint32_t)(g.nt[0] * g.nt[1]));
    for (int a = 0; a < 3; ++a) { int last = g.N[a] - (g.nt[a] - 1) * g.T[a]; G.mext[a] = last < g.T[a] ? last : g.T[a]; }
    return G;
}

// next_count of a block whose particles drifted inside their ranges: population per tile by the CURRENT cells
static int recount_tiles(ent_ctx *ctx, ent_ctx::SortedBlock *sb, const ent_particles *p) {
    const GridDev &g = ctx->g;
    const long long ntiles = (long long)g.nt[0] * g.nt[1] * g.nt[2];
    CK(cudaMemsetAsync(sb->next_count, 0, (size_t)(ntiles + 1) * 4, ctx->stream));
    rebin_count_kernel<<<(unsigned)ntiles, REBIN_TPB, 0, ctx->stream>>>(rebin_geom(g), p->cell, sb->tile_off, ctx->class_count, sb->next_count);
    int rc = launch_check(ctx, "rebin_count_kernel");
    if (rc == ENT_OK) sb->counts_valid = true;
    return rc;
}

// incremental ent_sort: `in` is tile-contiguous (src), particles have drifted; re-establish tile contiguity in `out`
static int sort_rebin(ent_ctx *ctx, ent_ctx::SortedBlock *src, const ent_particles *in, ent_particles *out) {
    const GridDev &g = ctx->g;
    const long long ntiles = (long long)g.nt[0] * g.nt[1] * g.nt[2];
    int rc;
    ent_ctx::SortedBlock *slot = claim_slot(ctx, src, out->cell);
    const RebinGeom G = rebin_geom(g);
    CK(cudaMemsetAsync(ctx->count, 0, (size_t)(ntiles + 1) * 4, ctx->stream));
    CK(cudaMemsetAsync(slot->tile_wmax, 0, (size_t)ntiles * 4, ctx->stream));
    rebin_count_kernel<<<(unsigned)ntiles, REBIN_TPB, 0, ctx->stream>>>(G, in->cell, src->tile_off, ctx->class_count, ctx->count);
    if ((rc = launch_check(ctx, "rebin_count_kernel"))) return rc;
    CK(cudaMemcpyAsync(slot->next_count, ctx->count, (size_t)ntiles * 4, cudaMemcpyDeviceToDevice, ctx->stream));
    if ((rc = exclusive_scan(ctx, ctx->count, ntiles, slot->tile_off, ctx->cursor))) return rc;
    if (g.kind == ENT_CART && g.tcells <= ORD_BINS && ctx->rebin_ordered) {
        if (!ctx->ord_attr_set) { CK(cudaFuncSetAttribute(rebin_scatter_ordered_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, ORD_CAP_MAX * ORD_REC_BYTES)); ctx->ord_attr_set = true; }
        // staging capacity: 25 % above the mean tile population (a fuller tile is placed unordered), as small as possible so
        // that several CTAs fit an SM
        long long cap = ((in->n / ntiles) * 5 / 4 + 64 + 3) & ~3LL;
        if (cap < 256) cap = 256;
        if (cap > ORD_CAP_MAX) cap = ORD_CAP_MAX;
        rebin_scatter_ordered_kernel<<<(unsigned)ntiles, ORD_TPB, (size_t)cap * ORD_REC_BYTES, ctx->stream>>>(G, g.tcells, (int)cap, src->tile_off, ctx->class_count,
                                                                                                 ctx->cursor, pp(in), pp(out), (unsigned *)slot->tile_wmax);
        if ((rc = launch_check(ctx, "rebin_scatter_ordered_kernel"))) return rc;
    } else {
        rebin_scatter_kernel<<<(unsigned)ntiles, REBIN_TPB, 0, ctx->stream>>>(G, src->tile_off, ctx->class_count, ctx->cursor, pp(in), pp(out),
                                                                            g.kind != ENT_CART, (unsigned *)slot->tile_wmax);
        if ((rc = launch_check(ctx, "rebin_scatter_kernel"))) return rc;
    }
    if ((rc = build_work_lists(ctx, slot, ntiles, in->n))) return rc;
    if (!in->tag && out->tag) CK(cudaMemsetAsync(out->tag, 1, (size_t)in->n, ctx->stream));       // as in the full sort: every particle is alive
    out->q = in->q; out->m = in->m;
    slot->cell = out->cell; slot->n = in->n; slot->stamp = ++ctx->sort_stamp; slot->wmax_valid = true; slot->counts_valid = true;
    ctx->last_sort_rebin = 1;
    return ENT_OK;
}

extern "C" int ent_sort(ent_ctx *ctx, const ent_particles *in, ent_particles *out, int32_t *key_offsets) {
    ENTER();
    int rc;
    if ((rc = check_particles(ctx, in, "in", false)) || (rc = check_particles(ctx, out, "out", false))) return rc;
    if (in->n != out->n) return fail(ctx, ENT_EINVAL, "in->n != out->n");
    if (in->n > 0 && (in->cell == out->cell || in->w == out->w)) return fail(ctx, ENT_EINVAL, "ent_sort is out-of-place: in and out overlap");
    if (in->tag && !out->tag) return fail(ctx, ENT_EINVAL, "in has tags but out->tag is NULL");
    const GridDev &g = ctx->g;
    const long long n = in->n;
    const long long nkeys = (long long)g.nt[0] * g.nt[1] * g.nt[2] * g.tcells;
    const long long ntiles = (long long)g.nt[0] * g.nt[1] * g.nt[2];
    if ((rc = reserve_pool(ctx, n))) return rc;
    ctx->last_sort_rebin = 0;
    if (ctx->sort_mode == 0 && !key_offsets && n > 0) {
        ent_ctx::SortedBlock *src = find_block(ctx, in);
        if (src) return sort_rebin(ctx, src, in, out);
    }
    forget_block(ctx, out->cell);
    CK(cudaMemsetAsync(ctx->count, 0, (size_t)(nkeys + 1) * 4, ctx->stream));
    if (n > 0) {
        if (g.D == 2) sort_hist_kernel<2><<<nblk(n), TPB, 0, ctx->stream>>>(g, in->cell, n, ctx->keys, ctx->count);
        else sort_hist_kernel<3><<<nblk(n), TPB, 0, ctx->stream>>>(g, in->cell, n, ctx->keys, ctx->count);
        if ((rc = launch_check(ctx, "sort_hist_kernel"))) return rc;
    }
    if ((rc = exclusive_scan(ctx, ctx->count, nkeys, ctx->offsets, ctx->cursor))) return rc;
    if (n > 0) {
        if (ctx->sort_staging) {                       // unordered input: full-sector writes to a side buffer, then a coalesced unpack
            if ((rc = ensure(ctx, &ctx->sbuf, &ctx->sbuf_cap, (size_t)n * 32))) return rc;
            sort_scatter_aos_kernel<<<nblk(n), TPB, 0, ctx->stream>>>(ctx->keys, ctx->cursor, pp(in), (float4 *)ctx->sbuf, out->tag, n, g.D, g.kind != ENT_CART);
            if ((rc = launch_check(ctx, "sort_scatter_aos_kernel"))) return rc;
            sort_unpack_aos_kernel<<<nblk(n), TPB, 0, ctx->stream>>>((const float4 *)ctx->sbuf, pp(out), n, g.D, g.kind != ENT_CART);
            if ((rc = launch_check(ctx, "sort_unpack_aos_kernel"))) return rc;
        } else {
            sort_scatter_kernel<<<nblk(n), TPB, 0, ctx->stream>>>(ctx->keys, ctx->cursor, pp(in), pp(out), n, g.D, g.kind != ENT_CART);
            if ((rc = launch_check(ctx, "sort_scatter_kernel"))) return rc;
        }
        // in has no tags but out has: every particle is alive (ent.h)
        if (!in->tag && out->tag) CK(cudaMemsetAsync(out->tag, 1, (size_t)n, ctx->stream));
    }
    if (key_offsets) CK(cudaMemcpyAsync(key_offsets, ctx->offsets, (size_t)(nkeys + 1) * 4, cudaMemcpyDeviceToDevice, ctx->stream));
    out->q = in->q; out->m = in->m;
    if (n > 0) {   // remember `out` as sorted, with its own layout (tile t = particles [tile_off[t], tile_off[t+1]))
        ent_ctx::SortedBlock *slot = claim_slot(ctx, nullptr, out->cell);
        tile_offsets_kernel<<<nblk(ntiles + 1), TPB, 0, ctx->stream>>>(ctx->offsets, g.tcells, ntiles, slot->tile_off, slot->next_count);
        if ((rc = launch_check(ctx, "tile_offsets_kernel"))) return rc;
        tile_wmax_kernel<<<(unsigned)ntiles, 128, 0, ctx->stream>>>(slot->tile_off, out->w, slot->tile_wmax);
        if ((rc = launch_check(ctx, "tile_wmax_kernel"))) return rc;
        if ((rc = build_work_lists(ctx, slot, ntiles, n))) return rc;
        slot->cell = out->cell; slot->n = n; slot->stamp = ++ctx->sort_stamp; slot->wmax_valid = true; slot->counts_valid = true;
    }
    return ENT_OK;
}

// ---- N4: tag sort ------------------------------------------------------------------------------------
extern "C" int ent_compact(ent_ctx *ctx, const ent_particles *in, ent_particles *out, int64_t *n_alive) {
    ENTER();
    int rc;
    if ((rc = check_particles(ctx, in, "in", false)) || (rc = check_particles(ctx, out, "out", false))) return rc;
    if (in->n != out->n) return fail(ctx, ENT_EINVAL, "in->n != out->n");
    if (in->n > 0 && (in->cell == out->cell || in->w == out->w)) return fail(ctx, ENT_EINVAL, "ent_compact is out-of-place: in and out overlap");
    if (!in->tag || !out->tag) return fail(ctx, ENT_EINVAL, "ent_compact needs tag arrays in both blocks");
    const GridDev &g = ctx->g;
    const long long n = in->n;
    out->q = in->q; out->m = in->m;
    forget_block(ctx, out->cell);
    if (n == 0) { if (n_alive) CK(cudaMemsetAsync(n_alive, 0, sizeof(int64_t), ctx->stream)); return ENT_OK; }
    const size_t slot = ((size_t)(n + 1) * 4 + 255) & ~(size_t)255;
    const size_t nch = ((size_t)((n + SCAN_CHUNK - 1) / SCAN_CHUNK) * 4 + 255) & ~(size_t)255;
    if ((rc = ensure(ctx, &ctx->cbuf, &ctx->cbuf_cap, 3 * slot + nch))) return rc;
    int32_t *flag = (int32_t *)ctx->cbuf, *pos = (int32_t *)((char *)ctx->cbuf + slot), *copy = (int32_t *)((char *)ctx->cbuf + 2 * slot);
    int32_t *chunk = (int32_t *)((char *)ctx->cbuf + 3 * slot);
    const int nchunks = (int)((n + SCAN_CHUNK - 1) / SCAN_CHUNK);
    compact_flag_kernel<<<nblk(n), TPB, 0, ctx->stream>>>(in->tag, n, flag);
    if ((rc = launch_check(ctx, "compact_flag_kernel"))) return rc;
    scan_reduce_kernel<<<nchunks, TPB, 0, ctx->stream>>>(flag, n, chunk);
    if ((rc = launch_check(ctx, "scan_reduce_kernel"))) return rc;
    scan_chunks_kernel<<<1, TPB, 0, ctx->stream>>>(chunk, nchunks);
    if ((rc = launch_check(ctx, "scan_chunks_kernel"))) return rc;
    scan_apply_kernel<<<nchunks, TPB, 0, ctx->stream>>>(flag, n, chunk, pos, copy);
    if ((rc = launch_check(ctx, "scan_apply_kernel"))) return rc;
    compact_scatter_kernel<<<nblk(n), TPB, 0, ctx->stream>>>(pos, pp(in), pp(out), n, g.D, g.kind != ENT_CART, (long long *)n_alive);
    return launch_check(ctx, "compact_scatter_kernel");
}

// ent_compact without any allocation: the scan's scratch is the module's static array (see compact_static_scratch above)
extern "C" int ent_compact_static(ent_ctx *ctx, const ent_particles *in, ent_particles *out, int64_t *n_alive) {
    ENTER();
    int rc;
    if ((rc = check_particles(ctx, in, "in", false)) || (rc = check_particles(ctx, out, "out", false))) return rc;
    if (in->n != out->n) return fail(ctx, ENT_EINVAL, "in->n != out->n");
    if (in->n > COMPACT_STATIC_MAX_N)
        return fail(ctx, ENT_EINVAL, "ent_compact_static: n = %lld exceeds the static scratch (ENT_COMPACT_STATIC_MAX_N = %lld particles); use ent_compact",
                    (long long)in->n, (long long)COMPACT_STATIC_MAX_N);
    if (in->n > 0 && (in->cell == out->cell || in->w == out->w)) return fail(ctx, ENT_EINVAL, "ent_compact_static is out-of-place: in and out overlap");
    if (!in->tag || !out->tag) return fail(ctx, ENT_EINVAL, "ent_compact_static needs tag arrays in both blocks");
    const GridDev &g = ctx->g;
    const long long n = in->n;
    out->q = in->q; out->m = in->m;
    forget_block(ctx, out->cell);
    if (n == 0) { if (n_alive) CK(cudaMemsetAsync(n_alive, 0, sizeof(int64_t), ctx->stream)); return ENT_OK; }
    void *base = nullptr;
    cudaError_t e = static_scratch_lookup(ctx->device, &base);
    if (e != cudaSuccess || !base) return fail(ctx, ENT_ECUDA, "cudaGetSymbolAddress of the static scratch failed: %s", cudaGetErrorString(e));
    // nothing has to start at zero: every element read below (flags 0 .. n-1, chunk sums, positions 0 .. n) is written by this call first
    const size_t slot = ((size_t)(n + 1) * 4 + 255) & ~(size_t)255;
    int32_t *flag = (int32_t *)base, *pos = (int32_t *)((char *)base + slot), *copy = (int32_t *)((char *)base + 2 * slot);
    int32_t *chunk = (int32_t *)((char *)base + 3 * slot);
    const int nchunks = (int)((n + SCAN_CHUNK - 1) / SCAN_CHUNK);
    compact_flag_kernel<<<nblk(n), TPB, 0, ctx->stream>>>(in->tag, n, flag);
    if ((rc = launch_check(ctx, "compact_flag_kernel"))) return rc;
    scan_reduce_kernel<<<nchunks, TPB, 0, ctx->stream>>>(flag, n, chunk);
    if ((rc = launch_check(ctx, "scan_reduce_kernel"))) return rc;
    scan_chunks_kernel<<<1, TPB, 0, ctx->stream>>>(chunk, nchunks);
    if ((rc = launch_check(ctx, "scan_chunks_kernel"))) return rc;
    scan_apply_kernel<<<nchunks, TPB, 0, ctx->stream>>>(flag, n, chunk, pos, copy);
    if ((rc = launch_check(ctx, "scan_apply_kernel"))) return rc;
    compact_scatter_kernel<<<nblk(n), TPB, 0, ctx->stream>>>(pos, pp(in), pp(out), n, g.D, g.kind != ENT_CART, (long long *)n_alive);
    return launch_check(ctx, "compact_scatter_kernel");
}

// ---- fused step + re-bin: the timed entry point on Cartesian grids ----------------------------------------------
extern "C" int ent_step_sorted(ent_ctx *ctx, const ent_fields *EB, const ent_particles *in, ent_particles *out, ent_current *J, float dt) {
    ENTER();
    int rc;
    if ((rc = check_fields(ctx, EB)) || (rc = check_current(ctx, J)) || (rc = check_particles(ctx, in, "in", false)) ||
        (rc = check_particles(ctx, out, "out", true))) return rc;
    if (in->n != out->n) return fail(ctx, ENT_EINVAL, "in->n != out->n");
    if (!(dt > 0.f)) return fail(ctx, ENT_EINVAL, "dt must be positive");
    ctx->g.gca_c = (float)(2.0 * ctx->gca_rho / (double)dt);      // hybrid pusher: rho_crit q/m = gca_c * eps
    if (!(in->m != 0.f)) return fail(ctx, ENT_EINVAL, "mass is zero");
    if (in->tag && !out->tag) return fail(ctx, ENT_EINVAL, "in has tags but out->tag is NULL");
    ctx->last_step_tiled = 0;
    out->q = in->q; out->m = in->m;
    if (in->n == 0) return ENT_OK;
    if (in->cell == out->cell || in->w == out->w || in->u[0] == out->u[0]) return fail(ctx, ENT_EINVAL, "ent_step_sorted is out-of-place: in and out overlap");
    if (!sorted_supported(ctx->tiled, ctx->g)) return fail(ctx, ENT_EUNSUPPORTED, "ent_step_sorted: Cartesian grids with N1 %% 4 == 0 only");
    ent_ctx::SortedBlock *src = find_block(ctx, in);
    if (!src) return fail(ctx, ENT_EINVAL, "ent_step_sorted: `in` is not a sorted block of this ctx (call ent_sort first)");
    const GridDev &g = ctx->g;
    const long long ntiles = (long long)g.nt[0] * g.nt[1] * g.nt[2];
    if (!src->counts_valid && (rc = recount_tiles(ctx, src, in))) return rc;
    if (!src->wmax_valid) {
        tile_wmax_kernel<<<(unsigned)ntiles, 128, 0, ctx->stream>>>(src->tile_off, in->w, src->tile_wmax);
        if ((rc = launch_check(ctx, "tile_wmax_kernel"))) return rc;
        src->wmax_valid = true;
    }
    ent_ctx::SortedBlock *dst = claim_slot(ctx, src, out->cell);
    // layout of `out`: exclusive scan of the populations by current tile; cursor = second copy, consumed by the kernel's reservations
    if ((rc = exclusive_scan(ctx, src->next_count, ntiles, dst->tile_off, ctx->cursor))) return rc;
    CK(cudaMemsetAsync(dst->next_count, 0, (size_t)(ntiles + 1) * 4, ctx->stream));
    CK(cudaMemsetAsync(dst->tile_wmax, 0, (size_t)(ntiles + 1) * 4, ctx->stream));
    CK(cudaMemsetAsync(ctx->counters + 1, 0, sizeof(unsigned long long), ctx->stream));         // strays of THIS step
    SortedArgs A;
    A.g = g; A.F = fp(EB); A.J = cp(J); A.in = pp(in); A.out = pp(out);
    A.tile_off = src->tile_off; A.chunk_off = src->chunk_off; A.tile_wmax = src->tile_wmax; A.cursor = ctx->cursor;
    A.next_count = dst->next_count; A.wmax_out = (unsigned *)dst->tile_wmax;
    A.n = in->n; A.chunk = tile_chunk_for(in->n); A.eps = 0.5f * (in->q / in->m) * dt; A.dt = dt; A.q = in->q; A.inv_dt = 1.0f / dt; A.counters = ctx->counters;
    if ((rc = sorted_step(ctx->tiled, A, dt, ctx->stream, ctx->err, sizeof(ctx->err)))) return rc;
    ctx->launches += 1;
    if ((rc = build_work_lists(ctx, dst, ntiles, in->n))) return rc;
    dst->cell = out->cell; dst->n = in->n; dst->stamp = ++ctx->sort_stamp; dst->wmax_valid = true; dst->counts_valid = true;
    ctx->last_step_tiled = 1;
    return ENT_OK;
}

extern "C" int ent_tile_offsets(ent_ctx *ctx, const ent_particles *block, int32_t *tile_offsets) {
    ENTER();
    if (!block || !tile_offsets) return fail(ctx, ENT_EINVAL, "NULL argument");
    const GridDev &g = ctx->g;
    const long long ntiles = (long long)g.nt[0] * g.nt[1] * g.nt[2];
    ent_ctx::SortedBlock *b = find_block(ctx, block);
    if (!b) return fail(ctx, ENT_EINVAL, "the block is not a sorted block of this ctx");
    CK(cudaMemcpyAsync(tile_offsets, b->tile_off, (size_t)(ntiles + 1) * 4, cudaMemcpyDeviceToDevice, ctx->stream));
    return ENT_OK;
}

extern "C" int ent_set_option(ent_ctx *ctx, int key, int64_t value) {
    if (!ctx) return ENT_EINVAL;
    switch (key) {
        case ENT_OPT_STEP_IMPL:
            if (value < 0 || value > 3) return fail(ctx, ENT_EINVAL, "ENT_OPT_STEP_IMPL must be 0, 1, 2 or 3");
            ctx->step_impl = (int)value; return ENT_OK;
        case ENT_OPT_SORT_MODE:
            if (value < 0 || value > 2) return fail(ctx, ENT_EINVAL, "ENT_OPT_SORT_MODE must be 0, 1 or 2");
            ctx->sort_mode = value == 1 ? 1 : 0; ctx->rebin_ordered = value != 2; return ENT_OK;
        case ENT_OPT_PUSHER:
            if (value < 0 || value > 3) return fail(ctx, ENT_EINVAL, "ENT_OPT_PUSHER must be 0 (Boris), 1 (Vay), 2 (Boris,GCA) or 3 (Vay,GCA)");
            ctx->pusher = (int)value; ctx->g.pusher = (int)value; return ENT_OK;
        case ENT_OPT_SORT_STAGING:
            if (value < 0 || value > 1) return fail(ctx, ENT_EINVAL, "ENT_OPT_SORT_STAGING must be 0 or 1");
            ctx->sort_staging = (int)value; return ENT_OK;
        case ENT_OPT_CURV_FP64:
            if (value < 0 || value > 1) return fail(ctx, ENT_EINVAL, "ENT_OPT_CURV_FP64 must be 0 or 1");
            ctx->curv_f64 = (int)value; ctx->g.curv_f64 = (int)value; return ENT_OK;
        case ENT_OPT_TILE_1: case ENT_OPT_TILE_2: case ENT_OPT_TILE_3:
            if (value < 0 || value > 64) return fail(ctx, ENT_EINVAL, "tile extent must be in 0..64 (0 = default)");
            ctx->tile_opt[key - ENT_OPT_TILE_1] = (int)value; return ENT_OK;
        default: return fail(ctx, ENT_EINVAL, "unknown option %d", key);
    }
}

extern "C" int ent_get_stat(ent_ctx *ctx, int key, int64_t *value) {
    if (!ctx) return ENT_EINVAL;
    if (!value) return fail(ctx, ENT_EINVAL, "value is NULL");
    const GridDev &g = ctx->g;
    switch (key) {
        case ENT_STAT_TILE_1: case ENT_STAT_TILE_2: case ENT_STAT_TILE_3:
            if (!ctx->have_grid) return fail(ctx, ENT_EINVAL, "no grid"); *value = g.T[key - ENT_STAT_TILE_1]; return ENT_OK;
        case ENT_STAT_NKEYS:
            if (!ctx->have_grid) return fail(ctx, ENT_EINVAL, "no grid"); *value = (int64_t)g.nt[0] * g.nt[1] * g.nt[2] * g.tcells; return ENT_OK;
        case ENT_STAT_NTILES:
            if (!ctx->have_grid) return fail(ctx, ENT_EINVAL, "no grid"); *value = (int64_t)g.nt[0] * g.nt[1] * g.nt[2]; return ENT_OK;
        case ENT_STAT_LAUNCHES: *value = ctx->launches; return ENT_OK;
        case ENT_STAT_BAD_MOVES: case ENT_STAT_STRAYS: case ENT_STAT_SLOT_ERRORS: case ENT_STAT_CARRIES: case ENT_STAT_GLOBAL_ADDS: {
            unsigned long long h[8];
            CK(cudaSetDevice(ctx->device));
            CK(cudaMemcpyAsync(h, ctx->counters, sizeof(h), cudaMemcpyDeviceToHost, ctx->stream));
            CK(cudaStreamSynchronize(ctx->stream));
            *value = (int64_t)h[key == ENT_STAT_BAD_MOVES ? 0 : key == ENT_STAT_STRAYS ? 1 : key == ENT_STAT_SLOT_ERRORS ? 3 : key == ENT_STAT_CARRIES ? 4 : 5]; return ENT_OK;
        }
        case ENT_STAT_SCRATCH_BYTES: *value = (int64_t)(ctx->pool_bytes + ctx->side_bytes); return ENT_OK;
        case ENT_STAT_LAST_STEP_TILED: *value = ctx->last_step_tiled; return ENT_OK;
        case ENT_STAT_LAST_SORT_REBIN: *value = ctx->last_sort_rebin; return ENT_OK;
        default: return fail(ctx, ENT_EINVAL, "unknown stat %d", key);
    }
}

// ---- host-buffer variant: H2D, ent_sort, nsteps x ent_step (tiled kernel), D2H, all inside the call (end-to-end measurement) ----
extern "C" int ent_step_host(ent_ctx *ctx, const ent_fields *EB, ent_particles *p, ent_current *J, float dt, int nsteps,
                             int64_t *h2d_bytes, int64_t *d2h_bytes) {
    ENTER();
    if (!EB || !p || !J) return fail(ctx, ENT_EINVAL, "NULL argument");
    if (nsteps < 0) return fail(ctx, ENT_EINVAL, "nsteps < 0");
    const GridDev &g = ctx->g;
    const size_t n = (size_t)p->n, pad = (size_t)padded_size(g);
    const size_t fslot = (pad * 4 + 255) & ~(size_t)255, pslot = (n * 4 + 255) & ~(size_t)255;
    const bool axisym = g.kind != ENT_CART;
    int rc;
    if ((rc = ensure(ctx, &ctx->hbuf, &ctx->hbuf_cap, fslot * 9 + pslot * 20))) return rc;      // fields, J, two particle blocks
    if ((rc = reserve_pool(ctx, (long long)n))) return rc;
    char *b = (char *)ctx->hbuf;
    int64_t up = 0, down = 0;
    ent_fields dEB; ent_current dJ; ent_particles dp = *p, ds = *p;
    for (int c = 0; c < 6; ++c) {
        if (!EB->comp[c]) return fail(ctx, ENT_EINVAL, "host field component %d is NULL", c);
        float *dst = (float *)(b + fslot * c);
        CK(cudaMemcpyAsync(dst, EB->comp[c], pad * 4, cudaMemcpyHostToDevice, ctx->stream)); up += (int64_t)pad * 4;
        dEB.comp[c] = dst;
    }
    for (int c = 0; c < 3; ++c) {
        if (!J->comp[c]) return fail(ctx, ENT_EINVAL, "host current component %d is NULL", c);
        dJ.comp[c] = (float *)(b + fslot * (6 + c));
    }
    char *pb = b + fslot * 9, *sb = pb + pslot * 10;          // staged block (as uploaded) and its sorted copy
    struct Arr { void **dev; void **srt; void *host; size_t bytes; bool back; };
    Arr arrs[10]; int na = 0;
    dp.cell = (int32_t *)(pb + pslot * 0); ds.cell = (int32_t *)(sb + pslot * 0); arrs[na++] = { (void **)&dp.cell, (void **)&ds.cell, p->cell, n * 4, true };
    for (int a = 0; a < 3; ++a) {
        if (a < g.D) { dp.d[a] = (float *)(pb + pslot * (1 + a)); ds.d[a] = (float *)(sb + pslot * (1 + a)); arrs[na++] = { (void **)&dp.d[a], (void **)&ds.d[a], p->d[a], n * 4, true }; }
        else dp.d[a] = ds.d[a] = nullptr;
        dp.u[a] = (float *)(pb + pslot * (4 + a)); ds.u[a] = (float *)(sb + pslot * (4 + a)); arrs[na++] = { (void **)&dp.u[a], (void **)&ds.u[a], p->u[a], n * 4, true };
    }
    dp.w = (float *)(pb + pslot * 7); ds.w = (float *)(sb + pslot * 7); arrs[na++] = { (void **)&dp.w, (void **)&ds.w, p->w, n * 4, true };
    if (axisym) { dp.phi = (float *)(pb + pslot * 8); ds.phi = (float *)(sb + pslot * 8); arrs[na++] = { (void **)&dp.phi, (void **)&ds.phi, p->phi, n * 4, true }; }
    else dp.phi = ds.phi = nullptr;
    if (p->tag) { dp.tag = (uint8_t *)(pb + pslot * 9); ds.tag = (uint8_t *)(sb + pslot * 9); arrs[na++] = { (void **)&dp.tag, (void **)&ds.tag, p->tag, n, true }; }
    else dp.tag = ds.tag = nullptr;
    for (int k = 0; k < na; ++k) {
        if (!arrs[k].host) return fail(ctx, ENT_EINVAL, "a required host particle array is NULL");
        if (arrs[k].bytes) CK(cudaMemcpyAsync(*arrs[k].dev, arrs[k].host, arrs[k].bytes, cudaMemcpyHostToDevice, ctx->stream));
        up += (int64_t)arrs[k].bytes;
    }
    if ((rc = ent_zero_current(ctx, &dJ))) return rc;
    // tile sort of the uploaded block, so that the steps run the tiled kernel (the block comes back in that order)
    forget_block(ctx, dp.cell);
    const int saved_mode = ctx->sort_mode;
    ctx->sort_mode = 1;
    rc = n ? ent_sort(ctx, &dp, &ds, nullptr) : ENT_OK;
    ctx->sort_mode = saved_mode;
    if (rc) return rc;
    for (int s = 0; s < nsteps; ++s)
        if ((rc = ent_step(ctx, &dEB, &ds, &dJ, dt))) return rc;
    forget_block(ctx, ds.cell);                               // the staging memory is reused by the next call
    for (int k = 0; k < na; ++k) {
        if (!arrs[k].back) continue;
        if (arrs[k].bytes) CK(cudaMemcpyAsync(arrs[k].host, *arrs[k].srt, arrs[k].bytes, cudaMemcpyDeviceToHost, ctx->stream));
        down += (int64_t)arrs[k].bytes;
    }
    for (int c = 0; c < 3; ++c) { CK(cudaMemcpyAsync(J->comp[c], dJ.comp[c], pad * 4, cudaMemcpyDeviceToHost, ctx->stream)); down += (int64_t)pad * 4; }
    CK(cudaStreamSynchronize(ctx->stream));
    if (h2d_bytes) *h2d_bytes = up;
    if (d2h_bytes) *d2h_bytes = down;
    return ENT_OK;
}

// Both species of a pair plasma from host buffers, pipelined over three streams.  Each species is cut into HOST_CHUNKS independent
// sub-blocks (particles are independent; J accumulates): while one sub-block is sorted and advanced, the next ones are still arriving
// over PCIe and the previous ones are already on their way back (the link is full duplex), so the call takes about the time of
// the larger of the two transfers plus one sub-block's work.  Fields go up once, J comes back once.
constexpr int HOST_CHUNKS = 8;
extern "C" int ent_step_host_pair(ent_ctx *ctx, const ent_fields *EB, ent_particles *p1, ent_particles *p2, ent_current *J, float dt, int nsteps,
                                  int64_t *h2d_bytes, int64_t *d2h_bytes) {
    ENTER();
    if (!EB || !p1 || !p2 || !J) return fail(ctx, ENT_EINVAL, "NULL argument");
    if (nsteps < 0) return fail(ctx, ENT_EINVAL, "nsteps < 0");
    const GridDev &g = ctx->g;
    ent_particles *hp[2] = { p1, p2 };
    const size_t pad = (size_t)padded_size(g), fslot = (pad * 4 + 255) & ~(size_t)255;
    const size_t nmax = (size_t)(p1->n > p2->n ? p1->n : p2->n);
    const size_t cmax = (nmax + HOST_CHUNKS - 1) / HOST_CHUNKS + 4, pslot = (cmax * 4 + 255) & ~(size_t)255;   // per sub-block and array
    const bool axisym = g.kind != ENT_CART;
    constexpr int NJOB = 2 * HOST_CHUNKS;
    int rc;
    if ((rc = ensure(ctx, &ctx->hbuf, &ctx->hbuf_cap, fslot * 9 + pslot * 20 * NJOB))) return rc;   // fields, J, per sub-block: staged + sorted copy
    if ((rc = reserve_pool(ctx, (long long)cmax))) return rc;
    if (!ctx->up_stream) {
        CK(cudaStreamCreateWithFlags(&ctx->up_stream, cudaStreamNonBlocking));
        CK(cudaStreamCreateWithFlags(&ctx->down_stream, cudaStreamNonBlocking));
        for (auto &e : ctx->ev) CK(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    }
    CK(cudaEventRecord(ctx->ev[2 * NJOB], ctx->stream));         // whatever the caller enqueued before must finish first
    CK(cudaStreamWaitEvent(ctx->up_stream, ctx->ev[2 * NJOB], 0));
    char *b = (char *)ctx->hbuf;
    int64_t up = 0, down = 0;
    ent_fields dEB; ent_current dJ;
    for (int c = 0; c < 6; ++c) {
        if (!EB->comp[c]) return fail(ctx, ENT_EINVAL, "host field component %d is NULL", c);
        float *dst = (float *)(b + fslot * c);
        CK(cudaMemcpyAsync(dst, EB->comp[c], pad * 4, cudaMemcpyHostToDevice, ctx->up_stream)); up += (int64_t)pad * 4;
        dEB.comp[c] = dst;
    }
    for (int c = 0; c < 3; ++c) {
        if (!J->comp[c]) return fail(ctx, ENT_EINVAL, "host current component %d is NULL", c);
        dJ.comp[c] = (float *)(b + fslot * (6 + c));
    }
    struct Arr { void *dev; void *srt; char *host; size_t bytes; };
    Arr arrs[NJOB][10]; int na[NJOB] = {};
    ent_particles dp[NJOB], ds[NJOB];
    for (int k = 0; k < NJOB; ++k) {                              // uploads, in the order the sub-blocks will be advanced
        const ent_particles *p = hp[k / HOST_CHUNKS];
        const int ch = k % HOST_CHUNKS;
        const size_t i0 = (size_t)p->n * ch / HOST_CHUNKS, i1 = (size_t)p->n * (ch + 1) / HOST_CHUNKS, n = i1 - i0;
        char *pb = b + fslot * 9 + pslot * 20 * k, *sb = pb + pslot * 10;
        dp[k] = *p; ds[k] = *p; dp[k].n = ds[k].n = (int64_t)n;
        auto add = [&](void **d, void **s_, void *host, int slot, size_t elem) {
            *d = pb + pslot * slot; *s_ = sb + pslot * slot;
            arrs[k][na[k]++] = { *d, *s_, host ? (char *)host + i0 * elem : nullptr, n * elem };
        };
        add((void **)&dp[k].cell, (void **)&ds[k].cell, p->cell, 0, 4);
        for (int a = 0; a < 3; ++a) {
            if (a < g.D) add((void **)&dp[k].d[a], (void **)&ds[k].d[a], p->d[a], 1 + a, 4); else dp[k].d[a] = ds[k].d[a] = nullptr;
            add((void **)&dp[k].u[a], (void **)&ds[k].u[a], p->u[a], 4 + a, 4);
        }
        add((void **)&dp[k].w, (void **)&ds[k].w, p->w, 7, 4);
        if (axisym) add((void **)&dp[k].phi, (void **)&ds[k].phi, p->phi, 8, 4); else dp[k].phi = ds[k].phi = nullptr;
        if (p->tag) add((void **)&dp[k].tag, (void **)&ds[k].tag, p->tag, 9, 1); else dp[k].tag = ds[k].tag = nullptr;
        for (int j = 0; j < na[k]; ++j) {
            if (!arrs[k][j].host) return fail(ctx, ENT_EINVAL, "a required host particle array is NULL");
            if (arrs[k][j].bytes) CK(cudaMemcpyAsync(arrs[k][j].dev, arrs[k][j].host, arrs[k][j].bytes, cudaMemcpyHostToDevice, ctx->up_stream));
            up += (int64_t)arrs[k][j].bytes;
        }
        CK(cudaEventRecord(ctx->ev[k], ctx->up_stream));         // sub-block k (and, for k = 0, the fields) has arrived
    }
    if ((rc = ent_zero_current(ctx, &dJ))) return rc;
    const int saved_mode = ctx->sort_mode;
    for (int k = 0; k < NJOB; ++k) {
        CK(cudaStreamWaitEvent(ctx->stream, ctx->ev[k], 0));
        if (dp[k].n > 0) {
            forget_block(ctx, dp[k].cell);
            ctx->sort_mode = 1;
            rc = ent_sort(ctx, &dp[k], &ds[k], nullptr);
            ctx->sort_mode = saved_mode;
            if (rc) return rc;
            for (int s_ = 0; s_ < nsteps; ++s_)
                if ((rc = ent_step(ctx, &dEB, &ds[k], &dJ, dt))) return rc;
            forget_block(ctx, ds[k].cell);                       // the staging memory is reused by the next call
        }
        CK(cudaEventRecord(ctx->ev[NJOB + k], ctx->stream));
        CK(cudaStreamWaitEvent(ctx->down_stream, ctx->ev[NJOB + k], 0));
        for (int j = 0; j < na[k]; ++j) {
            if (arrs[k][j].bytes) CK(cudaMemcpyAsync(arrs[k][j].host, arrs[k][j].srt, arrs[k][j].bytes, cudaMemcpyDeviceToHost, ctx->down_stream));
            down += (int64_t)arrs[k][j].bytes;
        }
    }
    for (int c = 0; c < 3; ++c) { CK(cudaMemcpyAsync(J->comp[c], dJ.comp[c], pad * 4, cudaMemcpyDeviceToHost, ctx->down_stream)); down += (int64_t)pad * 4; }
    CK(cudaStreamSynchronize(ctx->down_stream));
    CK(cudaStreamSynchronize(ctx->stream));
    if (h2d_bytes) *h2d_bytes = up;
    if (d2h_bytes) *d2h_bytes = down;
    return ENT_OK;
}
