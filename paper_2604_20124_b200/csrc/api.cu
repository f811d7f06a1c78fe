// api.cu -- the C-ABI of include/spray.h: argument checks, scratch ownership, kernel sequencing.
// Every step of the path runs in CUDA kernels enqueued on the caller's stream; nothing here touches particle
// data on the host and there is no CPU fallback.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "spray_internal.h"

using namespace spray;

namespace {

thread_local char g_noctx_err[256] = "";

int fail(Ctx* c, int code, const char* fmt, const char* a = "") {
    char buf[512];
    snprintf(buf, sizeof buf, fmt, a);
    if (c) c->err = buf;
    else { strncpy(g_noctx_err, buf, sizeof g_noctx_err - 1); }
    return code;
}
int cuda_fail(Ctx* c, cudaError_t e, const char* where) {
    char buf[512];
    snprintf(buf, sizeof buf, "CUDA error in %s: %s", where, cudaGetErrorString(e));
    if (c) c->err = buf;
    return SPRAY_ERR_CUDA;
}

template <class T>
bool dmalloc(T** p, int64_t count, Ctx* c = nullptr) {
    if (count < 1) count = 1;
    if (cudaMalloc((void**)p, sizeof(T) * (size_t)count) != cudaSuccess) return false;
    if (c) c->scratch_bytes += (int64_t)(sizeof(T) * (size_t)count);
    return true;
}

void free_all(Ctx* c) {
    for (int k = 0; k < 2; ++k) { cudaFree(c->key[k]); cudaFree(c->idx[k]); }
    cudaFree(c->hist); cudaFree(c->cell_start); cudaFree(c->cell_end); cudaFree(c->cell_hmax);
    cudaFree(c->hglob); cudaFree(c->dev_status); cudaFree(c->cell_tend); cudaFree(c->cell_hmin); cudaFree(c->left); cudaFree(c->hs_c); cudaFree(c->fast_c); cudaFree(c->fast_all);
    for (double* r : c->rad_scratch) cudaFree(r);
    cudaFree(c->s.x); cudaFree(c->s.y); cudaFree(c->s.z); cudaFree(c->s.h); cudaFree(c->s.hs);
    for (double* f : c->s.f) cudaFree(f);
    Packed& k = c->pk;
    cudaFree(k.p0); cudaFree(k.p1); cudaFree(k.hh); cudaFree(k.t0); cudaFree(k.me); cudaFree(k.e1);
    for (double2* r : k.s) cudaFree(r);
    Tiled& t = c->tl;
    cudaFree(t.tiles); cudaFree(t.bcount); cudaFree(t.pool); cudaFree(t.ctr); cudaFree(t.winfo); cudaFree(t.lcount);
    cudaFree(t.tflags); cudaFree(t.tiletab); cudaFree(t.fast);
}

// Scratch of the tiled path (tiles, tile tables, neighbour-list pool), allocated once by spray_create from n_max and
// ncell_max -- spray_build_cells never allocates, frees or synchronises.  Capacities: a bundle is a 2 x 2 block of cell
// rows, so a grid has ceil(ny/2) ceil(nz/2) of them: room for 4 ncell_max^(2/3) (at least 4096), which covers every
// grid whose x extent is not much shorter than the other two; tiles: twice n_max / TILE_T plus the partial tiles at bundle
// ends and column cuts (a tile cut into parts takes an entry per part; groups beyond the capacity are not served); list pool: 208 bytes per particle (two bytes per neighbour and list padding; ~100 neighbours).
// A build that needs more than this is served by the general kernels (whole grid or, for the pool, unit by unit).
// Failure to allocate is not an error either: the general kernels then serve every particle.
void alloc_tiled(Ctx* c) {
    Tiled& t = c->tl;
    const int64_t n = c->n_max;
    int64_t nb = 4 * (int64_t)ceil(pow((double)c->ncell_max, 2.0 / 3.0));
    nb = nb < 4096 ? 4096 : nb;
    nb = nb > c->ncell_max ? c->ncell_max : nb;
    const int64_t tiles = 2 * ((n + TILE_T - 1) / TILE_T) + 2 * nb + c->ncell_max / 64 + 256;   // (tiles in several parts take an entry per part)
    const int64_t rows = (n * 208) / 256 + 4096;
    bool ok = dmalloc(&t.tiles, tiles, c) && dmalloc(&t.bcount, nb + 4096 + 64, c) && dmalloc(&t.winfo, tiles * TILE_WARPS, c) &&
              dmalloc(&t.lcount, tiles * TILE_T, c) && dmalloc(&t.tflags, tiles, c) && dmalloc(&t.tiletab, tiles * TILES_WORDS, c) &&
              dmalloc(&t.pool, rows * 32, c) && dmalloc(&t.ctr, CTR_COUNT, c) && dmalloc(&t.fast, n, c);
    if (ok) ok = tiled_set_attributes(c) == cudaSuccess;
    if (!ok) {
        cudaGetLastError();
        cudaFree(t.tiles); cudaFree(t.bcount); cudaFree(t.pool); cudaFree(t.winfo); cudaFree(t.lcount); cudaFree(t.tflags); cudaFree(t.tiletab);
        cudaFree(t.ctr); cudaFree(t.fast);
        t = Tiled{};
        int sms = 0;
        if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device) == cudaSuccess && sms > 0) t.sms = sms;
        return;
    }
    t.tile_cap = tiles; t.bundle_cap = nb; t.pool_rows = rows > 0xFFFFFFF0ll ? 0xFFFFFFF0ll : rows;
}

// every entry point runs on the context's device and leaves the caller's current device as it found it
struct DeviceGuard {
    int prev = -1;
    bool ok = true;
    explicit DeviceGuard(int dev) {
        if (cudaGetDevice(&prev) != cudaSuccess) { prev = -1; cudaGetLastError(); }
        if (prev != dev) ok = cudaSetDevice(dev) == cudaSuccess;
        if (prev == dev) prev = -1;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

SweepArgs base_args(Ctx* c) {
    SweepArgs a;
    memset(&a, 0, sizeof a);
    a.x = c->s.x; a.y = c->s.y; a.z = c->s.z; a.h = c->s.h; a.hs = c->s.hs;
    return a;
}

// general-kernel arguments of a sweep that the tiled kernels ran first: skip what they served (levels = the call also ran the
// tiled kernels of the internal levels)
// the context whose grid and sorted copies the general kernels of a level-aware call use: with levels on, the finest level
// that was built (build_levels), else the context itself
Ctx* general_ctx(Ctx* c) { return (c->levels_on && c->general) ? c->general : c; }

SweepArgs fallback_args(Ctx* c, bool levels = false) {
    if (levels && c->levels_on && c->general) {
        Ctx* g = c->general;
        SweepArgs a = base_args(g);
        a.skip = g->fast_all; a.nfast = c->tl.ctr + CTR_NFAST_ALL; a.left = g->left; a.nleft = g->tl.ctr + CTR_NLEFT;
        return a;
    }
    SweepArgs a = base_args(c);
    if (levels && c->levels_on) { a.skip = c->fast_all; a.nfast = c->tl.ctr + CTR_NFAST_ALL; a.left = c->left; a.nleft = c->tl.ctr + CTR_NLEFT; }
    else if (c->tl.enabled) {
        a.skip = c->tl.fast; a.nfast = c->tl.ctr + CTR_NFAST;
        if (!c->levels_on) { a.left = c->left; a.nleft = c->tl.ctr + CTR_NLEFT; }   // (with levels the list holds what is left after them)
    }
    return a;
}

enum { F_M = 0, F_RHO, F_P, F_CS, F_VX, F_VY, F_VZ, F_ALPHA, F_E, F_KAPPA, F_MU, F_V, F_Q, F_AC };

// the per-call prologue of a level context: same caller arrays, the level's own sorted scratch
PrepJob level_job(const PrepJob& j, Ctx* v) {
    PrepJob r = j;
    double** f = v->s.f;
    if (j.sm) r.sm = f[F_M];
    if (j.srho) r.srho = f[F_RHO];
    if (j.sp) r.sp = f[F_P];
    if (j.scs) r.scs = f[F_CS];
    if (j.svx) r.svx = f[F_VX];
    if (j.svy) r.svy = f[F_VY];
    if (j.svz) r.svz = f[F_VZ];
    if (j.salpha) r.salpha = f[F_ALPHA];
    if (j.sE) r.sE = f[F_E];
    if (j.skx) r.skx = j.kx_is_mu ? f[F_MU] : f[F_KAPPA];
    if (j.sV) r.sV = f[F_V];
    if (j.sQ) r.sQ = f[F_Q];
    if (j.sAC) r.sAC = f[F_AC];
    return r;
}

// the contexts whose tiled kernels serve particles of this one: itself and its levels
struct TiledSet { Ctx* v[1 + SPRAY_MAX_LEVELS]; int n = 0; };
TiledSet tiled_set(Ctx* c) {
    TiledSet s;
    if (c->tl.enabled) s.v[s.n++] = c;
    if (c->levels_on)
        for (int k = 0; k < c->nlevels; ++k)
            if (c->child[k] && c->child[k]->built && c->child[k]->tl.enabled) s.v[s.n++] = c->child[k];
    return s;
}

#define CK(call, where) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) return cuda_fail(c, e__, where); } while (0)
#define NEED_BUILT() if (!ctx) return SPRAY_ERR_INVALID_ARG; \
    if (!ctx->c.built) return fail(&ctx->c, SPRAY_ERR_NOT_BUILT, "spray_build_cells has not succeeded on this context"); \
    DeviceGuard dev_guard__(ctx->c.device); \
    if (!dev_guard__.ok) { cudaGetLastError(); return fail(&ctx->c, SPRAY_ERR_CUDA, "cudaSetDevice failed"); }


}  // namespace

extern "C" {

const char* spray_version(void) { return "spray-b200 0.1 sm_100a"; }

int spray_create(spray_ctx** out, int64_t n_max, int64_t ncell_max, int device) {
    // n_max <= 2^28: the radix sort scans its digit histograms in two levels of 4096 (build.cu), which covers 2^28 keys
    if (!out || n_max < 0 || ncell_max < 1 || n_max > (1ll << 28) || ncell_max > 0x7FFFFFFFll)
        return fail(nullptr, SPRAY_ERR_INVALID_ARG, "spray_create: bad arguments (n_max <= 2^28, 1 <= ncell_max < 2^31)");
    DeviceGuard dg(device);
    if (!dg.ok) { cudaGetLastError(); return fail(nullptr, SPRAY_ERR_CUDA, "spray_create: cudaSetDevice failed"); }
    spray_ctx* h = new (std::nothrow) spray_ctx();
    if (!h) return SPRAY_ERR_ALLOC;
    Ctx* c = &h->c;
    c->device = device; c->n_max = n_max; c->ncell_max = ncell_max;
    c->path = 1;
    int sms = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device) == cudaSuccess && sms > 0) c->tl.sms = sms;
    c->hist_cap = 256 * ((n_max + 4095) / 4096 + 1) + 4096;   // radix histograms + block totals of their scan
    bool ok = true;
    for (int k = 0; k < 2; ++k) ok = ok && dmalloc(&c->key[k], n_max, c) && dmalloc(&c->idx[k], n_max, c);
    ok = ok && dmalloc(&c->hist, c->hist_cap, c) && dmalloc(&c->cell_start, ncell_max, c) && dmalloc(&c->cell_end, ncell_max, c) &&
         dmalloc(&c->cell_hmax, ncell_max, c) && dmalloc(&c->cell_tend, ncell_max, c) && dmalloc(&c->cell_hmin, ncell_max, c) && dmalloc(&c->left, n_max, c) &&
         dmalloc(&c->hs_c, n_max, c) &&
         dmalloc(&c->fast_c, n_max, c) && dmalloc(&c->fast_all, n_max, c) && dmalloc(&c->hglob, 4, c) && dmalloc(&c->dev_status, 1, c) && dmalloc(&c->s.x, n_max, c) &&
         dmalloc(&c->s.y, n_max, c) && dmalloc(&c->s.z, n_max, c) && dmalloc(&c->s.h, n_max, c) && dmalloc(&c->s.hs, n_max, c);
    for (double*& f : c->s.f) ok = ok && dmalloc(&f, n_max, c);
    Packed& k = c->pk;
    ok = ok && dmalloc(&k.p0, n_max, c) && dmalloc(&k.p1, n_max, c) && dmalloc(&k.hh, n_max, c) && dmalloc(&k.t0, n_max, c) &&
         dmalloc(&k.me, n_max, c) && dmalloc(&k.e1, n_max, c);
    for (double2*& r : k.s) ok = ok && dmalloc(&r, n_max, c);
    for (double*& r : c->rad_scratch) ok = ok && dmalloc(&r, n_max, c);     // rows N1, N2: y, Lambda, Gamma, chi / g, y of two species
    if (ok) ok = cudaMemset(c->dev_status, 0, sizeof(uint32_t)) == cudaSuccess;
    if (!ok) {
        cudaGetLastError();
        free_all(c);
        delete h;
        return fail(nullptr, SPRAY_ERR_ALLOC, "spray_create: device allocation failed");
    }
    alloc_tiled(c);
    for (cudaEvent_t& e : c->ev)
        if (cudaEventCreate(&e) != cudaSuccess) { cudaGetLastError(); e = nullptr; }
    *out = h;
    return SPRAY_OK;
}

static void destroy_levels(Ctx* c) {
    for (int k = 0; k < c->nlevels; ++k) {
        if (!c->child[k]) continue;
        spray_ctx* h = reinterpret_cast<spray_ctx*>(c->child[k]);     // Ctx is the first (only) member of spray_ctx
        for (cudaEvent_t e : h->c.ev) if (e) cudaEventDestroy(e);
        c->scratch_bytes -= h->c.scratch_bytes;
        free_all(&h->c);
        delete h;
        c->child[k] = nullptr;
    }
    c->nlevels = 0;
    c->levels_on = false;
    c->general = nullptr;
}

int spray_set_levels(spray_ctx* ctx, int nlevels, const double* edges, const int64_t* ncell_max) {
    if (!ctx) return SPRAY_ERR_INVALID_ARG;
    Ctx* c = &ctx->c;
    if (nlevels < 0 || nlevels > SPRAY_MAX_LEVELS || (nlevels > 0 && (!edges || !ncell_max)))
        return fail(c, SPRAY_ERR_INVALID_ARG, "spray_set_levels: 0 <= nlevels <= 16, edges and ncell_max non-NULL");
    for (int k = 0; k < nlevels; ++k)
        if (!(edges[k] > 0.0) || (k > 0 && !(edges[k] > edges[k - 1])) || ncell_max[k] < 1)
            return fail(c, SPRAY_ERR_INVALID_ARG, "spray_set_levels: edges must be positive and ascending, ncell_max >= 1");
    DeviceGuard dg(c->device);
    if (!dg.ok) { cudaGetLastError(); return fail(c, SPRAY_ERR_CUDA, "cudaSetDevice failed"); }
    cudaDeviceSynchronize();
    destroy_levels(c);
    c->built = false;
    for (int k = 0; k < nlevels; ++k) {
        spray_ctx* h = nullptr;
        const int rc = spray_create(&h, c->n_max, ncell_max[k], c->device);
        if (rc != SPRAY_OK) { destroy_levels(c); return fail(c, rc, "spray_set_levels: allocation of a level failed"); }
        h->c.is_level = true;
        c->child[k] = &h->c;
        c->level_edge[k] = edges[k];
        c->nlevels = k + 1;
        c->scratch_bytes += h->c.scratch_bytes;
    }
    return SPRAY_OK;
}

int spray_destroy(spray_ctx* ctx) {
    if (!ctx) return SPRAY_OK;
    DeviceGuard dg(ctx->c.device);
    cudaDeviceSynchronize();
    destroy_levels(&ctx->c);
    for (cudaEvent_t e : ctx->c.ev) if (e) cudaEventDestroy(e);
    free_all(&ctx->c);
    delete ctx;
    return SPRAY_OK;
}

const char* spray_last_error(const spray_ctx* ctx) { return ctx ? ctx->c.err.c_str() : g_noctx_err; }

int spray_check(spray_ctx* ctx, void* stream, uint32_t* dev_status) {
    if (!ctx) return SPRAY_ERR_INVALID_ARG;
    Ctx* c = &ctx->c;
    DeviceGuard dg(c->device);
    cudaStream_t st = (cudaStream_t)stream;
    CK(cudaStreamSynchronize(st), "spray_check (a kernel enqueued earlier faulted)");
    uint32_t v = 0;
    CK(cudaMemcpy(&v, c->dev_status, sizeof v, cudaMemcpyDeviceToHost), "spray_check");
    CK(cudaMemset(c->dev_status, 0, sizeof v), "spray_check");
    if (dev_status) *dev_status = v;
    return SPRAY_OK;
}

int64_t spray_launch_count(const spray_ctx* ctx) { return ctx ? ctx->c.launches : 0; }

int spray_set_path(spray_ctx* ctx, int path) {
    if (!ctx) return SPRAY_ERR_INVALID_ARG;
    if (path != 0 && path != 1) return fail(&ctx->c, SPRAY_ERR_INVALID_ARG, "spray_set_path: path must be 0 or 1");
    ctx->c.path = path;
    ctx->c.built = false;           // the neighbour lists belong to a path: rebuild the cells after switching
    return SPRAY_OK;
}

int spray_path_stats(spray_ctx* ctx, void* stream, int64_t* n_tiles, int64_t* n_fast, int64_t* n_nonuniform,
                     int64_t* scratch_bytes, int64_t* declined) {
    NEED_BUILT();
    Ctx* c = &ctx->c;
    cudaStream_t st = (cudaStream_t)stream;
    unsigned long long v[CTR_COUNT] = {};
    int64_t tiles = 0, nonuni = 0, dec[4] = {0, 0, 0, 0}, nfast = 0;
    if (c->n > 0 && (c->tl.enabled || c->levels_on)) {
        CK(cudaStreamSynchronize(st), "spray_path_stats");
        const TiledSet ts = tiled_set(c);
        for (int k = 0; k < ts.n; ++k) {
            CK(cudaMemcpy(v, ts.v[k]->tl.ctr, sizeof v, cudaMemcpyDeviceToHost), "spray_path_stats");
            tiles += (int64_t)v[CTR_NTILES]; nonuni += (int64_t)v[CTR_NNONUNI];
            if (getenv("SPRAY_DEBUG"))
                fprintf(stderr, "[spray] %s grid %d x %d x %d  2hs in (%.4g, %.4g]  tiles %llu  served %llu  nonuniform units %llu  declined %llu %llu %llu\n",
                        ts.v[k] == c ? "caller grid" : "level", ts.v[k]->grid.ncell[0], ts.v[k]->grid.ncell[1], ts.v[k]->grid.ncell[2],
                        ts.v[k]->level_lo, ts.v[k]->level_hi, v[CTR_NTILES], v[CTR_NFAST], v[CTR_NNONUNI], v[CTR_DECL + 1], v[CTR_DECL + 2], v[CTR_DECL + 3]);
            for (int r = 0; r < 4; ++r) dec[r] += (int64_t)v[CTR_DECL + r];
            if (!c->levels_on) nfast += (int64_t)v[CTR_NFAST];
        }
        if (c->levels_on) {
            CK(cudaMemcpy(v, c->tl.ctr, sizeof v, cudaMemcpyDeviceToHost), "spray_path_stats");
            nfast = (int64_t)v[CTR_NFAST_ALL];
        }
    }
    if (n_tiles) *n_tiles = tiles;
    if (n_fast) *n_fast = nfast;
    if (n_nonuniform) *n_nonuniform = nonuni;
    if (scratch_bytes) *scratch_bytes = c->scratch_bytes;
    if (declined) for (int k = 0; k < 4; ++k) declined[k] = dec[k];
    return SPRAY_OK;
}

// Internal levels of the tiled path (spray_set_levels; the search range follows from the ratio of a
// particle's smoothing length to the cell size, neighbours are mutual).  Level k is a grid over the caller's box with
// ncell_d = floor(L_d / edge_k) cells; it serves the particles a that nobody served yet with hi_(k-1) < 2 hs_a <= hi_k, where
// hs_a is the symmetric search length (max of h_a and of the h of everyone who sees a) and hi_k the smallest cell edge of
// the level: every mutual neighbour of such a particle lies within one cell of its own.  The level sorts ALL particles by
// (cell, served-here bit), so the targets of a cell come first and every particle is a candidate; tiles, lists and sweeps
// are those of tiles.cu / sweeps_tiled.cu unchanged.  What no level takes stays with the general kernels of this context.
static int build_levels(Ctx* c, const double* x, const double* y, const double* z, const double* h, cudaStream_t st) {
    CK(launch_to_caller_order(c, st), "levels: search lengths to caller order");
    double lo = 0.0;
    for (int k = 0; k < c->nlevels; ++k) {
        Ctx* v = c->child[k];
        v->built = false; v->tl.enabled = false; v->soa_ctr = nullptr;
        spray_grid_t g = c->grid;
        int64_t nc = 1;
        double emin = 1e300, emax = 0.0;
        bool ok = true;
        for (int d = 0; d < 3; ++d) {
            const double L = g.hi[d] - g.lo[d];
            int64_t m = (int64_t)floor(L / c->level_edge[k] * (1.0 + 1e-12));
            m = m < 1 ? 1 : (m > 32000 ? 32000 : m);
            g.ncell[d] = (int32_t)m;
            nc *= m;
            emin = fmin(emin, L / (double)m); emax = fmax(emax, L / (double)m);
        }
        if (nc > v->ncell_max) ok = false;
        const double hi = emin / (1.0 + 1e-9);
        if (!ok || !(hi > lo)) continue;                  // the level cannot be built on this box: its particles stay unserved
        v->grid = g; v->kernel = c->kernel; v->n = c->n; v->ncell = nc; v->path = 1;
        for (int d = 0; d < 3; ++d) {
            v->dg.lo[d] = g.lo[d]; v->dg.L[d] = g.hi[d] - g.lo[d]; v->dg.halfL[d] = 0.5 * v->dg.L[d];
            v->dg.inv[d] = (double)g.ncell[d] / v->dg.L[d]; v->dg.edge[d] = v->dg.L[d] / (double)g.ncell[d];
            v->dg.nc[d] = g.ncell[d]; v->dg.per[d] = g.periodic[d] ? 1 : 0;
        }
        v->level_lo = lo; v->level_hi = hi;
        v->level_rmax = (float)(3.5 * emax * (1.0 + 1e-6));   // every candidate of a window lies within 2 cells per dimension
        v->hs_caller = c->hs_c; v->fast_caller = c->fast_c;
        Ctx* keep = c;
        {
            Ctx* c = v;                                   // CK reports into the level's context
            CK(launch_cell_keys(c, x, y, z, st), "level: cell keys");
            CK(launch_radix_sort(c, st), "level: radix sort");
            CK(launch_cell_table(c, st), "level: cell table");
            CK(launch_reorder_build(c, x, y, z, h, st), "level: reorder");
            CK(launch_build_tiles(c, st), "level: tiles + neighbour lists");
            c->built = true;
        }
        c = keep;
        CK(launch_merge_served(c, v, st), "levels: served flags");
        lo = hi;
    }
    CK(launch_fast_from_caller(c, st), "levels: served flags to sorted order");
    CK(launch_compact_left(c, c->fast_all, st), "levels: list of the particles left to the general kernels");
    // The general kernels of the level-aware calls run on the finest level that was built: where particles are left over they
    // are dense for their search length (that is why no level could tile them), and the caller's grid (A14: 2 mean(h)) holds
    // ~140 of them per cell at config 4 against ~18 on the finest level's.  That context gets what the general kernels need on
    // top of a level's own: per-cell h_max / h_min, hs and the served flags in its sorted order, the list of the left-overs.
    c->general = nullptr;
    for (int k = 0; k < c->nlevels && !c->general; ++k) {
        Ctx* v = c->child[k];
        if (!v || !v->built || !v->tl.enabled) continue;
        CK(launch_cell_hmax(v, st), "levels: per-cell h_max of the general kernels' grid");
        CK(launch_general_from_parent(v, c, st), "levels: search lengths and served flags on the general kernels' grid");
        CK(launch_compact_left(v, v->fast_all, st), "levels: left-over list on the general kernels' grid");
        v->soa_ctr = c->tl.ctr + CTR_NFAST_ALL;
        c->general = v;
    }
    c->levels_on = true;
    return SPRAY_OK;
}

int spray_build_timing(spray_ctx* ctx, double* ms_cells, double* ms_tiles, double* ms_lists) {
    NEED_BUILT();
    Ctx* c = &ctx->c;
    for (cudaEvent_t e : c->ev) if (!e) return fail(c, SPRAY_ERR_CUDA, "spray_build_timing: no events");
    CK(cudaEventSynchronize(c->ev[3]), "spray_build_timing");
    float a = 0.f, b = 0.f, d = 0.f;
    CK(cudaEventElapsedTime(&a, c->ev[0], c->ev[1]), "spray_build_timing");
    if (c->tl.enabled) {
        CK(cudaEventElapsedTime(&b, c->ev[1], c->ev[2]), "spray_build_timing");
        CK(cudaEventElapsedTime(&d, c->ev[2], c->ev[3]), "spray_build_timing");
    }
    if (ms_cells) *ms_cells = a;
    if (ms_tiles) *ms_tiles = b;
    if (ms_lists) *ms_lists = d;
    return SPRAY_OK;
}

int spray_build_cells(spray_ctx* ctx, const spray_grid_t* g, spray_kernel_t kernel, int64_t n, const double* x,
                      const double* y, const double* z, const double* h, void* stream) {
    if (!ctx) return SPRAY_ERR_INVALID_ARG;
    Ctx* c = &ctx->c;
    c->built = false;
    c->chain_ok = false;
    DeviceGuard dg(c->device);
    if (!dg.ok) { cudaGetLastError(); return fail(c, SPRAY_ERR_CUDA, "cudaSetDevice failed"); }
    if (!g || n < 0 || (n > 0 && (!x || !y || !z || !h))) return fail(c, SPRAY_ERR_INVALID_ARG, "spray_build_cells: NULL argument or n < 0");
    if (kernel != SPRAY_KERNEL_CUBIC_SPLINE && kernel != SPRAY_KERNEL_WENDLAND_C2)
        return fail(c, SPRAY_ERR_INVALID_ARG, "spray_build_cells: unknown kernel id");
    if (n > c->n_max) return fail(c, SPRAY_ERR_CAPACITY, "spray_build_cells: n > n_max");
    int64_t nc = 1;
    for (int d = 0; d < 3; ++d) {
        if (g->ncell[d] < 1) return fail(c, SPRAY_ERR_GRID, "grid: ncell_d < 1");
        if (!(g->hi[d] > g->lo[d])) return fail(c, SPRAY_ERR_GRID, "grid: hi <= lo");
        nc *= g->ncell[d];
        if (nc > c->ncell_max) return fail(c, SPRAY_ERR_GRID, "grid: prod ncell_d > ncell_max");
        if (g->periodic[d] && !((g->hi[d] - g->lo[d]) >= 3.0 * (2.0 * g->h_max)))
            return fail(c, SPRAY_ERR_GRID, "grid: periodic extent L_d < 3*(2*h_max): the minimum image would be ambiguous");
    }
    if (!(g->h_max > 0.0)) return fail(c, SPRAY_ERR_GRID, "grid: h_max must be > 0");
    c->grid = *g; c->kernel = (int)kernel; c->n = n; c->ncell = nc;
    for (int d = 0; d < 3; ++d) {
        c->dg.lo[d] = g->lo[d];
        c->dg.L[d] = g->hi[d] - g->lo[d];
        c->dg.halfL[d] = 0.5 * c->dg.L[d];
        c->dg.edge[d] = c->dg.L[d] / (double)g->ncell[d];
        c->dg.inv[d] = (double)g->ncell[d] / c->dg.L[d];
        c->dg.nc[d] = g->ncell[d];
        c->dg.per[d] = g->periodic[d] ? 1 : 0;
    }
    cudaStream_t st = (cudaStream_t)stream;
    if (c->ev[0]) cudaEventRecord(c->ev[0], st);
    CK(launch_cell_keys(c, x, y, z, st), "cell keys");
    CK(launch_radix_sort(c, st), "radix sort");
    CK(launch_cell_table(c, st), "cell table");
    c->tl.enabled = false;
    CK(launch_reorder_build(c, x, y, z, h, st), "reorder");
    CK(launch_cell_hmax(c, st), "cell hmax");
    // symmetric search length: hs = h, then raised by every particle that sees me with a larger h
    if (n > 0) CK(cudaMemcpyAsync(c->s.hs, c->s.h, sizeof(double) * (size_t)n, cudaMemcpyDeviceToDevice, st), "hs init");
    SweepArgs a = base_args(c);
    a.o0 = c->s.hs;
    if (c->tl.pool && (int64_t)c->tl.pool_rows * 256 >= 16 * n) {
        // fp32 copies for the pre-test, in the list pool (free until the lists of this build are written)
        float4* f4 = reinterpret_cast<float4*>(c->tl.pool);
        CK(launch_pack_f4(c, f4, st), "search lengths: fp32 positions");
        a.f4 = f4;
        double cm = 0.0;
        for (int d = 0; d < 3; ++d) cm = fmax(cm, fmax(fabs(g->lo[d]), fabs(g->hi[d])));
        a.f4_cmax = (float)cm;
    }
    CK(launch_ref_sweep(c, SW_HSEARCH, a, st), "search-length sweep");
    if (c->ev[1]) cudaEventRecord(c->ev[1], st);
    if (c->path == 1) CK(launch_build_tiles(c, st), "tiles + neighbour lists");
    if (c->tl.enabled) CK(launch_compact_left(c, c->tl.fast, st), "list of the particles left to the general kernels");
    c->levels_on = false;
    if (c->path == 1 && c->nlevels > 0 && n > 0) {
        const int rc = build_levels(c, x, y, z, h, st);
        if (rc != SPRAY_OK) return rc;
    }
    if (c->ev[3]) cudaEventRecord(c->ev[3], st);
    c->built = true;
    return SPRAY_OK;
}

int spray_density(spray_ctx* ctx, const double* m, double* rho, uint32_t* nnbr, void* stream) {
    NEED_BUILT();
    Ctx* c = &ctx->c;
    c->chain_ok = false;
    if (c->n > 0 && (!m || !rho)) return fail(c, SPRAY_ERR_INVALID_ARG, "spray_density: NULL argument");
    cudaStream_t st = (cudaStream_t)stream;
    CK(launch_prep_density(c, m, st), "density prologue");
    const TiledSet ts = tiled_set(c);
    for (int k = 0; k < ts.n; ++k) {
        if (ts.v[k] != c) CK(launch_prep_density(ts.v[k], m, st), "density prologue (level)");
        TiledArgs t{};
        t.o0 = rho; t.ocount = nnbr;
        CK(launch_tiled_sweep(ts.v[k], SW_DENSITY, t, st), "tiled density sweep");
    }
    Ctx* gc = general_ctx(c);
    SweepArgs a = fallback_args(c, true);
    a.m = gc->s.f[F_M]; a.o0 = rho; a.ocount = nnbr;
    CK(launch_ref_sweep(gc, SW_DENSITY, a, st), "density sweep");
    return SPRAY_OK;
}

int spray_hydro_rhs(spray_ctx* ctx, const double* m, const double* rho, const double* p, const double* cs,
                    const double* vx, const double* vy, const double* vz, const double* alpha, double beta,
                    double* ax, double* ay, double* az, double* dudt, double* divv_sum, void* stream) {
    NEED_BUILT();
    Ctx* c = &ctx->c;
    c->chain_ok = false;
    if (c->n > 0 && (!m || !rho || !p || !cs || !vx || !vy || !vz || !alpha || !ax || !ay || !az || !dudt))
        return fail(c, SPRAY_ERR_INVALID_ARG, "spray_hydro_rhs: NULL argument");
    cudaStream_t st = (cudaStream_t)stream;
    double** f = c->s.f;
    PrepJob pj{};
    pj.m = m; pj.rho = rho; pj.p = p; pj.cs = cs; pj.vx = vx; pj.vy = vy; pj.vz = vz; pj.alpha = alpha;
    pj.sm = f[F_M]; pj.srho = f[F_RHO]; pj.sp = f[F_P]; pj.scs = f[F_CS]; pj.svx = f[F_VX]; pj.svy = f[F_VY]; pj.svz = f[F_VZ];
    pj.salpha = f[F_ALPHA]; pj.sV = f[F_V]; pj.sQ = f[F_Q]; pj.sAC = f[F_AC];
    CK(launch_prep_hydro(c, pj, st), "hydro prologue");
    const TiledSet ts = tiled_set(c);
    for (int k = 0; k < ts.n; ++k) {
        if (ts.v[k] != c) CK(launch_prep_hydro(ts.v[k], level_job(pj, ts.v[k]), st), "hydro prologue (level)");
        TiledArgs t{};
        t.beta = beta;
        t.o0 = ax; t.o1 = ay; t.o2 = az; t.o3 = dudt; t.o4 = divv_sum;
        CK(launch_tiled_sweep(ts.v[k], SW_HYDRO, t, st), "tiled hydro sweep");
    }
    Ctx* gc = general_ctx(c);
    f = gc->s.f;
    SweepArgs a = fallback_args(c, true);
    a.m = f[F_M]; a.rho = f[F_RHO]; a.p = f[F_P]; a.cs = f[F_CS];
    a.vx = f[F_VX]; a.vy = f[F_VY]; a.vz = f[F_VZ]; a.alpha = f[F_ALPHA];
    a.beta = beta;
    a.o0 = ax; a.o1 = ay; a.o2 = az; a.o3 = dudt; a.o4 = divv_sum;
    CK(launch_ref_sweep(gc, SW_HYDRO, a, st), "hydro sweep");
    return SPRAY_OK;
}

int spray_hydro_rhs_limiter(spray_ctx* ctx, const double* m, const double* rho, const double* p, const double* cs,
                            const double* vx, const double* vy, const double* vz, const double* alpha, double beta,
                            const double* E, const double* kappa, double c_light,
                            double* ax, double* ay, double* az, double* dudt, double* divv_sum, double* mu, double* gradE, void* stream) {
    NEED_BUILT();
    Ctx* c = &ctx->c;
    if (c->n > 0 && (!m || !rho || !p || !cs || !vx || !vy || !vz || !alpha || !E || !kappa || !ax || !ay || !az || !dudt || !mu))
        return fail(c, SPRAY_ERR_INVALID_ARG, "spray_hydro_rhs_limiter: NULL argument");
    cudaStream_t st = (cudaStream_t)stream;
    double** f = c->s.f;
    PrepJob pj{};
    pj.m = m; pj.rho = rho; pj.p = p; pj.cs = cs; pj.vx = vx; pj.vy = vy; pj.vz = vz; pj.alpha = alpha;
    pj.sm = f[F_M]; pj.srho = f[F_RHO]; pj.sp = f[F_P]; pj.scs = f[F_CS]; pj.svx = f[F_VX]; pj.svy = f[F_VY]; pj.svz = f[F_VZ];
    pj.salpha = f[F_ALPHA]; pj.sV = f[F_V]; pj.sQ = f[F_Q]; pj.sAC = f[F_AC];
    // the limiter's prologue rides along: E, and rho kappa parked in the (mu, E) record so that t0 stays the hydro's
    pj.E = E; pj.kx = kappa; pj.sE = f[F_E]; pj.skx = f[F_KAPPA];
    CK(launch_prep_hydro(c, pj, st), "hydro + limiter prologue");
    const TiledSet ts = tiled_set(c);
    for (int k = 0; k < ts.n; ++k) {
        if (ts.v[k] != c) CK(launch_prep_hydro(ts.v[k], level_job(pj, ts.v[k]), st), "hydro + limiter prologue (level)");
        TiledArgs t{};
        t.beta = beta; t.c_light = c_light;
        t.o0 = ax; t.o1 = ay; t.o2 = az; t.o3 = dudt; t.o4 = divv_sum; t.o5 = mu; t.o6 = gradE;
        CK(launch_tiled_sweep(ts.v[k], SW_HYDLIM, t, st), "tiled hydro + limiter sweep");
    }
    Ctx* gc = general_ctx(c);
    f = gc->s.f;
    SweepArgs a = fallback_args(c, true);
    a.m = f[F_M]; a.rho = f[F_RHO]; a.p = f[F_P]; a.cs = f[F_CS];
    a.vx = f[F_VX]; a.vy = f[F_VY]; a.vz = f[F_VZ]; a.alpha = f[F_ALPHA];
    a.beta = beta;
    a.o0 = ax; a.o1 = ay; a.o2 = az; a.o3 = dudt; a.o4 = divv_sum;
    CK(launch_ref_sweep(gc, SW_HYDRO, a, st), "hydro sweep");
    SweepArgs l = fallback_args(c, true);
    l.m = f[F_M]; l.rho = f[F_RHO]; l.E = f[F_E]; l.kappa = f[F_KAPPA]; l.mu = f[F_MU];
    l.c_light = c_light;
    l.o0 = mu; l.o1 = gradE; l.mu_sorted = f[F_MU]; l.me_sorted = gc->pk.me;
    CK(launch_ref_sweep(gc, SW_LIMITER, l, st), "limiter sweep");
    // the sorted (z, V) and (mu, E) records of every particle are in place: spray_fld_apply(SPRAY_FLD_FROZEN_CHAINED) may reuse them
    c->chain_ok = !c->levels_on;
    c->chain_m = m; c->chain_rho = rho; c->chain_E = E; c->chain_mu = mu;
    return SPRAY_OK;
}

int spray_fld_apply(spray_ctx* ctx, const double* m, const double* rho, const double* kappa, const double* E,
                    double c_light, spray_fld_kernel_mode_t kmode, spray_fld_limiter_mode_t lmode, double* mu, double* y,
                    double* diag, double* offd, double* gradE, void* stream) {
    NEED_BUILT();
    Ctx* c = &ctx->c;
    const bool update = (lmode == SPRAY_FLD_UPDATE_LIMITER);
    // FROZEN_CHAINED: FROZEN with the same m, rho, E and the mu that the spray_hydro_rhs_limiter call just before produced:
    // that call left the sorted records of the operator in place, so the prologue (a pass over all particles) is skipped
    bool chained = (lmode == SPRAY_FLD_FROZEN_CHAINED);
    if (chained && !(c->chain_ok && m == c->chain_m && rho == c->chain_rho && E == c->chain_E && mu == c->chain_mu)) {
        if (!c->levels_on) return fail(c, SPRAY_ERR_INVALID_ARG, "spray_fld_apply(FROZEN_CHAINED): not preceded by spray_hydro_rhs_limiter on the same arrays");
        chained = false;                                   // with internal levels the records are re-packed (FROZEN)
    }
    if (!chained) c->chain_ok = false;
    if (c->n > 0 && (!m || !rho || !E || !mu || !y || (update && !kappa)))
        return fail(c, SPRAY_ERR_INVALID_ARG, "spray_fld_apply: NULL argument");
    if ((kmode != SPRAY_FLD_SYMMETRIC && kmode != SPRAY_FLD_GATHER) ||
        (lmode != SPRAY_FLD_UPDATE_LIMITER && lmode != SPRAY_FLD_FROZEN && lmode != SPRAY_FLD_FROZEN_CHAINED))
        return fail(c, SPRAY_ERR_INVALID_ARG, "spray_fld_apply: unknown mode");
    cudaStream_t st = (cudaStream_t)stream;
    double** f = c->s.f;
    PrepJob pj{};
    pj.m = m; pj.rho = rho; pj.E = E; pj.kx = update ? kappa : mu; pj.kx_is_mu = update ? 0 : 1;
    pj.sm = f[F_M]; pj.srho = f[F_RHO]; pj.sE = f[F_E]; pj.skx = update ? f[F_KAPPA] : f[F_MU]; pj.sV = f[F_V];
    if (!chained) CK(launch_prep_fld(c, pj, st), "fld prologue");
    const TiledSet ts = tiled_set(c);
    for (int k = 0; k < ts.n; ++k)
        if (ts.v[k] != c) CK(launch_prep_fld(ts.v[k], level_job(pj, ts.v[k]), st), "fld prologue (level)");
    Ctx* gc = general_ctx(c);
    double** gf = gc->s.f;
    SweepArgs a = fallback_args(c, true);
    a.m = gf[F_M]; a.rho = gf[F_RHO]; a.E = gf[F_E]; a.kappa = gf[F_KAPPA]; a.mu = gf[F_MU];
    a.c_light = c_light;
    if (update) {
        for (int k = 0; k < ts.n; ++k) {
            TiledArgs t{};
            t.c_light = c_light; t.o0 = mu; t.o1 = gradE;
            CK(launch_tiled_sweep(ts.v[k], SW_LIMITER, t, st), "tiled limiter sweep");
        }
        SweepArgs l = a;
        l.o0 = mu; l.o1 = gradE; l.mu_sorted = gf[F_MU]; l.me_sorted = gc->pk.me;
        CK(launch_ref_sweep(gc, SW_LIMITER, l, st), "limiter sweep");
        if (c->levels_on) {
            // every context computed mu for the particles it serves only: the (mu, E) records and the sorted mu of all of them
            // are re-packed from the caller-order mu (as in FROZEN mode) before the apply
            PrepJob pm = pj;
            pm.kx = mu; pm.kx_is_mu = 1; pm.skx = f[F_MU];
            CK(launch_prep_fld(c, pm, st), "fld prologue (mu)");
            for (int k = 0; k < ts.n; ++k)
                if (ts.v[k] != c) CK(launch_prep_fld(ts.v[k], level_job(pm, ts.v[k]), st), "fld prologue (mu, level)");
        }
    }
    a.fld_sym = (kmode == SPRAY_FLD_SYMMETRIC) ? 1 : 0;
    for (int k = 0; k < ts.n; ++k) {
        TiledArgs t{};
        t.fld_sym = a.fld_sym;
        t.o0 = y; t.o1 = diag; t.o2 = offd;
        CK(launch_tiled_sweep(ts.v[k], SW_APPLY, t, st), "tiled apply sweep");
    }
    a.o0 = y; a.o1 = diag; a.o2 = offd;
    CK(launch_ref_sweep(gc, SW_APPLY, a, st), "apply sweep");
    return SPRAY_OK;
}

int spray_conduction(spray_ctx* ctx, const double* m, const double* rho, const double* k, const double* T, double* dudt,
                     void* stream) {
    NEED_BUILT();
    Ctx* c = &ctx->c;
    c->chain_ok = false;
    if (c->n > 0 && (!m || !rho || !k || !T || !dudt)) return fail(c, SPRAY_ERR_INVALID_ARG, "spray_conduction: NULL argument");
    cudaStream_t st = (cudaStream_t)stream;
    double** f = c->s.f;
    PrepJob pj{};                     // the frozen symmetric operator with mu = k, E = T
    pj.m = m; pj.rho = rho; pj.E = T; pj.kx = k; pj.kx_is_mu = 1;
    pj.sm = f[F_M]; pj.srho = f[F_RHO]; pj.sE = f[F_E]; pj.skx = f[F_MU]; pj.sV = f[F_V];
    CK(launch_prep_fld(c, pj, st), "conduction prologue");
    if (c->tl.enabled) {
        TiledArgs t{};
        t.fld_sym = 1; t.o0 = dudt;
        CK(launch_tiled_sweep(c, SW_APPLY, t, st), "conduction: tiled sweep");
    }
    SweepArgs a = fallback_args(c);
    a.m = f[F_M]; a.rho = f[F_RHO]; a.E = f[F_E]; a.mu = f[F_MU]; a.fld_sym = 1; a.o0 = dudt;
    CK(launch_ref_sweep(c, SW_APPLY, a, st), "conduction: sweep");
    CK(launch_div_by_rho(c, dudt, rho, st), "conduction: 1/rho");
    return SPRAY_OK;
}

// pair sum of the conduction operator for one species: y_a = sum_b V_b 4 k_a k_b/(k_a+k_b) (g_a - g_b) Fbar/r (not yet divided by rho_a)
static int cond_pair_sum(Ctx* c, const double* m, const double* rho, const double* k, const double* g, double* y, cudaStream_t st) {
    double** f = c->s.f;
    PrepJob pj{};
    pj.m = m; pj.rho = rho; pj.E = g; pj.kx = k; pj.kx_is_mu = 1;
    pj.sm = f[F_M]; pj.srho = f[F_RHO]; pj.sE = f[F_E]; pj.skx = f[F_MU]; pj.sV = f[F_V];
    CK(launch_prep_fld(c, pj, st), "implicit conduction: prologue");
    if (c->tl.enabled) {
        TiledArgs t{};
        t.fld_sym = 1; t.o0 = y;
        CK(launch_tiled_sweep(c, SW_APPLY, t, st), "implicit conduction: tiled sweep");
    }
    SweepArgs a = fallback_args(c);
    a.m = f[F_M]; a.rho = f[F_RHO]; a.E = f[F_E]; a.mu = f[F_MU]; a.fld_sym = 1; a.o0 = y;
    CK(launch_ref_sweep(c, SW_APPLY, a, st), "implicit conduction: sweep");
    return SPRAY_OK;
}

int spray_conduction_implicit(spray_ctx* ctx, const double* m, const double* rho, const double* k_i, const double* k_e,
                              const double* kei, const double* dTdu_i, const double* dTdu_e, const double* T_i, const double* T_e,
                              const double* u_i, const double* u_e, double dt, spray_cond_which_t which, double* out_i, double* out_e,
                              void* stream) {
    NEED_BUILT();
    Ctx* c = &ctx->c;
    c->chain_ok = false;
    if (which != SPRAY_COND_OPERATOR && which != SPRAY_COND_RHS) return fail(c, SPRAY_ERR_INVALID_ARG, "spray_conduction_implicit: unknown `which`");
    const bool rhs = which == SPRAY_COND_RHS;
    if (c->n > 0 && (!m || !rho || !k_i || !k_e || !kei || !dTdu_i || !dTdu_e || !u_i || !u_e || !out_i || !out_e || (rhs && (!T_i || !T_e))))
        return fail(c, SPRAY_ERR_INVALID_ARG, "spray_conduction_implicit: NULL argument");
    if (!(dt > 0.0)) return fail(c, SPRAY_ERR_INVALID_ARG, "spray_conduction_implicit: dt must be > 0");
    cudaStream_t st = (cudaStream_t)stream;
    CondArgs a{};
    a.rho = rho; a.kei = kei; a.tau_i = dTdu_i; a.tau_e = dTdu_e; a.T_i = T_i; a.T_e = T_e; a.u_i = u_i; a.u_e = u_e;
    a.g_i = c->rad_scratch[0]; a.g_e = c->rad_scratch[1]; a.y_i = c->rad_scratch[2]; a.y_e = c->rad_scratch[3];
    a.dt = dt; a.rhs = rhs ? 1 : 0; a.out_i = out_i; a.out_e = out_e;
    CK(launch_cond_form(c, a, st), "implicit conduction: g");
    int rc = cond_pair_sum(c, m, rho, k_i, a.g_i, c->rad_scratch[2], st);
    if (rc != SPRAY_OK) return rc;
    rc = cond_pair_sum(c, m, rho, k_e, a.g_e, c->rad_scratch[3], st);
    if (rc != SPRAY_OK) return rc;
    CK(launch_cond_combine(c, a, st), "implicit conduction: combine");
    return SPRAY_OK;
}

int spray_kgc_continuity(spray_ctx* ctx, const double* m, const double* rho, const double* vx, const double* vy,
                         const double* vz, double* drhodt, double* L, double* drhodt_raw, void* stream) {
    NEED_BUILT();
    Ctx* c = &ctx->c;
    c->chain_ok = false;
    if (c->n > 0 && (!m || !rho || !vx || !vy || !vz || !drhodt))
        return fail(c, SPRAY_ERR_INVALID_ARG, "spray_kgc_continuity: NULL argument");
    cudaStream_t st = (cudaStream_t)stream;
    double** f = c->s.f;
    PrepJob pj{};
    pj.m = m; pj.rho = rho; pj.vx = vx; pj.vy = vy; pj.vz = vz;
    pj.sm = f[F_M]; pj.srho = f[F_RHO]; pj.svx = f[F_VX]; pj.svy = f[F_VY]; pj.svz = f[F_VZ]; pj.sV = f[F_V];
    CK(launch_prep_kgc(c, pj, st), "kgc prologue");
    if (c->tl.enabled) {
        TiledArgs t{};
        t.o0 = drhodt; t.o1 = L; t.o2 = drhodt_raw;
        CK(launch_tiled_sweep(c, SW_KGC, t, st), "kgc: tiled sweep");
    }
    SweepArgs a = fallback_args(c);
    a.m = f[F_M]; a.rho = f[F_RHO]; a.vx = f[F_VX]; a.vy = f[F_VY]; a.vz = f[F_VZ];
    a.o0 = drhodt; a.o1 = L; a.o2 = drhodt_raw;
    CK(launch_ref_sweep(c, SW_KGC, a, st), "kgc: sweep");
    return SPRAY_OK;
}

int spray_rad_jacobi(spray_ctx* ctx, const double* m, const double* rho, const double* mu, const double* kappa_p,
                     const double* E_n, const double* u_n, const double* T_n, const double* dTdu, double dt, double c_light,
                     double a_rad, spray_fld_kernel_mode_t kmode, int niter, double* E, double* u, double* resid, void* stream) {
    NEED_BUILT();
    Ctx* c = &ctx->c;
    c->chain_ok = false;
    if (c->n > 0 && (!m || !rho || !mu || !kappa_p || !E_n || !u_n || !T_n || !dTdu || !E || !u))
        return fail(c, SPRAY_ERR_INVALID_ARG, "spray_rad_jacobi: NULL argument");
    if (!(dt > 0.0) || !(c_light > 0.0) || !(a_rad > 0.0) || niter < 1 || (kmode != SPRAY_FLD_SYMMETRIC && kmode != SPRAY_FLD_GATHER))
        return fail(c, SPRAY_ERR_INVALID_ARG, "spray_rad_jacobi: dt, c_light, a_rad must be > 0, niter >= 1, kmode valid");
    cudaStream_t st = (cudaStream_t)stream;
    double** f = c->s.f;
    // sorted records of the frozen operator: (z, V), (mu, E) with E = the starting iterate
    PrepJob pj{};
    pj.m = m; pj.rho = rho; pj.E = E; pj.kx = mu; pj.kx_is_mu = 1;
    pj.sm = f[F_M]; pj.srho = f[F_RHO]; pj.sE = f[F_E]; pj.skx = f[F_MU]; pj.sV = f[F_V];
    CK(launch_prep_fld(c, pj, st), "rad prologue");
    if (resid) CK(cudaMemsetAsync(resid, 0, sizeof(double) * (size_t)niter, st), "rad residuals");
    double *y = c->rad_scratch[0], *lam = c->rad_scratch[1], *gam = c->rad_scratch[2], *chi = c->rad_scratch[3];
    const int sym = (kmode == SPRAY_FLD_SYMMETRIC) ? 1 : 0;
    for (int k = 0; k < niter; ++k) {
        if (c->tl.enabled) {
            TiledArgs t{};
            t.fld_sym = sym; t.o0 = y; t.o1 = lam; t.o2 = gam;
            CK(launch_tiled_sweep(c, SW_APPLY, t, st), "rad: tiled apply sweep");
        }
        SweepArgs a = fallback_args(c);
        a.m = f[F_M]; a.rho = f[F_RHO]; a.E = f[F_E]; a.mu = f[F_MU]; a.c_light = c_light; a.fld_sym = sym;
        a.o0 = y; a.o1 = lam; a.o2 = gam;
        CK(launch_ref_sweep(c, SW_APPLY, a, st), "rad: apply sweep");
        RadArgs r{};
        r.rho = rho; r.kappa_p = kappa_p; r.E_n = E_n; r.u_n = u_n; r.T_n = T_n; r.dTdu = dTdu;
        r.lam = lam; r.gam = gam; r.dt = dt; r.c_light = c_light; r.a_rad = a_rad;
        r.E = E; r.u = u; r.chi = chi; r.me = c->pk.me; r.sE = f[F_E];
        r.resid = resid ? resid + k : nullptr; r.first = (k == 0) ? 1 : 0;
        CK(launch_rad_update(c, r, st), "rad: quartic update");
    }
    return SPRAY_OK;
}

int spray_ray_deposit(spray_ctx* ctx, const double* m, const double* rho, const double* f, const double* kib, int64_t nrays,
                      const double* rays_in, double dt, int64_t nsteps, double c_light, double pmin, double* gradn, double* edep,
                      double* rays_out, int64_t* steps_out, void* stream) {
    NEED_BUILT();
    Ctx* c = &ctx->c;
    c->chain_ok = false;
    if (c->n > 0 && (!m || !rho || !f || !kib || !edep)) return fail(c, SPRAY_ERR_INVALID_ARG, "spray_ray_deposit: NULL argument");
    if (nrays < 0 || nsteps < 0 || (nrays > 0 && (!rays_in || !rays_out)) || !(dt > 0.0) || !(c_light > 0.0))
        return fail(c, SPRAY_ERR_INVALID_ARG, "spray_ray_deposit: nrays, nsteps >= 0, dt, c_light > 0, ray buffers non-NULL");
    cudaStream_t st = (cudaStream_t)stream;
    double** fs = c->s.f;
    // (1) G_a = sum_b V_b f_b gradW(x_ab, h_a): the limiter-type sweep without the -f_a term; sorted records
    //     (z, V), f, (kib, f) from the FLD prologue with "mu" = kib, "E" = f
    PrepJob pj{};
    pj.m = m; pj.rho = rho; pj.E = f; pj.kx = kib; pj.kx_is_mu = 1;
    pj.sm = fs[F_M]; pj.srho = fs[F_RHO]; pj.sE = fs[F_E]; pj.skx = fs[F_MU]; pj.sV = fs[F_V];
    CK(launch_prep_fld(c, pj, st), "ray: prologue");
    if (c->tl.enabled) {
        TiledArgs t{};
        t.o1 = gradn;
        CK(launch_tiled_sweep(c, SW_GRADN, t, st), "ray: tiled gradient sweep");
    }
    SweepArgs a = fallback_args(c);
    a.m = fs[F_M]; a.rho = fs[F_RHO]; a.E = fs[F_E]; a.mu = fs[F_MU];
    a.o1 = gradn; a.me_sorted = c->pk.s[1]; a.g2_sorted = c->pk.s[2];
    CK(launch_ref_sweep(c, SW_GRADN, a, st), "ray: gradient sweep");
    // (2) rays: deposit into a sorted-order accumulator, then back to caller order
    double* dep = fs[15];
    if (c->n > 0) CK(cudaMemsetAsync(dep, 0, sizeof(double) * (size_t)c->n, st), "ray: deposit accumulator");
    RayArgs r{};
    r.nrays = nrays; r.rays_in = rays_in; r.dt = dt; r.c_light = c_light; r.pmin = pmin; r.nsteps = nsteps;
    r.dep_sorted = dep; r.rays_out = rays_out; r.steps_out = steps_out;
    CK(launch_ray_trace(c, r, st), "ray: trace");
    CK(launch_unsort(c, dep, edep, st), "ray: deposit to caller order");
    return SPRAY_OK;
}

int spray_get_cell_table(spray_ctx* ctx, uint32_t* sorted_key, uint32_t* perm, uint32_t* cell_start, uint32_t* cell_end,
                         void* stream) {
    NEED_BUILT();
    Ctx* c = &ctx->c;
    cudaStream_t st = (cudaStream_t)stream;
    size_t nb = sizeof(uint32_t) * (size_t)c->n, cb = sizeof(uint32_t) * (size_t)c->ncell;
    if (sorted_key && c->n) CK(cudaMemcpyAsync(sorted_key, c->sorted_key, nb, cudaMemcpyDeviceToDevice, st), "get_cell_table");
    if (perm && c->n) CK(cudaMemcpyAsync(perm, c->perm, nb, cudaMemcpyDeviceToDevice, st), "get_cell_table");
    if (cell_start) CK(cudaMemcpyAsync(cell_start, c->cell_start, cb, cudaMemcpyDeviceToDevice, st), "get_cell_table");
    if (cell_end) CK(cudaMemcpyAsync(cell_end, c->cell_end, cb, cudaMemcpyDeviceToDevice, st), "get_cell_table");
    return SPRAY_OK;
}

int spray_neighbor_counts(spray_ctx* ctx, int symmetric, uint32_t* count, void* stream) {
    NEED_BUILT();
    Ctx* c = &ctx->c;
    if (c->n > 0 && !count) return fail(c, SPRAY_ERR_INVALID_ARG, "spray_neighbor_counts: NULL argument");
    const TiledSet ts = tiled_set(c);
    for (int k = 0; k < ts.n; ++k)
        CK(launch_tiled_export(ts.v[k], 0, symmetric, count, nullptr, nullptr, nullptr, nullptr, (cudaStream_t)stream), "neighbour counts from the tiled lists");
    SweepArgs a = fallback_args(c, true);
    a.symmetric = symmetric; a.ocount = count;
    CK(launch_ref_sweep(general_ctx(c), SW_COUNT, a, (cudaStream_t)stream), "neighbour count sweep");
    return SPRAY_OK;
}

int spray_neighbor_lists(spray_ctx* ctx, int symmetric, const uint64_t* offsets, uint32_t* nbr, void* stream) {
    NEED_BUILT();
    Ctx* c = &ctx->c;
    if (c->n > 0 && (!offsets || !nbr)) return fail(c, SPRAY_ERR_INVALID_ARG, "spray_neighbor_lists: NULL argument");
    const TiledSet ts = tiled_set(c);
    for (int k = 0; k < ts.n; ++k)
        CK(launch_tiled_export(ts.v[k], 1, symmetric, nullptr, offsets, nbr, nullptr, nullptr, (cudaStream_t)stream), "neighbour lists from the tiled lists");
    SweepArgs a = fallback_args(c, true);
    a.symmetric = symmetric; a.offsets = offsets; a.onbr = nbr;
    CK(launch_ref_sweep(general_ctx(c), SW_LIST, a, (cudaStream_t)stream), "neighbour list sweep");
    return SPRAY_OK;
}

int spray_neighbor_digest(spray_ctx* ctx, int symmetric, uint64_t* dsum, uint64_t* dxor, void* stream) {
    NEED_BUILT();
    Ctx* c = &ctx->c;
    if (c->n > 0 && (!dsum || !dxor)) return fail(c, SPRAY_ERR_INVALID_ARG, "spray_neighbor_digest: NULL argument");
    const TiledSet ts = tiled_set(c);
    for (int k = 0; k < ts.n; ++k)
        CK(launch_tiled_export(ts.v[k], 2, symmetric, nullptr, nullptr, nullptr, dsum, dxor, (cudaStream_t)stream), "neighbour digests from the tiled lists");
    SweepArgs a = fallback_args(c, true);
    a.symmetric = symmetric; a.odsum = dsum; a.odxor = dxor;
    CK(launch_ref_sweep(general_ctx(c), SW_DIGEST, a, (cudaStream_t)stream), "neighbour digest sweep");
    return SPRAY_OK;
}

int spray_fp64_peak_probe(int device, int blocks, int threads, int64_t iters, double* out, void* stream) {
    if (!out || blocks < 1 || threads < 1 || threads > 256 || iters < 0) return SPRAY_ERR_INVALID_ARG;
    DeviceGuard dg(device);
    if (!dg.ok) { cudaGetLastError(); return SPRAY_ERR_CUDA; }
    return launch_fp64_probe(blocks, threads, iters, out, (cudaStream_t)stream) == cudaSuccess ? SPRAY_OK : SPRAY_ERR_CUDA;
}

}  // extern "C"
