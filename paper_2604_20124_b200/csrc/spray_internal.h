// spray_internal.h -- host-side context and launcher prototypes (C++ side of the C-ABI in include/spray.h)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>

#include "../../include/spray.h"
#include "common.cuh"
#include "tiles.cuh"

constexpr int SPRAY_MAX_LEVELS = 16;

namespace spray {

// Particle store in SORTED order, structure-of-arrays (BASELINE.json "reordered by cell after the sort"): used by
// the general one-thread-per-particle kernels (parity exports, search-length pre-pass, fallback of the tiled path).
struct Sorted {
    double *x, *y, *z, *h;      // built by spray_build_cells
    double* hs;                 // symmetric search length: max(h_a, max{h_b : a in N_gather(b)})
    double* f[16];              // per-call field scratch (m, rho, p, cs, vx, vy, vz, alpha, E, kappa, mu, V, Q, alpha*cs, ...)
};

// Particle store in SORTED order as 16-byte records (two fp64 fields per record): what the tiled kernels stage into
// shared memory and gather with one 128-bit load per record.
struct Packed {
    double2* p0;                // (x, y)                       built by spray_build_cells
    double2* p1;                // (z, h)                       built by spray_build_cells
    double2* hh;                // (1/h, FN_K / h^4)            built by spray_build_cells (FN_K: sweeps_tiled.cu)
    double2* s[4];              // per-call source-side records (meaning per sweep, sweeps_tiled.cu)
    double2* t0;                // per-call target-side record
    double2* me;                // (mu, E) of the FLD apply
    double* e1;                 // E of the limiter pre-sweep
};

// Tiled path (tiles.cuh): tiles + scheduled per-thread neighbour lists, rebuilt by every spray_build_cells.
struct Tiled {
    bool enabled = false;        // tiles and lists were built for the current cell table
    int sms = 148;               // SM count of the device (persistent grids)
    TileDesc* tiles = nullptr;
    int64_t tile_cap = 0;
    uint32_t* bcount = nullptr;  // [bundle_cap + 1 + scan scratch] tiles per bundle -> exclusive scan
    int64_t bundle_cap = 0;
    uint2* pool = nullptr;       // list storage: rows of 32 lanes x (4 u16 slots); a unit's warps take R/4 rows each, allocated
                                 // by the list builder from ctr[CTR_POOL]
    int64_t pool_rows = 0;       // capacity in rows (256 bytes each)
    unsigned long long* ctr = nullptr;   // CTR_*
    uint2* winfo = nullptr;      // [tile_cap][TILE_WARPS]: (first pool row, rounds)
    uint32_t* lcount = nullptr;  // [tile_cap][TILE_T]: n_gather | n_sym << 16
    uint32_t* tflags = nullptr;  // [tile_cap]: TILE_FLAG_*
    uint32_t* tiletab = nullptr; // [tile_cap][TILES_WORDS]: per-tile TileS tables
    uint8_t* fast = nullptr;     // [n_max] sorted order: 1 = particle is served by the tiled kernels
    int attr_device = -1;        // device on which the dynamic shared-memory opt-in of the tiled kernels was set
};
// CTR_NFAST: particles served by the tiled kernels; CTR_NTILES: tiles; CTR_NNONUNI: half-tile units that found non-uniform h;
// CTR_POOL: list-pool rows handed out
// CTR_DECL + k: warps / threads that declined their unit (general kernels), by reason k: 1 = list pool exhausted, 2 = list
// longer than LIST_RMAX rounds or more than LIST_BC neighbours in one bank, 3 = other (coincident particles, particle
// outside the tile's fp32 range)
// CTR_NALL: n (level contexts: the per-call prologues compare it with n and skip the structure-of-arrays copies)
// CTR_NFAST_ALL: particles served by the tiled kernels of the context or of one of its levels
enum { CTR_NFAST = 1, CTR_NTILES = 2, CTR_NNONUNI = 3, CTR_POOL = 4, CTR_NALL = 5, CTR_NFAST_ALL = 6, CTR_NLEFT = 7, CTR_DECL = 8, CTR_NMULTI = 12, CTR_COUNT = 16 };   // CTR_NMULTI: tile groups of more than one part (tiles.cuh)

struct Ctx {
    int device = 0;
    int64_t n_max = 0, ncell_max = 0;
    int64_t n = 0, ncell = 0;
    bool built = false;
    int path = 0;               // 0 = general kernels only, 1 = tiled kernels (+ general kernels for what they decline)
    int kernel = 0;
    spray_grid_t grid{};
    DevGrid dg{};
    // build scratch
    uint32_t *key[2] = {nullptr, nullptr}, *idx[2] = {nullptr, nullptr};
    uint32_t* hist = nullptr;   // radix histograms [256][nblocks]
    int64_t hist_cap = 0;
    uint32_t *sorted_key = nullptr, *perm = nullptr;   // aliases into key[]/idx[] after the last pass
    uint32_t *cell_start = nullptr, *cell_end = nullptr;
    uint32_t* cell_tend = nullptr;  // level contexts: end of the targets of a cell (they are sorted to the front of the cell)
    double* cell_hmax = nullptr;
    double* cell_hmin = nullptr;    // per-cell min h (search-length pre-pass: a cell whose particles all have h >= h_b cannot be raised by b)
    uint32_t* left = nullptr;       // sorted indices of the particles the tiled kernels (own + levels) do not serve: the general
                                    // kernels run over this compact list at full lane occupancy; count in tl.ctr[CTR_NLEFT]
    double* hglob = nullptr;    // [0] = min h, [1] = max h (device scalars)
    uint32_t* dev_status = nullptr;
    Sorted s{};
    Packed pk{};
    Tiled tl{};
    double* rad_scratch[4] = {nullptr, nullptr, nullptr, nullptr};   // N1: y, Lambda, Gamma, chi (caller order), allocated on first use
    bool chain_ok = false;      // the sorted records of the FLD operator are those of the last spray_hydro_rhs_limiter (FROZEN_CHAINED)
    const double *chain_m = nullptr, *chain_rho = nullptr, *chain_E = nullptr, *chain_mu = nullptr;
    int64_t launches = 0;       // kernels launched through this ctx (bench.py reports it as gpu_launches)
    int64_t scratch_bytes = 0;  // device memory held by this ctx
    // ---- internal levels of the tiled path (spray_set_levels): a level is a context of its own on a grid of the library's
    //      choosing (same box, cell edge >= level_edge), built from the same particles; it serves (tiles, lists, sweeps) only
    //      the particles a with level_lo < 2 hs_a <= level_hi that nobody served before; the parent keeps the general kernels
    int nlevels = 0;
    Ctx* child[SPRAY_MAX_LEVELS] = {};
    double level_edge[SPRAY_MAX_LEVELS] = {};
    bool is_level = false;
    Ctx* general = nullptr;                     // parent, levels on: the level context (finest built one) whose grid the general kernels use for
                                                // the particles no level serves -- the caller's grid may be far too coarse where they are dense
    const unsigned long long* soa_ctr = nullptr;// that level context: device word the prologues compare with n (parent's count of served particles)
    double level_lo = 0.0, level_hi = 0.0;      // of a level context: its range of 2 hs
    float level_rmax = 0.f;                     // of a level context: largest support radius it can meet (error bound of the fp32 prefilter)
    const double* hs_caller = nullptr;          // level context: the parent's arrays below
    const uint8_t* fast_caller = nullptr;
    double* hs_c = nullptr;                     // parent: hs in caller order
    uint8_t* fast_c = nullptr;                  // parent: 1 = served by the tiled kernels of the parent or of a level (caller order)
    uint8_t* fast_all = nullptr;                // parent: the same in the parent's sorted order (skip flags of its general kernels)
    bool levels_on = false;                     // the last build used the levels: fast_all / ctr[CTR_NFAST_ALL] are valid
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};   // recorded by spray_build_cells: start, cell list done, tiles done, lists done
    std::string err;
};

// ---- build.cu
cudaError_t launch_cell_keys(Ctx* c, const double* x, const double* y, const double* z, cudaStream_t st);
cudaError_t launch_to_caller_order(Ctx* c, cudaStream_t st);           // hs_c, fast_c from the sorted hs / fast of the parent
cudaError_t launch_merge_served(Ctx* parent, Ctx* child, cudaStream_t st);   // fast_c |= the child's served targets
cudaError_t launch_general_from_parent(Ctx* v, Ctx* parent, cudaStream_t st);   // level v: s.hs and fast_all in v's sorted order from the parent's caller-order arrays
cudaError_t launch_fast_from_caller(Ctx* c, cudaStream_t st);          // parent: fast_all[i] = fast_c[perm[i]], ctr[CTR_NFAST_ALL] = count
cudaError_t launch_radix_sort(Ctx* c, cudaStream_t st);      // sets c->sorted_key / c->perm
cudaError_t launch_cell_table(Ctx* c, cudaStream_t st);
cudaError_t launch_reorder_build(Ctx* c, const double* x, const double* y, const double* z, const double* h, cudaStream_t st);
cudaError_t launch_cell_hmax(Ctx* c, cudaStream_t st);
cudaError_t launch_pack_f4(Ctx* c, float4* f4, cudaStream_t st);             // (x, y, z, h) sorted, fp32 (skipped on the device when h is uniform)
cudaError_t launch_compact_left(Ctx* c, const uint8_t* fast, cudaStream_t st);   // c->left, ctr[CTR_NLEFT] from the served flags
cudaError_t launch_excl_scan_u32(Ctx* c, uint32_t* a, int64_t total, uint32_t* scratch, cudaStream_t st);

// ---- sweeps_ref.cu : general pair kernels (one thread per particle)
struct SweepArgs {
    // sorted inputs
    const double *x, *y, *z, *h, *hs;
    const double *m, *rho, *p, *cs, *vx, *vy, *vz, *alpha, *E, *kappa, *mu;
    double beta, c_light;
    int fld_sym;                // apply: 1 = symmetric (A17), 0 = literal gather
    // caller-order outputs (written through perm)
    double *o0, *o1, *o2, *o3, *o4, *o5;
    double* mu_sorted;          // limiter: also keeps mu in sorted order for the apply that follows
    double2* me_sorted;         // limiter: (mu, E) record of the tiled apply;  SW_GRADN: (G_x, G_y)
    double2* g2_sorted;         // SW_GRADN: (G_z, kappa^ib)
    uint32_t* ocount;
    const uint64_t* offsets;
    uint32_t* onbr;
    uint64_t *odsum, *odxor;
    int symmetric;              // count / list / digest: which set
    const uint8_t* skip;        // nullable: particles with skip[i] != 0 are served by the tiled kernels
    const uint32_t* left;       // nullable: the particles with skip[i] == 0, compacted (then the kernel runs over this list)
    const unsigned long long* nleft;
    const float4* f4;           // SW_HSEARCH, nullable: (x, y, z, h) of the sorted particles in fp32, for the pre-test of the pre-pass
    float f4_cmax;              // largest absolute coordinate of the box (bounds the fp32 rounding of a position)
    const unsigned long long* nfast;   // nullable: device count of such particles (== n: nothing to do)
};
cudaError_t launch_ref_sweep(Ctx* c, int sweep, const SweepArgs& a, cudaStream_t st);

// ---- build.cu : per-call prologues (caller order -> sorted order through perm, per-particle factors hoisted)
struct PrepJob {
    const double *m, *rho, *p, *cs, *vx, *vy, *vz, *alpha, *E, *kx;   // caller order (kx = kappa or mu)
    double *sm, *srho, *sp, *scs, *svx, *svy, *svz, *salpha, *sE, *skx, *sV, *sQ, *sAC;   // sorted order (general kernels)
    int kx_is_mu;
};
cudaError_t launch_prep_density(Ctx* c, const double* m, cudaStream_t st);
cudaError_t launch_prep_hydro(Ctx* c, const PrepJob& j, cudaStream_t st);
cudaError_t launch_prep_fld(Ctx* c, const PrepJob& j, cudaStream_t st);
cudaError_t launch_prep_kgc(Ctx* c, const PrepJob& j, cudaStream_t st);

// ---- tiles.cu / sweeps_tiled.cu : tiled path
struct TiledArgs {
    double beta, c_light;
    int fld_sym;
    double *o0, *o1, *o2, *o3, *o4;              // caller-order outputs
    double *o5 = nullptr, *o6 = nullptr;         // SW_HYDLIM: mu, gradE
    uint32_t* ocount;
};
cudaError_t launch_build_tiles(Ctx* c, cudaStream_t st);
cudaError_t tiled_set_attributes(Ctx* c);      // dynamic shared-memory opt-in of the tiled kernels, on the ctx's device (spray_create)
cudaError_t sweeps_set_attributes();

cudaError_t launch_tiled_sweep(Ctx* c, int sweep, const TiledArgs& a, cudaStream_t st);
// parity exports from the tiled lists: mode 0 = counts, 1 = CSR lists, 2 = digests (tiles.cu)
cudaError_t launch_tiled_export(Ctx* c, int mode, int symmetric, uint32_t* ocount, const uint64_t* offsets, uint32_t* onbr,
                                uint64_t* odsum, uint64_t* odxor, cudaStream_t st);

// ---- rad.cu : row N1, per-particle quartic solve of the Jacobi iteration (eqs. (54)-(57))
struct RadArgs {
    const double *rho, *kappa_p, *E_n, *u_n, *T_n, *dTdu;     // caller order
    const double *lam, *gam;                                   // caller order: Lambda, Gamma of the current iterate
    double dt, c_light, a_rad;
    double *E, *u;                                             // caller order: iterate out
    double *chi;                                               // caller order scratch: chi of the previous solve (residual)
    double2* me;                                               // sorted (mu, E) record of the tiled apply
    double* sE;                                                // sorted E of the general kernels
    double* resid;                                             // nullable: slot of this iteration
    int first;                                                 // iteration 0: no residual
};
cudaError_t launch_rad_update(Ctx* c, const RadArgs& a, cudaStream_t st);
cudaError_t launch_div_by_rho(Ctx* c, double* y, const double* rho, cudaStream_t st);   // N2
// N2 implicit system (eqs. (28)-(34)): g = tau u (rhs = 0) or T - tau u (rhs = 1) for both species; then
// out^i = u^i + s dt (y^i/rho + X), out^e = u^e + s dt (y^e/rho - X), X = kei (g^e - g^i), s = -1 (operator) or +1 (rhs)
struct CondArgs {
    const double *rho, *kei, *tau_i, *tau_e, *T_i, *T_e, *u_i, *u_e;   // caller order
    double *g_i, *g_e;                                                 // caller-order scratch
    const double *y_i, *y_e;                                           // caller-order pair sums of the two species
    double dt;
    int rhs;
    double *out_i, *out_e;
};
cudaError_t launch_cond_form(Ctx* c, const CondArgs& a, cudaStream_t st);
cudaError_t launch_cond_combine(Ctx* c, const CondArgs& a, cudaStream_t st);

// ---- ray.cu : row N4, mesh-free laser ray tracing and deposition
struct RayArgs {
    int64_t nrays;
    const double* rays_in;      // [7 nrays] planes x y z vx vy vz P
    double dt, c_light, pmin;
    int64_t nsteps;
    double* dep_sorted;         // [n] sorted order, zeroed: deposited energy (fp64 atomics)
    double* rays_out;           // [7 nrays]
    int64_t* steps_out;         // nullable
};
cudaError_t launch_ray_trace(Ctx* c, const RayArgs& a, cudaStream_t st);
cudaError_t launch_unsort(Ctx* c, const double* sorted, double* caller, cudaStream_t st);   // caller[perm[i]] = sorted[i]

// ---- probe.cu
cudaError_t launch_fp64_probe(int blocks, int threads, int64_t iters, double* out, cudaStream_t st);

}  // namespace spray

struct spray_ctx {
    spray::Ctx c;
};
