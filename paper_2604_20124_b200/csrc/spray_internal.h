// spray_internal.h -- host-side context and launcher prototypes (C++ side of the C-ABI in include/spray.h)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>

#include "../../include/spray.h"
#include "common.cuh"
#include "tiles.cuh"

namespace spray {

// Particle store in SORTED order (structure-of-arrays; BASELINE.json "reordered by cell after the sort").
struct Sorted {
    double *x, *y, *z, *h;      // built by spray_build_cells
    double* hs;                 // symmetric search length: max(h_a, max{h_b : a in N_gather(b)})
    double* f[16];              // per-call field scratch (m, rho, p, cs, vx, vy, vz, alpha, E, kappa, mu, V, Q, alpha*cs, ...)
};

// Tiled path (tiles.cuh): tiles + per-target neighbour lists, rebuilt by every spray_build_cells.
struct Tiled {
    bool enabled = false;        // tiles and lists were built for the current cell table
    int sms = 148;               // SM count of the device (persistent grids)
    int grid = 148;              // CTAs of the list builder
    TileDesc* tiles = nullptr;
    uint32_t* ntiles = nullptr;  // device counter
    int64_t tile_cap = 0;
    uint2* lists = nullptr;      // [tile_cap][TILE_WARPS][LIST_CAP/4][32] x 4 u16 slots
    uint32_t* lcount = nullptr;  // [tile_cap][TILE_T]: n_gather | n_sym << 16
    uint32_t* tile_ok = nullptr; // [tile_cap]
    uint8_t* fast = nullptr;     // [n_max] sorted order: 1 = particle is served by the tiled kernels
};

struct Ctx {
    int device = 0;
    int64_t n_max = 0, ncell_max = 0;
    int64_t n = 0, ncell = 0;
    bool built = false;
    int path = 0;               // 0 = reference kernels, 1 = tiled kernels
    int kernel = 0;
    spray_grid_t grid{};
    DevGrid dg{};
    // build scratch
    uint32_t *key[2] = {nullptr, nullptr}, *idx[2] = {nullptr, nullptr};
    uint32_t* hist = nullptr;   // radix histograms [256][nblocks]
    int64_t hist_cap = 0;
    uint32_t *sorted_key = nullptr, *perm = nullptr;   // aliases into key[]/idx[] after the last pass
    uint32_t *cell_start = nullptr, *cell_end = nullptr;
    double* cell_hmax = nullptr;
    double* hglob = nullptr;    // [0] = min h, [1] = max h (device scalars)
    uint32_t* dev_status = nullptr;
    Sorted s{};
    Tiled tl{};
    int64_t launches = 0;       // kernels launched through this ctx (bench.py reports it as gpu_launches)
    std::string err;
};

struct GatherJob {              // out[k][i] = in[k][perm[i]] for k < count
    const double* in[12];
    double* out[12];
    int count;
};

// ---- build.cu
cudaError_t launch_cell_keys(Ctx* c, const double* x, const double* y, const double* z, cudaStream_t st);
cudaError_t launch_radix_sort(Ctx* c, cudaStream_t st);      // sets c->sorted_key / c->perm
cudaError_t launch_cell_table(Ctx* c, cudaStream_t st);
cudaError_t launch_gather(Ctx* c, const GatherJob& job, cudaStream_t st);
cudaError_t launch_cell_hmax(Ctx* c, cudaStream_t st);

// ---- sweeps_ref.cu : reference pair kernels (one thread per particle)
struct SweepArgs {
    // sorted inputs
    const double *x, *y, *z, *h, *hs;
    const double *m, *rho, *p, *cs, *vx, *vy, *vz, *alpha, *E, *kappa, *mu;
    double beta, c_light;
    int fld_sym;                // apply: 1 = symmetric (A17), 0 = literal gather
    // caller-order outputs (written through perm)
    double *o0, *o1, *o2, *o3, *o4, *o5;
    double* mu_sorted;          // limiter: also keeps mu in sorted order for the apply that follows
    uint32_t* ocount;
    const uint64_t* offsets;
    uint32_t* onbr;
    uint64_t *odsum, *odxor;
    int symmetric;              // count / list / digest: which set
    const uint8_t* skip;        // nullable: particles with skip[i] != 0 are served by the tiled kernels
};
cudaError_t launch_ref_sweep(Ctx* c, int sweep, const SweepArgs& a, cudaStream_t st);

// ---- build.cu : per-call prologues (caller order -> sorted order through perm, per-particle factors hoisted)
struct PrepJob {
    const double *m, *rho, *p, *cs, *vx, *vy, *vz, *alpha, *E, *kx;   // caller order (kx = kappa or mu)
    double *sm, *srho, *sp, *scs, *svx, *svy, *svz, *salpha, *sE, *skx, *sV, *sQ, *sAC;   // sorted order
};
cudaError_t launch_prep_hydro(Ctx* c, const PrepJob& j, cudaStream_t st);
cudaError_t launch_prep_fld(Ctx* c, const PrepJob& j, cudaStream_t st);

// ---- tiles.cu / sweeps_tiled.cu : tiled path
struct TiledArgs {
    const double *x, *y, *z, *h;                 // sorted (filled by the launcher)
    const double *f0, *f1, *f2, *f3, *f4, *f5, *f6;   // sorted per-call fields, meaning per sweep (sweeps_tiled.cu)
    const double *g0, *g1;                       // sorted target-side fields (rho, p | rho, kappa)
    double beta, c_light;
    int fld_sym;
    double *o0, *o1, *o2, *o3, *o4;              // caller-order outputs
    double* mu_sorted;
    uint32_t* ocount;
    const uint32_t* perm;
    const TileDesc* tiles;
    const uint32_t* ntiles;
    const uint2* lists;
    const uint32_t* lcount;
    const uint32_t* tile_ok;
    int64_t n;
};
cudaError_t launch_build_tiles(Ctx* c, cudaStream_t st);
cudaError_t launch_count_fast(Ctx* c, cudaStream_t st);
cudaError_t launch_tiled_sweep(Ctx* c, int sweep, TiledArgs a, cudaStream_t st);

// ---- probe.cu
cudaError_t launch_fp64_probe(int blocks, int threads, int64_t iters, double* out, cudaStream_t st);

}  // namespace spray

struct spray_ctx {
    spray::Ctx c;
};
