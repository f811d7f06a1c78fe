// tiles.cu -- tile construction and the neighbour-list builder of the tiled path (run once per spray_build_cells).
//
// NNPS, PAPER.md L434-L446 (§2.6): the cell list identifies the particles of the 27 cells around a target; "a
// majority of computational time is spent on searching and identifying neighboring particles" (L436).  Here the
// search is done ONCE per cell build and its result -- for every target the list of its mutual neighbours N_sym
// (L442 "ensure all neighbors are mutual"), gather neighbours first -- is kept as u16 slots of the tile's
// candidate layout (tiles.cuh), so the four pair sweeps that follow (and every later spray_fld_apply of an
// implicit solve, L327) run their pair bodies at full lane occupancy with no distance test on rejected candidates.
//
// The candidate test is done in two steps: an fp32 prefilter on tile-relative coordinates (conservative margin,
// off the FP64 pipe), then the exact contract predicate in fp64 (common.cuh: r2_exact / support2 / min_image) on the
// survivors, so the sets are bit-identical to the definition.
#include "spray_internal.h"
#include "tiles.cuh"

namespace spray {

// ------------------------------------------------------------------------------------------- tile construction
// One thread per bundle of 2 x 2 rows walks the columns and emits tiles greedily: up to TILE_T targets, at most
// TILE_CMAX candidate slots, at most TILE_BXMAX columns.  A column whose own candidate set does not fit is left to
// the general kernels (its particles keep fast[i] = 0).
__device__ uint32_t bundle_col_count(const DevGrid& g, const CellTable& ct, int y0, int nyr, int z0, int nzr, int cx) {
    uint32_t c = 0;
    for (int rz = 0; rz < nzr; ++rz)
        for (int ry = 0; ry < nyr; ++ry) {
            const uint32_t id = cell_id(g, cx, y0 + ry, z0 + rz);
            c += ct.cell_end[id] - ct.cell_start[id];
        }
    return c;
}
__device__ uint32_t tile_ncand(const TileDesc& td, const DevGrid& g, const CellTable& ct) {
    uint32_t tot = 0;
    RangeGeo R;
    for (int q = 0; q < 32; ++q)
        if (tile_range(td, g, ct, q >> 1, q & 1, R)) tot += range_padded_len(R.vs, R.ve);
    return tot;
}

__global__ void k_make_tiles(DevGrid g, CellTable ct, const double* __restrict__ hglob, TileDesc* __restrict__ tiles,
                             uint32_t* __restrict__ ntiles, uint32_t cap, uint32_t* __restrict__ status) {
    const int nby = (g.nc[1] + 1) / 2, nbz = (g.nc[2] + 1) / 2;
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= nby * nbz) return;
    // every neighbour within one cell: 2 h_max <= cell edge in every dimension (tiny safety margin)
    const double hmax = hglob[1];
    for (int d = 0; d < 3; ++d)
        if (!(2.0 * hmax * g.inv[d] * (1.0 + 1e-9) <= 1.0)) return;
    const int nx = g.nc[0];
    TileDesc td;
    td.y0 = (int16_t)(2 * (b % nby)); td.z0 = (int16_t)(2 * (b / nby));
    td.nyr = (uint8_t)min(2, g.nc[1] - td.y0); td.nzr = (uint8_t)min(2, g.nc[2] - td.z0);
    td.pad = 0; td.pad2 = 0;
    int cxa = 0;
    uint32_t skip = 0;
    while (cxa < nx) {
        td.cxa = (int16_t)cxa; td.cxb = (int16_t)cxa; td.skip = skip;
        if (tile_ncand(td, g, ct) > (uint32_t)TILE_CMAX) { ++cxa; skip = 0; continue; }   // column not tileable
        uint32_t nt = 0;
        int next_cxa = nx;
        uint32_t next_skip = 0;
        for (int cx = cxa; cx < nx; ++cx) {
            if (cx > cxa) {
                const int ext = cx - cxa + 1;
                TileDesc t2 = td;
                t2.cxb = (int16_t)cx;
                if (ext > TILE_BXMAX || (g.per[0] && ext + 2 > nx) || tile_ncand(t2, g, ct) > (uint32_t)TILE_CMAX) {
                    next_cxa = cx; next_skip = 0; break;
                }
            }
            uint32_t c = bundle_col_count(g, ct, td.y0, td.nyr, td.z0, td.nzr, cx);
            if (cx == cxa) c -= skip;
            const uint32_t take = min(c, (uint32_t)TILE_T - nt);
            nt += take;
            td.cxb = (int16_t)cx;
            if (take < c) { next_cxa = cx; next_skip = (cx == cxa ? skip : 0u) + take; break; }
            if (nt == (uint32_t)TILE_T) { next_cxa = cx + 1; next_skip = 0; break; }
        }
        if (nt > 0) {
            td.nt = nt;
            const uint32_t idx = atomicAdd(ntiles, 1u);
            if (idx < cap) tiles[idx] = td;
            else atomicOr(status, (uint32_t)SPRAY_DEV_LIST_OVERFLOW);   // dropped tile: its particles use the general kernels
        }
        cxa = next_cxa; skip = next_skip;
    }
}
__global__ void k_clamp_ntiles(uint32_t* ntiles, uint32_t cap) { if (*ntiles > cap) *ntiles = cap; }

// ------------------------------------------------------------------------------------------- list builder
struct ListArgs {
    const double *x, *y, *z, *h;       // sorted
    const TileDesc* tiles;
    const uint32_t* ntiles;
    uint2* lists;                      // [tile][warp][LIST_CAP/4][32] x 4 u16
    uint32_t* lcount;                  // [tile][TILE_T]: n_gather | n_sym << 16
    uint8_t* fast;                     // [n] sorted order: 1 = served by the tiled kernels
    uint32_t* tile_ok;                 // [tile]
    uint32_t* status;
    int64_t n;
};

constexpr size_t BL_OFF_F4 = 0;                                             // float4 [CMAX]
constexpr size_t BL_OFF_XYZH = BL_OFF_F4 + sizeof(float4) * TILE_CMAX;      // double [4][CMAX]
constexpr size_t BL_OFF_L2 = 0;                                             // second list buffer aliases f4 + xyzh
constexpr size_t BL_OFF_GIDX = BL_OFF_XYZH + sizeof(double) * 4 * TILE_CMAX;// uint32 [CMAX]
constexpr size_t BL_OFF_L = BL_OFF_GIDX + sizeof(uint32_t) * TILE_CMAX;     // uint16 [LIST_CAPP][TILE_T]
constexpr size_t BL_OFF_COL = BL_OFF_L + sizeof(uint16_t) * LIST_CAPP * TILE_T;   // uint16 [MAXR][BXMAX + 3]
constexpr size_t BL_SMEM = BL_OFF_COL + sizeof(uint16_t) * TILE_MAXR * (TILE_BXMAX + 4);
static_assert(sizeof(uint16_t) * LIST_CAP * TILE_T <= BL_OFF_GIDX, "second list buffer must fit under gidx");
static_assert(BL_SMEM + sizeof(TileS) + 64 <= 227 * 1024, "list builder shared memory");

__global__ void __launch_bounds__(TILE_T, 1)
k_build_lists(DevGrid g, CellTable ct, ListArgs A) {
    extern __shared__ __align__(16) unsigned char smem[];
    __shared__ TileS S;
    __shared__ int s_bad;
    float4* f4 = reinterpret_cast<float4*>(smem + BL_OFF_F4);
    double* sx = reinterpret_cast<double*>(smem + BL_OFF_XYZH);
    double* sy = sx + TILE_CMAX;
    double* sz = sy + TILE_CMAX;
    double* sh = sz + TILE_CMAX;
    uint32_t* gidx = reinterpret_cast<uint32_t*>(smem + BL_OFF_GIDX);
    uint16_t* L = reinterpret_cast<uint16_t*>(smem + BL_OFF_L);        // [k][tid]
    uint16_t* L2 = reinterpret_cast<uint16_t*>(smem + BL_OFF_L2);      // [k][tid], valid after the exact phase
    uint16_t* colofs = reinterpret_cast<uint16_t*>(smem + BL_OFF_COL); // [range][TILE_BXMAX + 4]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t ntiles = *A.ntiles;

    for (uint32_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const TileDesc td = A.tiles[tile];
        __syncthreads();                                                // previous tile done with smem
        if (tid == 0) s_bad = 0;
        tile_setup(td, g, ct, S);
        const uint32_t ncand = S.ncand;
        const int ncolv = td.cxb - td.cxa + 3;                          // virtual columns 0 .. ncolv-1
        // tile origin (centre of the tile's cell block) for the fp32 relative coordinates
        const double ox = g.lo[0] + (0.5 * (td.cxa + td.cxb + 1)) / g.inv[0];
        const double oy = g.lo[1] + (td.y0 + 0.5 * td.nyr) / g.inv[1];
        const double oz = g.lo[2] + (td.z0 + 0.5 * td.nzr) / g.inv[2];
        // bound on the absolute error of an fp32 relative coordinate difference: 2 roundings of magnitude <= ext
        const float ext = (float)fmax(fmax((0.5 * ncolv + 0.5) / g.inv[0], 2.5 / g.inv[1]), 2.5 / g.inv[2]);
        const float E = ext * 2.4e-7f;                                  // 4 * 2^-24 * ext

        // ---- per-range column offsets (slot of the first particle of each column, relative to r_base)
        for (int w = tid; w < (int)S.nranges * (TILE_BXMAX + 4); w += TILE_T) {
            const int q = w / (TILE_BXMAX + 4), j = w % (TILE_BXMAX + 4);
            const int4 ge = S.r_geo[q];
            if (j <= ge.y) {
                const uint32_t gs = (j < ge.y) ? ct.cell_start[ge.w + j] : S.r_vend[q];
                colofs[q * (TILE_BXMAX + 4) + j] = (uint16_t)(gs - S.r_start[q]);
            }
        }
        // ---- stage the candidates
        for (uint32_t s = tid; s < ncand; s += TILE_T) {
            const int q = tile_slot_range(S, s);
            const uint32_t gi = S.r_start[q] + (s - S.r_base[q]);
            const bool valid = gi >= S.r_vstart[q] && gi < S.r_vend[q];
            if (valid) {
                const double xb = A.x[gi], yb = A.y[gi], zb = A.z[gi], hb = A.h[gi];
                sx[s] = xb; sy[s] = yb; sz[s] = zb; sh[s] = hb;
                gidx[s] = gi | ((uint32_t)q << 27);                     // n < 2^27 guaranteed by the launcher
                // image position next to the tile: x_b - shift*L
                const float fx = (float)((xb - S.r_shift[q][0] * g.L[0]) - ox);
                const float fy = (float)((yb - S.r_shift[q][1] * g.L[1]) - oy);
                const float fz = (float)((zb - S.r_shift[q][2] * g.L[2]) - oz);
                const float Rb = 2.0f * (float)hb * 1.000001f;
                f4[s] = make_float4(fx, fy, fz, Rb * Rb * 1.00001f + 4.4f * Rb * E + 5.0f * E * E);
            } else {
                gidx[s] = 0xFFFFFFFFu;
                f4[s] = make_float4(3.0e18f, 3.0e18f, 3.0e18f, 0.0f);
            }
        }
        // ---- this thread's target
        const bool active = tid < (int)td.nt;
        uint32_t i = 0;
        double xa = 0, ya = 0, za = 0, ha = 0;
        int tcol = 0, trow = 0;
        if (active) {
            const uint32_t p = td.skip + (uint32_t)tid;
            int lo = 0, hi = (int)S.ncells;
            while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (S.c_pre[mid] <= p) lo = mid; else hi = mid; }
            i = S.c_first[lo] + (p - S.c_pre[lo]);
            const int nrows = td.nyr * td.nzr;
            tcol = lo / nrows; trow = lo % nrows;
            xa = A.x[i]; ya = A.y[i]; za = A.z[i]; ha = A.h[i];
        }
        const float fax = (float)(xa - ox), fay = (float)(ya - oy), faz = (float)(za - oz);
        const float Ra = 2.0f * (float)ha * 1.000001f;
        const float thr_a = active ? Ra * Ra * 1.00001f + 4.4f * Ra * E + 5.0f * E * E : -1.0f;
        // warp window in virtual columns / candidate rows
        int cmin = active ? tcol : 1 << 20, cmax = active ? tcol : -1;
        int ymin = active ? trow % td.nyr : 4, ymax = active ? trow % td.nyr : -1;
        int zmin = active ? trow / td.nyr : 4, zmax = active ? trow / td.nyr : -1;
#pragma unroll
        for (int o = 16; o; o >>= 1) {
            cmin = min(cmin, __shfl_xor_sync(0xFFFFFFFFu, cmin, o)); cmax = max(cmax, __shfl_xor_sync(0xFFFFFFFFu, cmax, o));
            ymin = min(ymin, __shfl_xor_sync(0xFFFFFFFFu, ymin, o)); ymax = max(ymax, __shfl_xor_sync(0xFFFFFFFFu, ymax, o));
            zmin = min(zmin, __shfl_xor_sync(0xFFFFFFFFu, zmin, o)); zmax = max(zmax, __shfl_xor_sync(0xFFFFFFFFu, zmax, o));
        }
        __syncthreads();

        // ---- phase 1: fp32 prefilter, all lanes test the same candidate (shared-memory broadcast)
        uint32_t cnt = 0;
        if (cmax >= 0) {
            const int wv_lo = cmin, wv_hi = cmax + 2;                   // virtual columns [tcol, tcol + 2] around each target
            for (int q = 0; q < (int)S.nranges; ++q) {
                const int row = S.r_shift[q][3], ry = row & 3, rz = row >> 2;
                if (ry < ymin || ry > ymax + 2 || rz < zmin || rz > zmax + 2) continue;
                const int4 ge = S.r_geo[q];
                const int jlo = max(0, min(ge.y, wv_lo - ge.z)), jhi = max(0, min(ge.y, wv_hi + 1 - ge.z));
                if (jhi <= jlo) continue;
                const uint32_t sa = S.r_base[q] + colofs[q * (TILE_BXMAX + 4) + jlo];
                const uint32_t sb = S.r_base[q] + colofs[q * (TILE_BXMAX + 4) + jhi];
#pragma unroll 4
                for (uint32_t s = sa; s < sb; ++s) {
                    const float4 c = f4[s];
                    const float dx = fax - c.x, dy = fay - c.y, dz = faz - c.z;
                    const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                    if (r2 < fmaxf(thr_a, c.w)) {
                        if (cnt < (uint32_t)LIST_CAPP) L[cnt * TILE_T + tid] = (uint16_t)s;
                        ++cnt;
                    }
                }
            }
        }
        if (cnt > (uint32_t)LIST_CAPP) s_bad = 1;
        // ---- phase 2: exact predicate (contract O2/A12) on the survivors, compacted in place
        const double sup_a = support2(ha);
        uint32_t m = 0, ng = 0;
        if (active) {
            const uint32_t nn = min(cnt, (uint32_t)LIST_CAPP);
            const bool anysh = S.any_shift != 0;
            for (uint32_t k = 0; k < nn; ++k) {
                const uint32_t s = L[k * TILE_T + tid];
                const uint32_t gq = gidx[s];
                if ((gq & 0x07FFFFFFu) == i) continue;                  // self
                double dx = __dsub_rn(xa, sx[s]), dy = __dsub_rn(ya, sy[s]), dz = __dsub_rn(za, sz[s]);
                if (anysh) {
                    dx = min_image(dx, g.per[0], g.L[0], g.halfL[0]);
                    dy = min_image(dy, g.per[1], g.L[1], g.halfL[1]);
                    dz = min_image(dz, g.per[2], g.L[2], g.halfL[2]);
                }
                const double r2 = r2_exact(dx, dy, dz);
                const double hb = sh[s];
                if (r2 < support2(fmax(ha, hb))) {
                    const bool ing = r2 < sup_a;
                    L[m * TILE_T + tid] = (uint16_t)(s | (ing ? LIST_GATHER_BIT : 0));
                    ++m; ng += ing ? 1u : 0u;
                }
            }
            if (m > (uint32_t)LIST_CAP) s_bad = 1;
        }
        __syncthreads();                                                // coordinates no longer needed: L2 may alias them
        const bool bad = s_bad != 0;
        if (!bad) {
            // ---- phase 3: gather neighbours first, then the symmetric-only ones
            uint32_t pos = 0;
            for (uint32_t k = 0; k < m; ++k) { const uint16_t e = L[k * TILE_T + tid]; if (e & LIST_GATHER_BIT) L2[(pos++) * TILE_T + tid] = e & 0x7FFFu; }
            for (uint32_t k = 0; k < m; ++k) { const uint16_t e = L[k * TILE_T + tid]; if (!(e & LIST_GATHER_BIT)) L2[(pos++) * TILE_T + tid] = e; }
            // pad to a multiple of 4 with slot 0 (never evaluated: the sweeps stop at the counts)
            for (uint32_t k = m; k < ((m + 3u) & ~3u); ++k) L2[k * TILE_T + tid] = 0;
            uint32_t mx = m;
#pragma unroll
            for (int o = 16; o; o >>= 1) mx = max(mx, __shfl_xor_sync(0xFFFFFFFFu, mx, o));
            uint2* blk = A.lists + list_block_u2(tile, warp);
            for (uint32_t k4 = 0; k4 * 4 < mx; ++k4) {
                uint2 v = make_uint2(0u, 0u);
                if (k4 * 4 < m) {
                    const uint32_t e0 = L2[(k4 * 4 + 0) * TILE_T + tid], e1 = L2[(k4 * 4 + 1) * TILE_T + tid];
                    const uint32_t e2 = L2[(k4 * 4 + 2) * TILE_T + tid], e3 = L2[(k4 * 4 + 3) * TILE_T + tid];
                    v = make_uint2(e0 | (e1 << 16), e2 | (e3 << 16));
                }
                blk[k4 * 32 + lane] = v;
            }
            A.lcount[(size_t)tile * TILE_T + tid] = active ? (ng | (m << 16)) : 0u;
            if (active) A.fast[i] = 1;
        }
        if (tid == 0) A.tile_ok[tile] = bad ? 0u : 1u;
    }
}

__global__ void k_count_fast(const uint8_t* __restrict__ fast, int64_t n, unsigned long long* out) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const uint32_t b = __ballot_sync(0xFFFFFFFFu, i < n && fast[i]);
    if ((threadIdx.x & 31) == 0 && b) atomicAdd(out, (unsigned long long)__popc(b));
}

// ------------------------------------------------------------------------------------------- launchers
cudaError_t launch_count_fast(Ctx* c, cudaStream_t st) {
    unsigned long long* out = reinterpret_cast<unsigned long long*>(c->hglob + 2);
    cudaError_t e = cudaMemsetAsync(out, 0, sizeof(unsigned long long), st);
    if (e != cudaSuccess) return e;
    k_count_fast<<<(unsigned)((c->n + 255) / 256), 256, 0, st>>>(c->tl.fast, c->n, out);
    return cudaGetLastError();
}

cudaError_t launch_build_tiles(Ctx* c, cudaStream_t st) {
    Tiled& t = c->tl;
    t.enabled = false;
    if (c->n == 0 || !t.tiles) return cudaSuccess;
    // host-side guards: small periodic grids (a candidate row would appear twice), index width
    const spray_grid_t& gr = c->grid;
    if (c->n >= (1ll << 27)) return cudaSuccess;
    if (gr.periodic[0] && gr.ncell[0] < 3) return cudaSuccess;
    if (gr.periodic[1] && gr.ncell[1] < 4) return cudaSuccess;
    if (gr.periodic[2] && gr.ncell[2] < 4) return cudaSuccess;
    if (gr.ncell[0] > 32000 || gr.ncell[1] > 32000 || gr.ncell[2] > 32000) return cudaSuccess;
    cudaError_t e;
    if ((e = cudaMemsetAsync(t.ntiles, 0, sizeof(uint32_t), st)) != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(t.fast, 0, (size_t)c->n, st)) != cudaSuccess) return e;
    CellTable ct{c->cell_start, c->cell_end};
    const int nb = ((gr.ncell[1] + 1) / 2) * ((gr.ncell[2] + 1) / 2);
    k_make_tiles<<<(nb + 63) / 64, 64, 0, st>>>(c->dg, ct, c->hglob, t.tiles, t.ntiles, (uint32_t)t.tile_cap, c->dev_status);
    k_clamp_ntiles<<<1, 1, 0, st>>>(t.ntiles, (uint32_t)t.tile_cap);
    static bool attr_done = false;
    if (!attr_done) {
        if ((e = cudaFuncSetAttribute(k_build_lists, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)BL_SMEM)) != cudaSuccess) return e;
        attr_done = true;
    }
    ListArgs A{c->s.x, c->s.y, c->s.z, c->s.h, t.tiles, t.ntiles, t.lists, t.lcount, t.fast, t.tile_ok, c->dev_status, c->n};
    k_build_lists<<<t.grid, TILE_T, BL_SMEM, st>>>(c->dg, ct, A);
    c->launches += 3;
    t.enabled = true;
    return cudaGetLastError();
}

}  // namespace spray
