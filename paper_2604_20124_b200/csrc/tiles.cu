// tiles.cu -- tile construction and the neighbour-list builder of the tiled path (run once per spray_build_cells).
//
// NNPS, PAPER.md L434-L446 (§2.6): the cell list identifies the particles of the 27 cells around a target; "a
// majority of computational time is spent on searching and identifying neighboring particles" (L436).  Here the
// search is done ONCE per cell build and its result -- for every target the list of its mutual neighbours N_sym
// (L442 "ensure all neighbors are mutual") -- is kept as u16 slots of the tile's candidate layout (tiles.cuh), so
// the four pair sweeps that follow (and every later spray_fld_apply of an implicit solve, L327) run their pair
// bodies at full lane occupancy with no distance test on rejected candidates.
//
// The candidate test is an fp32 prefilter on tile-relative coordinates; a hit closer to a support boundary than
// the fp32 error bound (or to r = 0) is re-tested with the exact contract predicate in fp64 (common.cuh:
// r2_exact / support2 / min_image), so the sets are bit-identical to the definition.
//
// SCHEDULED LISTS.  The pair kernels gather 16-byte records of their neighbours from shared memory; 8 lanes form
// one 128-byte wavefront and conflict when two of them read different records of the same bank (slot & 7).  A
// target's neighbours are therefore split between its two threads bank by bank, and each thread's half-list is
// emitted in an order that walks the banks in phase with the other lanes of its 8-lane group: lane j spends
// rounds [t R / 8, (t + 1) R / 8) in bank (j + t) & 7, entries that do not fit their phase fill the holes of other
// phases, the remaining holes are dummy slots (records that contribute exactly zero).
#include "spray_internal.h"
#include "tiles.cuh"

namespace spray {

// ------------------------------------------------------------------------------------------- tile construction
// One warp per bundle of 2 x 2 rows walks the columns and cuts tiles greedily: up to TILE_T targets, at most
// TILE_CMAX candidate slots, at most TILE_BXMAX columns.  Lane l < 16 owns candidate row l (rz * 4 + ry).  A column
// whose own candidate set does not fit is left to the general kernels.  Run twice: EMIT = false counts the tiles
// of every bundle, EMIT = true writes them at the scanned offsets, so the tile order is deterministic and follows
// the grid (consecutive tiles share candidate rows in L2).
struct RowRef {                      // one candidate row of a bundle
    const uint32_t *cs, *ce, *te;    // cell_start / cell_end / cell_tend of the row (indexed by column)
    bool valid;
    bool target;                     // the row is one of the bundle's own rows
};
// slots the candidates of columns [xlo, xhi] of the row take in a tile's layout: every contiguous piece is padded to a
// multiple of 8 slots (tile_setup)
__device__ __forceinline__ uint32_t pad8(uint32_t c) { return (c + 7u) & ~7u; }
__device__ __forceinline__ uint32_t row_count(const RowRef& r, int xlo, int xhi, int nx, bool per) {
    if (!r.valid) return 0u;
    if (per) {
        if (xlo < 0) return pad8(r.ce[nx - 1] - r.cs[xlo + nx]) + pad8(r.ce[xhi] - r.cs[0]);
        if (xhi >= nx) return pad8(r.ce[nx - 1] - r.cs[xlo]) + pad8(r.ce[xhi - nx] - r.cs[0]);
    } else {
        xlo = xlo < 0 ? 0 : xlo;
        xhi = xhi > nx - 1 ? nx - 1 : xhi;
    }
    return pad8(r.ce[xhi] - r.cs[xlo]);
}
__device__ __forceinline__ uint32_t warp_sum(uint32_t v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
    return v;
}

template <bool EMIT>
__global__ void __launch_bounds__(256)
k_make_tiles(DevGrid g, CellTable ct, const double* __restrict__ hglob, uint32_t* __restrict__ bcount,
             TileDesc* __restrict__ tiles, uint32_t cap, unsigned long long* __restrict__ ctr, int level, unsigned long long n_all, int brows,
             int parts) {
    // a bundle is brows x brows cell rows: 2 x 2 on the caller's grid (cells of ~18 particles: 4 x 4 candidate rows), 1 x 1 on the
    // internal levels, whose cells hold up to ~60 particles (3 x 3 candidate rows fit the staging budget)
    const int nby = (g.nc[1] + brows - 1) / brows, nbz = (g.nc[2] + brows - 1) / brows;
    const int b = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (b >= nby * nbz) return;
    // every neighbour within one cell: 2 h_max <= cell edge in every dimension (tiny safety margin)
    // (a level context serves only particles whose 2 hs fits its cells: api.cu)
    const double hmax = level ? 0.0 : hglob[1];
    bool ok = true;
    for (int d = 0; d < 3; ++d)
        if (!(2.0 * hmax * g.inv[d] * (1.0 + 1e-9) <= 1.0)) ok = false;
    const int nx = g.nc[0];
    const int y0 = brows * (b % nby), z0 = brows * (b / nby);
    const int nyr = min(brows, g.nc[1] - y0), nzr = min(brows, g.nc[2] - z0);
    RowRef row;
    {
        const int ry = lane & 3, rz = (lane >> 2) & 3;
        int cy = y0 - 1 + ry, cz = z0 - 1 + rz;
        row.valid = lane < 16 && ry < nyr + 2 && rz < nzr + 2;
        if (cy < 0) { if (g.per[1]) cy += g.nc[1]; else row.valid = false; }
        else if (cy >= g.nc[1]) { if (g.per[1]) cy -= g.nc[1]; else row.valid = false; }
        if (cz < 0) { if (g.per[2]) cz += g.nc[2]; else row.valid = false; }
        else if (cz >= g.nc[2]) { if (g.per[2]) cz -= g.nc[2]; else row.valid = false; }
        row.target = row.valid && ry >= 1 && ry <= nyr && rz >= 1 && rz <= nzr;
        const uint32_t base = row.valid ? cell_id(g, 0, cy, cz) : 0u;
        row.cs = ct.cell_start + base; row.ce = ct.cell_end + base; row.te = ct.cell_tend + base;
    }
    const bool per = g.per[0] != 0;
    uint32_t ntl = 0;
    const uint32_t obase = EMIT ? bcount[b] : 0u;
    int cxa = 0;
    uint32_t skip = 0;
    while (ok && cxa < nx) {
        {
            const uint32_t myc = row_count(row, cxa - 1, cxa + 1, nx, per);             // lane l < 16: candidates of row l; others 0
            if (warp_sum(myc) > (uint32_t)TILE_CMAX) {
                // The column's own candidates do not fit one tile (cells holding a few hundred particles: the levels' junction
                // zones): its targets still get tiles -- one column, up to TILE_T targets -- in several PARTS, each with a
                // subset of the candidate rows that fits (greedy in row order).  A single row over the budget is hopeless.
                // (parts = 0: the caller's grid when internal levels are set -- a finer level serves such a column far cheaper)
                if (!parts || !__all_sync(0xFFFFFFFFu, myc <= (uint32_t)TILE_CMAX)) { ++cxa; skip = 0; continue; }
                uint32_t accr = 0, part = 0, mypart = 0xFFu;
                for (int l = 0; l < 16; ++l) {
                    const uint32_t cl = __shfl_sync(0xFFFFFFFFu, myc, l);
                    if (cl == 0u) continue;
                    if (accr + cl > (uint32_t)TILE_CMAX) { ++part; accr = 0; }
                    accr += cl;
                    if (lane == l) mypart = part;
                }
                const uint32_t nparts = part + 1u;
                uint32_t c = warp_sum(row.target ? row.te[cxa] - row.cs[cxa] : 0u) - skip;
                const uint32_t take = min(c, (uint32_t)TILE_T);
                if (take > 0) {
                    for (uint32_t p = 0; p < nparts; ++p) {
                        const uint32_t mask = __ballot_sync(0xFFFFFFFFu, mypart == p) & 0xFFFFu;
                        if (EMIT && lane == 0 && obase + ntl + p < cap) {
                            TileDesc td;
                            td.y0 = (int16_t)y0; td.z0 = (int16_t)z0; td.cxa = (int16_t)cxa; td.cxb = (int16_t)cxa;
                            td.nyr = (uint8_t)nyr; td.nzr = (uint8_t)nzr; td.part = (uint8_t)p; td.nparts = (uint8_t)nparts;
                            td.skip = skip; td.nt = take; td.rowmask = mask;
                            tiles[obase + ntl + p] = td;
                        }
                    }
                    ntl += nparts;
                    if (EMIT && lane == 0) atomicAdd(&ctr[CTR_NMULTI], 1ull);
                }
                if (take < c) skip += take; else { ++cxa; skip = 0; }
                continue;
            }
        }
        uint32_t nt = 0;
        int cxb = cxa, next_cxa = nx;
        uint32_t next_skip = 0;
        for (int cx = cxa; cx < nx; ++cx) {
            if (cx > cxa) {
                const int ext = cx - cxa + 1;
                if (ext > TILE_BXMAX || (per && ext + 2 > nx) ||
                    warp_sum(row_count(row, cxa - 1, cx + 1, nx, per)) > (uint32_t)TILE_CMAX) {
                    next_cxa = cx; next_skip = 0; break;
                }
            }
            uint32_t c = warp_sum(row.target ? row.te[cx] - row.cs[cx] : 0u);
            if (cx == cxa) c -= skip;
            const uint32_t take = min(c, (uint32_t)TILE_T - nt);
            nt += take;
            cxb = cx;
            if (take < c) { next_cxa = cx; next_skip = (cx == cxa ? skip : 0u) + take; break; }
            if (nt == (uint32_t)TILE_T) { next_cxa = cx + 1; next_skip = 0; break; }
        }
        if (nt > 0) {
            if (EMIT && lane == 0 && obase + ntl < cap) {
                TileDesc td;
                td.y0 = (int16_t)y0; td.z0 = (int16_t)z0; td.cxa = (int16_t)cxa; td.cxb = (int16_t)cxb;
                td.nyr = (uint8_t)nyr; td.nzr = (uint8_t)nzr; td.part = 0; td.nparts = 1; td.skip = skip; td.nt = nt; td.rowmask = 0xFFFFu;
                tiles[obase + ntl] = td;
            }
            ++ntl;
        }
        cxa = next_cxa; skip = next_skip;
    }
    if (!EMIT) {
        if (lane == 0) bcount[b] = ntl;
    } else if (b == nby * nbz - 1 && lane == 0) {
        const uint32_t total = obase + ntl;
        ctr[CTR_NTILES] = total < cap ? total : cap;
        if (total > cap) ctr[CTR_NTILES] = cap;      // dropped tiles: their particles use the general kernels
        ctr[CTR_NALL] = n_all;
    }
}

// ------------------------------------------------------------------------------------------- tile tables
// TileS of every tile, computed once per build and kept in global memory: the list builder and every sweep copy
// them into shared memory instead of recomputing them.
__global__ void __launch_bounds__(128)
k_tile_tables(DevGrid g, CellTable ct, const TileDesc* __restrict__ tiles, const unsigned long long* __restrict__ ctr,
              uint32_t* __restrict__ tiletab) {
    __shared__ TileS S;
    const uint32_t ntiles = (uint32_t)ctr[CTR_NTILES];
    for (uint32_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const TileDesc td = tiles[tile];
        __syncthreads();
        tile_setup(td, g, ct, S);
        uint32_t* dst = tiletab + (size_t)tile * TILES_WORDS;
        const uint32_t* src = reinterpret_cast<const uint32_t*>(&S);
        for (int w = threadIdx.x; w < TILES_WORDS; w += blockDim.x) dst[w] = src[w];
    }
}

// ------------------------------------------------------------------------------------------- list builder
// One CTA of BL_THREADS threads builds the lists of HALF a tile (targets [128 half, 128 half + 128), i.e. warps
// 8 half .. 8 half + 7 of the sweeps' CTA), so that two CTAs fit on an SM and one's barriers and staging latencies are
// covered by the other's scan.  Work unit w = 2 tile + half.
//
// THE SCAN.  Candidates are staged as fp32 coordinates relative to the tile centre, one array per component, indexed
// by slot; candidate ranges start on multiples of 8 slots, so an aligned BLOCK of 8 slots holds one slot of every
// shared-memory bank of the sweeps (slot & 7).  The two threads of a target split the banks: thread u tests slots
// 8 b + 4 u .. 8 b + 4 u + 3 of every block b of its warp's window with two packed (sm_100 FADD2/FFMA2) chains,
//     t = dz^2 + (dy^2 + (dx^2 - T_hi)),   T_hi = (2 h)^2 (1 + 1e-5) + Am   (error bound Am below),
// and a candidate with t < 0 is appended -- one predicated 16-bit store of the block number and one predicated
// pointer increment -- to the thread's bucket of the candidate's bank.  The thread keeps min |t| over everything
// it tested: if that stays above the width of the uncertainty band, every decision of the fp32 test was certain
// and the buckets are final (only the target itself has to be taken out); otherwise, and in tiles with variable h,
// every bucket entry is classified again (fp32 bounds first, then the exact fp64 contract predicate, O2/A12), so the
// sets are bit-identical to the definition.  A hit is never lost: t < 0 is a superset of the support.
struct ListArgs {
    const double2 *p0, *p1;            // sorted (x, y), (z, h)
    const TileDesc* tiles;
    unsigned long long* ctr;           // CTR_*
    uint2* pool;                       // list storage, rows of 32 lanes x 4 u16 slots, allocated from ctr[CTR_POOL]
    uint32_t pool_rows;                // capacity in rows
    uint2* winfo;                      // [tile][warp]: (first pool row, rounds)
    uint32_t* lcount;                  // [tile][TILE_T]: n_gather | n_sym << 16
    uint32_t* tflags;                  // [tile], zeroed before the launch; each half ORs its bits in
    const uint32_t* tiletab;           // [tile][TILES_WORDS]
    uint8_t* fast;                     // [n] sorted order: 1 = served by the tiled kernels
    uint8_t* fail;                     // [n] sorted order, zeroed before the launch: a target of a multi-part tile that some part declined
    const double* hglob;
    uint32_t* status;
    float rmax;                        // > 0: largest support radius the unit can meet (level contexts); else 2 max h from hglob
};

constexpr int BL_THREADS = TILE_THREADS / 2;
constexpr int BL_WARPS = BL_THREADS / 32;
constexpr int BL_TGT = TILE_T / 2;
constexpr int COLW = TILE_BXMAX + 4;
constexpr int LIST_TRASH = 4;                // trash rows of a bucket: the scan clamps its row pointers once per 4 blocks
constexpr int LIST_BS = LIST_BC + LIST_TRASH;
constexpr int LIST_LCAP = LIST_RMAX;         // rounds of the schedule staging area
constexpr int WBLK_CAP = TILE_CMAXP / 8 + 8; // a warp's block list: every staged block at most, padded to a multiple of 4
constexpr size_t BL_OFF_X = 0;                                                          // float [CMAXP] each: x, y, z relative to the
constexpr size_t BL_OFF_Y = BL_OFF_X + sizeof(float) * TILE_CMAXP;                      // tile centre, T = (2 h)^2
constexpr size_t BL_OFF_Z = BL_OFF_Y + sizeof(float) * TILE_CMAXP;
constexpr size_t BL_OFF_T = BL_OFF_Z + sizeof(float) * TILE_CMAXP;
constexpr size_t BL_CAND_END = BL_OFF_T + sizeof(float) * TILE_CMAXP;
constexpr size_t BL_OFF_L = 0;                                                          // uint2 [LIST_LCAP / 4][BL_THREADS]: the schedule, 4 rounds per
                                                                                        // word pair, written after the scan is over -- shares the
                                                                                        // space of the candidates
constexpr size_t BL_L_END = BL_OFF_L + sizeof(uint16_t) * LIST_LCAP * BL_THREADS;
constexpr size_t BL_OFF_B = BL_CAND_END > BL_L_END ? BL_CAND_END : BL_L_END;             // u16 [4][LIST_BS][BL_THREADS]
constexpr size_t BL_OFF_COL = BL_OFF_B + sizeof(uint16_t) * 4 * LIST_BS * BL_THREADS;   // u16 [MAXR][COLW]
constexpr size_t BL_OFF_WB = BL_OFF_COL + sizeof(uint16_t) * TILE_MAXR * COLW;          // u16 [BL_WARPS][WBLK_CAP]
constexpr size_t BL_SMEM = BL_OFF_WB + sizeof(uint16_t) * BL_WARPS * WBLK_CAP;
static_assert(2 * (BL_SMEM + 2 * sizeof(TileS) + 1280) <= 228 * 1024, "list builder: two CTAs per SM");
static_assert(TILE_CMAXP % 8 == 0 && TILE_CMAX % 8 == 0, "blocks of 8 slots");
static_assert(TILES_WORDS <= 2 * BL_THREADS, "tile table prefetch: two words per thread");
static_assert(sizeof(TileDesc) == 24, "tile descriptor prefetch: six words");
static_assert(BL_OFF_WB % 8 == 0 && WBLK_CAP % 4 == 0, "block list rows are read four entries at a time");

// packed fp32 pairs (sm_100 FADD2 / FMUL2 / FFMA2): one instruction tests two candidates
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float a, float b) { f32x2 r; asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ void unpk2(f32x2 v, float& a, float& b) { asm("mov.b64 {%0,%1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); }
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b) { f32x2 r; asm("sub.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) { f32x2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }

// One candidate of the scan: if t < 0 store the block number at the bucket row pointer and advance it.  No branches; the
// caller clamps the pointer at the first trash row of the bucket once per LIST_TRASH blocks.
__device__ __forceinline__ void append_if_neg(float t, uint32_t& addr, uint32_t blk) {
    asm volatile("{\n\t.reg .pred p;\n\t"
                 "setp.lt.f32 p, %1, 0f00000000;\n\t"
                 "@p st.shared.u16 [%0], %2;\n\t"
                 "@p add.u32 %0, %0, %3;\n\t}"
                 : "+r"(addr) : "f"(t), "r"(blk), "n"(2 * BL_THREADS));
    // no memory clobber: the loads of the next blocks must be free to move above the store; the buckets are read back
    // only after the fence that follows the scan
}
__device__ __forceinline__ uint32_t lds_u16(uint32_t addr) { uint32_t v; asm volatile("ld.shared.u16 %0, [%1];" : "=r"(v) : "r"(addr)); return v; }
__device__ __forceinline__ void sts_u16(uint32_t addr, uint32_t v) { asm volatile("st.shared.u16 [%0], %1;" :: "r"(addr), "r"(v)); }

// Which thread of a target owns bank beta in the scan (thread u tests slots 8 b + 4 u .. 8 b + 4 u + 3), and the index
// of that bank among the owner's four buckets.
__device__ __forceinline__ int bank_owner(int beta) { return beta >> 2; }
__device__ __forceinline__ int bank_local(int beta) { return beta & 3; }


__global__ void __launch_bounds__(BL_THREADS, 2)
k_build_lists(DevGrid g, CellTable ct, ListArgs A) {
    extern __shared__ __align__(16) unsigned char smem[];
    __shared__ TileS Sb[2];                                             // this unit's tile table / the next unit's, prefetched
    __shared__ uint32_t s_td[2][6];
    __shared__ int s_bad, s_nonuni, s_clo, s_chi;
    __shared__ double s_h0;
    float* X = reinterpret_cast<float*>(smem + BL_OFF_X);
    float* Y = reinterpret_cast<float*>(smem + BL_OFF_Y);
    float* Z = reinterpret_cast<float*>(smem + BL_OFF_Z);
    float* Tc = reinterpret_cast<float*>(smem + BL_OFF_T);
    uint16_t* Lf = reinterpret_cast<uint16_t*>(smem + BL_OFF_L);       // [k * BL_THREADS + tid]
    uint16_t* B = reinterpret_cast<uint16_t*>(smem + BL_OFF_B);        // [(b * LIST_BS + k) * BL_THREADS + tid]
    uint16_t* colofs = reinterpret_cast<uint16_t*>(smem + BL_OFF_COL); // [range][COLW]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    uint16_t* wblk = reinterpret_cast<uint16_t*>(smem + BL_OFF_WB) + warp * WBLK_CAP;
    const int u = tid & 1, j = lane & 7;
    const uint32_t nunits = 2u * (uint32_t)A.ctr[CTR_NTILES];
    const float Rmax = A.rmax > 0.f ? A.rmax : 2.0f * (float)A.hglob[1] * 1.000001f;
    constexpr uint32_t BROW = 2u * BL_THREADS;                        // bytes per bucket row

    // tile table and descriptor of the first unit; afterwards each unit prefetches the next one's while it works
    if (blockIdx.x < nunits) {
        const uint32_t tile = blockIdx.x >> 1;
        const uint32_t* src = A.tiletab + (size_t)tile * TILES_WORDS;
        uint32_t* dst = reinterpret_cast<uint32_t*>(&Sb[0]);
        for (int w = tid; w < TILES_WORDS; w += BL_THREADS) dst[w] = src[w];
        if (tid < 6) s_td[0][tid] = reinterpret_cast<const uint32_t*>(A.tiles + tile)[tid];
    }
    int buf = 0;
    for (uint32_t unit = blockIdx.x; unit < nunits; unit += gridDim.x, buf ^= 1) {
        __syncthreads();                                                // previous unit done with smem; this unit's table is in place
        const TileS& S = Sb[buf];
        const uint32_t tile = unit >> 1;
        const int half = (int)(unit & 1u);
        TileDesc td;
        {
            uint32_t* w = reinterpret_cast<uint32_t*>(&td);
#pragma unroll
            for (int k = 0; k < 6; ++k) w[k] = s_td[buf][k];
        }
        // prefetch: two table words (and one descriptor word) per thread, parked in registers until the end of the unit
        const uint32_t nunit = unit + gridDim.x;
        uint32_t pf0 = 0, pf1 = 0, pfd = 0;
        if (nunit < nunits) {
            const uint32_t* src = A.tiletab + (size_t)(nunit >> 1) * TILES_WORDS;
            pf0 = __ldg(src + tid);
            if (tid + BL_THREADS < TILES_WORDS) pf1 = __ldg(src + tid + BL_THREADS);
            if (tid < 6) pfd = __ldg(reinterpret_cast<const uint32_t*>(A.tiles + (nunit >> 1)) + tid);
        }
        const int tgt = half * BL_TGT + (tid >> 1);                     // target index within the tile
        const int twarp = half * BL_WARPS + warp;                       // warp index within the tile
        if (half * BL_TGT >= (int)td.nt) {                              // no target in this half: empty lists
            if (lane == 0) A.winfo[(size_t)tile * TILE_WARPS + twarp] = make_uint2(0u, 0u);
            if (u == 0) A.lcount[(size_t)tile * TILE_T + tgt] = 0u;
            if (tid == 0) atomicOr(&A.tflags[tile], TILE_FLAG_OK0 << half);
        } else {
        if (tid == 0) { s_bad = 0; s_nonuni = 0; s_clo = 1 << 20; s_chi = -1; }
        const int ncolv = td.cxb - td.cxa + 3;                          // virtual columns 0 .. ncolv-1
        // tile origin (centre of the tile's cell block) for the fp32 relative coordinates
        const double ox = g.lo[0] + (0.5 * (td.cxa + td.cxb + 1)) * g.edge[0];
        const double oy = g.lo[1] + (td.y0 + 0.5 * td.nyr) * g.edge[1];
        const double oz = g.lo[2] + (td.z0 + 0.5 * td.nzr) * g.edge[2];
        // Bound on the absolute error of an fp32 relative coordinate difference: every staged coordinate lies within
        // ext of the origin (checked while staging: particles clamped into an edge cell from outside an open box do not,
        // and send the unit to the general kernels), so each of the two operands carries one rounding <= 2^-24 ext and
        // the difference another one: 3 x 2^-24 ext < E.
        const float ext = (float)fmax(fmax((0.5 * ncolv + 0.5) * g.edge[0], 2.5 * g.edge[1]), 2.5 * g.edge[2]);
        const float extc = ext * 1.0001f;
        const float E = ext * 2.4e-7f;                                  // 4 * 2^-24 * ext
        // |r2_fp32 - r2| <= 2 (|dx| + |dy| + |dz|) E + 3 E^2 + the roundings of the three fused steps (relative 2^-24 each,
        // of max(r2, T) <= 1.1 T: covered by the relative margin 1e-5 of the thresholds) <= 2 sqrt(3) Rmax' E + 3 E^2 near a
        // support boundary
        const float Am = 4.4f * Rmax * E + 5.0f * E * E;

        // ---- per-range column offsets (slot of the first particle of each column, relative to r_base)
        for (int w = tid; w < (int)S.nranges * COLW; w += BL_THREADS) {
            const int q = w / COLW, jj = w % COLW;
            const int4 ge = S.r_geo[q];
            if (jj <= ge.y) {
                const uint32_t gs = (jj < ge.y) ? ct.cell_start[ge.w + jj] : S.r_vend[q];
                colofs[q * COLW + jj] = (uint16_t)(gs - S.r_vstart[q]);
            }
        }
        // ---- this thread's target
        const bool active = tgt < (int)td.nt;
        uint32_t i = 0, s_self = 0xFFFFFFFFu;
        double xa = 0, ya = 0, za = 0, ha = 0;
        int tcol = 0, try_ = 0, trz = 0;
        bool tbad = false;
        if (active) {
            int e;
            i = tile_target(td, S, tgt, &e);
            int cxe;
            tile_cell_rc(td, e, cxe, try_, trz);
            tcol = cxe - td.cxa;
            const double2 xy = A.p0[i], zh = A.p1[i];
            xa = xy.x; ya = xy.y; za = zh.x; ha = zh.y;
            // the target's own slot: its row is candidate row (trz + 1, try_ + 1), one or two (wrapped x-range) pieces
            const int row = (trz + 1) * 4 + (try_ + 1);
            int q = S.r_row[row];
            if (q != 0xFF) {
                if (!(i >= S.r_vstart[q] && i < S.r_vend[q]) && q + 1 < (int)S.nranges && S.r_shift[q + 1][3] == row) ++q;
                if (i >= S.r_vstart[q] && i < S.r_vend[q]) s_self = S.r_base[q] + (i - S.r_vstart[q]);
            }
        }
        // an inactive thread sits far away from everything: it never hits
        const float fax = active ? (float)(xa - ox) : -3.0e18f, fay = (float)(ya - oy), faz = (float)(za - oz);
        if (active && !(fabsf(fax) <= extc && fabsf(fay) <= extc && fabsf(faz) <= extc)) tbad = true;
        const bool multi = td.nparts > 1;                               // one of several entries that share these targets (tiles.cuh)
        if (active && s_self == 0xFFFFFFFFu && !multi) tbad = true;     // cannot happen: the target's cell is among the candidates
        if (multi && tile - td.part + td.nparts > (nunits >> 1)) tbad = true;   // a group cut off at the tile capacity: nobody is served
        const float Ra = 2.0f * (float)ha;
        const float Ta = Ra * Ra;
        const float Ta_hi = fmaf(Ta, 1.00001f, Am), Ta_lo = fmaf(Ta, 0.99999f, -Am);
        // warp window in virtual columns / candidate rows; the union over the warps is what this CTA stages
        int cmin = active ? tcol : 1 << 20, cmax = active ? tcol : -1;
        int ymin = active ? try_ : 4, ymax = active ? try_ : -1;
        int zmin = active ? trz : 4, zmax = active ? trz : -1;
#pragma unroll
        for (int o = 16; o; o >>= 1) {
            cmin = min(cmin, __shfl_xor_sync(0xFFFFFFFFu, cmin, o)); cmax = max(cmax, __shfl_xor_sync(0xFFFFFFFFu, cmax, o));
            ymin = min(ymin, __shfl_xor_sync(0xFFFFFFFFu, ymin, o)); ymax = max(ymax, __shfl_xor_sync(0xFFFFFFFFu, ymax, o));
            zmin = min(zmin, __shfl_xor_sync(0xFFFFFFFFu, zmin, o)); zmax = max(zmax, __shfl_xor_sync(0xFFFFFFFFu, zmax, o));
        }
        __syncthreads();                                                // flags reset by thread 0 above; column offsets written
        // (a target that cannot be served -- tbad here, bucket overflow or a list that is too long below -- is declined on its
        //  own: empty lists, fast[i] stays 0, the general kernels compute it after the tiled sweeps and overwrite what they wrote)
        if (lane == 0 && cmax >= 0) { atomicMin(&s_clo, cmin); atomicMax(&s_chi, cmax); }
        if (tid == 0) s_h0 = ha;                                        // the half's first target: always there
        // ---- the warp's block list: lane q takes candidate range q, its blocks inside the warp's window (rows
        //      [ymin, ymax + 2] x [zmin, zmax + 2], virtual columns [cmin, cmax + 2]: one cell around every target), whole
        //      blocks of 8 slots; the list is padded to a multiple of 4 entries with the block of the dummy slots, which
        //      is staged out of reach.  A block that reaches over the window's columns brings in slots of the same row
        //      two or more cells away (never a neighbour); slots past the end of a range are put out of reach.
        uint32_t nwb = 0;
        {
            uint32_t b0 = 0, nb = 0;
            if (lane < (int)S.nranges && cmax >= 0) {
                const int row = S.r_shift[lane][3], ry = row & 3, rz = row >> 2;
                if (!(ry < ymin || ry > ymax + 2 || rz < zmin || rz > zmax + 2)) {
                    const int4 ge = S.r_geo[lane];
                    const int jlo = max(0, min(ge.y, cmin - ge.z)), jhi = max(0, min(ge.y, cmax + 3 - ge.z));
                    if (jhi > jlo) {
                        const uint32_t sa = S.r_base[lane] + colofs[lane * COLW + jlo];
                        const uint32_t sb = S.r_base[lane] + colofs[lane * COLW + jhi];
                        b0 = sa >> 3; nb = ((sb + 7u) >> 3) - b0;
                    }
                }
            }
            uint32_t incl = nb;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
                if (lane >= o) incl += v;
            }
            nwb = __shfl_sync(0xFFFFFFFFu, incl, 31);
            for (uint32_t k = 0, at = incl - nb; k < nb; ++k) wblk[at + k] = (uint16_t)(b0 + k);
            if (lane < 4) wblk[nwb + lane] = (uint16_t)(TILE_CMAX / 8);  // pad (up to 3 used)
        }
        __syncthreads();

        // ---- stage the candidates of virtual columns [s_clo, s_chi + 2], whole blocks of 8 slots: one warp per range
        {
            const unsigned long long h0 = (unsigned long long)__double_as_longlong(s_h0);
            const int clo = s_clo, chi = s_chi + 2;
            bool nonuni = false, far = false;
            for (int q = warp; q < (int)S.nranges; q += BL_WARPS) {
                const int4 ge = S.r_geo[q];
                const int jlo = max(0, min(ge.y, clo - ge.z)), jhi = max(0, min(ge.y, chi + 1 - ge.z));
                if (jhi <= jlo) continue;
                const uint32_t vs = S.r_vstart[q], len = S.r_vend[q] - vs, base = S.r_base[q];
                const uint32_t ka = (uint32_t)colofs[q * COLW + jlo] & ~7u, kb = ((uint32_t)colofs[q * COLW + jhi] + 7u) & ~7u;
                const double shx = S.r_shift[q][0] * g.L[0], shy = S.r_shift[q][1] * g.L[1], shz = S.r_shift[q][2] * g.L[2];
                for (uint32_t k = ka + lane; k < kb; k += 32) {
                    float fx = 3.0e18f, fy = 3.0e18f, fz = 3.0e18f, T = 0.0f;
                    if (k < len) {
                        const double2 xy = A.p0[vs + k], zh = A.p1[vs + k];
                        fx = (float)((xy.x - shx) - ox);                // image position next to the tile: x_b - shift*L
                        fy = (float)((xy.y - shy) - oy);
                        fz = (float)((zh.x - shz) - oz);
                        const float Rb = 2.0f * (float)zh.y;
                        T = Rb * Rb;
                        nonuni |= (unsigned long long)__double_as_longlong(zh.y) != h0;
                        far |= !(fabsf(fx) <= extc && fabsf(fy) <= extc && fabsf(fz) <= extc);
                    }
                    const uint32_t s = base + k;
                    X[s] = fx; Y[s] = fy; Z[s] = fz; Tc[s] = T;
                }
            }
            if (tid < TILE_NDUMMY) { X[TILE_CMAX + tid] = 3.0e18f; Y[TILE_CMAX + tid] = 3.0e18f; Z[TILE_CMAX + tid] = 3.0e18f; Tc[TILE_CMAX + tid] = 0.0f; }
            if (nonuni) s_nonuni = 1;                                   // some staged candidate differs from the first target's h
            if (far) { s_bad = 1; atomicAdd(&A.ctr[CTR_DECL + 3], 1ull); }   // the error bound does not hold: general kernels
        }
        __syncthreads();
        const bool uni = s_nonuni == 0;

        // ---- scan (see the header).  All lanes of one parity read the same 16 bytes (shared-memory broadcast).
        const uint32_t bk0 = (uint32_t)__cvta_generic_to_shared(B + tid);
        uint32_t bp0 = bk0, bp1 = bk0 + LIST_BS * BROW, bp2 = bk0 + 2 * LIST_BS * BROW, bp3 = bk0 + 3 * LIST_BS * BROW;
        const uint32_t e0 = bk0 + LIST_BC * BROW, e1 = e0 + LIST_BS * BROW, e2 = e1 + LIST_BS * BROW, e3 = e2 + LIST_BS * BROW;
        float tmin = 3.0e38f;                                           // min |t| over the tested candidates
        float zb0 = 0.f, zb1 = 0.f, zb2 = 0.f, zb3 = 0.f;               // max -t per bank: T_hi exactly = a candidate at fp32 distance 0
        {
            const f32x2 ax2 = pk2(fax, fax), ay2 = pk2(fay, fay), az2 = pk2(faz, faz);
            const f32x2 nT2 = pk2(-Ta_hi, -Ta_hi);
            const float4* X4 = reinterpret_cast<const float4*>(X) + u;   // [2 b]: slots 8 b + 4 u ..
            const float4* Y4 = reinterpret_cast<const float4*>(Y) + u;
            const float4* Z4 = reinterpret_cast<const float4*>(Z) + u;
            const float4* T4 = reinterpret_cast<const float4*>(Tc) + u;
            auto block_uni = [&](uint32_t b) {
                const float4 x = X4[2 * b], y = Y4[2 * b], z = Z4[2 * b];
                const f32x2 dx0 = sub2(ax2, pk2(x.x, x.y)), dy0 = sub2(ay2, pk2(y.x, y.y)), dz0 = sub2(az2, pk2(z.x, z.y));
                const f32x2 dx1 = sub2(ax2, pk2(x.z, x.w)), dy1 = sub2(ay2, pk2(y.z, y.w)), dz1 = sub2(az2, pk2(z.z, z.w));
                float t0, t1, t2, t3;
                unpk2(fma2(dz0, dz0, fma2(dy0, dy0, fma2(dx0, dx0, nT2))), t0, t1);
                unpk2(fma2(dz1, dz1, fma2(dy1, dy1, fma2(dx1, dx1, nT2))), t2, t3);
                append_if_neg(t0, bp0, b); append_if_neg(t1, bp1, b); append_if_neg(t2, bp2, b); append_if_neg(t3, bp3, b);
                tmin = fminf(fminf(tmin, fabsf(t0)), fminf(fabsf(t1), fminf(fabsf(t2), fabsf(t3))));
                zb0 = fmaxf(zb0, -t0); zb1 = fmaxf(zb1, -t1); zb2 = fmaxf(zb2, -t2); zb3 = fmaxf(zb3, -t3);
            };
            auto block_gen = [&](uint32_t b) {
                const float4 x = X4[2 * b], y = Y4[2 * b], z = Z4[2 * b], T = T4[2 * b];
                const f32x2 dx0 = sub2(ax2, pk2(x.x, x.y)), dy0 = sub2(ay2, pk2(y.x, y.y)), dz0 = sub2(az2, pk2(z.x, z.y));
                const f32x2 dx1 = sub2(ax2, pk2(x.z, x.w)), dy1 = sub2(ay2, pk2(y.z, y.w)), dz1 = sub2(az2, pk2(z.z, z.w));
                // support of the larger h, error bound added
                const float n0 = -fmaf(fmaxf(Ta, T.x), 1.00001f, Am), n1 = -fmaf(fmaxf(Ta, T.y), 1.00001f, Am);
                const float n2 = -fmaf(fmaxf(Ta, T.z), 1.00001f, Am), n3 = -fmaf(fmaxf(Ta, T.w), 1.00001f, Am);
                float t0, t1, t2, t3;
                unpk2(fma2(dz0, dz0, fma2(dy0, dy0, fma2(dx0, dx0, pk2(n0, n1)))), t0, t1);
                unpk2(fma2(dz1, dz1, fma2(dy1, dy1, fma2(dx1, dx1, pk2(n2, n3)))), t2, t3);
                append_if_neg(t0, bp0, b); append_if_neg(t1, bp1, b); append_if_neg(t2, bp2, b); append_if_neg(t3, bp3, b);
            };
            const uint2* wb4 = reinterpret_cast<const uint2*>(wblk);
            if (uni) {
                for (uint32_t k = 0; k < nwb; k += 4) {
                    const uint2 w = wb4[k >> 2];
                    block_uni(w.x & 0xFFFFu); block_uni(w.x >> 16); block_uni(w.y & 0xFFFFu); block_uni(w.y >> 16);
                    bp0 = min(bp0, e0); bp1 = min(bp1, e1); bp2 = min(bp2, e2); bp3 = min(bp3, e3);
                }
            } else {
                for (uint32_t k = 0; k < nwb; k += 4) {
                    const uint2 w = wb4[k >> 2];
                    block_gen(w.x & 0xFFFFu); block_gen(w.x >> 16); block_gen(w.y & 0xFFFFu); block_gen(w.y >> 16);
                    bp0 = min(bp0, e0); bp1 = min(bp1, e1); bp2 = min(bp2, e2); bp3 = min(bp3, e3);
                }
            }
        }
        asm volatile("" ::: "memory");                                  // the appends above wrote the buckets
        // ---- settle.  An entry is the block number of a hit of the fp32 test; its slot is 8 block + 4 u + bucket.
        uint32_t cnt = 0, ng = 0;                                       // cnt: 4 x 8-bit bucket fills
        bool ovf = (bp0 >= e0) || (bp1 >= e1) || (bp2 >= e2) || (bp3 >= e3), coinc = false;
        // Certain scan: no tested candidate within the uncertainty band of the support boundary, i.e. every fp32 decision
        // holds for the exact predicate too.  |t| >= band  <=>  r2_fp32 outside [T_lo, T_hi + (T_hi - T_lo)).
        const bool certain = uni && tmin >= (Ta_hi - Ta_lo);
        const bool sees_self = active && s_self != 0xFFFFFFFFu && ((s_self >> 2) & 1u) == (uint32_t)u;   // (a part may not hold the target's own row)
        const bool full_settle = __any_sync(0xFFFFFFFFu, !certain && !ovf);
        if (!full_settle) {
            // the target itself (r = 0) is met by the thread that owns its bank: take that one entry out of its bucket
            const uint32_t n0 = (bp0 - bk0) / BROW, n1 = (bp1 - (bk0 + LIST_BS * BROW)) / BROW;
            const uint32_t n2 = (bp2 - (bk0 + 2 * LIST_BS * BROW)) / BROW, n3 = (bp3 - (bk0 + 3 * LIST_BS * BROW)) / BROW;
            cnt = n0 | (n1 << 8) | (n2 << 16) | (n3 << 24);
            // A candidate at fp32 distance 0 (t = -T_hi exactly) is the target itself or a twin -- another particle at the same
            // place up to fp32 resolution, possibly at fp64 distance 0, where the pair bodies are not defined (A11): the target
            // is then declined (general kernels).  Only the bank of the target's own slot needs a look into the bucket.
            const uint32_t kself = sees_self ? (s_self & 3u) : 4u;
            if (active && ((zb0 == Ta_hi && kself != 0u) || (zb1 == Ta_hi && kself != 1u) || (zb2 == Ta_hi && kself != 2u) ||
                           (zb3 == Ta_hi && kself != 3u))) coinc = true;
            if (sees_self && !ovf) {
                const int b = (int)(s_self & 3u);
                uint16_t* bb = B + (size_t)b * LIST_BS * BL_THREADS + tid;
                const uint32_t nb = (cnt >> (8 * b)) & 0xFFu, want = s_self >> 3;
                uint32_t k = nb;
                for (uint32_t e = 0; e < nb; ++e) {
                    const uint32_t blk = bb[e * BL_THREADS];
                    if (blk == want) { k = e; continue; }
                    const uint32_t s = (blk << 3) + 4u * (uint32_t)u + (uint32_t)b;
                    if (X[s] == fax && Y[s] == fay && Z[s] == faz) coinc = true;
                }
                if (k < nb) {                                           // the last entry takes its place (order is free)
                    bb[k * BL_THREADS] = bb[(nb - 1) * BL_THREADS];
                    cnt -= 1u << (8 * b);
                }
            }
            ng = (cnt & 0xFFu) + ((cnt >> 8) & 0xFFu) + ((cnt >> 16) & 0xFFu) + (cnt >> 24);
        } else if (!ovf) {
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                const uint32_t nb = ((b == 0 ? bp0 : b == 1 ? bp1 : b == 2 ? bp2 : bp3) - (bk0 + b * LIST_BS * BROW)) / BROW;
                uint16_t* bb = B + (size_t)b * LIST_BS * BL_THREADS + tid;
                uint32_t w = 0;
                for (uint32_t k = 0; k < nb; ++k) {
                    const uint32_t blk = bb[k * BL_THREADS], s = (blk << 3) + 4u * (uint32_t)u + (uint32_t)b;
                    bool in_s = true, in_g = true;
                    const float dx = fax - X[s], dy = fay - Y[s], dz = faz - Z[s];
                    const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                    const float Tm = fmaxf(Ta, Tc[s]);
                    if (r2 < fmaf(Tm, 0.99999f, -Am) && (r2 < Ta_lo || r2 >= Ta_hi) && r2 > 0.0f) {
                        in_g = r2 < Ta_lo;                              // certain member of N_sym; N_gather decided with the same margin
                    } else if (s == s_self) {
                        in_s = false;
                    } else {
                        int q = 0;
                        while (q + 1 < (int)S.nranges && S.r_base[q + 1] <= s) ++q;
                        const uint32_t k2 = s - S.r_base[q];
                        if (k2 >= S.r_vend[q] - S.r_vstart[q]) {
                            in_s = false;                               // pad slot (cannot hit; kept for safety)
                        } else {
                            const uint32_t gi = S.r_vstart[q] + k2;
                            const double2 xy = A.p0[gi], zh = A.p1[gi];
                            const double ex2 = min_image(__dsub_rn(xa, xy.x), g.per[0], g.L[0], g.halfL[0]);
                            const double ey2 = min_image(__dsub_rn(ya, xy.y), g.per[1], g.L[1], g.halfL[1]);
                            const double ez2 = min_image(__dsub_rn(za, zh.x), g.per[2], g.L[2], g.halfL[2]);
                            const double e2x = r2_exact(ex2, ey2, ez2);
                            in_s = gi != i && e2x < support2(fmax(ha, zh.y));
                            in_g = in_s && e2x < support2(ha);
                            if (in_s && !(e2x > 1.0e-290)) coinc = true;    // (near-)coincident particles: left to the general kernels (A11)
                        }
                    }
                    if (in_s) bb[w * BL_THREADS] = (uint16_t)blk;
                    w += in_s ? 1u : 0u;
                    ng += (in_s && in_g) ? 1u : 0u;
                }
                cnt |= w << (8 * b);
            }
        }
        if (active && (ovf || coinc || (tbad && u == 0))) atomicAdd(&A.ctr[CTR_DECL + (ovf ? 2 : 3)], 1ull);
        bool tdecl = ovf || coinc || tbad;                              // decline this target (both of its threads agree below)
        tdecl = __shfl_xor_sync(0xFFFFFFFFu, (int)tdecl, 1) != 0 || tdecl;
        if (tdecl) { cnt = 0; ng = 0; }
        // ---- split every bank bucket of the target between its two threads (alternate entries)
        const uint32_t cnt_o = __shfl_xor_sync(0xFFFFFFFFu, cnt, 1);
        ng += __shfl_xor_sync(0xFFFFFFFFu, ng, 1);
        uint32_t cu = 0;                                                // 8 x 4-bit: entries of bank beta that are mine (<= LIST_BC / 2)
        uint32_t n_lane = 0, nsym = 0;
#pragma unroll
        for (int beta = 0; beta < 8; ++beta) {
            const uint32_t cb = ((bank_owner(beta) == u ? cnt : cnt_o) >> (8 * bank_local(beta))) & 0xFFu;
            const uint32_t f = (uint32_t)(u + beta) & 1u;
            const uint32_t mine = (cb + 1u - f) >> 1;
            cu |= mine << (4 * beta);
            n_lane += mine; nsym += cb;
        }
        {   // a list longer than the schedule can hold: decline the target
            bool toolong = n_lane > (uint32_t)LIST_RMAX;
            toolong = __shfl_xor_sync(0xFFFFFFFFu, (int)toolong, 1) != 0 || toolong;
            if (toolong) {
                if (active && u == 0) atomicAdd(&A.ctr[CTR_DECL + 2], 1ull);
                tdecl = true; cu = 0; n_lane = 0; nsym = 0; ng = 0;
            }
        }
        uint32_t R = n_lane;
#pragma unroll
        for (int o = 16; o; o >>= 1) R = max(R, __shfl_xor_sync(0xFFFFFFFFu, R, o));
        R = (R + 3u) & ~3u;
        __syncthreads();                                                // every warp is done with the staged candidates: the schedule
                                                                        // staging area below shares their space
        // list storage: rows of 32 lanes x 4 slots, R / 4 rows per warp, taken from the pool counter.  Placement depends on
        // the order in which warps get there; the contents of the rows do not.  If another warp sends the unit to the general
        // kernels after this one has emitted (list too long, pool exhausted), the rows stay unused.
        uint32_t row0 = 0;
        bool wbad = s_bad != 0;
        if (lane == 0 && !wbad && R) {
            const unsigned long long r0 = atomicAdd(&A.ctr[CTR_POOL], (unsigned long long)(R >> 2));
            if (r0 + (R >> 2) > (unsigned long long)A.pool_rows) { wbad = true; atomicAdd(&A.ctr[CTR_DECL + 1], 1ull); }   // pool exhausted
            row0 = (uint32_t)r0;
        }
        wbad = __shfl_sync(0xFFFFFFFFu, (int)wbad, 0) != 0;
        row0 = __shfl_sync(0xFFFFFFFFu, row0, 0);
        if (wbad) {
            if (lane == 0) s_bad = 1;
        } else {
            // ---- emit my half-list in scheduled order (see the header): phase t = rounds [tR/8, (t+1)R/8) in bank
            //      (j + t) & 7; what a phase cannot hold (overflow) fills the holes of other phases; the rest are dummies.
            // R = 8 m + 4 e (e = 0, 1): phase t starts at t m + e (t >> 1) and holds m + e (t & 1) rounds.
            const uint32_t m8 = R >> 3, e4 = (R >> 2) & 1u;
            uint16_t* out = Lf + tid;                                   // my column of the schedule: out[r * BL_THREADS]
            const uint16_t* Bp = B + (tid & ~1);
            uint32_t own[8], ovr[8];                                    // per phase: entries placed in the phase / left over
            const uint16_t* bq[8];                                      // per phase: my entries of its bank (stride 2 rows)
            uint32_t Hw = 0;                                            // 8 x 4-bit: holes of each phase
#pragma unroll
            for (int t = 0; t < 8; ++t) {
                const int beta = (j + t) & 7;
                const uint32_t cap = m8 + (e4 & (uint32_t)(t & 1));
                const uint32_t c = (cu >> (4 * beta)) & 15u;
                own[t] = min(c, cap);
                ovr[t] = c - own[t];
                Hw |= (cap - own[t]) << (4 * t);
                // my entries of bank beta: indices f, f+2, ... of the bucket of thread bank_owner(beta)
                bq[t] = Bp + (bank_local(beta) * LIST_BS + ((u + beta) & 1)) * BL_THREADS + bank_owner(beta);
            }
            // pass 1 (lockstep): every phase takes its own bank's entries up to its capacity (an entry is a block number:
            // slot = 8 block + bank); a hole gets the dummy slot of the phase's bank
            for (uint32_t k = 0; k < m8; ++k) {
#pragma unroll
                for (int t = 0; t < 8; ++t) {
                    const uint32_t beta = (uint32_t)(j + t) & 7u;
                    uint32_t item = (uint32_t)TILE_CMAX + beta;
                    if (k < own[t]) item = ((uint32_t)bq[t][2 * k * BL_THREADS] << 3) + beta;
                    out[((uint32_t)t * m8 + (e4 ? (uint32_t)(t >> 1) : 0u) + k) * BL_THREADS] = (uint16_t)item;
                }
            }
            if (e4) {
#pragma unroll
                for (int t = 1; t < 8; t += 2) {
                    const uint32_t beta = (uint32_t)(j + t) & 7u;
                    uint32_t item = (uint32_t)TILE_CMAX + beta;
                    if (m8 < own[t]) item = ((uint32_t)bq[t][2 * m8 * BL_THREADS] << 3) + beta;
                    out[((uint32_t)t * m8 + (uint32_t)(t >> 1) + m8) * BL_THREADS] = (uint16_t)item;
                }
            }
            // the left-over entries go into the holes (a phase has either holes or left-overs): one left-over per iteration,
            // its phase and the phase of the next hole are the first non-zero 4-bit fields
            {
                uint32_t Ov = 0;
#pragma unroll
                for (int t = 0; t < 8; ++t) Ov |= ovr[t] << (4 * t);
                const uint32_t Ov0 = Ov;
                while (Ov != 0u && Hw != 0u) {                          // Hw runs out only after Ov: n_lane <= R
                    const uint32_t ts = (uint32_t)(__ffs((int)Ov) - 1) >> 2, th = (uint32_t)(__ffs((int)Hw) - 1) >> 2;
                    const uint32_t beta = ((uint32_t)j + ts) & 7u;
                    const uint32_t cap_s = m8 + (e4 & ts & 1u);         // a phase with left-overs is full: own = cap
                    const uint32_t taken = ((Ov0 >> (4 * ts)) & 15u) - ((Ov >> (4 * ts)) & 15u);
                    const uint16_t* src = Bp + (bank_local((int)beta) * LIST_BS + ((u + (int)beta) & 1)) * BL_THREADS + bank_owner((int)beta);
                    const uint32_t hrem = (Hw >> (4 * th)) & 15u;
                    const uint32_t pos = (((th + 1u) * R) >> 3) - hrem;
                    out[pos * BL_THREADS] = (uint16_t)(((uint32_t)src[2 * (cap_s + taken) * BL_THREADS] << 3) + beta);
                    Ov -= 1u << (4 * ts); Hw -= 1u << (4 * th);
                }
            }
            // pass 2: pack 4 rounds per 8-byte store
            uint2* blk = A.pool + (size_t)row0 * 32 + lane;
            for (uint32_t r4 = 0; r4 < R; r4 += 4) {
                const uint32_t e0 = out[r4 * BL_THREADS], e1 = out[(r4 + 1) * BL_THREADS];
                const uint32_t e2 = out[(r4 + 2) * BL_THREADS], e3 = out[(r4 + 3) * BL_THREADS];
                blk[(size_t)(r4 >> 2) * 32] = make_uint2(e0 | (e1 << 16), e2 | (e3 << 16));
            }
            if (u == 0) A.lcount[(size_t)tile * TILE_T + tgt] = (active && !tdecl) ? (ng | (nsym << 16)) : 0u;
            if (lane == 0) A.winfo[(size_t)tile * TILE_WARPS + twarp] = make_uint2(row0, R);
        }
        const int served = __syncthreads_count(active && u == 0 && !tdecl);
        const bool bad = s_bad != 0;
        // served = every part served: part 0 sets the flag and counts, any part that declines marks the target, and the pass
        // after this kernel (k_apply_fail) takes the marked ones back
        if (active && u == 0) {
            if (!bad && !tdecl) { if (td.part == 0) A.fast[i] = 1; }
            else if (multi) A.fail[i] = 1;
        }
        if (tid == 0) {
            const uint32_t bits = (bad ? 0u : (TILE_FLAG_OK0 << half)) | (s_nonuni ? TILE_FLAG_NONUNI : 0u);
            if (bits) atomicOr(&A.tflags[tile], bits);
            if (s_nonuni && td.part) atomicOr(&A.tflags[tile - td.part], TILE_FLAG_NONUNI);   // the sweeps pick a group's pair bodies by its first entry
            if (s_nonuni) atomicAdd(&A.ctr[CTR_NNONUNI], 1ull);
            if (!bad && td.part == 0) atomicAdd(&A.ctr[CTR_NFAST], (unsigned long long)served);
        }
        }
        // the next unit's table goes into the other buffer (read after the barrier at the top of the loop)
        if (nunit < nunits) {
            uint32_t* dst = reinterpret_cast<uint32_t*>(&Sb[buf ^ 1]);
            dst[tid] = pf0;
            if (tid + BL_THREADS < TILES_WORDS) dst[tid + BL_THREADS] = pf1;
            if (tid < 6) s_td[buf ^ 1][tid] = pfd;
        }
    }
}

// targets of multi-part tiles that one of the parts declined: not served after all
__global__ void k_apply_fail(uint8_t* __restrict__ fast, const uint8_t* __restrict__ fail, int64_t n, unsigned long long* __restrict__ ctr) {
    if (ctr[CTR_NMULTI] == 0) return;                 // no tile in several parts: nothing can be marked
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const bool back = i < n && fail[i] && fast[i];
    if (back) fast[i] = 0;
    const unsigned m = __ballot_sync(0xFFFFFFFFu, back);
    if ((threadIdx.x & 31) == 0 && m) atomicAdd(&ctr[CTR_NFAST], (unsigned long long)(0ll - (long long)__popc(m)));
}

// ------------------------------------------------------------------------------------------- parity exports
// spray_neighbor_counts / _lists / _digest served FROM THE TILED LISTS for the particles the tiled kernels serve, so
// that the parity tests compare the very lists the sweeps run on with the oracle's sets (the general kernel does the
// rest).  N_sym is the list itself; N_gather(a) is its subset with r2 < 4 h_a^2, decided by the exact contract
// predicate on the fp64 coordinates (O2/A12).  Not on the hot path.
struct ExportArgs {
    const double2 *p0, *p1;
    const uint32_t* perm;
    const TileDesc* tiles;
    const uint32_t* tiletab;
    const unsigned long long* ctr;
    const uint2* pool;
    const uint2* winfo;
    const uint32_t* tflags;
    int symmetric;
    uint32_t* ocount;                  // mode 0
    const uint64_t* offsets;           // mode 1
    uint32_t* onbr;
    uint64_t *odsum, *odxor;           // mode 2
};

template <int MODE>
__global__ void __launch_bounds__(TILE_THREADS, 1)
k_tiled_export(DevGrid g, ExportArgs A) {
    __shared__ TileS S;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int u = tid & 1, tgt = tid >> 1;
    const uint32_t ntiles = (uint32_t)A.ctr[CTR_NTILES];
    // (a tile entry is part 0 of nparts, tiles.cuh: the parts' lists of a target are one list)
    for (uint32_t tile0 = blockIdx.x; tile0 < ntiles; tile0 += gridDim.x) {
        const TileDesc td0 = A.tiles[tile0];
        if (td0.part != 0) continue;
        const uint32_t np = td0.nparts > 1 ? min((uint32_t)td0.nparts, ntiles - tile0) : 1u;
        bool active = false, grp_ok = true;
        uint32_t i = 0;
        double xa = 0, ya = 0, za = 0, ha = 0;
        uint32_t cnt = 0;
        uint64_t dsum = 0, dxr = 0;
        // mode 1 needs the first thread's count before the second thread writes: two passes (count, then write)
        for (int pass = 0; pass < (MODE == 1 ? 2 : 1); ++pass) {
            uint32_t wpos = 0;
            if (MODE == 1 && pass == 1) {
                const uint32_t other = __shfl_xor_sync(0xFFFFFFFFu, cnt, 1);
                wpos = u ? other : 0u;                     // thread 1 writes after thread 0's entries
            }
            uint32_t c2 = 0;
            for (uint32_t part = 0; part < np; ++part) {
                const uint32_t tile = tile0 + part;
                const uint32_t flags = A.tflags[tile];
                const bool half_ok = ((flags >> (warp / (TILE_WARPS / 2))) & 1u) != 0;
                const TileDesc td = A.tiles[tile];
                __syncthreads();
                {
                    const uint32_t* src = A.tiletab + (size_t)tile * TILES_WORDS;
                    uint32_t* dst = reinterpret_cast<uint32_t*>(&S);
                    for (int w = tid; w < TILES_WORDS; w += TILE_THREADS) dst[w] = src[w];
                }
                __syncthreads();
                if (part == 0 && pass == 0) {
                    active = half_ok && tgt < (int)td.nt;
                    if (active) {
                        i = tile_target(td, S, tgt);
                        const double2 xy = A.p0[i], zh = A.p1[i];
                        xa = xy.x; ya = xy.y; za = zh.x; ha = zh.y;
                    }
                }
                if (!half_ok) grp_ok = false;
                uint2 wi = A.winfo[(size_t)tile * TILE_WARPS + warp];
                if (!half_ok || !active) wi.y = 0u;
                const uint2* lp = A.pool + (size_t)wi.x * 32 + lane;
                const uint64_t lbase = (MODE == 1 && active) ? A.offsets[A.perm[i]] : 0;
                for (uint32_t r = 0; r < wi.y; ++r) {
                    const uint2 w4 = lp[(size_t)(r >> 2) * 32];
                    const uint32_t half = (r & 2u) ? w4.y : w4.x;
                    const uint32_t s = (r & 1u) ? (half >> 16) : (half & 0xFFFFu);
                    if (s >= (uint32_t)TILE_CMAX) continue;                          // dummy entry
                    int q = 0;
                    while (q + 1 < (int)S.nranges && S.r_base[q + 1] <= s) ++q;
                    const uint32_t gi = S.r_vstart[q] + (s - S.r_base[q]);
                    if (!A.symmetric) {
                        const double2 xy = A.p0[gi], zh = A.p1[gi];
                        const double ex = min_image(__dsub_rn(xa, xy.x), g.per[0], g.L[0], g.halfL[0]);
                        const double ey = min_image(__dsub_rn(ya, xy.y), g.per[1], g.L[1], g.halfL[1]);
                        const double ez = min_image(__dsub_rn(za, zh.x), g.per[2], g.L[2], g.halfL[2]);
                        if (!(r2_exact(ex, ey, ez) < support2(ha))) continue;
                    }
                    const uint32_t id = A.perm[gi];
                    if (MODE == 1 && pass == 1) A.onbr[lbase + wpos + c2] = id;
                    if (MODE == 2) { const uint64_t hsh = mix64((uint64_t)id); dsum += hsh; dxr ^= hsh; }
                    ++c2;
                }
            }
            cnt = c2;
        }
        const uint32_t total = cnt + __shfl_xor_sync(0xFFFFFFFFu, cnt, 1);
        if (MODE == 2) {
            dsum += __shfl_xor_sync(0xFFFFFFFFu, dsum, 1);
            dxr ^= __shfl_xor_sync(0xFFFFFFFFu, dxr, 1);
        }
        if (MODE == 1) __syncwarp();
        if (active && grp_ok && u == 0) {
            const uint32_t ia = A.perm[i];
            if (MODE == 0) A.ocount[ia] = total;
            if (MODE == 2) { A.odsum[ia] = dsum; A.odxor[ia] = dxr; }
            if (MODE == 1) {               // ascending caller ids (debug export: insertion sort of this particle's segment)
                __threadfence_block();
                uint32_t* L = A.onbr + A.offsets[ia];
                for (uint32_t a = 1; a < total; ++a) {
                    uint32_t v = L[a]; int b = (int)a - 1;
                    while (b >= 0 && L[b] > v) { L[b + 1] = L[b]; --b; }
                    L[b + 1] = v;
                }
            }
        }
    }
}

cudaError_t launch_tiled_export(Ctx* c, int mode, int symmetric, uint32_t* ocount, const uint64_t* offsets, uint32_t* onbr,
                                uint64_t* odsum, uint64_t* odxor, cudaStream_t st) {
    if (c->n == 0 || !c->tl.enabled) return cudaSuccess;
    const Tiled& t = c->tl;
    ExportArgs A{c->pk.p0, c->pk.p1, c->perm, t.tiles, t.tiletab, t.ctr, t.pool, t.winfo, t.tflags, symmetric,
                 ocount, offsets, onbr, odsum, odxor};
    const int grid = t.sms * 2;
    if (mode == 0) k_tiled_export<0><<<grid, TILE_THREADS, 0, st>>>(c->dg, A);
    else if (mode == 1) k_tiled_export<1><<<grid, TILE_THREADS, 0, st>>>(c->dg, A);
    else k_tiled_export<2><<<grid, TILE_THREADS, 0, st>>>(c->dg, A);
    c->launches += 1;
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------- launcher
cudaError_t tiled_set_attributes(Ctx* c) {
    cudaError_t e = cudaFuncSetAttribute(k_build_lists, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)BL_SMEM);
    if (e == cudaSuccess) e = sweeps_set_attributes();
    if (e == cudaSuccess) c->tl.attr_device = c->device;
    return e;
}

cudaError_t launch_build_tiles(Ctx* c, cudaStream_t st) {
    Tiled& t = c->tl;
    t.enabled = false;
    if (c->n == 0 || !t.tiles) return cudaSuccess;
    // host-side guards: small periodic grids (a candidate row would appear twice), index width
    const spray_grid_t& gr = c->grid;
    if (c->n >= (1ll << 31)) return cudaSuccess;
    if (gr.periodic[0] && gr.ncell[0] < 3) return cudaSuccess;
    if (gr.periodic[1] && gr.ncell[1] < 4) return cudaSuccess;
    if (gr.periodic[2] && gr.ncell[2] < 4) return cudaSuccess;
    if (gr.ncell[0] > 32000 || gr.ncell[1] > 32000 || gr.ncell[2] > 32000) return cudaSuccess;
    const int brows = c->is_level ? 1 : 2;
    const int64_t nb = (int64_t)((gr.ncell[1] + brows - 1) / brows) * ((gr.ncell[2] + brows - 1) / brows);
    if (nb > t.bundle_cap) return cudaSuccess;
    cudaError_t e;
    if ((e = cudaMemsetAsync(t.ctr, 0, sizeof(unsigned long long) * CTR_COUNT, st)) != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(t.fast, 0, (size_t)c->n, st)) != cudaSuccess) return e;
    uint8_t* fail = c->fast_c;                        // free at this point of every build (written later, by the levels' bookkeeping, on the parent only)
    if ((e = cudaMemsetAsync(fail, 0, (size_t)c->n, st)) != cudaSuccess) return e;
    CellTable ct{c->cell_start, c->cell_end, c->is_level ? c->cell_tend : c->cell_end};
    const int blocks = (int)((nb * 32 + 255) / 256);
    const int lvl = c->is_level ? 1 : 0;
    const int parts = (c->is_level || c->nlevels == 0) ? 1 : 0;
    k_make_tiles<false><<<blocks, 256, 0, st>>>(c->dg, ct, c->hglob, t.bcount, t.tiles, (uint32_t)t.tile_cap, t.ctr, lvl, (unsigned long long)c->n, brows, parts);
    if ((e = launch_excl_scan_u32(c, t.bcount, nb, t.bcount + t.bundle_cap, st)) != cudaSuccess) return e;
    k_make_tiles<true><<<blocks, 256, 0, st>>>(c->dg, ct, c->hglob, t.bcount, t.tiles, (uint32_t)t.tile_cap, t.ctr, lvl, (unsigned long long)c->n, brows, parts);
    k_tile_tables<<<t.sms * 8, 128, 0, st>>>(c->dg, ct, t.tiles, t.ctr, t.tiletab);
    if ((e = cudaMemsetAsync(t.tflags, 0, sizeof(uint32_t) * (size_t)t.tile_cap, st)) != cudaSuccess) return e;
    if (c->ev[2]) cudaEventRecord(c->ev[2], st);
    ListArgs A{c->pk.p0, c->pk.p1, t.tiles, t.ctr, t.pool, (uint32_t)t.pool_rows, t.winfo, t.lcount, t.tflags, t.tiletab, t.fast, fail,
               c->hglob, c->dev_status, c->is_level ? c->level_rmax : 0.f};
    k_build_lists<<<t.sms * 2, BL_THREADS, BL_SMEM, st>>>(c->dg, ct, A);
    k_apply_fail<<<(int)((c->n + 255) / 256), 256, 0, st>>>(t.fast, fail, c->n, t.ctr);
    c->launches += 5;
    t.enabled = true;
    return cudaGetLastError();
}

}  // namespace spray
