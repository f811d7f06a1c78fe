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
    const uint32_t *cs, *ce;         // cell_start / cell_end of the row (indexed by column)
    bool valid;
    bool target;                     // the row is one of the bundle's own rows
};
__device__ __forceinline__ uint32_t row_count(const RowRef& r, int xlo, int xhi, int nx, bool per) {
    if (!r.valid) return 0u;
    if (per) {
        if (xlo < 0) return (r.ce[nx - 1] - r.cs[xlo + nx]) + (r.ce[xhi] - r.cs[0]);
        if (xhi >= nx) return (r.ce[nx - 1] - r.cs[xlo]) + (r.ce[xhi - nx] - r.cs[0]);
    } else {
        xlo = xlo < 0 ? 0 : xlo;
        xhi = xhi > nx - 1 ? nx - 1 : xhi;
    }
    return r.ce[xhi] - r.cs[xlo];
}
__device__ __forceinline__ uint32_t warp_sum(uint32_t v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
    return v;
}

template <bool EMIT>
__global__ void __launch_bounds__(256)
k_make_tiles(DevGrid g, CellTable ct, const double* __restrict__ hglob, uint32_t* __restrict__ bcount,
             TileDesc* __restrict__ tiles, uint32_t cap, unsigned long long* __restrict__ ctr) {
    const int nby = (g.nc[1] + 1) / 2, nbz = (g.nc[2] + 1) / 2;
    const int b = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (b >= nby * nbz) return;
    // every neighbour within one cell: 2 h_max <= cell edge in every dimension (tiny safety margin)
    const double hmax = hglob[1];
    bool ok = true;
    for (int d = 0; d < 3; ++d)
        if (!(2.0 * hmax * g.inv[d] * (1.0 + 1e-9) <= 1.0)) ok = false;
    const int nx = g.nc[0];
    const int y0 = 2 * (b % nby), z0 = 2 * (b / nby);
    const int nyr = min(2, g.nc[1] - y0), nzr = min(2, g.nc[2] - z0);
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
        row.cs = ct.cell_start + base; row.ce = ct.cell_end + base;
    }
    const bool per = g.per[0] != 0;
    uint32_t ntl = 0;
    const uint32_t obase = EMIT ? bcount[b] : 0u;
    int cxa = 0;
    uint32_t skip = 0;
    while (ok && cxa < nx) {
        if (warp_sum(row_count(row, cxa - 1, cxa + 1, nx, per)) > (uint32_t)(TILE_CMAX - TILE_MAXR)) { ++cxa; skip = 0; continue; }   // column not tileable
        uint32_t nt = 0;
        int cxb = cxa, next_cxa = nx;
        uint32_t next_skip = 0;
        for (int cx = cxa; cx < nx; ++cx) {
            if (cx > cxa) {
                const int ext = cx - cxa + 1;
                if (ext > TILE_BXMAX || (per && ext + 2 > nx) ||
                    warp_sum(row_count(row, cxa - 1, cx + 1, nx, per)) > (uint32_t)(TILE_CMAX - TILE_MAXR)) {
                    next_cxa = cx; next_skip = 0; break;
                }
            }
            uint32_t c = warp_sum(row.target ? row.ce[cx] - row.cs[cx] : 0u);
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
                td.nyr = (uint8_t)nyr; td.nzr = (uint8_t)nzr; td.pad = 0; td.skip = skip; td.nt = nt; td.pad2 = 0;
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
struct ListArgs {
    const double2 *p0, *p1;            // sorted (x, y), (z, h)
    const TileDesc* tiles;
    unsigned long long* ctr;           // CTR_*
    uint2* pool;
    uint2* winfo;                      // [tile][warp]: (pool offset, rounds)
    uint32_t* lcount;                  // [tile][TILE_T]: n_gather | n_sym << 16
    uint32_t* tflags;                  // [tile], zeroed before the launch; each half ORs its bits in
    const uint32_t* tiletab;           // [tile][TILES_WORDS]
    uint8_t* fast;                     // [n] sorted order: 1 = served by the tiled kernels
    const double* hglob;
    uint32_t* status;
};

constexpr int BL_THREADS = TILE_THREADS / 2;
constexpr int BL_WARPS = BL_THREADS / 32;
constexpr int BL_TGT = TILE_T / 2;
constexpr int COLW = TILE_BXMAX + 4;
constexpr uint32_t LIST_RECHECK = 0x8000u;   // bucket-entry flag: classify this hit again (fp32 bounds, then exact fp64)
constexpr int LIST_BS = LIST_BC + 1;        // rows of a (thread, bank) bucket incl. the trash row
constexpr int LIST_LCAP = LIST_RMAX;       // rows of the schedule staging area (one column per thread)
constexpr size_t BL_OFF_XY = 0;                                                         // float4 [CMAXP/2]: (x0, x1, y0, y1) of slots 2p, 2p+1
constexpr size_t BL_OFF_ZT = BL_OFF_XY + sizeof(float4) * (TILE_CMAXP / 2);             // float4 [CMAXP/2]: (z0, z1, T0, T1), T = (2h)^2
constexpr size_t BL_OFF_L = 0;                                                          // u16 [LIST_LCAP][BL_THREADS]: the schedule, written after
                                                                                        // the scan is over -- shares the space of XY / ZT
constexpr size_t BL_CAND_END = BL_OFF_ZT + sizeof(float4) * (TILE_CMAXP / 2);
constexpr size_t BL_L_END = BL_OFF_L + sizeof(uint16_t) * LIST_LCAP * BL_THREADS;
constexpr size_t BL_OFF_B = BL_CAND_END > BL_L_END ? BL_CAND_END : BL_L_END;             // u16 [4][LIST_BS][BL_THREADS]
constexpr size_t BL_OFF_COL = BL_OFF_B + sizeof(uint16_t) * 4 * LIST_BS * BL_THREADS;   // u16 [MAXR][COLW]
constexpr size_t BL_SMEM = BL_OFF_COL + sizeof(uint16_t) * TILE_MAXR * COLW;
static_assert(2 * (BL_SMEM + sizeof(TileS) + 1280) <= 228 * 1024, "list builder: two CTAs per SM");

// packed fp32 pairs (sm_100 FADD2 / FMUL2 / FFMA2): one instruction tests two candidates
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float a, float b) { f32x2 r; asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ void unpk2(f32x2 v, float& a, float& b) { asm("mov.b64 {%0,%1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); }
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b) { f32x2 r; asm("sub.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) { f32x2 r; asm("mul.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) { f32x2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }

// One candidate of the scan: if r2 < hi, store (value | LIST_RECHECK unless 0 < r2 < 2 half_lo) at the bucket row pointer and
// advance it, clamped at `end` (the bucket's trash row: a pointer that reaches it reports the overflow); nflag counts
// the flagged hits.  No branches.
__device__ __forceinline__ void append_flag(float r2, float hi, float half_lo, uint32_t& addr, uint32_t end, uint32_t v, uint32_t& nflag) {
    asm volatile("{\n\t.reg .pred p, s, q;\n\t.reg .f32 t;\n\t.reg .b32 w;\n\t"
                 "setp.lt.f32 p, %2, %3;\n\t"
                 "sub.f32 t, %2, %4;\n\t"
                 "abs.f32 t, t;\n\t"
                 "setp.lt.f32 s, t, %4;\n\t"
                 "setp.ge.and.f32 q, t, %4, p;\n\t"
                 "selp.b32 w, %6, %7, s;\n\t"
                 "@p st.shared.u16 [%0], w;\n\t"
                 "@p add.u32 %0, %0, %8;\n\t"
                 "@q add.u32 %1, %1, 1;\n\t"
                 "min.u32 %0, %0, %5;\n\t}"
                 : "+r"(addr), "+r"(nflag) : "f"(r2), "f"(hi), "f"(half_lo), "r"(end), "r"(v), "r"(v | LIST_RECHECK), "n"(2 * BL_THREADS));
    // no memory clobber: the loads of the next pairs must be free to move above the store; the buckets are read back
    // only after the fence that follows the scan
}

// Which thread of a target owns bank beta in the scan (threads split the candidate PAIRS: slots 4i+2u, 4i+2u+1), and
// the index of that bank among the owner's four buckets.
__device__ __forceinline__ int bank_owner(int beta) { return (beta >> 1) & 1; }
__device__ __forceinline__ int bank_local(int beta) { return ((beta >> 2) << 1) | (beta & 1); }


__global__ void __launch_bounds__(BL_THREADS, 2)
k_build_lists(DevGrid g, CellTable ct, ListArgs A) {
    extern __shared__ __align__(16) unsigned char smem[];
    __shared__ TileS S;
    __shared__ int s_bad, s_nonuni, s_clo, s_chi;
    __shared__ double s_h0;
    float4* XY = reinterpret_cast<float4*>(smem + BL_OFF_XY);
    float4* ZT = reinterpret_cast<float4*>(smem + BL_OFF_ZT);
    float* XYf = reinterpret_cast<float*>(XY);
    float* ZTf = reinterpret_cast<float*>(ZT);
    uint16_t* Lf = reinterpret_cast<uint16_t*>(smem + BL_OFF_L);       // [k * BL_THREADS + tid]
    uint16_t* B = reinterpret_cast<uint16_t*>(smem + BL_OFF_B);        // [(b * LIST_BS + k) * BL_THREADS + tid]
    uint16_t* colofs = reinterpret_cast<uint16_t*>(smem + BL_OFF_COL); // [range][COLW]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int u = tid & 1, j = lane & 7;
    const uint32_t nunits = 2u * (uint32_t)A.ctr[CTR_NTILES];
    const float Rmax = 2.0f * (float)A.hglob[1] * 1.000001f;

    for (uint32_t unit = blockIdx.x; unit < nunits; unit += gridDim.x) {
        const uint32_t tile = unit >> 1;
        const int half = (int)(unit & 1u);
        const TileDesc td = A.tiles[tile];
        const int tgt = half * BL_TGT + (tid >> 1);                     // target index within the tile
        const int twarp = half * BL_WARPS + warp;                       // warp index within the tile
        if (half * BL_TGT >= (int)td.nt) {                              // no target in this half: empty lists
            if (lane == 0) A.winfo[(size_t)tile * TILE_WARPS + twarp] = make_uint2(0u, 0u);
            if (u == 0) A.lcount[(size_t)tile * TILE_T + tgt] = 0u;
            if (tid == 0) atomicOr(&A.tflags[tile], TILE_FLAG_OK0 << half);
            continue;
        }
        __syncthreads();                                                // previous unit done with smem
        if (tid == 0) { s_bad = 0; s_nonuni = 0; s_clo = 1 << 20; s_chi = -1; }
        {   // tile tables (k_tile_tables)
            const uint32_t* src = A.tiletab + (size_t)tile * TILES_WORDS;
            uint32_t* dst = reinterpret_cast<uint32_t*>(&S);
            for (int w = tid; w < TILES_WORDS; w += BL_THREADS) dst[w] = src[w];
        }
        const int ncolv = td.cxb - td.cxa + 3;                          // virtual columns 0 .. ncolv-1
        // tile origin (centre of the tile's cell block) for the fp32 relative coordinates
        const double ox = g.lo[0] + (0.5 * (td.cxa + td.cxb + 1)) / g.inv[0];
        const double oy = g.lo[1] + (td.y0 + 0.5 * td.nyr) / g.inv[1];
        const double oz = g.lo[2] + (td.z0 + 0.5 * td.nzr) / g.inv[2];
        // bound on the absolute error of an fp32 relative coordinate difference: 2 roundings of magnitude <= ext
        const float ext = (float)fmax(fmax((0.5 * ncolv + 0.5) / g.inv[0], 2.5 / g.inv[1]), 2.5 / g.inv[2]);
        const float E = ext * 2.4e-7f;                                  // 4 * 2^-24 * ext
        const float Am = 4.4f * Rmax * E + 5.0f * E * E;
        __syncthreads();

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
        if (active) {
            int e;
            i = tile_target(td, S, tgt, &e);
            int cxe;
            tile_cell_rc(td, e, cxe, try_, trz);
            tcol = cxe - td.cxa;
            const double2 xy = A.p0[i], zh = A.p1[i];
            xa = xy.x; ya = xy.y; za = zh.x; ha = zh.y;
            for (int q = 0; q < (int)S.nranges; ++q)
                if (i >= S.r_vstart[q] && i < S.r_vend[q]) s_self = S.r_base[q] + (i - S.r_vstart[q]);
        }
        // an inactive thread sits far away from everything: it never hits
        const float fax = active ? (float)(xa - ox) : -3.0e18f, fay = (float)(ya - oy), faz = (float)(za - oz);
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
        if (lane == 0 && cmax >= 0) { atomicMin(&s_clo, cmin); atomicMax(&s_chi, cmax); }
        if (tid == 0) s_h0 = ha;                                        // the half's first target: always there
        __syncthreads();

        // ---- stage the candidates of virtual columns [s_clo, s_chi + 2] as slot pairs: one warp per range; whole pairs
        //      only (a pair cut by the window's edge is staged in full), the odd pad slot of a range is put out of reach
        {
            const unsigned long long h0 = (unsigned long long)__double_as_longlong(s_h0);
            const int clo = s_clo, chi = s_chi + 2;
            bool nonuni = false;
            for (int q = warp; q < (int)S.nranges; q += BL_WARPS) {
                const int4 ge = S.r_geo[q];
                const int jlo = max(0, min(ge.y, clo - ge.z)), jhi = max(0, min(ge.y, chi + 1 - ge.z));
                if (jhi <= jlo) continue;
                const uint32_t vs = S.r_vstart[q], len = S.r_vend[q] - vs, base = S.r_base[q];
                const uint32_t ka = (uint32_t)colofs[q * COLW + jlo] & ~1u, kb = ((uint32_t)colofs[q * COLW + jhi] + 1u) & ~1u;
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
                    }
                    const uint32_t s = base + k, o = (s >> 1) * 4 + (s & 1);
                    XYf[o] = fx; XYf[o + 2] = fy; ZTf[o] = fz; ZTf[o + 2] = T;
                }
            }
            if (nonuni) s_nonuni = 1;                                   // some staged candidate differs from the first target's h
        }
        __syncthreads();
        const bool uni = s_nonuni == 0;

        // ---- scan: fp32 prefilter on slot pairs (FADD2/FFMA2: two candidates per instruction).  The two threads of a
        //      target take alternate pairs (slots 4i+2u, 4i+2u+1); all lanes of the same parity read the same pair
        //      (shared-memory broadcast).  A hit (r2 below the support of the larger h, error bound added) goes straight
        //      to the thread's bucket of the slot's bank: pair p feeds buckets (p & 2) and (p & 2) + 1, so with the loop
        //      unrolled by two pairs the bucket of every append is a compile-time choice.  A hit that is not certain
        //      (0 < r2 < Ta_lo, uniform-h tiles only) carries LIST_RECHECK.
        const uint32_t bk0 = (uint32_t)__cvta_generic_to_shared(B + tid);
        constexpr uint32_t BROW = 2u * BL_THREADS;                    // bytes per bucket row
        uint32_t nflag = 0;                                             // flagged hits of this thread
        uint32_t bp0 = bk0, bp1 = bk0 + LIST_BS * BROW, bp2 = bk0 + 2 * LIST_BS * BROW, bp3 = bk0 + 3 * LIST_BS * BROW;
        const uint32_t e0 = bk0 + LIST_BC * BROW, e1 = e0 + LIST_BS * BROW, e2 = e1 + LIST_BS * BROW, e3 = e2 + LIST_BS * BROW;
        if (cmax >= 0) {
            const int wv_lo = cmin, wv_hi = cmax + 2;                   // virtual columns [tcol, tcol + 2] around each target
            const f32x2 ax2 = pk2(fax, fax), ay2 = pk2(fay, fay), az2 = pk2(faz, faz);
            const f32x2 one_eps = pk2(1.00001f, 1.00001f), am2 = pk2(Am, Am);
            const float half_lo = 0.5f * Ta_lo;
            // one pair: test both slots, append to buckets (pa_, pb_) whose row pointers are clamped at the trash row
            auto pair_uni = [&](uint32_t p, const float4 c0, const float4 c1, uint32_t& qa, uint32_t qa_end, uint32_t& qb, uint32_t qb_end) {
                const f32x2 dx = sub2(ax2, pk2(c0.x, c0.y)), dy = sub2(ay2, pk2(c0.z, c0.w)), dz = sub2(az2, pk2(c1.x, c1.y));
                float r0, r1;
                unpk2(fma2(dz, dz, fma2(dy, dy, mul2(dx, dx))), r0, r1);
                append_flag(r0, Ta_hi, half_lo, qa, qa_end, 2 * p, nflag);
                append_flag(r1, Ta_hi, half_lo, qb, qb_end, 2 * p + 1, nflag);
            };
            auto pair_gen = [&](uint32_t p, uint32_t& qa, uint32_t qa_end, uint32_t& qb, uint32_t qb_end) {
                const float4 c0 = XY[p], c1 = ZT[p];
                const f32x2 dx = sub2(ax2, pk2(c0.x, c0.y)), dy = sub2(ay2, pk2(c0.z, c0.w)), dz = sub2(az2, pk2(c1.x, c1.y));
                float r0, r1, h0, h1;
                unpk2(fma2(dz, dz, fma2(dy, dy, mul2(dx, dx))), r0, r1);
                unpk2(fma2(pk2(fmaxf(Ta, c1.z), fmaxf(Ta, c1.w)), one_eps, am2), h0, h1);
                append_flag(r0, h0, -1.0f, qa, qa_end, 2 * p, nflag);    // half_lo < 0: always flagged
                append_flag(r1, h1, -1.0f, qb, qb_end, 2 * p + 1, nflag);
            };
            for (int q = 0; q < (int)S.nranges; ++q) {
                const int row = S.r_shift[q][3], ry = row & 3, rz = row >> 2;
                if (ry < ymin || ry > ymax + 2 || rz < zmin || rz > zmax + 2) continue;
                const int4 ge = S.r_geo[q];
                const int jlo = max(0, min(ge.y, wv_lo - ge.z)), jhi = max(0, min(ge.y, wv_hi + 1 - ge.z));
                if (jhi <= jlo) continue;
                const uint32_t sa = S.r_base[q] + colofs[q * COLW + jlo];
                const uint32_t sb = S.r_base[q] + colofs[q * COLW + jhi];
                // pairs [sa/2, (sb+1)/2): a pair cut by a column boundary brings in a slot of the same row two or
                // more cells away (never a neighbour, never scanned twice); a range's pad slot is out of reach
                const uint32_t pa = sa >> 1, pb = (sb + 1u) >> 1;
                uint32_t p = pa + ((pa ^ (uint32_t)u) & 1u);
                if (uni) {
                    if ((p & 2u) && p < pb) { pair_uni(p, XY[p], ZT[p], bp2, e2, bp3, e3); p += 2; }
                    // software pipeline: the records of the next two pairs are loaded while the current two are tested
                    // (indices clamped to the staged arrays; a clamped load is never used)
                    constexpr uint32_t PLAST = TILE_CMAXP / 2 - 1;
                    float4 a0 = XY[min(p, PLAST)], a1 = ZT[min(p, PLAST)], b0 = XY[min(p + 2, PLAST)], b1 = ZT[min(p + 2, PLAST)];
#pragma unroll 2
                    for (; p + 2 < pb; p += 4) {
                        const uint32_t pn = min(p + 4, PLAST), pm = min(p + 6, PLAST);
                        const float4 na0 = XY[pn], na1 = ZT[pn], nb0 = XY[pm], nb1 = ZT[pm];
                        pair_uni(p, a0, a1, bp0, e0, bp1, e1);
                        pair_uni(p + 2, b0, b1, bp2, e2, bp3, e3);
                        a0 = na0; a1 = na1; b0 = nb0; b1 = nb1;
                    }
                    if (p < pb) pair_uni(p, a0, a1, bp0, e0, bp1, e1);
                } else {
                    if ((p & 2u) && p < pb) { pair_gen(p, bp2, e2, bp3, e3); p += 2; }
#pragma unroll 2
                    for (; p + 2 < pb; p += 4) { pair_gen(p, bp0, e0, bp1, e1); pair_gen(p + 2, bp2, e2, bp3, e3); }
                    if (p < pb) pair_gen(p, bp0, e0, bp1, e1);
                }
            }
        }
        asm volatile("" ::: "memory");                                  // the appends above wrote the buckets
        // ---- settle the flagged hits, bucket by bucket, in place.  Certain when the fp32 r2 is clear of every support
        //      boundary by more than the error bound; otherwise (and at r = 0, which includes the target itself) the
        //      exact fp64 contract predicate decides (O2/A12).
        uint32_t cnt = 0, ng = 0;                                       // cnt: 4 x 8-bit bucket fills
        bool ovf = (bp0 >= e0) || (bp1 >= e1) || (bp2 >= e2) || (bp3 >= e3), coinc = false;
        // In a uniform-h tile the target itself (r = 0) is normally the only flagged hit, met by the thread that scans its
        // slot pair: then the settle pass is a removal of that one entry from its bucket.
        const bool sees_self = active && (((s_self >> 1) & 1u) == (uint32_t)u);
        const bool full_settle = __any_sync(0xFFFFFFFFu, nflag != (sees_self ? 1u : 0u));
        if (!full_settle) {
            const uint32_t n0 = (bp0 - bk0) / BROW, n1 = (bp1 - (bk0 + LIST_BS * BROW)) / BROW;
            const uint32_t n2 = (bp2 - (bk0 + 2 * LIST_BS * BROW)) / BROW, n3 = (bp3 - (bk0 + 3 * LIST_BS * BROW)) / BROW;
            cnt = n0 | (n1 << 8) | (n2 << 16) | (n3 << 24);
            if (sees_self) {
                const int b = bank_local((int)(s_self & 7u));
                uint16_t* bb = B + (size_t)b * LIST_BS * BL_THREADS + tid;
                const uint32_t nb = (cnt >> (8 * b)) & 0xFFu;
                uint32_t k = 0;
                while (k < nb && (bb[k * BL_THREADS] & 0x7FFFu) != s_self) ++k;
                if (k < nb) {                                           // the last entry takes its place (order is free)
                    bb[k * BL_THREADS] = bb[(nb - 1) * BL_THREADS];
                    cnt -= 1u << (8 * b);
                }
            }
            ng = (cnt & 0xFFu) + ((cnt >> 8) & 0xFFu) + ((cnt >> 16) & 0xFFu) + (cnt >> 24);
        } else
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const uint32_t nb = ((b == 0 ? bp0 : b == 1 ? bp1 : b == 2 ? bp2 : bp3) - (bk0 + b * LIST_BS * BROW)) / BROW;
            uint16_t* bb = B + (size_t)b * LIST_BS * BL_THREADS + tid;
            uint32_t w = 0;
            for (uint32_t k = 0; k < nb; ++k) {
                const uint32_t v = bb[k * BL_THREADS], s = v & 0x7FFFu;
                bool in_s = true, in_g = true;
                if (v & LIST_RECHECK) {
                    const float4 c0 = XY[s >> 1], c1 = ZT[s >> 1];
                    const bool od = (s & 1u) != 0;
                    const float dx = fax - (od ? c0.y : c0.x), dy = fay - (od ? c0.w : c0.z), dz = faz - (od ? c1.y : c1.x);
                    const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                    const float Tm = fmaxf(Ta, od ? c1.w : c1.z);
                    if (r2 < fmaf(Tm, 0.99999f, -Am) && (r2 < Ta_lo || r2 >= Ta_hi) && r2 > 0.0f) {
                        in_g = r2 < Ta_lo;
                    } else if (s == s_self) {
                        in_s = false;
                    } else {
                        int q = 0;
                        while (q + 1 < (int)S.nranges && S.r_base[q + 1] <= s) ++q;
                        const uint32_t gi = S.r_vstart[q] + (s - S.r_base[q]);
                        const double2 xy = A.p0[gi], zh = A.p1[gi];
                        const double ex = min_image(__dsub_rn(xa, xy.x), g.per[0], g.L[0], g.halfL[0]);
                        const double ey = min_image(__dsub_rn(ya, xy.y), g.per[1], g.L[1], g.halfL[1]);
                        const double ez = min_image(__dsub_rn(za, zh.x), g.per[2], g.L[2], g.halfL[2]);
                        const double e2x = r2_exact(ex, ey, ez);
                        in_s = gi != i && e2x < support2(fmax(ha, zh.y));
                        in_g = in_s && e2x < support2(ha);
                        if (in_s && !(e2x > 0.0)) coinc = true;         // coincident particles: left to the general kernels (A11)
                    }
                    if (in_s) bb[w * BL_THREADS] = (uint16_t)s;
                } else if (w != k) {
                    bb[w * BL_THREADS] = (uint16_t)s;
                }
                w += in_s ? 1u : 0u;
                ng += (in_s && in_g) ? 1u : 0u;
            }
            cnt |= w << (8 * b);
        }
        if (ovf || coinc) s_bad = 1;
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
        uint32_t R = n_lane;
#pragma unroll
        for (int o = 16; o; o >>= 1) R = max(R, __shfl_xor_sync(0xFFFFFFFFu, R, o));
        R = (R + 3u) & ~3u;
        // list storage: one fixed block of LIST_RMAX rounds per (tile, warp) -- no allocation, placement is deterministic
        const unsigned long long off = ((unsigned long long)tile * TILE_WARPS + twarp) * (unsigned long long)(LIST_RMAX / 4) * 32;
        if (lane == 0 && R > (uint32_t)LIST_RMAX) s_bad = 1;
        __syncthreads();
        const bool bad = s_bad != 0;
        if (!bad) {
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
            // pass 1 (lockstep): every phase takes its own bank's entries up to its capacity; a hole gets the dummy slot
            // of the phase's bank
            for (uint32_t k = 0; k < m8; ++k) {
#pragma unroll
                for (int t = 0; t < 8; ++t) {
                    uint16_t item = (uint16_t)(TILE_CMAX + ((j + t) & 7));
                    if (k < own[t]) item = bq[t][2 * k * BL_THREADS];
                    out[((uint32_t)t * m8 + (e4 ? (uint32_t)(t >> 1) : 0u) + k) * BL_THREADS] = item;
                }
            }
            if (e4) {
#pragma unroll
                for (int t = 1; t < 8; t += 2) {
                    uint16_t item = (uint16_t)(TILE_CMAX + ((j + t) & 7));
                    if (m8 < own[t]) item = bq[t][2 * m8 * BL_THREADS];
                    out[((uint32_t)t * m8 + (uint32_t)(t >> 1) + m8) * BL_THREADS] = item;
                }
            }
            // the left-over entries go into the holes, phase by phase (a phase has either holes or left-overs)
            {
                int th = -1;
                uint32_t hrem = 0;
#pragma unroll
                for (int t = 0; t < 8; ++t) {
                    for (uint32_t e = 0; e < ovr[t]; ++e) {
                        while (hrem == 0 && th < 7) { ++th; hrem = (Hw >> (4 * th)) & 15u; }
                        if (hrem == 0) break;                           // cannot happen: n_lane <= R
                        const uint32_t pos = (((uint32_t)(th + 1) * R) >> 3) - hrem;
                        --hrem;
                        out[pos * BL_THREADS] = bq[t][2 * (own[t] + e) * BL_THREADS];
                    }
                }
            }
            // pass 2: pack 4 rounds per 8-byte store
            uint2* blk = A.pool + off + lane;
            for (uint32_t r4 = 0; r4 < R; r4 += 4) {
                const uint32_t e0 = out[r4 * BL_THREADS], e1 = out[(r4 + 1) * BL_THREADS];
                const uint32_t e2 = out[(r4 + 2) * BL_THREADS], e3 = out[(r4 + 3) * BL_THREADS];
                blk[(size_t)(r4 >> 2) * 32] = make_uint2(e0 | (e1 << 16), e2 | (e3 << 16));
            }
            if (u == 0) A.lcount[(size_t)tile * TILE_T + tgt] = active ? (ng | (nsym << 16)) : 0u;
            if (active && u == 0) A.fast[i] = 1;
            if (lane == 0) A.winfo[(size_t)tile * TILE_WARPS + twarp] = make_uint2((uint32_t)off, R);
        }
        if (tid == 0) {
            const uint32_t bits = (bad ? 0u : (TILE_FLAG_OK0 << half)) | (s_nonuni ? TILE_FLAG_NONUNI : 0u);
            if (bits) atomicOr(&A.tflags[tile], bits);
            if (s_nonuni) atomicAdd(&A.ctr[CTR_NNONUNI], 1ull);
            if (!bad) atomicAdd(&A.ctr[CTR_NFAST], (unsigned long long)min((int)td.nt - half * BL_TGT, BL_TGT));
        }
    }
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
    for (uint32_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const uint32_t flags = A.tflags[tile];
        if (!(flags & TILE_FLAG_OK)) continue;
        const bool half_ok = ((flags >> (warp / (TILE_WARPS / 2))) & 1u) != 0;
        const TileDesc td = A.tiles[tile];
        __syncthreads();
        {
            const uint32_t* src = A.tiletab + (size_t)tile * TILES_WORDS;
            uint32_t* dst = reinterpret_cast<uint32_t*>(&S);
            for (int w = tid; w < TILES_WORDS; w += TILE_THREADS) dst[w] = src[w];
        }
        __syncthreads();
        const bool active = half_ok && tgt < (int)td.nt;
        uint32_t i = 0;
        double xa = 0, ya = 0, za = 0, ha = 0;
        if (active) {
            i = tile_target(td, S, tgt);
            const double2 xy = A.p0[i], zh = A.p1[i];
            xa = xy.x; ya = xy.y; za = zh.x; ha = zh.y;
        }
        uint2 wi = A.winfo[(size_t)tile * TILE_WARPS + warp];
        if (!half_ok) wi.y = 0u;
        const uint2* lp = A.pool + wi.x + lane;
        uint32_t cnt = 0;
        uint64_t dsum = 0, dxr = 0;
        // mode 1 needs the first half's count before the second half writes: two passes (count, then write)
        for (int pass = 0; pass < (MODE == 1 ? 2 : 1); ++pass) {
            uint32_t wpos = 0;
            if (MODE == 1 && pass == 1) {
                const uint32_t other = __shfl_xor_sync(0xFFFFFFFFu, cnt, 1);
                wpos = u ? other : 0u;                     // thread 1 writes after thread 0's entries
            }
            const uint64_t lbase = (MODE == 1 && active) ? A.offsets[A.perm[i]] : 0;
            uint32_t c2 = 0;
            for (uint32_t r = 0; r < wi.y; ++r) {
                const uint2 w4 = lp[(size_t)(r >> 2) * 32];
                const uint32_t half = (r & 2u) ? w4.y : w4.x;
                const uint32_t s = (r & 1u) ? (half >> 16) : (half & 0xFFFFu);
                if (s >= (uint32_t)TILE_CMAX || !active) continue;             // dummy entry
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
            cnt = c2;
        }
        const uint32_t total = cnt + __shfl_xor_sync(0xFFFFFFFFu, cnt, 1);
        if (MODE == 2) {
            dsum += __shfl_xor_sync(0xFFFFFFFFu, dsum, 1);
            dxr ^= __shfl_xor_sync(0xFFFFFFFFu, dxr, 1);
        }
        if (MODE == 1) __syncwarp();
        if (active && u == 0) {
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
    const int64_t nb = (int64_t)((gr.ncell[1] + 1) / 2) * ((gr.ncell[2] + 1) / 2);
    if (nb > t.bundle_cap) return cudaSuccess;
    cudaError_t e;
    if ((e = cudaMemsetAsync(t.ctr, 0, sizeof(unsigned long long) * CTR_COUNT, st)) != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(t.fast, 0, (size_t)c->n, st)) != cudaSuccess) return e;
    CellTable ct{c->cell_start, c->cell_end};
    const int blocks = (int)((nb * 32 + 255) / 256);
    k_make_tiles<false><<<blocks, 256, 0, st>>>(c->dg, ct, c->hglob, t.bcount, t.tiles, (uint32_t)t.tile_cap, t.ctr);
    if ((e = launch_excl_scan_u32(c, t.bcount, nb, t.bcount + t.bundle_cap, st)) != cudaSuccess) return e;
    k_make_tiles<true><<<blocks, 256, 0, st>>>(c->dg, ct, c->hglob, t.bcount, t.tiles, (uint32_t)t.tile_cap, t.ctr);
    k_tile_tables<<<t.sms * 8, 128, 0, st>>>(c->dg, ct, t.tiles, t.ctr, t.tiletab);
    if ((e = cudaMemsetAsync(t.tflags, 0, sizeof(uint32_t) * (size_t)t.tile_cap, st)) != cudaSuccess) return e;
    static bool attr_done = false;
    if (!attr_done) {
        if ((e = cudaFuncSetAttribute(k_build_lists, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)BL_SMEM)) != cudaSuccess) return e;
        attr_done = true;
    }
    ListArgs A{c->pk.p0, c->pk.p1, t.tiles, t.ctr, t.pool, t.winfo, t.lcount, t.tflags, t.tiletab, t.fast,
               c->hglob, c->dev_status};
    k_build_lists<<<t.sms * 2, BL_THREADS, BL_SMEM, st>>>(c->dg, ct, A);
    c->launches += 4;
    t.enabled = true;
    return cudaGetLastError();
}

}  // namespace spray
