// tiles.cuh -- tile geometry shared by the neighbour-list builder (tiles.cu) and the tiled pair kernels
// (sweeps_tiled.cu).  Not shared with oracle/.
//
// A TILE is the unit of work of one CTA: up to TILE_T target particles taken from a "bundle" of 2 x 2 cell rows
// (rows run along x; after the sort the cells of a row are one contiguous index range), enumerated column-major
// (for cx: for row: particles of the cell), plus the candidate particles of every cell within one cell of the
// tile's cells: (nyr + 2) x (nzr + 2) rows, x-range [cxa - 1, cxb + 1].  Each candidate row contributes one
// contiguous range of sorted slots (two when the x-range wraps in a periodic box); the ranges are laid out
// back-to-back in shared memory and a candidate is addressed by its SLOT in that layout.  The slot numbering is a
// pure function of (TileDesc, cell table), so the neighbour lists built once per spray_build_cells (u16 slots)
// stay valid for every later sweep.
//
// Valid only when every neighbour of a target lies within one cell: 2 * h_max <= min cell edge (checked on the
// device when the tiles are made; otherwise no tile is emitted and the general one-thread-per-particle kernels
// serve every particle).
//
// Threads: TILE_TPT = 2 threads per target (thread tid serves target tid >> 1 with the half-list tid & 1), so a
// warp holds 16 targets and an aligned group of 8 lanes (one 128-byte shared-memory wavefront of 16-byte loads)
// holds 4 targets x 2 half-lists.  The lists are SCHEDULED per lane (tiles.cu) so that in most rounds the 8 lanes
// of such a group read 8 different 16-byte banks.
#pragma once
#include "common.cuh"

namespace spray {

constexpr int TILE_T = 256;          // max targets per tile
constexpr int TILE_TPT = 2;          // threads per target
constexpr int TILE_THREADS = TILE_T * TILE_TPT;
constexpr int TILE_WARPS = TILE_THREADS / 32;
constexpr int TILE_CMAX = 2232;      // max candidate slots per tile
constexpr int TILE_NDUMMY = 8;       // dummy slots (one per 16-byte bank) appended after the candidates
constexpr int TILE_CMAXP = TILE_CMAX + TILE_NDUMMY;   // 2240: multiple of 8, so slot & 7 is the bank of a 16-byte record
constexpr int TILE_MAXR = 32;        // candidate ranges: 4 x 4 rows x (1 or 2 pieces, at most 16 rows wrap)
constexpr int TILE_BXMAX = 24;       // max columns (cells along x) of a tile
constexpr int TILE_MAXCELL = 4 * TILE_BXMAX;
constexpr int LIST_BC = 24;          // builder: capacity of one (target, bank) bucket
constexpr int LIST_RMAX = 80;        // max rounds of a warp's schedule = builder's flat-list rows (longer -> tile served by the general kernels)

struct TileDesc {                    // 24 bytes
    int16_t y0, z0;                  // first row of the bundle
    int16_t cxa, cxb;                // first / last column
    uint8_t nyr, nzr;                // rows of the bundle present (1 or 2 each)
    uint8_t part, nparts;            // a column whose candidates exceed TILE_CMAX is cut into nparts consecutive tile entries with the same
                                     // targets and disjoint sets of candidate rows (rowmask): a sweep's CTA runs them one after the other
                                     // and keeps its sums; each part has lists of its own.  Ordinary tiles: part 0 of 1, every row.
    uint32_t skip;                   // targets of column cxa (column-major order) that belong to earlier tiles
    uint32_t nt;                     // targets of this tile (<= TILE_T)
    uint32_t rowmask;                // bit rz * 4 + ry: candidate row of this entry
};

// Tile flags.  The lists of a tile are built in two halves (targets [0, TILE_T/2) and [TILE_T/2, TILE_T), i.e. the
// first and the second TILE_WARPS/2 warps of a sweep's CTA); each half reports on its own.
constexpr uint32_t TILE_FLAG_OK0 = 1u;       // lists of the first half were built: the tiled kernels serve those targets
constexpr uint32_t TILE_FLAG_OK1 = 2u;       // same for the second half (= TILE_FLAG_OK0 << 1)
constexpr uint32_t TILE_FLAG_OK = 3u;        // mask: any half
constexpr uint32_t TILE_FLAG_NONUNI = 4u;    // NOT every target and candidate of the tile has the same h (bitwise)

struct CellTable {
    const uint32_t* cell_start;
    const uint32_t* cell_end;
    const uint32_t* cell_tend;       // the TARGETS of a cell are the slots [cell_start, cell_tend); = cell_end unless the grid is an
                                     // internal level of the tiled path, which serves only the particles of its h range (api.cu)
};

// Per-CTA tile tables in shared memory (filled by tile_setup)
struct TileS {
    // candidate ranges
    uint32_t r_vstart[TILE_MAXR];    // first global slot of the range
    uint32_t r_vend[TILE_MAXR];      // one past the last global slot
    uint32_t r_base[TILE_MAXR + 1];  // first shared-memory slot of the range (exclusive scan of the lengths rounded up to even)
    int8_t r_shift[TILE_MAXR][4];    // [0..2] periodic image: dx = (x_a - x_b) + shift * L (-1, 0, +1); [3] candidate row id
    int4 r_geo[TILE_MAXR];           // (first cell column, number of columns, virtual column of the first, first cell id)
    uint8_t r_row[16];               // candidate row id (rz * 4 + ry) -> index of its first range, 0xFF when the row has none
    uint32_t nranges, ncand;
    // targets
    uint32_t c_first[TILE_MAXCELL];  // global slot of the first particle of cell e (column-major enumeration)
    uint32_t c_pre[TILE_MAXCELL + 1];// exclusive scan of the cell counts
    uint32_t ncells;
};

static_assert(sizeof(TileS) % 16 == 0, "TileS is copied in 16-byte pieces");
constexpr int TILES_WORDS = (int)(sizeof(TileS) / 4);

__device__ __forceinline__ uint32_t cell_id(const DevGrid& g, int cx, int cy, int cz) {
    return (uint32_t)((cz * g.nc[1] + cy) * g.nc[0] + cx);
}

// Candidate range (row, piece) of a tile: row = rz * 4 + ry enumerates the (nyr + 2) x (nzr + 2) candidate rows,
// piece = 0/1 the two parts of an x-range that wraps in a periodic box.  Returns false when the range does not
// exist or is empty.  [vs, ve) = global slots, (xlo, ncol) = its first cell column (actual index) and number
// of columns, vlo = position of that column in the tile's virtual column axis (0 = column cxa - 1),
// sh = periodic image so that dx = (x_a - x_b) + sh * L.
struct RangeGeo { uint32_t vs, ve; int xlo, ncol, vlo, cy, cz; int sh[3]; };
__device__ __forceinline__ bool tile_range(int y0, int z0, int nyr, int nzr, int cxa, int cxb, const DevGrid& g,
                                           const CellTable& ct, int row, int piece, RangeGeo& R) {
    const int nyc = nyr + 2, nzc = nzr + 2;
    const int ry = row % 4, rz = row / 4;
    if (ry >= nyc || rz >= nzc) return false;
    int cy = y0 - 1 + ry, cz = z0 - 1 + rz;
    int sy = 0, sz = 0, sx = 0;
    if (cy < 0) { if (g.per[1]) { cy += g.nc[1]; sy = 1; } else return false; }
    else if (cy >= g.nc[1]) { if (g.per[1]) { cy -= g.nc[1]; sy = -1; } else return false; }
    if (cz < 0) { if (g.per[2]) { cz += g.nc[2]; sz = 1; } else return false; }
    else if (cz >= g.nc[2]) { if (g.per[2]) { cz -= g.nc[2]; sz = -1; } else return false; }
    int xlo = cxa - 1, xhi = cxb + 1, vlo = 0;
    const int nx = g.nc[0];
    if (g.per[0]) {
        if (xlo < 0) {               // piece 0 = wrapped tail of the row, piece 1 = [0, xhi]
            if (piece == 0) { xlo += nx; xhi = nx - 1; sx = 1; } else { vlo = -xlo; xlo = 0; }
        } else if (xhi >= nx) {      // piece 0 = [xlo, nx-1], piece 1 = wrapped head of the row
            if (piece == 0) { xhi = nx - 1; } else { vlo = nx - xlo; xlo = 0; xhi -= nx; sx = -1; }
        } else if (piece == 1) return false;
    } else {
        if (piece == 1) return false;
        if (xlo < 0) { vlo = -xlo; xlo = 0; }
        xhi = xhi > nx - 1 ? nx - 1 : xhi;
    }
    if (xhi < xlo) return false;
    R.vs = ct.cell_start[cell_id(g, xlo, cy, cz)];
    R.ve = ct.cell_end[cell_id(g, xhi, cy, cz)];
    R.xlo = xlo; R.ncol = xhi - xlo + 1; R.vlo = vlo; R.cy = cy; R.cz = cz;
    R.sh[0] = sx; R.sh[1] = sy; R.sh[2] = sz;
    return R.ve > R.vs;
}
__device__ __forceinline__ bool tile_range(const TileDesc& td, const DevGrid& g, const CellTable& ct, int row, int piece,
                                           RangeGeo& R) {
    if (!((td.rowmask >> row) & 1u)) return false;
    return tile_range(td.y0, td.z0, td.nyr, td.nzr, td.cxa, td.cxb, g, ct, row, piece, R);
}

// Cell e of the tile's target enumeration: column-major, and within a column the 2 x 2 rows in serpentine (Gray)
// order, reversed in odd columns, so that consecutive cells always share a face.  A warp's 16 consecutive targets
// then straddle two face-adjacent cells at worst and its candidate window is 36 cells instead of up to 64.
__device__ __forceinline__ void tile_cell_rc(const TileDesc& td, int e, int& cx, int& ry, int& rz) {
    const int nrows = td.nyr * td.nzr;
    cx = td.cxa + e / nrows;
    int r = e % nrows;
    if (cx & 1) r = nrows - 1 - r;
    rz = r / td.nyr; ry = r % td.nyr;
    if (rz & 1) ry = td.nyr - 1 - ry;
}

// Fills S.  Must be called by all threads of the CTA (blockDim.x >= 32 + TILE_MAXCELL); ends with __syncthreads().
__device__ __forceinline__ void tile_setup(const TileDesc& td, const DevGrid& g, const CellTable& ct, TileS& S) {
    const int tid = threadIdx.x;
    if (tid < 32) {
        RangeGeo R;
        const bool valid = tile_range(td, g, ct, tid >> 1, tid & 1, R);
        const uint32_t len = valid ? ((R.ve - R.vs + 7u) & ~7u) : 0u;  // every range starts on a slot that is a multiple of 8 (list builder: blocks of 8 slots = the 8 banks)
        // compact the valid ranges to the front, keeping order (ballot + popc), and scan the padded lengths
        const uint32_t mask = __ballot_sync(0xFFFFFFFFu, valid);
        const int pos = __popc(mask & ((1u << tid) - 1u));
        uint32_t incl = len;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
            if (tid >= o) incl += v;
        }
        if (valid) {
            S.r_vstart[pos] = R.vs; S.r_vend[pos] = R.ve; S.r_base[pos] = incl - len;
            S.r_shift[pos][0] = (int8_t)R.sh[0]; S.r_shift[pos][1] = (int8_t)R.sh[1]; S.r_shift[pos][2] = (int8_t)R.sh[2];
            S.r_shift[pos][3] = (int8_t)(tid >> 1);                    // candidate row id (rz * 4 + ry)
            S.r_geo[pos] = make_int4(R.xlo, R.ncol, R.vlo, (int)cell_id(g, R.xlo, R.cy, R.cz));
        }
        const uint32_t total = __shfl_sync(0xFFFFFFFFu, incl, 31);
        if (tid == 0) { S.nranges = __popc(mask); S.ncand = total; S.r_base[__popc(mask)] = total; }
        if ((tid & 1) == 0) {                                          // first valid piece of candidate row tid >> 1
            const bool v1 = (mask >> (tid + 1)) & 1u;
            S.r_row[tid >> 1] = valid ? (uint8_t)pos : (v1 ? (uint8_t)__popc(mask & ((2u << tid) - 1u)) : (uint8_t)0xFF);
        }
    }
    // target cells, column-major with serpentine rows (tile_cell_rc)
    const int nrows = td.nyr * td.nzr;
    const int ncells = (td.cxb - td.cxa + 1) * nrows;
    if (tid >= 32 && tid < 32 + TILE_MAXCELL) {
        const int e = tid - 32;
        if (e < ncells) {
            int cx, ry, rz;
            tile_cell_rc(td, e, cx, ry, rz);
            const uint32_t c = cell_id(g, cx, td.y0 + ry, td.z0 + rz);
            const uint32_t a = ct.cell_start[c], b = ct.cell_tend[c];
            S.c_first[e] = a;
            S.c_pre[e + 1] = b - a;          // counts, scanned below
        }
    }
    __syncthreads();
    if (tid < 32) {                          // exclusive scan of <= 96 counts by one warp
        uint32_t run = 0;
        for (int b0 = 0; b0 < ncells; b0 += 32) {
            const int e = b0 + tid;
            uint32_t v = e < ncells ? S.c_pre[e + 1] : 0u, incl = v;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                uint32_t u = __shfl_up_sync(0xFFFFFFFFu, incl, o);
                if (tid >= o) incl += u;
            }
            if (e < ncells) S.c_pre[e + 1] = run + incl;
            run += __shfl_sync(0xFFFFFFFFu, incl, 31);
        }
        if (tid == 0) { S.c_pre[0] = 0; S.ncells = ncells; }
    }
    __syncthreads();
}

// global sorted slot of target t of the tile (t < td.nt); *cell_e = index of its cell in the column-major enumeration
__device__ __forceinline__ uint32_t tile_target(const TileDesc& td, const TileS& S, int t, int* cell_e = nullptr) {
    const uint32_t p = td.skip + (uint32_t)t;
    int lo = 0, hi = (int)S.ncells;          // find e with c_pre[e] <= p < c_pre[e+1]
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (S.c_pre[mid] <= p) lo = mid; else hi = mid;
    }
    if (cell_e) *cell_e = lo;
    return S.c_first[lo] + (p - S.c_pre[lo]);
}

}  // namespace spray
