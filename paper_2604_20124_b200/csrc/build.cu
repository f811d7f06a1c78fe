// build.cu -- (a1)-(a4) of the hot path: cell key, stable LSD radix sort, cell table, SoA reorder.
// NNPS by a cell list, PAPER.md L438 (§2.6): "the index of the cell that each particle resides in can be easily
// computed ... the particles are sorted based on their cell indices, so that the particles in any arbitrary cell
// can be identified directly".
#include "spray_internal.h"

#include <cstdio>
#include <mutex>

namespace spray {

// ------------------------------------------------------------------------------------------- K1: cell key
// c_d = (int) floor((x_d - lo_d) * inv_d) clamped to [0, nc_d-1]; key = (c_z*nc_y + c_y)*nc_x + c_x.
// Subtract then multiply (two roundings, nothing to contract).  24 B read + 8 B written per particle.
// Level contexts (api.cu) append one bit: 0 for the particles the level serves (2 hs in (lvl_lo, lvl_hi], not served before),
// 1 for the others, so that the sort puts the targets of a cell in front of its other particles.
__global__ void k_cell_key(DevGrid g, int64_t n, const double* __restrict__ x, const double* __restrict__ y,
                           const double* __restrict__ z, uint32_t* __restrict__ key, uint32_t* __restrict__ idx,
                           uint32_t* __restrict__ status, const double* __restrict__ hs_caller, const uint8_t* __restrict__ fast_caller,
                           double lvl_lo, double lvl_hi) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    double p[3] = {x[i], y[i], z[i]};
    int c[3];
    bool bad = false;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        double t = floor(__dmul_rn(__dsub_rn(p[d], g.lo[d]), g.inv[d]));
        int ci = (t < 0.0) ? 0 : (t >= (double)g.nc[d] ? g.nc[d] - 1 : (int)t);
        if (!(t == t)) { ci = 0; bad = true; }
        if (g.per[d] && !(p[d] >= g.lo[d] && p[d] < g.lo[d] + g.L[d])) bad = true;
        c[d] = ci;
    }
    uint32_t k = (uint32_t)((c[2] * g.nc[1] + c[1]) * g.nc[0] + c[0]);
    if (hs_caller) {
        const double r = 2.0 * hs_caller[i];
        const bool target = !fast_caller[i] && r > lvl_lo && r <= lvl_hi && !bad;
        k = (k << 1) | (target ? 0u : 1u);
    }
    key[i] = k;
    idx[i] = (uint32_t)i;
    if (bad) atomicOr(status, (uint32_t)SPRAY_DEV_OUTSIDE_BOX);
}

// ------------------------------------------------------------------------------------------- K2: radix sort
// Stable LSD radix sort of (key, idx), 8 bits per pass, ceil(bits(ncell-1)/8) passes.
// Per pass: per-tile digit histogram -> exclusive scan over [digit][tile] -> stable scatter.
// Stability inside a tile: each warp owns a contiguous run of the tile and ranks its keys round by round with
// __match_any_sync, so equal digits keep ascending position; warps are then offset in warp order.
constexpr int RS_THREADS = 256;
constexpr int RS_ITEMS = 16;
constexpr int RS_TILE = RS_THREADS * RS_ITEMS;   // 4096 keys per CTA
constexpr int RS_WARPS = RS_THREADS / 32;

__global__ void __launch_bounds__(RS_THREADS)
k_rs_hist(const uint32_t* __restrict__ key, int64_t n, int shift, uint32_t* __restrict__ hist, int nblk) {
    __shared__ uint32_t sh[256];
    sh[threadIdx.x] = 0;
    __syncthreads();
    int64_t base = (int64_t)blockIdx.x * RS_TILE;
#pragma unroll
    for (int j = 0; j < RS_ITEMS; ++j) {
        int64_t i = base + j * RS_THREADS + threadIdx.x;
        if (i < n) atomicAdd(&sh[(key[i] >> shift) & 255u], 1u);
    }
    __syncthreads();
    hist[(int64_t)threadIdx.x * nblk + blockIdx.x] = sh[threadIdx.x];
}

// exclusive scan, in place, of `total` u32 counters (total = 256 * ntiles ~ 1.05 M at 16.7 M keys) in three small kernels:
// per-block scan of SC_TILE counters + block totals, single-CTA scan of the <= SC_TILE totals, add-back.
constexpr int SC_THREADS = 256;
constexpr int SC_ITEMS = 16;
constexpr int SC_TILE = SC_THREADS * SC_ITEMS;

__device__ __forceinline__ uint32_t block_excl_scan_256(uint32_t v, uint32_t* total) {
    __shared__ uint32_t wsum[SC_THREADS / 32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    uint32_t incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t u = __shfl_up_sync(0xFFFFFFFFu, incl, o);
        if (lane >= o) incl += u;
    }
    if (lane == 31) wsum[w] = incl;
    __syncthreads();
    if (w == 0) {
        uint32_t t = lane < SC_THREADS / 32 ? wsum[lane] : 0u, ti = t;
#pragma unroll
        for (int o = 1; o < SC_THREADS / 32; o <<= 1) {
            uint32_t u = __shfl_up_sync(0xFFFFFFFFu, ti, o);
            if (lane >= o) ti += u;
        }
        if (lane < SC_THREADS / 32) wsum[lane] = ti - t;
        if (lane == SC_THREADS / 32 - 1) *total = ti;
    }
    __syncthreads();
    return wsum[w] + incl - v;
}

__global__ void __launch_bounds__(SC_THREADS) k_scan_blocks(uint32_t* __restrict__ a, int64_t total, uint32_t* __restrict__ btot) {
    __shared__ uint32_t tot;
    const int64_t base = (int64_t)blockIdx.x * SC_TILE + (int64_t)threadIdx.x * SC_ITEMS;
    uint32_t v[SC_ITEMS], s = 0;
#pragma unroll
    for (int j = 0; j < SC_ITEMS; ++j) { v[j] = (base + j < total) ? a[base + j] : 0u; s += v[j]; }
    uint32_t run = block_excl_scan_256(s, &tot);
#pragma unroll
    for (int j = 0; j < SC_ITEMS; ++j) { if (base + j < total) a[base + j] = run; run += v[j]; }
    if (threadIdx.x == 0) btot[blockIdx.x] = tot;
}
__global__ void __launch_bounds__(SC_THREADS) k_scan_totals(uint32_t* __restrict__ btot, int nb) {   // nb <= SC_TILE
    __shared__ uint32_t tot;
    const int base = threadIdx.x * SC_ITEMS;
    uint32_t v[SC_ITEMS], s = 0;
#pragma unroll
    for (int j = 0; j < SC_ITEMS; ++j) { v[j] = (base + j < nb) ? btot[base + j] : 0u; s += v[j]; }
    uint32_t run = block_excl_scan_256(s, &tot);
#pragma unroll
    for (int j = 0; j < SC_ITEMS; ++j) { if (base + j < nb) btot[base + j] = run; run += v[j]; }
}
__global__ void __launch_bounds__(SC_THREADS) k_scan_add(uint32_t* __restrict__ a, int64_t total, const uint32_t* __restrict__ btot) {
    const uint32_t off = btot[blockIdx.x];
    const int64_t base = (int64_t)blockIdx.x * SC_TILE;
#pragma unroll
    for (int j = 0; j < SC_ITEMS; ++j) {
        const int64_t i = base + j * SC_THREADS + threadIdx.x;
        if (i < total) a[i] += off;
    }
}

__global__ void __launch_bounds__(RS_THREADS)
k_rs_scatter(const uint32_t* __restrict__ key_in, const uint32_t* __restrict__ idx_in, uint32_t* __restrict__ key_out,
             uint32_t* __restrict__ idx_out, int64_t n, int shift, const uint32_t* __restrict__ hist, int nblk) {
    __shared__ uint32_t wh[RS_WARPS][256];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (int i = threadIdx.x; i < RS_WARPS * 256; i += RS_THREADS) (&wh[0][0])[i] = 0;
    __syncthreads();
    const int64_t base = (int64_t)blockIdx.x * RS_TILE + (int64_t)w * (RS_ITEMS * 32);
    uint32_t k[RS_ITEMS], v[RS_ITEMS], rank[RS_ITEMS];
    const uint32_t lt = (1u << lane) - 1u;
#pragma unroll
    for (int r = 0; r < RS_ITEMS; ++r) {
        int64_t i = base + r * 32 + lane;
        bool ok = i < n;
        k[r] = ok ? key_in[i] : 0xFFFFFFFFu;
        v[r] = ok ? idx_in[i] : 0u;
        uint32_t d = ok ? ((k[r] >> shift) & 255u) : 256u;       // 256 = padding lane, its own match group
        uint32_t peers = __match_any_sync(0xFFFFFFFFu, d);
        int leader = __ffs(peers) - 1;
        uint32_t old = 0;
        if (lane == leader && ok) { old = wh[w][d]; wh[w][d] = old + __popc(peers); }
        old = __shfl_sync(0xFFFFFFFFu, old, leader);
        rank[r] = old + __popc(peers & lt);
        __syncwarp();
    }
    __syncthreads();
    {   // per digit: global offset of this tile, then warps in order
        int d = threadIdx.x;
        uint32_t run = hist[(int64_t)d * nblk + blockIdx.x];
#pragma unroll
        for (int ww = 0; ww < RS_WARPS; ++ww) { uint32_t t = wh[ww][d]; wh[ww][d] = run; run += t; }
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < RS_ITEMS; ++r) {
        int64_t i = base + r * 32 + lane;
        if (i < n) {
            uint32_t d = (k[r] >> shift) & 255u;
            uint32_t pos = wh[w][d] + rank[r];
            key_out[pos] = k[r];
            idx_out[pos] = v[r];
        }
    }
}

// ------------------------------------------------------------------------------------------- K3: cell table
// cell_start[c] = #{key < c} = lower_bound(sorted_key, c); cell_end[c] = lower_bound(sorted_key, c+1).
__device__ __forceinline__ uint32_t lower_bound_u32(const uint32_t* __restrict__ a, uint32_t n, uint32_t v) {
    uint32_t lo = 0, hi = n;
    while (lo < hi) {
        uint32_t mid = (lo + hi) >> 1;
        if (__ldg(a + mid) < v) lo = mid + 1; else hi = mid;
    }
    return lo;
}
__global__ void k_cell_table(const uint32_t* __restrict__ sorted_key, uint32_t n, uint32_t ncell,
                             uint32_t* __restrict__ cell_start, uint32_t* __restrict__ cell_end) {
    uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c > ncell) return;
    uint32_t lb = lower_bound_u32(sorted_key, n, c);
    if (c < ncell) cell_start[c] = lb;
    if (c > 0) cell_end[c - 1] = lb;
}
// level contexts: keys are 2 cell + (0 target | 1 other)
__global__ void k_cell_table_level(const uint32_t* __restrict__ sorted_key, uint32_t n, uint32_t ncell, uint32_t* __restrict__ cell_start,
                                   uint32_t* __restrict__ cell_tend, uint32_t* __restrict__ cell_end) {
    uint32_t v = blockIdx.x * blockDim.x + threadIdx.x;
    if (v > 2u * ncell) return;
    uint32_t lb = lower_bound_u32(sorted_key, n, v);
    if (v & 1u) { cell_tend[v >> 1] = lb; return; }
    if (v < 2u * ncell) cell_start[v >> 1] = lb;
    if (v > 0) cell_end[(v >> 1) - 1] = lb;
}

// ------------------------------------------------------------------------------------------- K4: reorder by cell
// Sorted copies of (x, y, z, h): structure-of-arrays for the general kernels and 16-byte records (x,y), (z,h),
// (1/h, FN_K/h^4) for the tiled kernels.  64 B written per particle and layout.
__global__ void k_reorder_build(const uint32_t* __restrict__ perm, int64_t n, const double* __restrict__ x,
                                const double* __restrict__ y, const double* __restrict__ z, const double* __restrict__ h,
                                double* __restrict__ sx, double* __restrict__ sy, double* __restrict__ sz, double* __restrict__ sh,
                                double2* __restrict__ p0, double2* __restrict__ p1, double2* __restrict__ hh, double fnk) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint32_t p = perm[i];
    const double xv = __ldg(x + p), yv = __ldg(y + p), zv = __ldg(z + p), hv = __ldg(h + p);
    sx[i] = xv; sy[i] = yv; sz[i] = zv; sh[i] = hv;
    p0[i] = make_double2(xv, yv);
    p1[i] = make_double2(zv, hv);
    const double hinv = 1.0 / hv, h2 = hinv * hinv;
    hh[i] = make_double2(hinv, fnk * (h2 * h2));
}

// per-call prologues: caller order -> sorted order, with the per-particle factors of the pair formulas hoisted
// (V = m/rho, Q = V p, alpha*c, p/rho, 1/rho): one division per particle instead of one per pair.  The packed
// records feed the tiled kernels; the structure-of-arrays copies feed the general kernels and are written only
// when some particle is left to them (*nfast != n).
struct PackedOut { double2 *s0, *s1, *s2, *s3, *t0, *me; double* e1; const double2* p1; };

__global__ void k_prep_density(const double* __restrict__ m, const uint32_t* __restrict__ perm, int64_t n, PackedOut o,
                               double* __restrict__ sm, const unsigned long long* __restrict__ nfast) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double mv = __ldg(m + perm[i]);
    o.s0[i] = make_double2(o.p1[i].x, mv);
    if (!nfast || *nfast != (unsigned long long)n) sm[i] = mv;
}
__global__ void k_prep_hydro(PrepJob j, const uint32_t* __restrict__ perm, int64_t n, PackedOut o,
                             const unsigned long long* __restrict__ nfast) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint32_t p = perm[i];
    const double m = __ldg(j.m + p), rho = __ldg(j.rho + p), pr = __ldg(j.p + p), cs = __ldg(j.cs + p), al = __ldg(j.alpha + p);
    const double vx = __ldg(j.vx + p), vy = __ldg(j.vy + p), vz = __ldg(j.vz + p);
    const double ia = 1.0 / rho;
    const double V = m / rho;
    o.s0[i] = make_double2(o.p1[i].x, V);
    o.s1[i] = make_double2(V * pr, vx);
    o.s2[i] = make_double2(vy, vz);
    o.s3[i] = make_double2(m, al * cs);
    o.t0[i] = make_double2(pr * ia, ia);
    const bool soa = !nfast || *nfast != (unsigned long long)n;
    if (soa) {
        j.sm[i] = m; j.srho[i] = rho; j.sp[i] = pr; j.scs[i] = cs; j.salpha[i] = al;
        j.svx[i] = vx; j.svy[i] = vy; j.svz[i] = vz;
        j.sV[i] = V; j.sQ[i] = V * pr; j.sAC[i] = al * cs;
    }
    if (j.E) {   // spray_hydro_rhs_limiter: the limiter's prologue in the same pass over the particles
        const double E = __ldg(j.E + p), kx = __ldg(j.kx + p);
        o.e1[i] = E;
        o.me[i] = make_double2(rho * kx, E);
        if (soa) { j.sE[i] = E; j.skx[i] = kx; }
    }
}
__global__ void k_prep_fld(PrepJob j, const uint32_t* __restrict__ perm, int64_t n, PackedOut o,
                           const unsigned long long* __restrict__ nfast) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint32_t p = perm[i];
    const double m = __ldg(j.m + p), rho = __ldg(j.rho + p), E = __ldg(j.E + p), kx = __ldg(j.kx + p);
    const double V = m / rho;
    o.s0[i] = make_double2(o.p1[i].x, V);
    o.e1[i] = E;
    if (j.kx_is_mu) o.me[i] = make_double2(kx, E);
    else o.t0[i] = make_double2(rho * kx, 0.0);
    if (!nfast || *nfast != (unsigned long long)n) {
        j.sm[i] = m; j.srho[i] = rho; j.sE[i] = E; j.skx[i] = kx;
        j.sV[i] = V;
    }
}

// N3: (z, V), (vx, vy), (vz, -), target record (rho, -)
__global__ void k_prep_kgc(PrepJob j, const uint32_t* __restrict__ perm, int64_t n, PackedOut o,
                           const unsigned long long* __restrict__ nfast) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint32_t p = perm[i];
    const double m = __ldg(j.m + p), rho = __ldg(j.rho + p);
    const double vx = __ldg(j.vx + p), vy = __ldg(j.vy + p), vz = __ldg(j.vz + p);
    const double V = m / rho;
    o.s0[i] = make_double2(o.p1[i].x, V);
    o.s1[i] = make_double2(vx, vy);
    o.s2[i] = make_double2(vz, 0.0);
    o.t0[i] = make_double2(rho, 0.0);
    if (!nfast || *nfast != (unsigned long long)n) {
        j.sm[i] = m; j.srho[i] = rho; j.svx[i] = vx; j.svy[i] = vy; j.svz[i] = vz; j.sV[i] = V;
    }
}

// per-cell max h (fp64 max is exact and order independent), global min/max of h, and the h <= h_max check
__global__ void k_init_hglob(double* hglob) { hglob[0] = __longlong_as_double(0x7FF0000000000000ll); hglob[1] = 0.0; }

__global__ void k_cell_hmax(const uint32_t* __restrict__ cell_start, const uint32_t* __restrict__ cell_end,
                            const double* __restrict__ h, uint32_t ncell, double hmax_decl,
                            double* __restrict__ cell_hmax, double* __restrict__ cell_hmin, double* __restrict__ hglob, uint32_t* __restrict__ status) {
    uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
    double mx = 0.0, mn = __longlong_as_double(0x7FF0000000000000ll);
    if (c < ncell) {
        for (uint32_t j = cell_start[c]; j < cell_end[c]; ++j) { double v = h[j]; mx = fmax(mx, v); mn = fmin(mn, v); }
        cell_hmax[c] = mx;
        cell_hmin[c] = mn;
    }
    // warp reduce, then one atomic per warp on the bit patterns (positive doubles order like integers)
    for (int o = 16; o; o >>= 1) {
        mx = fmax(mx, __shfl_xor_sync(0xFFFFFFFFu, mx, o));
        mn = fmin(mn, __shfl_xor_sync(0xFFFFFFFFu, mn, o));
    }
    if ((threadIdx.x & 31) == 0) {
        if (mx > 0.0) atomicMax((unsigned long long*)&hglob[1], (unsigned long long)__double_as_longlong(mx));
        if (mn > 0.0) atomicMin((unsigned long long*)&hglob[0], (unsigned long long)__double_as_longlong(mn));
        if (mx > hmax_decl) atomicOr(status, (uint32_t)SPRAY_DEV_H_EXCEEDS_HMAX);
    }
}

// ---- levels (api.cu): per-particle data between the parent (sorted order) and the level contexts (caller order)
__global__ void k_to_caller(const uint32_t* __restrict__ perm, int64_t n, const double* __restrict__ hs, const uint8_t* __restrict__ fast,
                            double* __restrict__ hs_c, uint8_t* __restrict__ fast_c) {
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint32_t p = perm[i];
    hs_c[p] = hs[i];
    fast_c[p] = fast ? fast[i] : (uint8_t)0;
}
__global__ void k_merge_served(const uint32_t* __restrict__ perm_child, int64_t n, const uint8_t* __restrict__ fast_child,
                               uint8_t* __restrict__ fast_c) {
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    if (fast_child[i]) fast_c[perm_child[i]] = 1;
}
__global__ void k_fast_from_caller(const uint32_t* __restrict__ perm, int64_t n, const uint8_t* __restrict__ fast_c, uint8_t* __restrict__ fast,
                                   unsigned long long* __restrict__ nfast) {
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const bool f = i < n && fast_c[perm[i]] != 0;
    if (i < n) fast[i] = f ? 1 : 0;
    const unsigned m = __ballot_sync(0xFFFFFFFFu, f);
    if ((threadIdx.x & 31) == 0 && m) atomicAdd(nfast, (unsigned long long)__popc(m));
}

__global__ void k_general_from_parent(const uint32_t* __restrict__ perm, int64_t n, const double* __restrict__ hs_c, const uint8_t* __restrict__ fast_c,
                                      double* __restrict__ hs, uint8_t* __restrict__ fast) {
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint32_t p = perm[i];
    hs[i] = hs_c[p];
    fast[i] = fast_c[p] ? 1 : 0;
}

// ------------------------------------------------------------------------------------------- launchers
static inline int cdiv64(int64_t a, int64_t b) { return (int)((a + b - 1) / b); }

// the particles the tiled kernels do not serve, compacted in ascending sorted order within a block's 256 (blocks in the order
// they get to the counter: the order of the list changes nothing in the results, each particle's sums are its own)
__global__ void k_compact_left(const uint8_t* __restrict__ fast, int64_t n, uint32_t* __restrict__ left, unsigned long long* __restrict__ nleft) {
    __shared__ uint32_t wbase[8];
    __shared__ unsigned long long base;
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const bool keep = i < n && fast[i] == 0;
    const unsigned m = __ballot_sync(0xFFFFFFFFu, keep);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) wbase[w] = __popc(m);
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t run = 0;
        for (int k = 0; k < 8; ++k) { const uint32_t t = wbase[k]; wbase[k] = run; run += t; }
        base = run ? atomicAdd(nleft, (unsigned long long)run) : 0ull;
    }
    __syncthreads();
    if (keep) left[base + wbase[w] + __popc(m & ((1u << lane) - 1u))] = (uint32_t)i;
}
cudaError_t launch_compact_left(Ctx* c, const uint8_t* fast, cudaStream_t st) {
    if (c->n == 0 || !c->left) return cudaSuccess;
    cudaError_t e = cudaMemsetAsync(c->tl.ctr + CTR_NLEFT, 0, sizeof(unsigned long long), st);
    if (e != cudaSuccess) return e;
    k_compact_left<<<cdiv64(c->n, 256), 256, 0, st>>>(fast, c->n, c->left, c->tl.ctr + CTR_NLEFT);
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_to_caller_order(Ctx* c, cudaStream_t st) {
    if (c->n == 0) return cudaSuccess;
    k_to_caller<<<cdiv64(c->n, 256), 256, 0, st>>>(c->perm, c->n, c->s.hs, c->tl.enabled ? c->tl.fast : nullptr, c->hs_c, c->fast_c);
    c->launches += 1;
    return cudaGetLastError();
}
cudaError_t launch_merge_served(Ctx* parent, Ctx* child, cudaStream_t st) {
    if (child->n == 0 || !child->tl.enabled) return cudaSuccess;
    k_merge_served<<<cdiv64(child->n, 256), 256, 0, st>>>(child->perm, child->n, child->tl.fast, parent->fast_c);
    parent->launches += 1;
    return cudaGetLastError();
}
cudaError_t launch_fast_from_caller(Ctx* c, cudaStream_t st) {
    if (c->n == 0) return cudaSuccess;
    cudaError_t e = cudaMemsetAsync(c->tl.ctr + CTR_NFAST_ALL, 0, sizeof(unsigned long long), st);
    if (e != cudaSuccess) return e;
    k_fast_from_caller<<<cdiv64(c->n, 256), 256, 0, st>>>(c->perm, c->n, c->fast_c, c->fast_all, c->tl.ctr + CTR_NFAST_ALL);
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_general_from_parent(Ctx* v, Ctx* parent, cudaStream_t st) {
    if (v->n == 0) return cudaSuccess;
    k_general_from_parent<<<cdiv64(v->n, 256), 256, 0, st>>>(v->perm, v->n, parent->hs_c, parent->fast_c, v->s.hs, v->fast_all);
    v->launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_cell_keys(Ctx* c, const double* x, const double* y, const double* z, cudaStream_t st) {
    if (c->n == 0) return cudaSuccess;
    k_cell_key<<<cdiv64(c->n, 256), 256, 0, st>>>(c->dg, c->n, x, y, z, c->key[0], c->idx[0], c->dev_status,
                                                 c->is_level ? c->hs_caller : nullptr, c->fast_caller, c->level_lo, c->level_hi);
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_radix_sort(Ctx* c, cudaStream_t st) {
    int bits = 0;
    while (((int64_t)1 << bits) < c->ncell * (c->is_level ? 2 : 1)) ++bits;
    int passes = (bits + 7) / 8;
    int cur = 0;
    int nblk = cdiv64(c->n, RS_TILE);
    for (int p = 0; p < passes && c->n > 0; ++p) {
        int shift = 8 * p;
        k_rs_hist<<<nblk, RS_THREADS, 0, st>>>(c->key[cur], c->n, shift, c->hist, nblk);
        {
            const int64_t total = (int64_t)256 * nblk;
            const int nb = cdiv64(total, SC_TILE);          // <= SC_TILE for n <= 2^32 keys
            uint32_t* btot = c->hist + total;
            k_scan_blocks<<<nb, SC_THREADS, 0, st>>>(c->hist, total, btot);
            k_scan_totals<<<1, SC_THREADS, 0, st>>>(btot, nb);
            k_scan_add<<<nb, SC_THREADS, 0, st>>>(c->hist, total, btot);
        }
        k_rs_scatter<<<nblk, RS_THREADS, 0, st>>>(c->key[cur], c->idx[cur], c->key[cur ^ 1], c->idx[cur ^ 1], c->n, shift,
                                                  c->hist, nblk);
        cur ^= 1;
        c->launches += 5;
    }
    c->sorted_key = c->key[cur];
    c->perm = c->idx[cur];
    return cudaGetLastError();
}

cudaError_t launch_cell_table(Ctx* c, cudaStream_t st) {
    if (c->is_level)
        k_cell_table_level<<<cdiv64(2 * c->ncell + 1, 256), 256, 0, st>>>(c->sorted_key, (uint32_t)c->n, (uint32_t)c->ncell, c->cell_start,
                                                                         c->cell_tend, c->cell_end);
    else
        k_cell_table<<<cdiv64(c->ncell + 1, 256), 256, 0, st>>>(c->sorted_key, (uint32_t)c->n, (uint32_t)c->ncell, c->cell_start,
                                                               c->cell_end);
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_reorder_build(Ctx* c, const double* x, const double* y, const double* z, const double* h, cudaStream_t st) {
    if (c->n == 0) return cudaSuccess;
    k_reorder_build<<<cdiv64(c->n, 256), 256, 0, st>>>(c->perm, c->n, x, y, z, h, c->s.x, c->s.y, c->s.z, c->s.h, c->pk.p0, c->pk.p1,
                                                       c->pk.hh, c->kernel == SPRAY_KERNEL_WENDLAND_C2 ? kFnWend : kFnCubic);
    c->launches += 1;
    return cudaGetLastError();
}

// device word the prologues compare with n: equal = nobody needs the structure-of-arrays copies (general kernels idle).
// A level context never runs general kernels: its word is CTR_NALL = n.
static const unsigned long long* nfast_ptr(Ctx* c) {
    if (c->soa_ctr) return c->soa_ctr;               // the level context that runs the parent's general kernels
    if (c->is_level) return c->tl.ctr + CTR_NALL;
    return c->tl.enabled ? c->tl.ctr + CTR_NFAST : nullptr;
}
static PackedOut packed_out(Ctx* c) {
    PackedOut o{c->pk.s[0], c->pk.s[1], c->pk.s[2], c->pk.s[3], c->pk.t0, c->pk.me, c->pk.e1, c->pk.p1};
    return o;
}

cudaError_t launch_prep_density(Ctx* c, const double* m, cudaStream_t st) {
    if (c->n == 0) return cudaSuccess;
    k_prep_density<<<cdiv64(c->n, 256), 256, 0, st>>>(m, c->perm, c->n, packed_out(c), c->s.f[0], nfast_ptr(c));
    c->launches += 1;
    return cudaGetLastError();
}
cudaError_t launch_prep_hydro(Ctx* c, const PrepJob& j, cudaStream_t st) {
    if (c->n == 0) return cudaSuccess;
    k_prep_hydro<<<cdiv64(c->n, 256), 256, 0, st>>>(j, c->perm, c->n, packed_out(c), nfast_ptr(c));
    c->launches += 1;
    return cudaGetLastError();
}
cudaError_t launch_prep_fld(Ctx* c, const PrepJob& j, cudaStream_t st) {
    if (c->n == 0) return cudaSuccess;
    k_prep_fld<<<cdiv64(c->n, 256), 256, 0, st>>>(j, c->perm, c->n, packed_out(c), nfast_ptr(c));
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_prep_kgc(Ctx* c, const PrepJob& j, cudaStream_t st) {
    if (c->n == 0) return cudaSuccess;
    k_prep_kgc<<<cdiv64(c->n, 256), 256, 0, st>>>(j, c->perm, c->n, packed_out(c), nfast_ptr(c));
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_excl_scan_u32(Ctx* c, uint32_t* a, int64_t total, uint32_t* scratch, cudaStream_t st) {
    if (total <= 0) return cudaSuccess;
    const int nb = cdiv64(total, SC_TILE);            // <= SC_TILE
    k_scan_blocks<<<nb, SC_THREADS, 0, st>>>(a, total, scratch);
    k_scan_totals<<<1, SC_THREADS, 0, st>>>(scratch, nb);
    k_scan_add<<<nb, SC_THREADS, 0, st>>>(a, total, scratch);
    c->launches += 3;
    return cudaGetLastError();
}

// fp32 copies of the sorted positions and smoothing lengths for the pre-test of the search-length pre-pass (sweeps_ref.cu)
__global__ void k_pack_f4(const double* __restrict__ x, const double* __restrict__ y, const double* __restrict__ z, const double* __restrict__ h,
                          const double* __restrict__ hglob, int64_t n, float4* __restrict__ f4) {
    if (!(hglob[0] < hglob[1])) return;               // uniform h: the pre-pass has nothing to do and reads nothing
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i < n) f4[i] = make_float4((float)x[i], (float)y[i], (float)z[i], (float)h[i]);
}
cudaError_t launch_pack_f4(Ctx* c, float4* f4, cudaStream_t st) {
    if (c->n == 0) return cudaSuccess;
    k_pack_f4<<<cdiv64(c->n, 256), 256, 0, st>>>(c->s.x, c->s.y, c->s.z, c->s.h, c->hglob, c->n, f4);
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_cell_hmax(Ctx* c, cudaStream_t st) {
    k_init_hglob<<<1, 1, 0, st>>>(c->hglob);
    k_cell_hmax<<<cdiv64(c->ncell, 256), 256, 0, st>>>(c->cell_start, c->cell_end, c->s.h, (uint32_t)c->ncell, c->grid.h_max,
                                                      c->cell_hmax, c->cell_hmin, c->hglob, c->dev_status);
    c->launches += 2;
    return cudaGetLastError();
}

}  // namespace spray

// ------------------------------------------------------------------------------------------- spray_cell_list_static
// Rows a1-a3 (cell key, stable radix sort, cell table) for callers that cannot allocate: no context, no
// cudaMalloc / cudaFree / allocating library routine.  The sort's scratch -- two (key, index) buffers and the radix
// histograms -- lives in the file-scope device array below, which every GPU that loads the library holds until the process
// exits.  Same kernels, launch order and pass count as spray_build_cells, so the results are bit-identical to
// spray_build_cells + spray_get_cell_table.  The last radix pass scatters straight into the caller's sorted_key / perm.
namespace spray {
constexpr int64_t STATIC_NMAX = SPRAY_STATIC_NMAX;
constexpr int64_t STATIC_HIST = 256 * (STATIC_NMAX / RS_TILE + 1) + SC_TILE;   // [digit][tile] counters + block totals of their scan
constexpr int64_t STATIC_OFF_KEY0 = 0, STATIC_OFF_IDX0 = STATIC_NMAX, STATIC_OFF_KEY1 = 2 * STATIC_NMAX, STATIC_OFF_IDX1 = 3 * STATIC_NMAX;
constexpr int64_t STATIC_OFF_HIST = 4 * STATIC_NMAX, STATIC_OFF_STATUS = STATIC_OFF_HIST + STATIC_HIST;
constexpr int64_t STATIC_WORDS = STATIC_OFF_STATUS + 64;
static_assert(STATIC_NMAX % RS_TILE == 0, "whole sort tiles");
static_assert(STATIC_WORDS * 4 <= (int64_t)SPRAY_STATIC_SCRATCH_BYTES, "spray.h states the size of the static scratch");

// In host code this name is a host-side stand-in, not a device address: kernels get the pointer cudaGetSymbolAddress returns.
static __device__ __align__(256) uint32_t g_static_scratch[STATIC_WORDS];

constexpr int STATIC_MAX_DEVICES = 64;
static uint32_t* g_static_ptr[STATIC_MAX_DEVICES] = {};     // per device, set once with that device current
static std::mutex g_static_mu;
static thread_local char g_static_err[256] = "";

static int static_fail(int code, const char* what, cudaError_t e = cudaSuccess) {
    if (e != cudaSuccess) snprintf(g_static_err, sizeof g_static_err, "%s: %s", what, cudaGetErrorString(e));
    else snprintf(g_static_err, sizeof g_static_err, "%s", what);
    return code;
}
}  // namespace spray

extern "C" const char* spray_static_last_error(void) { return spray::g_static_err; }

extern "C" int spray_cell_list_static(const spray_grid_t* grid, int64_t n, const double* x, const double* y, const double* z,
                                      uint32_t* sorted_key, uint32_t* perm, uint32_t* cell_start, uint32_t* cell_end,
                                      uint32_t* dev_status, void* stream) {
    using namespace spray;
    g_static_err[0] = 0;
    if (!grid || n < 0 || !cell_start || !cell_end || (n > 0 && (!x || !y || !z || !sorted_key || !perm)))
        return static_fail(SPRAY_ERR_INVALID_ARG, "spray_cell_list_static: NULL argument or n < 0");
    if (n > STATIC_NMAX) {
        snprintf(g_static_err, sizeof g_static_err, "spray_cell_list_static: n = %lld exceeds SPRAY_STATIC_NMAX = %lld (the static scratch "
                 "holds no more; use spray_create + spray_build_cells)", (long long)n, (long long)STATIC_NMAX);
        return SPRAY_ERR_CAPACITY;
    }
    DevGrid dg;
    int64_t ncell = 1;
    for (int d = 0; d < 3; ++d) {
        if (grid->ncell[d] < 1) return static_fail(SPRAY_ERR_GRID, "spray_cell_list_static: grid: ncell_d < 1");
        if (!(grid->hi[d] > grid->lo[d])) return static_fail(SPRAY_ERR_GRID, "spray_cell_list_static: grid: hi <= lo");
        ncell *= grid->ncell[d];
        if (ncell > (int64_t)SPRAY_STATIC_NCELL_MAX) return static_fail(SPRAY_ERR_GRID, "spray_cell_list_static: grid: prod ncell_d > SPRAY_STATIC_NCELL_MAX");
        dg.lo[d] = grid->lo[d];
        dg.L[d] = grid->hi[d] - grid->lo[d];
        dg.halfL[d] = 0.5 * dg.L[d];
        dg.edge[d] = dg.L[d] / (double)grid->ncell[d];
        dg.inv[d] = (double)grid->ncell[d] / dg.L[d];
        dg.nc[d] = grid->ncell[d];
        dg.per[d] = grid->periodic[d] != 0;
    }
    // the scratch's device address: once per device, with that device current (the caller's current device is the one whose
    // stream and pointers it passes)
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return static_fail(SPRAY_ERR_CUDA, "spray_cell_list_static: cudaGetDevice", e);
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return static_fail(SPRAY_ERR_INVALID_ARG, "spray_cell_list_static: device index out of range");
    uint32_t* S = nullptr;
    {
        std::lock_guard<std::mutex> lk(g_static_mu);
        if (!g_static_ptr[dev]) {
            void* p = nullptr;
            e = cudaGetSymbolAddress(&p, g_static_scratch);
            if (e != cudaSuccess || !p) return static_fail(SPRAY_ERR_CUDA, "spray_cell_list_static: cudaGetSymbolAddress", e);
            g_static_ptr[dev] = static_cast<uint32_t*>(p);
        }
        S = g_static_ptr[dev];
    }
    cudaStream_t st = (cudaStream_t)stream;
    uint32_t* status = S + STATIC_OFF_STATUS;
    uint32_t* hist = S + STATIC_OFF_HIST;
    // the array keeps the last call's contents: the status word must start at zero (the histograms and block totals are
    // overwritten in full by every pass, the key / index buffers by the key kernel and the scatters)
    e = cudaMemsetAsync(status, 0, sizeof(uint32_t), st);
    if (e != cudaSuccess) return static_fail(SPRAY_ERR_CUDA, "spray_cell_list_static: clearing the status word", e);
    if (n > 0) {
        int bits = 0;
        while (((int64_t)1 << bits) < ncell) ++bits;
        const int passes = (bits + 7) / 8;                              // as launch_radix_sort; 0 when the grid has one cell
        uint32_t* kbuf[2] = {S + STATIC_OFF_KEY0, S + STATIC_OFF_KEY1};
        uint32_t* ibuf[2] = {S + STATIC_OFF_IDX0, S + STATIC_OFF_IDX1};
        // with no pass to run the keys (all 0) and the identity permutation are the result
        uint32_t* k0 = passes ? kbuf[0] : sorted_key;
        uint32_t* i0 = passes ? ibuf[0] : perm;
        k_cell_key<<<cdiv64(n, 256), 256, 0, st>>>(dg, n, x, y, z, k0, i0, status, nullptr, nullptr, 0.0, 0.0);
        const int nblk = cdiv64(n, RS_TILE);
        int cur = 0;
        for (int p = 0; p < passes; ++p) {
            const int shift = 8 * p;
            const bool last = p == passes - 1;
            uint32_t* kd = last ? sorted_key : kbuf[cur ^ 1];
            uint32_t* id = last ? perm : ibuf[cur ^ 1];
            k_rs_hist<<<nblk, RS_THREADS, 0, st>>>(kbuf[cur], n, shift, hist, nblk);
            const int64_t total = (int64_t)256 * nblk;
            const int nb = cdiv64(total, SC_TILE);
            uint32_t* btot = hist + total;
            k_scan_blocks<<<nb, SC_THREADS, 0, st>>>(hist, total, btot);
            k_scan_totals<<<1, SC_THREADS, 0, st>>>(btot, nb);
            k_scan_add<<<nb, SC_THREADS, 0, st>>>(hist, total, btot);
            k_rs_scatter<<<nblk, RS_THREADS, 0, st>>>(kbuf[cur], ibuf[cur], kd, id, n, shift, hist, nblk);
            cur ^= 1;
        }
    }
    k_cell_table<<<cdiv64(ncell + 1, 256), 256, 0, st>>>(sorted_key, (uint32_t)n, (uint32_t)ncell, cell_start, cell_end);
    e = cudaGetLastError();
    if (e != cudaSuccess) return static_fail(SPRAY_ERR_CUDA, "spray_cell_list_static: kernel launch", e);
    if (dev_status) {
        e = cudaMemcpyAsync(dev_status, status, sizeof(uint32_t), cudaMemcpyDeviceToDevice, st);
        if (e != cudaSuccess) return static_fail(SPRAY_ERR_CUDA, "spray_cell_list_static: status copy", e);
    }
    return SPRAY_OK;
}
