// sweeps_ref.cu -- reference pair kernels: one CUDA thread per particle walking the cell table, the scheme the
// paper describes ("each CUDA thread carries out relevant SPH calculation for one particle, looping
// over neighbor particles").  General in every respect (any search range, any grid, variable h); used for the
// parity exports, for the symmetric-search-length pre-pass, and as the fallback of the tiled kernels.
#include "spray_internal.h"

namespace spray {

constexpr int REF_THREADS = 128;                 // threads per CTA of k_ref_sweep: the per-warp shared-memory areas below are sized for it
constexpr int REF_WARPS = REF_THREADS / 32;

struct CellTabs {
    const uint32_t *sorted_key, *perm, *cell_start, *cell_end;
    const double* hglob;
    const double* cell_hmin;
    int key_shift;                // 1 on a level context, whose sort keys carry a served-here bit below the cell index
    const double* cell_hmax;      // per-cell max h: a cell farther from the target than 2 max(h_a, cell_hmax) holds no mutual neighbour
};

// cells to visit along one dimension: `cnt` cells starting at `start` (wrapped when periodic)
struct Span { int start, cnt; };
__device__ __forceinline__ Span cell_span(const DevGrid& g, int d, int c, double reach) {
    int nc = g.nc[d];
    double rr = reach * g.inv[d] * (1.0 + 1e-12);
    int R = rr < (double)nc ? (int)ceil(rr) : nc;
    Span s;
    if (g.per[d]) {
        if (2 * R + 1 >= nc) { s.start = 0; s.cnt = nc; }
        else { s.start = c - R; s.cnt = 2 * R + 1; }
    } else {
        int a = c - R < 0 ? 0 : c - R, b = c + R > nc - 1 ? nc - 1 : c + R;
        s.start = a; s.cnt = b - a + 1;
    }
    return s;
}
__device__ __forceinline__ int wrap_cell(int c, int nc) { return c < 0 ? c + nc : (c >= nc ? c - nc : c); }

// Cell culling.  t = (x_a - lo_d) * inv_d as k_cell_key computes it (cell units), ca = the target's cell, o = the (unwrapped)
// offset of a visited cell: every particle b of that cell has (x_b - lo_d) * inv_d in [ca + o, ca + o + 1) (or beyond the outer
// face when it was clamped into a boundary cell), so |x_a - x_b| >= gap / inv_d with gap = o - f (o > 0), f + |o| - 1 (o < 0),
// 0 (o = 0), f = t - ca.  In a periodic dimension the image at offset o is the nearest one as long as the span does not cover
// the whole dimension (2R + 1 < nc); when it does, `full` switches the bound off.  1e-9 cell units cover the rounding of t.
// A cell farther than the reach in this bound holds no neighbour and is skipped: the neighbour sets do not change.
__device__ __forceinline__ double cell_gap2(int o, double f, bool full, double edge) {
    double gp = 0.0;
    if (!full) {
        if (o > 0) gp = (double)o - f;
        else if (o < 0) gp = f - (double)(o + 1);
    }
    gp = gp - 1e-9;
    gp = gp > 0.0 ? gp * edge : 0.0;
    return gp * gp;
}

// WARP = false: one thread per particle (the paper's scheme).  WARP = true: one WARP per particle -- the lanes share the
// particle and split the candidates of every cell it visits; the partial sums are added by a fixed shuffle butterfly (so the
// result does not depend on the launch) and lane 0 writes.  Used for the compact list of particles the tiled kernels leave
// over, which are few and expensive (long search ranges through dense cells): 32 times the parallelism, coalesced candidates.
template <class V>
__device__ __forceinline__ V warp_add(V v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
    return v;
}
template <int SWEEP, int KERNEL, bool WARP>
__device__ __forceinline__ void ref_particle(const DevGrid& g, int64_t n, const CellTabs& T, const SweepArgs& A, int64_t i) {
    if (A.skip && A.skip[i]) return;        // served by the tiled kernels
    const double xa = A.x[i], ya = A.y[i], za = A.z[i], ha = A.h[i];
    const uint32_t ia = T.perm[i];

    bool sym;
    if (SWEEP == SW_HYDRO) sym = true;
    else if (SWEEP == SW_APPLY) sym = A.fld_sym != 0;
    else if (SWEEP == SW_COUNT || SWEEP == SW_LIST || SWEEP == SW_DIGEST) sym = A.symmetric != 0;
    else sym = false;
    if (SWEEP == SW_HSEARCH) {
        if (!(ha > T.hglob[0])) return;      // nobody has a smaller h: nothing to raise
    }
    const double reach = 2.0 * (sym ? A.hs[i] : ha);
    const double sup_a = support2(ha);

    const uint32_t key = T.sorted_key[i] >> T.key_shift;
    const int cx = key % g.nc[0], cy = (key / g.nc[0]) % g.nc[1], cz = key / (g.nc[0] * g.nc[1]);
    const Span sx = cell_span(g, 0, cx, reach), sy = cell_span(g, 1, cy, reach), sz = cell_span(g, 2, cz, reach);
    const double fcx = __dmul_rn(__dsub_rn(xa, g.lo[0]), g.inv[0]) - (double)cx;
    const double fcy = __dmul_rn(__dsub_rn(ya, g.lo[1]), g.inv[1]) - (double)cy;
    const double fcz = __dmul_rn(__dsub_rn(za, g.lo[2]), g.inv[2]) - (double)cz;
    const double ex = 1.0 / g.inv[0], ey = 1.0 / g.inv[1], ez = 1.0 / g.inv[2];
    const bool fullx = sx.cnt == g.nc[0] && g.per[0], fully = sy.cnt == g.nc[1] && g.per[1], fullz = sz.cnt == g.nc[2] && g.per[2];
    const double reach2 = (reach * reach) * (1.0 + 1e-9);

    // per-particle constants
    const double hinv = 1.0 / ha;
    double acc0 = 0, acc1 = 0, acc2 = 0, acc3 = 0, acc4 = 0;
    uint32_t cnt = 0;
    uint64_t dsum = 0, dxr = 0;
    double rho_a = 0, p_a = 0, vxa = 0, vya = 0, vza = 0, ac_a = 0, E_a = 0, mu_a = 0, Wn = 0, Fn = 0;
    double km[6] = {0, 0, 0, 0, 0, 0}, kq[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};   // SW_KGC: sum c x_i x_j, sum c dv_i x_j
    Wn = sigma<KERNEL>() * hinv * hinv * hinv;          // sigma / h^3
    Fn = Wn * hinv;                                      // sigma / h^4
    if (SWEEP == SW_HYDRO) {
        rho_a = A.rho[i]; p_a = A.p[i]; vxa = A.vx[i]; vya = A.vy[i]; vza = A.vz[i]; ac_a = A.alpha[i] * A.cs[i];
    }
    if (SWEEP == SW_LIMITER) { E_a = A.E[i]; }
    if (SWEEP == SW_GRADN) { E_a = 0.0; }      // row N4: sum_b V_b f_b gradW(x_ab, h_a), no -f_a term
    if (SWEEP == SW_KGC) { rho_a = A.rho[i]; vxa = A.vx[i]; vya = A.vy[i]; vza = A.vz[i]; }
    if (SWEEP == SW_APPLY) { E_a = A.E[i]; mu_a = A.mu[i]; }
    uint64_t lbase = 0;
    if (SWEEP == SW_LIST) lbase = A.offsets[ia];

    // One candidate j: geometry and set membership (contract expressions), then the pair term of the sweep.
    struct Pair { double dx, dy, dz, r2, hb; bool self, in_g, in_s, in_set; };
    auto geometry = [&](uint32_t j) {
        Pair P;
        P.dx = min_image(__dsub_rn(xa, __ldg(A.x + j)), g.per[0], g.L[0], g.halfL[0]);
        P.dy = min_image(__dsub_rn(ya, __ldg(A.y + j)), g.per[1], g.L[1], g.halfL[1]);
        P.dz = min_image(__dsub_rn(za, __ldg(A.z + j)), g.per[2], g.L[2], g.halfL[2]);
        P.r2 = r2_exact(P.dx, P.dy, P.dz);
        P.hb = __ldg(A.h + j);
        P.self = (j == (uint32_t)i);
        P.in_g = P.r2 < sup_a;
        P.in_s = !P.self && (P.r2 < support2(fmax(ha, P.hb)));
        P.in_set = sym ? P.in_s : (P.in_g && !P.self);
        return P;
    };
    // does candidate j contribute anything to this sweep?  (the conditions of the pair terms below)
    auto contributes = [&](const Pair& P) {
        if (SWEEP == SW_DENSITY) return P.in_g;
        if (SWEEP == SW_HYDRO) return P.in_s && P.r2 > 0.0;
        if (SWEEP == SW_LIMITER || SWEEP == SW_GRADN || SWEEP == SW_KGC) return P.in_g && !P.self && P.r2 > 0.0;
        if (SWEEP == SW_APPLY) return P.in_set && P.r2 > 0.0;
        return true;
    };
    auto pair_term = [&](uint32_t j, const Pair& P) {
        const double dx = P.dx, dy = P.dy, dz = P.dz, r2 = P.r2, hb = P.hb;
        const bool self = P.self, in_g = P.in_g, in_s = P.in_s, in_set = P.in_set;
        (void)in_s; (void)in_set; (void)self; (void)hb; (void)dx; (void)dy; (void)dz;

            if (SWEEP == SW_DENSITY) {
                // eq. (35), self term included (A11)
                if (in_g) {
                    double q = sqrt(r2) * hinv;
                    acc0 += A.m[j] * shape_w<KERNEL>(q);
                    cnt += self ? 0u : 1u;
                }
            } else if (SWEEP == SW_HSEARCH) {
                // make neighbours mutual -- raise the search length of every a that I see but that may not see me
                if (in_g && !self && hb < ha)
                    atomicMax((unsigned long long*)(A.o0 + j), (unsigned long long)__double_as_longlong(ha));
            } else if (SWEEP == SW_COUNT) {
                cnt += in_set ? 1u : 0u;
            } else if (SWEEP == SW_LIST) {
                if (in_set) A.onbr[lbase + cnt++] = T.perm[j];
            } else if (SWEEP == SW_DIGEST) {
                if (in_set) { uint64_t hsh = mix64((uint64_t)T.perm[j]); dsum += hsh; dxr ^= hsh; }
            } else if (SWEEP == SW_HYDRO) {
                if (in_s && r2 > 0.0) {
                    const double r = sqrt(r2), rinv = 1.0 / r;
                    const double hbinv = 1.0 / hb;
                    const double Fa = Fn * shape_f<KERNEL>(r * hinv);
                    const double Fb = sigma<KERNEL>() * (hbinv * hbinv) * (hbinv * hbinv) * shape_f<KERNEL>(r * hbinv);
                    const double mb = A.m[j], rho_b = A.rho[j], p_b = A.p[j];
                    const double w = ((vxa - A.vx[j]) * dx + (vya - A.vy[j]) * dy + (vza - A.vz[j]) * dz) * rinv;
                    // eq. (11) P:L98 with the sign of eq. (5) (A3)
                    double coef = -(mb / (rho_a * rho_b)) * (p_a * Fa + p_b * Fb);
                    if (w < 0.0) {   // eqs. (41)-(43) P:L236-L242 (A6, A7, A8)
                        const double aw = -w;
                        const double vsa = ac_a + A.beta * aw;
                        const double vsb = A.alpha[j] * A.cs[j] + A.beta * aw;
                        coef += 0.5 * mb * (vsa * Fa / rho_a + vsb * Fb / rho_b) * w;
                        acc4 += 0.5 * mb * vsa * (w * w) * Fa;
                    }
                    const double cr = coef * rinv;
                    acc0 += cr * dx; acc1 += cr * dy; acc2 += cr * dz;
                    acc3 += (mb / rho_b) * w * Fa;      // eq. (37)
                }
            } else if (SWEEP == SW_LIMITER || SWEEP == SW_GRADN) {
                if (in_g && !self && r2 > 0.0) {
                    // eq. (9) phi = 1 with f = E (A19)
                    const double r = sqrt(r2);
                    const double cc = (A.m[j] / A.rho[j]) * (A.E[j] - E_a) * (Fn * shape_f<KERNEL>(r * hinv)) / r;
                    acc0 += cc * dx; acc1 += cc * dy; acc2 += cc * dz;
                }
            } else if (SWEEP == SW_KGC) {
                if (in_g && !self && r2 > 0.0) {
                    // eqs. (37), (39), (40) P:L213-L228: moment sums over N_gather(a), h_a only
                    const double r = sqrt(r2);
                    const double cc = (A.m[j] / A.rho[j]) * (Fn * shape_f<KERNEL>(r * hinv)) / r;
                    const double cx = cc * dx, cy = cc * dy, cz = cc * dz;
                    const double dvx = vxa - A.vx[j], dvy = vya - A.vy[j], dvz = vza - A.vz[j];
                    km[0] += cx * dx; km[1] += cx * dy; km[2] += cx * dz; km[3] += cy * dy; km[4] += cy * dz; km[5] += cz * dz;
                    kq[0] += dvx * cx; kq[1] += dvx * cy; kq[2] += dvx * cz;
                    kq[3] += dvy * cx; kq[4] += dvy * cy; kq[5] += dvy * cz;
                    kq[6] += dvz * cx; kq[7] += dvz * cy; kq[8] += dvz * cz;
                }
            } else if (SWEEP == SW_APPLY) {
                if (in_set && r2 > 0.0) {
                    // eq. (47) first term P:L270 on eq. (16); Fbar as P:L134 (A17)
                    const double r = sqrt(r2);
                    double Fbar = Fn * shape_f<KERNEL>(r * hinv);
                    if (sym) {
                        const double hbinv = 1.0 / hb;
                        Fbar = 0.5 * (Fbar + sigma<KERNEL>() * (hbinv * hbinv) * (hbinv * hbinv) * shape_f<KERNEL>(r * hbinv));
                    }
                    const double mu_b = A.mu[j], E_b = A.E[j];
                    const double cab = (A.m[j] / A.rho[j]) * (4.0 * mu_a * mu_b / (mu_a + mu_b)) * (Fbar / r);
                    acc0 += cab * (E_a - E_b);
                    acc1 += cab;
                    acc2 -= cab * E_b;
                }
            }
    };
    // One warp per particle: the lanes test 32 candidates at a time and QUEUE the contributing ones (ballot compaction into
    // a per-warp shared-memory queue, in candidate order: deterministic); a pair term is evaluated only when 32 are waiting,
    // so its long fp64 body (divisions, square roots) runs with every lane busy instead of the few per cent that hit.
    constexpr bool QUEUED = WARP && (SWEEP == SW_DENSITY || SWEEP == SW_HYDRO || SWEEP == SW_LIMITER || SWEEP == SW_GRADN ||
                                     SWEEP == SW_KGC || SWEEP == SW_APPLY);
    __shared__ uint32_t s_queue[QUEUED ? REF_WARPS : 1][64];
    uint32_t* queue = s_queue[QUEUED ? (threadIdx.x >> 5) : 0];
    uint32_t qn = 0;
    const uint32_t lane = threadIdx.x & 31u;
    auto drain = [&](uint32_t count) {                                  // the first `count` (<= 32) queued candidates
        __syncwarp();
        const uint32_t j = queue[lane < count ? lane : 0u];
        const uint32_t moved = queue[32u + lane];
        if (lane < count) pair_term(j, geometry(j));
        __syncwarp();
        queue[lane] = moved;
        __syncwarp();
    };

    // does cell c (gap2 = squared distance bound between the target and the cell) have to be visited?
    auto cell_wanted = [&](uint32_t c, double gap2) {
        if (gap2 > reach2) return false;
        if (SWEEP == SW_HSEARCH && !(__ldg(T.cell_hmin + c) < ha)) return false;   // nobody in the cell has a smaller h
        if (sym) {
            // symmetric sets: b in N_sym(a) needs r < 2 max(h_a, h_b) <= 2 max(h_a, max h of b's cell), and r >= the gap
            const double rc = 2.0 * fmax(ha, __ldg(T.cell_hmax + c));
            if (gap2 > (rc * rc) * (1.0 + 1e-9)) return false;
        }
        return true;
    };
    // SW_HSEARCH, fp32 pre-test: a position carries a rounding of at most cmax 2^-24, so a distance r ~ 2 h_a is off by less than
    // 4 cmax 2^-24 and r^2 by the relative 4 cmax 2^-24 / h_a; four times that is allowed for (and the fp64 path is taken when
    // even this is not small, i.e. h tiny against the box)
    const float tolf = 16.0f * 5.97e-8f * A.f4_cmax / (float)ha;
    const bool use_f4 = SWEEP == SW_HSEARCH && !WARP && A.f4 != nullptr && tolf < 0.25f &&
                        fmax(fabs(xa), fmax(fabs(ya), fabs(za))) <= 2.0 * (double)A.f4_cmax;   // (a particle far outside an open box: fp64)
    const float xaf = (float)xa, yaf = (float)ya, zaf = (float)za, haf = (float)ha;
    const float supf = (float)sup_a * (1.0f + tolf) * 1.000001f;
    const float Lf[3] = {(float)g.L[0], (float)g.L[1], (float)g.L[2]}, hLf[3] = {(float)g.halfL[0], (float)g.halfL[1], (float)g.halfL[2]};
    if (WARP) {
        // The lanes take one cell ROW (fixed y, z; the cells of a row are consecutive ranges of sorted slots) each and cull
        // its cells in parallel -- the per-cell loads of the culling are then 32 wide instead of one dependent chain per
        // cell -- and leave the slot range from the first to the last cell wanted, per unwrapped piece of the row (two when
        // the x-span crosses a periodic face), in a per-warp list; the warp then runs through the listed ranges together.
        __shared__ uint2 s_ranges[REF_WARPS][64];
        __shared__ uint32_t s_rstart[REF_WARPS][64];
        uint2* ranges = s_ranges[threadIdx.x >> 5];
        uint32_t* rstart = s_rstart[threadIdx.x >> 5];
        const int nrows = sy.cnt * sz.cnt;
        for (int r0 = 0; r0 < nrows; r0 += 32) {
            uint2 ra = make_uint2(0u, 0u), rb = make_uint2(0u, 0u);
            const int r = r0 + (int)lane;
            if (r < nrows) {
                const int kz = r / sy.cnt, ky = r - kz * sy.cnt;
                const int czz = g.per[2] ? wrap_cell(sz.start + kz, g.nc[2]) : sz.start + kz;
                const int cyy = g.per[1] ? wrap_cell(sy.start + ky, g.nc[1]) : sy.start + ky;
                const double gyz2 = cell_gap2(sz.start + kz - cz, fcz, fullz, ez) + cell_gap2(sy.start + ky - cy, fcy, fully, ey);
                if (!(gyz2 > reach2)) {
                    const uint32_t crow = (uint32_t)((czz * g.nc[1] + cyy) * g.nc[0]);
                    int fa = -1, la = -1, fb = -1, lb = -1;              // first / last wanted cell of the two pieces (wrapped x index)
                    for (int kx = 0; kx < sx.cnt; ++kx) {
                        const int ox = sx.start + kx;
                        const int cxx = g.per[0] ? wrap_cell(ox, g.nc[0]) : ox;
                        if (!cell_wanted(crow + (uint32_t)cxx, gyz2 + cell_gap2(ox - cx, fcx, fullx, ex))) continue;
                        if (ox == cxx) { if (fa < 0) fa = cxx; la = cxx; }     // the piece inside [0, nc)
                        else { if (fb < 0) fb = cxx; lb = cxx; }               // the piece beyond a periodic face
                    }
                    if (fa >= 0) ra = make_uint2(__ldg(T.cell_start + crow + fa), __ldg(T.cell_end + crow + la));
                    if (fb >= 0) rb = make_uint2(__ldg(T.cell_start + crow + fb), __ldg(T.cell_end + crow + lb));
                }
            }
            const uint32_t ma = __ballot_sync(0xFFFFFFFFu, ra.y > ra.x), mb = __ballot_sync(0xFFFFFFFFu, rb.y > rb.x);
            const uint32_t lt = (1u << lane) - 1u;
            __syncwarp();
            if (ra.y > ra.x) ranges[__popc(ma & lt)] = ra;
            if (rb.y > rb.x) ranges[__popc(ma) + __popc(mb & lt)] = rb;
            const uint32_t nr = __popc(ma) + __popc(mb);
            __syncwarp();
            // The listed ranges are walked as ONE stream of candidates (exclusive prefix sums of their lengths; a lane finds
            // the range of its flat index by bisection), 128 candidates per step: short ranges -- a row of a fine grid holds a
            // few dozen particles -- would otherwise leave most lanes idle, and every step costs a full memory round trip.
            {
                const uint32_t l0 = lane < nr ? ranges[lane].y - ranges[lane].x : 0u;
                const uint32_t l1 = lane + 32u < nr ? ranges[lane + 32u].y - ranges[lane + 32u].x : 0u;
                uint32_t i0 = l0, i1 = l1;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const uint32_t v0 = __shfl_up_sync(0xFFFFFFFFu, i0, o), v1 = __shfl_up_sync(0xFFFFFFFFu, i1, o);
                    if ((int)lane >= o) { i0 += v0; i1 += v1; }
                }
                const uint32_t t0 = __shfl_sync(0xFFFFFFFFu, i0, 31), total = t0 + __shfl_sync(0xFFFFFFFFu, i1, 31);
                rstart[lane] = i0 - l0;
                rstart[lane + 32u] = t0 + i1 - l1;
                __syncwarp();
                auto candidate = [&](uint32_t fidx) {                   // flat index -> sorted slot
                    uint32_t lo = 0u, hi = nr;                          // largest q with rstart[q] <= fidx
                    while (hi - lo > 1u) {
                        const uint32_t mid = (lo + hi) >> 1;
                        if (rstart[mid] <= fidx) lo = mid; else hi = mid;
                    }
                    return ranges[lo].x + (fidx - rstart[lo]);
                };
                if (QUEUED) {
                    for (uint32_t f0 = 0; f0 < total; f0 += 128u) {
                        uint32_t jc[4];
                        bool hit[4];
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            const uint32_t fidx = f0 + 32u * e + lane;
                            hit[e] = false;
                            jc[e] = 0u;
                            if (fidx < total) { jc[e] = candidate(fidx); hit[e] = contributes(geometry(jc[e])); }
                        }
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            const uint32_t m = __ballot_sync(0xFFFFFFFFu, hit[e]);
                            if (hit[e]) queue[qn + __popc(m & lt)] = jc[e];
                            qn += __popc(m);
                            if (qn >= 32u) { drain(32u); qn -= 32u; }
                        }
                    }
                } else {
                    for (uint32_t fidx = lane; fidx < total; fidx += 32u) { const uint32_t j = candidate(fidx); pair_term(j, geometry(j)); }
                }
                __syncwarp();
            }
        }
    } else {
        for (int kz = 0; kz < sz.cnt; ++kz) {
            const int czz = g.per[2] ? wrap_cell(sz.start + kz, g.nc[2]) : sz.start + kz;
            const double gz2 = cell_gap2(sz.start + kz - cz, fcz, fullz, ez);
            if (gz2 > reach2) continue;
            for (int ky = 0; ky < sy.cnt; ++ky) {
                const int cyy = g.per[1] ? wrap_cell(sy.start + ky, g.nc[1]) : sy.start + ky;
                const double gyz2 = gz2 + cell_gap2(sy.start + ky - cy, fcy, fully, ey);
                if (gyz2 > reach2) continue;
                for (int kx = 0; kx < sx.cnt; ++kx) {
                    const int cxx = g.per[0] ? wrap_cell(sx.start + kx, g.nc[0]) : sx.start + kx;
                    const double gap2 = gyz2 + cell_gap2(sx.start + kx - cx, fcx, fullx, ex);
                    const uint32_t c = (uint32_t)((czz * g.nc[1] + cyy) * g.nc[0] + cxx);
                    if (!cell_wanted(c, gap2)) continue;
                    const uint32_t jb = __ldg(T.cell_start + c), je = __ldg(T.cell_end + c);
                    if (SWEEP == SW_HSEARCH && use_f4) {
                        // pre-test in fp32 (one 16-byte load per candidate instead of four 8-byte ones): only a candidate that
                        // cannot be excluded -- h_b > h_a even after rounding, or farther than the support widened by the
                        // rounding bound -- is looked at in fp64.  The widened test can only add to the particles raised: the
                        // search length is an upper bound by nature (it bounds a search range and picks a level).
                        for (uint32_t j = jb; j < je; ++j) {
                            const float4 b = __ldg(A.f4 + j);
                            if (b.w > haf) continue;
                            float dx = xaf - b.x, dy = yaf - b.y, dz = zaf - b.z;
                            if (g.per[0]) { if (dx > hLf[0]) dx -= Lf[0]; else if (dx < -hLf[0]) dx += Lf[0]; }
                            if (g.per[1]) { if (dy > hLf[1]) dy -= Lf[1]; else if (dy < -hLf[1]) dy += Lf[1]; }
                            if (g.per[2]) { if (dz > hLf[2]) dz -= Lf[2]; else if (dz < -hLf[2]) dz += Lf[2]; }
                            if (fmaf(dz, dz, fmaf(dy, dy, dx * dx)) > supf) continue;
                            if (__ldg(A.h + j) < ha) atomicMax((unsigned long long*)(A.o0 + j), (unsigned long long)__double_as_longlong(ha));
                        }
                    } else {
                        for (uint32_t j = jb; j < je; ++j) pair_term(j, geometry(j));
                    }
                }
            }
        }

    }

    if (QUEUED && qn) drain(qn);
    if (WARP) {
        acc0 = warp_add(acc0); acc1 = warp_add(acc1); acc2 = warp_add(acc2); acc3 = warp_add(acc3); acc4 = warp_add(acc4);
        cnt = warp_add(cnt);
        if (SWEEP == SW_DIGEST) {
            dsum = warp_add(dsum);
#pragma unroll
            for (int o = 16; o; o >>= 1) dxr ^= __shfl_xor_sync(0xFFFFFFFFu, dxr, o);
        }
        if (SWEEP == SW_KGC) {
#pragma unroll
            for (int e = 0; e < 6; ++e) km[e] = warp_add(km[e]);
#pragma unroll
            for (int e = 0; e < 9; ++e) kq[e] = warp_add(kq[e]);
        }
        if ((threadIdx.x & 31u) != 0u) return;
    }
    if (SWEEP == SW_DENSITY) {
        A.o0[ia] = Wn * acc0;
        if (A.ocount) A.ocount[ia] = cnt;
    } else if (SWEEP == SW_COUNT) {
        A.ocount[ia] = cnt;
    } else if (SWEEP == SW_DIGEST) {
        A.odsum[ia] = dsum; A.odxor[ia] = dxr;
    } else if (SWEEP == SW_LIST) {
        // ascending caller ids (debug export: insertion sort of this particle's segment)
        uint32_t* L = A.onbr + lbase;
        for (uint32_t a = 1; a < cnt; ++a) {
            uint32_t v = L[a]; int b = (int)a - 1;
            while (b >= 0 && L[b] > v) { L[b + 1] = L[b]; --b; }
            L[b + 1] = v;
        }
    } else if (SWEEP == SW_HYDRO) {
        A.o0[ia] = acc0; A.o1[ia] = acc1; A.o2[ia] = acc2;
        A.o3[ia] = (p_a / rho_a) * acc3 - acc4 / rho_a;       // eq. (17) 1st term P:L129 + eq. (42)
        if (A.o4) A.o4[ia] = acc3;
    } else if (SWEEP == SW_LIMITER) {
        // Larsen limiter, k = 2 (A20)
        const double rk = A.rho[i] * A.kappa[i];
        const double gn = sqrt(acc0 * acc0 + acc1 * acc1 + acc2 * acc2);
        const double R = gn / (rk * E_a);
        const double mu = A.c_light * (1.0 / sqrt(9.0 + R * R)) / rk;
        A.o0[ia] = mu;
        A.mu_sorted[i] = mu;
        if (A.me_sorted) A.me_sorted[i] = make_double2(mu, E_a);
        if (A.o1) { A.o1[ia] = acc0; A.o1[n + ia] = acc1; A.o1[2 * n + ia] = acc2; }
    } else if (SWEEP == SW_GRADN) {
        A.me_sorted[i] = make_double2(acc0, acc1);
        A.g2_sorted[i] = make_double2(acc2, A.mu[i]);   // (G_z, kappa^ib)
        if (A.o1) { A.o1[ia] = acc0; A.o1[n + ia] = acc1; A.o1[2 * n + ia] = acc2; }
    } else if (SWEEP == SW_APPLY) {
        A.o0[ia] = acc0;
        if (A.o1) A.o1[ia] = acc1;
        if (A.o2) A.o2[ia] = acc2;
    } else if (SWEEP == SW_KGC) {
        // M_a = -sum c x (x) x, L_a = M_a^-1 by cofactors; singular -> L_a = I (A28)
        const double m00 = -km[0], m01 = -km[1], m02 = -km[2], m11 = -km[3], m12 = -km[4], m22 = -km[5];
        const double c00 = m11 * m22 - m12 * m12, c01 = m02 * m12 - m01 * m22, c02 = m01 * m12 - m02 * m11;
        const double det = m00 * c00 + m01 * c01 + m02 * c02;
        double l00 = 1.0, l01 = 0.0, l02 = 0.0, l11 = 1.0, l12 = 0.0, l22 = 1.0;
        if (fabs(det) > 1e-12) {
            const double id = 1.0 / det;
            l00 = c00 * id; l01 = c01 * id; l02 = c02 * id;
            l11 = (m00 * m22 - m02 * m02) * id; l12 = (m01 * m02 - m00 * m12) * id; l22 = (m00 * m11 - m01 * m01) * id;
        }
        const double corr = l00 * kq[0] + l11 * kq[4] + l22 * kq[8] + l01 * (kq[1] + kq[3]) + l02 * (kq[2] + kq[6]) + l12 * (kq[5] + kq[7]);
        A.o0[ia] = rho_a * corr;
        if (A.o1) {
            double* Lo = A.o1 + ia;
            Lo[0] = l00; Lo[n] = l01; Lo[2 * n] = l02; Lo[3 * n] = l01; Lo[4 * n] = l11; Lo[5 * n] = l12;
            Lo[6 * n] = l02; Lo[7 * n] = l12; Lo[8 * n] = l22;
        }
        if (A.o2) A.o2[ia] = rho_a * (kq[0] + kq[4] + kq[8]);
    }
}

// Grid-stride over the particles with a bounded grid: when the tiled kernels served every particle (the usual
// case) the launch costs a few microseconds instead of n/128 empty blocks.
template <int SWEEP, int KERNEL>
__global__ void __launch_bounds__(REF_THREADS)
k_ref_sweep(DevGrid g, int64_t n, CellTabs T, SweepArgs A) {
    if (A.nfast && *A.nfast == (unsigned long long)n) return;   // the tiled kernels serve every particle
    if (A.left) {                                               // the rest, compacted: one warp per particle (SW_LIST: one thread)
        const int64_t nl = (int64_t)*A.nleft;
        if (SWEEP == SW_LIST) {
            for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < nl; t += (int64_t)gridDim.x * blockDim.x)
                ref_particle<SWEEP, KERNEL, false>(g, n, T, A, (int64_t)A.left[t]);
        } else {
            const int64_t nw = ((int64_t)gridDim.x * blockDim.x) >> 5;
            for (int64_t t = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5; t < nl; t += nw)
                ref_particle<SWEEP, KERNEL, true>(g, n, T, A, (int64_t)A.left[t]);
        }
        return;
    }
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        ref_particle<SWEEP, KERNEL, false>(g, n, T, A, i);
}

template <int SWEEP>
static cudaError_t launch_k(Ctx* c, const SweepArgs& a, cudaStream_t st) {
    if (c->n == 0) return cudaSuccess;
    CellTabs T{c->sorted_key, c->perm, c->cell_start, c->cell_end, c->hglob, c->cell_hmin, c->is_level ? 1 : 0, c->cell_hmax};
    const int64_t want = (c->n + REF_THREADS - 1) / REF_THREADS;
    const int blocks = (int)(want < 148 * 64 ? want : 148 * 64);
    if (c->kernel == SPRAY_KERNEL_WENDLAND_C2) k_ref_sweep<SWEEP, 1><<<blocks, REF_THREADS, 0, st>>>(c->dg, c->n, T, a);
    else k_ref_sweep<SWEEP, 0><<<blocks, REF_THREADS, 0, st>>>(c->dg, c->n, T, a);
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_ref_sweep(Ctx* c, int sweep, const SweepArgs& a, cudaStream_t st) {
    switch (sweep) {
        case SW_DENSITY: return launch_k<SW_DENSITY>(c, a, st);
        case SW_HYDRO: return launch_k<SW_HYDRO>(c, a, st);
        case SW_LIMITER: return launch_k<SW_LIMITER>(c, a, st);
        case SW_APPLY: return launch_k<SW_APPLY>(c, a, st);
        case SW_HSEARCH: return launch_k<SW_HSEARCH>(c, a, st);
        case SW_COUNT: return launch_k<SW_COUNT>(c, a, st);
        case SW_LIST: return launch_k<SW_LIST>(c, a, st);
        case SW_DIGEST: return launch_k<SW_DIGEST>(c, a, st);
        case SW_KGC: return launch_k<SW_KGC>(c, a, st);
        case SW_GRADN: return launch_k<SW_GRADN>(c, a, st);
    }
    return cudaErrorInvalidValue;
}

}  // namespace spray
