// ray.cu -- row N4: mesh-free laser ray tracing and inverse-bremsstrahlung deposition,
// PAPER.md section 2.5.  "Each ray is treated as a particle": position x, velocity v, power P.
//
// One WARP per ray (rays are independent).  Per step of the fixed dt the warp
//   (i)   finds the cells that can hold a particle a with |x - x_a| < 2 h_a: the cell table of the last
//         spray_build_cells, reach 2 max(h) (device scalar hglob[1]), rows (cy, cz) culled by their distance to the ray
//         and the x-range of a row narrowed to the chord of the reach sphere; after the sort the cells of a row are
//         one contiguous range of sorted slots (two when the range wraps in a periodic box);
//   (ii)  numbers the candidates of up to 32 rows consecutively (one lane per row reads the cell table, warp scan) and
//         strides its 32 lanes over that numbering: 16-byte records (x,y) (z,h) for the test r^2 < 4 h_a^2 in the contract
//         form (common.cuh), and for the accepted ones (z,V) (G_x,G_y) (G_z,kappa^ib) -- the last two written by the
//         SW_GRADN sweep -- to accumulate  G(x) = sum V_a G_a W,  kappa(x) = sum V_a kib_a W,  wsum = sum V_a W
//         (standard SPH interpolation with the particles' own h; reading A30);
//   (iii) compacts the accepted candidates into a per-warp hit list (slot, r^2) in shared memory and evaluates that list
//         densely (all lanes busy with accepted particles, their four records loaded together), reduces the five sums with
//         a shuffle butterfly (every lane ends with the same bits), and every lane advances the ray redundantly:
//         v <- v - (c^2/2) G dt (eq. (72)), ds = |v| dt, dE = P (1 - exp(-kappa ds)) (eq. (71)), P <- P - dE,
//         x <- x + v dt (semi-implicit Euler, A31), periodic wrap / exit test (A34);
//   (iv)  deposits dE w_a / wsum ("based on the kernel weight", A33) with fp64 atomics into a SORTED-order
//         accumulator (neighbouring rays hit neighbouring slots), from the hit list -- or by a second traversal in the
//         rare step whose support holds more than RAY_CAP particles.
// The atomics make the deposit's summation order, hence its last bits, vary from run to run.
#include "spray_internal.h"

namespace spray {

constexpr int RAY_WARPS = 4;        // rays per CTA
constexpr int RAY_CAP = 320;        // cached (slot, weight) pairs per ray and step
#ifndef RAY_MINB
#define RAY_MINB 6    // CTAs per SM the register budget is set for (80 registers): 8 -> 33.1 ms, 6 -> 31.7 ms, 4 (128 registers) -> 39.2 ms at c5
#endif

struct RayIn {
    const double2 *p0, *p1, *s0, *gA, *gB;      // sorted records: (x,y) (z,h) (z,V) (G_x,G_y) (G_z,kappa^ib)
    const uint32_t *cell_start, *cell_end;
    const double* hglob;                        // [1] = max h over the particles
};

struct RSpan { int start, cnt; bool all; };     // cells start .. start+cnt-1 (unwrapped when periodic); all: every cell of the dimension

// cells of dimension d that intersect [pd - reach, pd + reach]
__device__ __forceinline__ RSpan ray_span(const DevGrid& g, int d, double pd, double reach) {
    const int nc = g.nc[d];
    double a = (pd - reach - g.lo[d]) * g.inv[d] - 1e-9, b = (pd + reach - g.lo[d]) * g.inv[d] + 1e-9;
    RSpan s;
    s.all = false;
    if (g.per[d]) {
        if (!(b - a < (double)(nc - 1)) || !(fabs(a) < 1.0e9)) { s.start = 0; s.cnt = nc; s.all = true; return s; }
        const int ia = (int)floor(a), ib = (int)floor(b);
        s.start = ia; s.cnt = ib - ia + 1;
        if (s.cnt >= nc) { s.start = 0; s.cnt = nc; s.all = true; }
    } else {
        // particles outside the box sit in the edge cells (clamped keys): clamp the span instead of dropping it
        a = fmin(fmax(a, 0.0), (double)(nc - 1)); b = fmin(fmax(b, 0.0), (double)(nc - 1));
        if (!(a == a)) { a = 0.0; b = (double)(nc - 1); }
        const int ia = (int)floor(a), ib = (int)floor(b);
        s.start = ia; s.cnt = ib - ia + 1;
        s.all = (s.cnt == nc);
    }
    return s;
}
// distance from pd to the slab of (unwrapped) cell cu in dimension d; edge cells of an open dimension are unbounded
__device__ __forceinline__ double slab_dist(const DevGrid& g, int d, int cu, double pd, bool all) {
    if (all && g.per[d]) return 0.0;            // every cell visited: the unwrapped index is not the nearest image
    const double w = g.L[d] / (double)g.nc[d];
    const double lo = g.lo[d] + (double)cu * w, hi = lo + w;
    double dist = 0.0;
    if (pd < lo && (g.per[d] || cu > 0)) dist = lo - pd;
    else if (pd > hi && (g.per[d] || cu < g.nc[d] - 1)) dist = pd - hi;
    return dist * (1.0 - 1e-9);
}
__device__ __forceinline__ int wrap_mod(int c, int nc) { c %= nc; return c < 0 ? c + nc : c; }

struct RaySums { double gx, gy, gz, kap, wsum; };

// Per-warp table of the rows of one chunk (32 rows, one per lane): up to two contiguous pieces of sorted slots per row and
// the row's offset in the chunk's flattened candidate numbering.
struct RowTab {
    uint32_t jb0[32], len0[32], jb1[32], off[33];
};

// Dense evaluation of a hit list (slot, r^2): lanes stride over it, the four records of a hit are loaded together.
// PASS 0: w_a = V_a W(r; h_a) replaces r^2 in the list and the interpolation sums are accumulated.
// PASS 1: deposit sc * w_a (second traversal of a step whose hits did not fit one list).
template <int KERNEL, int PASS>
__device__ __forceinline__ void ray_eval(const RayIn& A, int lane, uint32_t cnt, const uint32_t* __restrict__ c_idx, double* __restrict__ c_w,
                                         RaySums& S, double sc, double* __restrict__ dep) {
    __syncwarp();
    for (uint32_t t = lane; t < cnt; t += 32) {
        const uint32_t j = c_idx[t];
        const double r2 = c_w[t];
        const double ha = __ldg(A.p1 + j).y, V = __ldg(A.s0 + j).y;
        const double hinv = 1.0 / ha;
        const double wa = V * ((sigma<KERNEL>() * hinv * hinv * hinv) * shape_w<KERNEL>(sqrt(r2) * hinv));
        if (PASS == 0) {
            const double2 ga = __ldg(A.gA + j), gb = __ldg(A.gB + j);
            S.gx = fma(wa, ga.x, S.gx); S.gy = fma(wa, ga.y, S.gy); S.gz = fma(wa, gb.x, S.gz);
            S.kap = fma(wa, gb.y, S.kap);
            S.wsum += wa;
            c_w[t] = wa;
        } else {
            if (wa != 0.0) atomicAdd(dep + j, sc * wa);
        }
    }
    __syncwarp();
}

// One traversal of the particles around the ray at (px, py, pz): tests every candidate and compacts the accepted ones into
// the hit list (slot, r^2); returns the number of hits left in the list for the caller to evaluate (ray_eval).  When the list
// fills up it is evaluated on the spot and `overflow` is set: the list then no longer holds the whole step, and the
// deposit needs a second traversal (PASS 1, which evaluates with the deposit scale sc instead of accumulating).
// The rows (cy, cz) in reach are taken 32 at a time: lane l works out the slot ranges of row l (cell-table reads of all
// rows in flight together), a warp scan numbers the candidates of the chunk consecutively, and the lanes then stride over
// that numbering, so all 32 lanes stay busy whatever the row lengths, with the next candidate's records loaded before the
// current one is evaluated.
template <int KERNEL, int PASS>
__device__ __forceinline__ uint32_t ray_visit(const DevGrid& g, const RayIn& A, double px, double py, double pz, double reach, int lane,
                                              RaySums& S, RowTab& RT, uint32_t* __restrict__ c_idx, double* __restrict__ c_w, double sc,
                                              double* __restrict__ dep, bool& overflow) {
    uint32_t cnt = 0;
    const double reach2 = reach * reach;
    const RSpan sy = ray_span(g, 1, py, reach), sz = ray_span(g, 2, pz, reach);
    const int nrows = sy.cnt * sz.cnt;
    for (int r0 = 0; r0 < nrows; r0 += 32) {
        // ---- this lane's row
        uint32_t jb0 = 0, len0 = 0, jb1 = 0, len1 = 0;
        const int rr = r0 + lane;
        if (rr < nrows) {
            const int kz = rr / sy.cnt, ky = rr - kz * sy.cnt;
            const int czu = sz.start + kz, cyu = sy.start + ky;
            const double dz0 = slab_dist(g, 2, czu, pz, sz.all), dy0 = slab_dist(g, 1, cyu, py, sy.all);
            const double rem = reach2 - (dy0 * dy0 + dz0 * dz0);
            if (rem > 0.0) {                                   // else the row is out of reach
                const int czz = g.per[2] ? wrap_mod(czu, g.nc[2]) : czu;
                const int cyy = g.per[1] ? wrap_mod(cyu, g.nc[1]) : cyu;
                const RSpan sx = ray_span(g, 0, px, sqrt(rem));
                const uint32_t row = (uint32_t)((czz * g.nc[1] + cyy) * g.nc[0]);
                const int c0 = g.per[0] ? wrap_mod(sx.start, g.nc[0]) : sx.start;
                const int take = min(sx.cnt, g.nc[0] - c0);
                jb0 = __ldg(A.cell_start + row + c0);
                len0 = __ldg(A.cell_end + row + c0 + take - 1) - jb0;
                if (take < sx.cnt) {                           // the range wraps: second piece from column 0
                    jb1 = __ldg(A.cell_start + row);
                    len1 = __ldg(A.cell_end + row + (sx.cnt - take) - 1) - jb1;
                }
            }
        }
        // ---- number the candidates of the chunk
        const uint32_t len = len0 + len1;
        uint32_t inc = len;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t v = __shfl_up_sync(0xFFFFFFFFu, inc, o);
            if (lane >= o) inc += v;
        }
        const uint32_t total = __shfl_sync(0xFFFFFFFFu, inc, 31);
        __syncwarp();
        RT.jb0[lane] = jb0; RT.len0[lane] = len0; RT.jb1[lane] = jb1; RT.off[lane] = inc - len;
        if (lane == 31) RT.off[32] = total;
        __syncwarp();
        // ---- stride over them: the test only (contract predicate); accepted candidates are compacted into the hit list
        int row = 0;
        auto slot_of = [&](uint32_t t) -> uint32_t {
            while (RT.off[row + 1] <= t) ++row;                // t < total = off[32]: terminates; rows of length 0 are skipped
            const uint32_t k = t - RT.off[row], l0 = RT.len0[row];
            return k < l0 ? RT.jb0[row] + k : RT.jb1[row] + (k - l0);
        };
        uint32_t j = 0;
        double2 a0 = make_double2(0.0, 0.0), a1 = a0;
        if ((uint32_t)lane < total) { j = slot_of(lane); a0 = __ldg(A.p0 + j); a1 = __ldg(A.p1 + j); }
        for (uint32_t base = 0; base < total; base += 32) {
            const uint32_t t = base + lane;
            const uint32_t jc = j;
            const double2 b0 = a0, b1 = a1;
            if (t + 32 < total) { j = slot_of(t + 32); a0 = __ldg(A.p0 + j); a1 = __ldg(A.p1 + j); }
            bool hit = false;
            double r2 = 0.0;
            if (t < total) {
                const double dx = min_image(__dsub_rn(px, b0.x), g.per[0], g.L[0], g.halfL[0]);
                const double dy = min_image(__dsub_rn(py, b0.y), g.per[1], g.L[1], g.halfL[1]);
                const double dz = min_image(__dsub_rn(pz, b1.x), g.per[2], g.L[2], g.halfL[2]);
                r2 = r2_exact(dx, dy, dz);
                hit = r2 < support2(b1.y);
            }
            if (cnt > (uint32_t)(RAY_CAP - 32)) {              // warp-uniform: the list may not take 32 more -- evaluate it now
                ray_eval<KERNEL, PASS>(A, lane, cnt, c_idx, c_w, S, sc, dep);
                overflow = true;
                cnt = 0;
            }
            const uint32_t mask = __ballot_sync(0xFFFFFFFFu, hit);
            if (hit) {
                const uint32_t pos = cnt + __popc(mask & ((1u << lane) - 1u));
                c_idx[pos] = jc; c_w[pos] = r2;
            }
            cnt += __popc(mask);
        }
    }
    return cnt;
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
    return v;
}

template <int KERNEL>
__global__ void __launch_bounds__(32 * RAY_WARPS, RAY_MINB)
k_ray_trace(DevGrid g, RayIn A, RayArgs R) {
    __shared__ uint32_t s_idx[RAY_WARPS][RAY_CAP];
    __shared__ double s_w[RAY_WARPS][RAY_CAP];
    __shared__ RowTab s_rt[RAY_WARPS];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t q = (int64_t)blockIdx.x * RAY_WARPS + warp;
    if (q >= R.nrays) return;                                   // warp-uniform; no CTA-wide barrier below
    const int64_t nr = R.nrays;
    double p[3] = {R.rays_in[q], R.rays_in[nr + q], R.rays_in[2 * nr + q]};
    double v[3] = {R.rays_in[3 * nr + q], R.rays_in[4 * nr + q], R.rays_in[5 * nr + q]};
    double P = R.rays_in[6 * nr + q];
    const double reach = 2.0 * A.hglob[1];
    const double acc = -0.5 * R.c_light * R.c_light * R.dt;
    uint32_t* c_idx = s_idx[warp];
    double* c_w = s_w[warp];
    int64_t k = 0;
    for (; k < R.nsteps && P > R.pmin; ++k) {
        RaySums S{0.0, 0.0, 0.0, 0.0, 0.0};
        bool overflow = false;
        const uint32_t cnt = ray_visit<KERNEL, 0>(g, A, p[0], p[1], p[2], reach, lane, S, s_rt[warp], c_idx, c_w, 0.0, nullptr, overflow);
        ray_eval<KERNEL, 0>(A, lane, cnt, c_idx, c_w, S, 0.0, nullptr);
        S.gx = warp_sum(S.gx); S.gy = warp_sum(S.gy); S.gz = warp_sum(S.gz); S.kap = warp_sum(S.kap); S.wsum = warp_sum(S.wsum);
        // eq. (72), then the track length of this step with the new v (A31)
        v[0] = fma(acc, S.gx, v[0]); v[1] = fma(acc, S.gy, v[1]); v[2] = fma(acc, S.gz, v[2]);
        const double ds = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]) * R.dt;
        if (S.wsum > 0.0) {
            const double dE = P * (1.0 - exp(-S.kap * ds));     // eq. (71), kappa held over the step (A32)
            P -= dE;
            const double sc = dE / S.wsum;                      // normalised kernel weights (A33)
            if (!overflow) {
                for (uint32_t t = lane; t < cnt; t += 32) {
                    const double wa = c_w[t];
                    if (wa != 0.0) atomicAdd(R.dep_sorted + c_idx[t], sc * wa);
                }
                __syncwarp();
            } else {
                RaySums dummy{};
                bool o2 = false;
                const uint32_t c2 = ray_visit<KERNEL, 1>(g, A, p[0], p[1], p[2], reach, lane, dummy, s_rt[warp], c_idx, c_w, sc, R.dep_sorted, o2);
                ray_eval<KERNEL, 1>(A, lane, c2, c_idx, c_w, dummy, sc, R.dep_sorted);
            }
        }
        bool out = false;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            p[d] = fma(v[d], R.dt, p[d]);
            if (g.per[d]) {
                const double hi = g.lo[d] + g.L[d];
                if (p[d] < g.lo[d]) p[d] += g.L[d]; else if (p[d] >= hi) p[d] -= g.L[d];
            } else if (p[d] < g.lo[d] || p[d] >= g.lo[d] + g.L[d]) out = true;
        }
        if (out) { ++k; break; }
    }
    if (lane == 0) {
#pragma unroll
        for (int d = 0; d < 3; ++d) { R.rays_out[d * nr + q] = p[d]; R.rays_out[(3 + d) * nr + q] = v[d]; }
        R.rays_out[6 * nr + q] = P;
        if (R.steps_out) R.steps_out[q] = k;
    }
}

__global__ void k_unsort(const double* __restrict__ sorted, const uint32_t* __restrict__ perm, int64_t n, double* __restrict__ caller) {
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i < n) caller[perm[i]] = sorted[i];
}

cudaError_t launch_ray_trace(Ctx* c, const RayArgs& a, cudaStream_t st) {
    if (a.nrays == 0) return cudaSuccess;
    RayIn in{c->pk.p0, c->pk.p1, c->pk.s[0], c->pk.s[1], c->pk.s[2], c->cell_start, c->cell_end, c->hglob};
    const int64_t blocks = (a.nrays + RAY_WARPS - 1) / RAY_WARPS;
    if (blocks > 0x7FFFFFFFll) return cudaErrorInvalidValue;
    if (c->kernel == SPRAY_KERNEL_WENDLAND_C2) k_ray_trace<1><<<(unsigned)blocks, 32 * RAY_WARPS, 0, st>>>(c->dg, in, a);
    else k_ray_trace<0><<<(unsigned)blocks, 32 * RAY_WARPS, 0, st>>>(c->dg, in, a);
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_unsort(Ctx* c, const double* sorted, double* caller, cudaStream_t st) {
    if (c->n == 0) return cudaSuccess;
    k_unsort<<<(unsigned)((c->n + 255) / 256), 256, 0, st>>>(sorted, c->perm, c->n, caller);
    c->launches += 1;
    return cudaGetLastError();
}

}  // namespace spray
