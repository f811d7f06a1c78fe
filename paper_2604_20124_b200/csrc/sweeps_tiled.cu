// sweeps_tiled.cu -- the tiled pair kernels: density (eq. (35)), hydro RHS (eqs. (11), (17), (37), (41)-(43)),
// FLD limiter pre-sweep (eq. (9)) and FLD operator apply (eqs. (16), (47), (51)-(52)) of PAPER.md.
//
// One persistent CTA of 512 threads per SM walks the tiles of tiles.cuh.  Per tile it stages the candidate
// particles' fields as 16-byte records (two fp64 fields each, positions moved to the periodic image next to the
// tile) into shared memory; then two threads share ONE target particle, each running down its scheduled half-list
// (u16 slots, tiles.cu): no distance test on rejected candidates, all 32 lanes busy with accepted pairs, one
// 128-bit shared-memory load per record with the 8 lanes of a wavefront mostly in 8 different banks, one
// reciprocal square root per pair (MUFU.RSQ64H seed + Newton), per-particle factors hoisted into the prologue
// kernels, kernel normalisations hoisted out of the pair loop where h is uniform over the tile.  Results are
// written to caller order through the sort permutation.  No floating-point atomics: each half-list is summed in
// list order and the two halves are added by a shuffle, so results are bitwise reproducible.
#include "spray_internal.h"
#include "tiles.cuh"

#ifndef SPRAY_NEWTON_ORDER
#define SPRAY_NEWTON_ORDER 3
#endif

namespace spray {

// 1/sqrt(x) for normal positive x: hardware seed and one Newton step of order SPRAY_NEWTON_ORDER
// (2: y (1 + e/2); 3: y (1 + e/2 + 3 e^2/8)), e = 1 - x y^2.
__device__ __forceinline__ double rsqrt_fast(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double t = x * y;
    const double e = fma(-t, y, 1.0);
#if SPRAY_NEWTON_ORDER == 2
    return fma(0.5 * y, e, y);
#else
    const double p = fma(0.375, e, 0.5);
    return fma(y * e, p, y);
#endif
}
// 1/x for normal positive x: hardware seed and one step y (1 + e [+ e^2]), e = 1 - x y.
__device__ __forceinline__ double rcp_fast(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x, y, 1.0);
#if SPRAY_NEWTON_ORDER == 2
    return fma(y, e, y);
#else
    return fma(y, fma(e, e, e), y);
#endif
}

// 16- and 8-byte asynchronous global -> shared copies (LDGSTS)
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"((uint32_t)__cvta_generic_to_shared(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async8(void* smem_dst, const void* gsrc) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" :: "r"((uint32_t)__cvta_generic_to_shared(smem_dst)), "l"(gsrc) : "memory");
}

// Rescaled shape functions (common.cuh): W = kWn / h^3 * wshape(q), F = dW/dr = kFn / h^4 * gshape(q).
// CLAMP = false is used where every listed pair is known to be inside the support (uniform h over the tile):
// rounding can then leave 2 - q at -1e-13 at worst, which contributes nothing at the tolerance of the pass.
template <int KERNEL, bool CLAMP>
__device__ __forceinline__ double wshape(double q) {
    if (KERNEL == 1) {                       // Wendland C2, eq. (3): (1-q/2)^4 (2q+1)
        double t = fma(-0.5, q, 1.0);
        if (CLAMP) t = dmax0_fast(t);
        const double t2 = t * t;
        return (t2 * t2) * fma(2.0, q, 1.0);
    } else {                                 // cubic spline (A1): (2-q)^3 - 4 (1-q)_+^3
        constexpr double C = 1.5874010519681994748;      // cbrt(4)
        double t2 = 2.0 - q;
        if (CLAMP) t2 = dmax0_fast(t2);
        const double t1 = dmax0_fast(fma(-C, q, C));
        return fma(t2 * t2, t2, -((t1 * t1) * t1));
    }
}
template <int KERNEL, bool CLAMP>
__device__ __forceinline__ double gshape(double q) {
    if (KERNEL == 1) {                       // q (1-q/2)^3
        double t = fma(-0.5, q, 1.0);
        if (CLAMP) t = dmax0_fast(t);
        return (q * t) * (t * t);
    } else {                                 // (2-2q)_+^2 - (2-q)^2
        double t2 = 2.0 - q;
        if (CLAMP) t2 = dmax0_fast(t2);
        const double s1 = dmax0_fast(fma(-2.0, q, 2.0));
        return fma(s1, s1, -(t2 * t2));
    }
}
template <int KERNEL> __device__ __forceinline__ double wn_k() { return KERNEL == 1 ? kWnWend : kWnCubic; }
template <int KERNEL> __device__ __forceinline__ double w0_k() { return KERNEL == 1 ? 1.0 : 4.0; }   // wshape(0)

// Records staged per candidate (16 bytes each) and extra fp64 arrays
template <int SWEEP> struct NRec;
template <> struct NRec<SW_DENSITY> { static constexpr int v = 2, e = 0; };   // (x,y) (z,m)
template <> struct NRec<SW_HYDRO> { static constexpr int v = 6, e = 0; };     // (x,y) (z,V) (Q,vx) (vy,vz) (m,alpha c) (1/h,Fn)
template <> struct NRec<SW_LIMITER> { static constexpr int v = 2, e = 1; };   // (x,y) (z,V) | E
template <> struct NRec<SW_APPLY> { static constexpr int v = 4, e = 0; };     // (x,y) (z,V) (mu,E) (1/h,Fn)
template <> struct NRec<SW_KGC> { static constexpr int v = 4, e = 0; };       // (x,y) (z,V) (vx,vy) (vz,-)
template <> struct NRec<SW_GRADN> { static constexpr int v = 2, e = 1; };     // (x,y) (z,V) | f = n_e/n_c   (row N4)
// hydro RHS + FLD limiter sum in one sweep (spray_hydro_rhs_limiter): the hydro records and the limiter's E.  Launched on
// uniform-h tiles only (MODE 1: no (1/h,Fn) record, 5 records + E = 197 KB); there N_gather = N_sym, so both sums walk the same list.
template <> struct NRec<SW_HYDLIM> { static constexpr int v = 6, e = 1; };    // (x,y) (z,V) (Q,vx) (vy,vz) (m,alpha c) (1/h,Fn) | E

struct SweepIn {
    const double2* rec[6];           // sorted global records, in the order of NRec
    const double* e1;                // sorted E (limiter)
    const double2* p1;               // (z, h)
    const double2* hh;               // (1/h, Fn)
    const double2* t0;               // per-call target record
    const double2* me;               // (mu, E); limiter with rk_in_me: (rho kappa, E) on entry
    double2* me_out;                 // limiter: (mu, E) for the apply
    double2* g_out[2];               // SW_GRADN: (G_x, G_y), (G_z, kappa^ib) in sorted order for the ray kernel (ray.cu)
    double* mu_sorted;               // limiter: mu in sorted order for the general kernels
    const uint32_t* perm;
    const TileDesc* tiles;
    const uint32_t* tiletab;         // [tile][TILES_WORDS]: TileS as built by tile_setup
    const unsigned long long* ctr;
    const uint2* pool;
    const uint2* winfo;
    const uint32_t* lcount;
    const uint32_t* tflags;
    int64_t n;
    double beta, c_light;
    int fld_sym;
    double *o0, *o1, *o2, *o3, *o4;
    double *o5, *o6;                 // SW_HYDLIM: mu, gradE (nullable)
    int rk_in_me;                    // limiter epilogue reads rho_a kappa_a from me[i].x instead of t0[i].x
    uint32_t* ocount;
};

struct Acc {
    double a0, a1, a2, a3, a4;
    double k[15];                    // SW_KGC: sum c x_i x_j (xx, xy, xz, yy, yz, zz), then sum c dv_i x_j (row-major 3 x 3)
};
struct Tgt {                         // per-target constants
    double x, y, z, hinv, fn;
    double c0, c1, c2, c3, c4, c5;   // per sweep (see k_tiled_sweep)
    double e, rk;                    // SW_HYDLIM: E_a, rho_a kappa_a
};

// One pair (target, slot s).  F = staged records ([record][TILE_CMAXP] double2), Ee = staged E (limiter).
// UNI: every particle of the tile has the target's h, so F(r;h_b) = F(r;h_a), the normalisation kFn/h^4 is applied
// once per target after the loop (k_tiled_sweep) and no support clamp is needed.
template <int SWEEP, int KERNEL, bool UNI>
__device__ __forceinline__ void pair_body(const double2* __restrict__ F, const double* __restrict__ Ee, uint32_t s, const double2 d0,
                                          const double2 d1, const Tgt& T, double beta, bool sym, Acc& acc) {
    const double dx = T.x - d0.x, dy = T.y - d0.y, dz = T.z - d1.x;
    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    const double y = rsqrt_fast(r2);                     // 1/r  (r2 > 0: coincident pairs never reach the tiled lists)
    const double r = r2 * y;
    const double qa = r * T.hinv;
    if (SWEEP == SW_DENSITY) {
        // eq. (35)
        acc.a0 = fma(d1.y, wshape<KERNEL, !UNI>(qa), acc.a0);
    } else if (SWEEP == SW_HYDRO) {
        const double2 d2 = F[2 * TILE_CMAXP + s], d3 = F[3 * TILE_CMAXP + s];
        const double Vb = d1.y, Qb = d2.x;
        const double dvx = T.c3 - d2.y, dvy = T.c4 - d3.x, dvz = T.c5 - d3.y;
        const double vr = fma(dvz, dz, fma(dvy, dy, dvx * dx));           // v_ab . x_ab = w r
        if (UNI) {
            const double G = gshape<KERNEL, false>(qa) * y;               // F / (r kFn/h^4)
            // eq. (11) P:L98 with the sign of eq. (5) (A3): -(m_b/(rho_a rho_b)) (p_a F_a + p_b F_b) x_ab / r
            double c = fma(Vb, T.c0, Qb * T.c1);
            if (vr < 0.0) {                  // eqs. (41)-(43) P:L236-L242 (A6, A7, A8)
                const double2 d4 = F[4 * TILE_CMAXP + s];
                const double w = vr * y, hw = 0.5 * w;
                const double vsa = fma(-beta, w, T.c2), vsb = fma(-beta, w, d4.y);
                c = fma(-hw, fma(d4.x * T.c1, vsa, Vb * vsb), c);
                acc.a4 = fma((hw * w) * (d4.x * vsa), G * r, acc.a4);
            }
            const double cg = c * G;
            acc.a0 = fma(cg, dx, acc.a0); acc.a1 = fma(cg, dy, acc.a1); acc.a2 = fma(cg, dz, acc.a2);
            acc.a3 = fma(Vb * G, vr, acc.a3);                             // eq. (37)
        } else {
            const double2 d5 = F[5 * TILE_CMAXP + s];
            const double Ga = (gshape<KERNEL, true>(qa) * y) * T.fn;
            const double Gb = (gshape<KERNEL, true>(r * d5.x) * y) * d5.y;
            double c = fma(Vb * T.c0, Ga, (Qb * T.c1) * Gb);
            if (vr < 0.0) {
                const double2 d4 = F[4 * TILE_CMAXP + s];
                const double w = vr * y, hw = 0.5 * w;
                const double vsa = fma(-beta, w, T.c2), vsb = fma(-beta, w, d4.y);
                c = fma(-hw, fma((d4.x * T.c1) * vsa, Ga, (Vb * vsb) * Gb), c);
                acc.a4 = fma((hw * w) * (d4.x * vsa), Ga * r, acc.a4);
            }
            acc.a0 = fma(c, dx, acc.a0); acc.a1 = fma(c, dy, acc.a1); acc.a2 = fma(c, dz, acc.a2);
            acc.a3 = fma(Vb * Ga, vr, acc.a3);
        }
    } else if (SWEEP == SW_LIMITER || SWEEP == SW_GRADN) {
        // eq. (9) phi = 1 with f = E (A19): h_a only.  SW_GRADN (row N4) is the same sum without
        // the -E_a term (T.c0 = 0): G_a = sum_b V_b f_b gradW(x_ab, h_a), literally as printed.
        const double G = gshape<KERNEL, !UNI>(qa) * y;
        const double cc = (d1.y * (Ee[s] - T.c0)) * G;
        acc.a0 = fma(cc, dx, acc.a0); acc.a1 = fma(cc, dy, acc.a1); acc.a2 = fma(cc, dz, acc.a2);
    } else if (SWEEP == SW_KGC) {
        // eq. (40): M_a = sum V_b gradW (x) x_ba = -(kFn/h_a^4) sum c x_ab (x) x_ab, c = V_b F/(r kFn/h_a^4);
        // eq. (37) with eq. (39): L_a : sum V_b v_ab (x) gradW = (kFn/h_a^4) L_a : sum c v_ab (x) x_ab.  h_a only.
        const double2 d2 = F[2 * TILE_CMAXP + s], d3 = F[3 * TILE_CMAXP + s];
        const double c = d1.y * (gshape<KERNEL, !UNI>(qa) * y);
        const double cx = c * dx, cy = c * dy, cz = c * dz;
        const double dvx = T.c3 - d2.x, dvy = T.c4 - d2.y, dvz = T.c5 - d3.x;
        acc.k[0] = fma(cx, dx, acc.k[0]); acc.k[1] = fma(cx, dy, acc.k[1]); acc.k[2] = fma(cx, dz, acc.k[2]);
        acc.k[3] = fma(cy, dy, acc.k[3]); acc.k[4] = fma(cy, dz, acc.k[4]); acc.k[5] = fma(cz, dz, acc.k[5]);
        acc.k[6] = fma(dvx, cx, acc.k[6]); acc.k[7] = fma(dvx, cy, acc.k[7]); acc.k[8] = fma(dvx, cz, acc.k[8]);
        acc.k[9] = fma(dvy, cx, acc.k[9]); acc.k[10] = fma(dvy, cy, acc.k[10]); acc.k[11] = fma(dvy, cz, acc.k[11]);
        acc.k[12] = fma(dvz, cx, acc.k[12]); acc.k[13] = fma(dvz, cy, acc.k[13]); acc.k[14] = fma(dvz, cz, acc.k[14]);
    } else {
        // eq. (47) first term P:L270 on eq. (16); Fbar as P:L134 (A17)
        const double2 d2 = F[2 * TILE_CMAXP + s];
        double G;
        if (UNI) {
            G = gshape<KERNEL, false>(qa) * y;
        } else {
            double Fbar = gshape<KERNEL, true>(qa) * T.fn;
            if (sym) {
                const double2 d3 = F[3 * TILE_CMAXP + s];
                Fbar = 0.5 * fma(gshape<KERNEL, true>(r * d3.x), d3.y, Fbar);
            }
            G = Fbar * y;
        }
        const double hm = (T.c2 * d2.x) * rcp_fast(T.c1 + d2.x);          // 4 mu_a mu_b / (mu_a + mu_b)
        const double cab = (d1.y * hm) * G;
        acc.a0 = fma(cab, T.c0 - d2.y, acc.a0);                           // difference form (O7)
        acc.a1 += cab;
    }
}

// Hydro pairs in groups: the branch-free part of every pair of the group first (so the compiler can interleave
// their dependency chains), then ONE branch for the group's viscous corrections (taken only if some pair approaches),
// then the accumulations.  Same arithmetic as pair_body<SW_HYDRO>.
struct HydroPair { double dx, dy, dz, y, r, Ga, Gb, c, vr, Vb, dE; uint32_t s; };

template <int KERNEL, bool UNI, bool LIM>
__device__ __forceinline__ void hydro_common(const double2* __restrict__ F, const double* __restrict__ Ee, uint32_t s, const Tgt& T, HydroPair& h) {
    if (LIM) h.dE = Ee[s] - T.e;
    const double2 d0 = F[s], d1 = F[TILE_CMAXP + s];
    const double2 d2 = F[2 * TILE_CMAXP + s], d3 = F[3 * TILE_CMAXP + s];
    h.s = s;
    h.dx = T.x - d0.x; h.dy = T.y - d0.y; h.dz = T.z - d1.x;
    const double r2 = fma(h.dz, h.dz, fma(h.dy, h.dy, h.dx * h.dx));
    h.y = rsqrt_fast(r2);
    h.r = r2 * h.y;
    h.Vb = d1.y;
    const double dvx = T.c3 - d2.y, dvy = T.c4 - d3.x, dvz = T.c5 - d3.y;
    h.vr = fma(dvz, h.dz, fma(dvy, h.dy, dvx * h.dx));                   // v_ab . x_ab = w r
    if (UNI) {
        h.Ga = gshape<KERNEL, false>(h.r * T.hinv) * h.y;                // F / (r kFn/h^4)
        h.Gb = h.Ga;
        // eq. (11) P:L98 with the sign of eq. (5) (A3): -(m_b/(rho_a rho_b)) (p_a F_a + p_b F_b) x_ab / r
        h.c = fma(h.Vb, T.c0, d2.x * T.c1);
    } else {
        const double2 d5 = F[5 * TILE_CMAXP + s];
        h.Ga = (gshape<KERNEL, true>(h.r * T.hinv) * h.y) * T.fn;
        h.Gb = (gshape<KERNEL, true>(h.r * d5.x) * h.y) * d5.y;
        h.c = fma(h.Vb * T.c0, h.Ga, (d2.x * T.c1) * h.Gb);
    }
}
template <bool UNI>
__device__ __forceinline__ void hydro_visc(const double2* __restrict__ F, const Tgt& T, double beta, HydroPair& h, Acc& acc) {
    // eqs. (41)-(43) P:L236-L242 (A6, A7, A8)
    const double2 d4 = F[4 * TILE_CMAXP + h.s];
    const double w = h.vr * h.y, hw = 0.5 * w;
    const double vsa = fma(-beta, w, T.c2), vsb = fma(-beta, w, d4.y);
    if (UNI) h.c = fma(-hw, fma(d4.x * T.c1, vsa, h.Vb * vsb), h.c);
    else h.c = fma(-hw, fma((d4.x * T.c1) * vsa, h.Ga, (h.Vb * vsb) * h.Gb), h.c);
    acc.a4 = fma((hw * w) * (d4.x * vsa), h.Ga * h.r, acc.a4);
}
template <bool UNI, bool LIM>
__device__ __forceinline__ void hydro_accum(const HydroPair& h, Acc& acc) {
    const double cg = UNI ? h.c * h.Ga : h.c;
    acc.a0 = fma(cg, h.dx, acc.a0); acc.a1 = fma(cg, h.dy, acc.a1); acc.a2 = fma(cg, h.dz, acc.a2);
    acc.a3 = fma(h.Vb * h.Ga, h.vr, acc.a3);                             // eq. (37)
    if (LIM) {                           // eq. (9) phi = 1 with f = E: the pair term of pair_body<SW_LIMITER>, same order (uniform h)
        const double cc = (h.Vb * h.dE) * h.Ga;
        acc.k[0] = fma(cc, h.dx, acc.k[0]); acc.k[1] = fma(cc, h.dy, acc.k[1]); acc.k[2] = fma(cc, h.dz, acc.k[2]);
    }
}
template <int KERNEL, bool UNI, bool LIM>
__device__ __forceinline__ void hydro_group2(const double2* __restrict__ F, const double* __restrict__ Ee, uint32_t s0, uint32_t s1, const Tgt& T, double beta, Acc& acc) {
    HydroPair h0, h1;
    hydro_common<KERNEL, UNI, LIM>(F, Ee, s0, T, h0);
    hydro_common<KERNEL, UNI, LIM>(F, Ee, s1, T, h1);
    if (fmin(h0.vr, h1.vr) < 0.0) {
        if (h0.vr < 0.0) hydro_visc<UNI>(F, T, beta, h0, acc);
        if (h1.vr < 0.0) hydro_visc<UNI>(F, T, beta, h1, acc);
    }
    hydro_accum<UNI, LIM>(h0, acc);
    hydro_accum<UNI, LIM>(h1, acc);
}

template <int SWEEP, int KERNEL, bool UNI>
__device__ __forceinline__ void pair_body(const double2* __restrict__ F, const double* __restrict__ Ee, uint32_t s, const Tgt& T,
                                          double beta, bool sym, Acc& acc) {
    pair_body<SWEEP, KERNEL, UNI>(F, Ee, s, F[s], F[TILE_CMAXP + s], T, beta, sym, acc);
}

template <int SWEEP, int KERNEL, bool UNI>
__device__ __forceinline__ void pair_loop(const double2* __restrict__ F, const double* __restrict__ Ee, const uint2* __restrict__ lp,
                                          uint32_t R, uint2 cur, uint2 nxt, uint2 nx2, const Tgt& T, double beta, bool sym, Acc& acc) {
    // list rows are read three iterations ahead of their use (the compiler sinks the load to the end of the iteration, which
    // leaves two full iterations of this warp to cover the DRAM latency of the streamed lists)
    // Density and limiter (two records per pair, the lightest pair bodies): the position records of the first pair of an
    // iteration are read from shared memory during the iteration before (slot 0 when there is none: read and not used), so
    // that the shared-memory round trip, long when the data pipe is busy, is not exposed at the top of every iteration.
    // Measured: -5 % for these two sweeps, +1-2 % for the heavier ones, which therefore do not do it.
    constexpr bool PIPE_FIRST = SWEEP == SW_DENSITY || SWEEP == SW_LIMITER || SWEEP == SW_GRADN;
    double2 q0 = F[cur.x & 0xFFFFu], q1 = F[TILE_CMAXP + (cur.x & 0xFFFFu)];
    for (uint32_t r4 = 0; r4 < R; r4 += 4) {
        const uint2 nx3 = (r4 + 12 < R) ? __ldcs(lp + (size_t)(r4 / 4 + 3) * 32) : make_uint2(0u, 0u);
        const uint32_t sn = nxt.x & 0xFFFFu;
        if (SWEEP == SW_HYDRO || SWEEP == SW_HYDLIM) {
            hydro_group2<KERNEL, UNI, SWEEP == SW_HYDLIM>(F, Ee, cur.x & 0xFFFFu, cur.x >> 16, T, beta, acc);
            hydro_group2<KERNEL, UNI, SWEEP == SW_HYDLIM>(F, Ee, cur.y & 0xFFFFu, cur.y >> 16, T, beta, acc);
        } else {
            if (PIPE_FIRST) {
                pair_body<SWEEP, KERNEL, UNI>(F, Ee, cur.x & 0xFFFFu, q0, q1, T, beta, sym, acc);
                q0 = F[sn]; q1 = F[TILE_CMAXP + sn];
            } else {
                pair_body<SWEEP, KERNEL, UNI>(F, Ee, cur.x & 0xFFFFu, T, beta, sym, acc);
            }
            pair_body<SWEEP, KERNEL, UNI>(F, Ee, cur.x >> 16, T, beta, sym, acc);
            pair_body<SWEEP, KERNEL, UNI>(F, Ee, cur.y & 0xFFFFu, T, beta, sym, acc);
            pair_body<SWEEP, KERNEL, UNI>(F, Ee, cur.y >> 16, T, beta, sym, acc);
        }
        cur = nxt; nxt = nx2; nx2 = nx3;
    }
}

// MODE 0: every tile.  MODE 1: only the tiles with uniform h, whose pair bodies never read the (1/h, Fn) record -- the
// apply then needs 3 records per candidate, 105 KB, and two CTAs fit an SM.  MODE 2: only the other tiles.
template <int SWEEP, int MODE> struct NRecM {
    static constexpr int v = (SWEEP == SW_APPLY && MODE == 1) ? 3 : ((SWEEP == SW_HYDLIM && MODE == 1) ? 5 : NRec<SWEEP>::v);
};
template <int SWEEP, int MODE> struct MinBlocks {
    static constexpr int v = (SWEEP == SW_DENSITY || SWEEP == SW_LIMITER || SWEEP == SW_GRADN || (SWEEP == SW_APPLY && MODE == 1)) ? 2 : 1;
};

// PARTS = false: the tiles that are one entry (nearly all; every tile of a particle set with uniform h).  PARTS = true: the
// groups of several parts (tiles.cuh), in a launch of their own that returns at once when the build cut none -- carrying a
// target and its sums from part to part costs registers that the 64-register kernels do not have to spare.
template <int SWEEP, int KERNEL, int MODE, bool PARTS>
__global__ void __launch_bounds__(TILE_THREADS, MinBlocks<SWEEP, MODE>::v)
k_tiled_sweep(DevGrid g, CellTable ct, SweepIn A) {
    constexpr int NV = NRecM<SWEEP, MODE>::v;
    extern __shared__ __align__(16) unsigned char smem[];
    // this tile's tables / the next tile's, fetched under the pair loop: ranges and target cells, the warps' list rows, descriptor, flags
    struct TileHdr { uint2 winfo[TILE_WARPS]; TileDesc td; uint32_t flags, pad; };
    __shared__ __align__(16) TileS Sb[2];
    __shared__ __align__(16) TileHdr Hb[2];
    double2* F = reinterpret_cast<double2*>(smem);               // F[record * TILE_CMAXP + slot]
    double* Ee = reinterpret_cast<double*>(F + (size_t)NV * TILE_CMAXP);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int u = tid & 1, tgt = tid >> 1;
    const uint32_t ntiles = (uint32_t)A.ctr[CTR_NTILES];
    if (MODE == 2 && A.ctr[CTR_NNONUNI] == 0) return;          // no tile with variable h (the usual case): nothing for this launch
    if (PARTS && A.ctr[CTR_NMULTI] == 0) return;               // no group of several parts (the usual case)
    constexpr bool HYD = SWEEP == SW_HYDRO || SWEEP == SW_HYDLIM;
    const bool sym = HYD || (SWEEP == SW_APPLY && A.fld_sym != 0);
    // dummy slots: far away, every weight zero, so that a padded list entry adds exactly nothing
    if (tid < TILE_NDUMMY) {
        const double far = g.lo[0] - 1.0e4 * g.L[0];
#pragma unroll
        for (int v = 0; v < NV; ++v) F[v * TILE_CMAXP + TILE_CMAX + tid] = make_double2(0.0, 0.0);
        F[TILE_CMAX + tid] = make_double2(far, g.lo[1]);
        F[TILE_CMAXP + TILE_CMAX + tid] = make_double2(g.lo[2], 0.0);
        if (SWEEP == SW_APPLY) F[2 * TILE_CMAXP + TILE_CMAX + tid] = make_double2(1.0, 0.0);
        if (NRec<SWEEP>::e) Ee[TILE_CMAX + tid] = 0.0;
    }

    auto fetch_tables = [&](uint32_t t, int b) {
        if (t < ntiles) {
            if (tid < TILES_WORDS / 4)
                cp_async16(reinterpret_cast<uint4*>(&Sb[b]) + tid, reinterpret_cast<const uint4*>(A.tiletab + (size_t)t * TILES_WORDS) + tid);
            else if (tid >= 128 && tid < 128 + TILE_WARPS / 2)
                cp_async16(reinterpret_cast<uint4*>(Hb[b].winfo) + (tid - 128), reinterpret_cast<const uint4*>(A.winfo + (size_t)t * TILE_WARPS) + (tid - 128));
            else if (tid >= 160 && tid < 163)
                cp_async8(reinterpret_cast<uint2*>(&Hb[b].td) + (tid - 160), reinterpret_cast<const uint2*>(A.tiles + t) + (tid - 160));
            else if (tid == 192)
                asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" :: "r"((uint32_t)__cvta_generic_to_shared(&Hb[b].flags)), "l"(A.tflags + t) : "memory");
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    fetch_tables(blockIdx.x, 0);
    int buf = 1;
    // A tile entry is part 0 of nparts (tiles.cuh): the CTA that meets part 0 runs all the parts one after the other -- same
    // targets, another set of candidate rows and lists each -- and keeps its sums; a CTA whose stride lands on a later part passes.
    for (uint32_t tile0 = blockIdx.x; tile0 < ntiles; tile0 += gridDim.x) {
      uint32_t np = 1;
      bool pass_group = false, active = false, grp_ok = true, uni = true;
      uint32_t i = 0, ia = 0, ngat = 0;
      Tgt T{};
      Acc acc{};
      for (uint32_t part = 0; part < (PARTS ? np : 1u); ++part) {
        const uint32_t tile = tile0 + part;
        buf ^= 1;
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        __syncthreads();                                         // tables in place; previous tile done with the staged records
        const TileS& S = Sb[buf];
        const uint32_t flags = Hb[buf].flags;
        const TileDesc td = Hb[buf].td;
        if (part == 0) {
            const bool tile_uni = (flags & TILE_FLAG_NONUNI) == 0;   // (of a group: the builder ORs every part's bit into part 0)
            uni = MODE == 1 ? true : (MODE == 2 ? false : tile_uni);
            if (td.part != 0 || (td.nparts > 1) != PARTS || (MODE != 0 && tile_uni != (MODE == 1))) pass_group = true;   // not mine / not this launch's kind
            else if (PARTS) np = min((uint32_t)td.nparts, ntiles - tile0);
        }
        fetch_tables(PARTS && part + 1 < np ? tile + 1 : tile0 + gridDim.x, buf ^ 1);     // (a group that is passed has np = 1)
        if (pass_group) break;
        const bool half_ok = ((flags >> (warp / (TILE_WARPS / 2))) & 1u) != 0;   // this warp's half of the tile has lists
        if (part == 0) active = half_ok && tgt < (int)td.nt;
        if (!half_ok) grp_ok = false;                            // (the builder marked these targets: the general kernels redo them)
        if (!(flags & TILE_FLAG_OK)) continue;
        // first three list rows: in flight while the records are staged
        uint2 wi = Hb[buf].winfo[warp];
        if (!half_ok || !active) wi.y = 0u;
        const uint2* lp = A.pool + (size_t)wi.x * 32 + lane;
        const uint2 l0 = wi.y ? __ldcs(lp) : make_uint2(0u, 0u);
        const uint2 l1 = wi.y > 4 ? __ldcs(lp + 32) : make_uint2(0u, 0u);
        const uint2 l2 = wi.y > 8 ? __ldcs(lp + 64) : make_uint2(0u, 0u);
        // ---- this thread's target.  Except in the hydro kernel (register pressure: measured slower) its loads go out before
        //      the staging traffic, so they are back when the pair loop starts.
        constexpr bool EARLY_TARGET = !HYD;
        auto load_target = [&]() {
            if (!active || part != 0) return;
            i = tile_target(td, S, tgt);
            ia = A.perm[i];                                      // caller index of the target: needed only in the epilogue
            const double2 xy = A.rec[0][i], zh = A.p1[i], hv = A.hh[i];
            T.x = xy.x; T.y = xy.y; T.z = zh.x; T.hinv = hv.x; T.fn = hv.y;
            if (SWEEP == SW_DENSITY) T.c0 = A.rec[1][i].y;                                   // m_a
            if (SWEEP == SW_HYDLIM) { const double2 re = A.me[i]; T.rk = re.x; T.e = re.y; }  // (rho_a kappa_a, E_a), parked there by k_prep_hydro
            if (HYD) {
                const double2 t0 = A.t0[i], q1 = A.rec[2][i], q2 = A.rec[3][i];
                T.c0 = t0.x; T.c1 = t0.y;                                                    // p_a/rho_a, 1/rho_a
                T.c2 = A.rec[4][i].y;                                                        // alpha_a c_a
                T.c3 = q1.y; T.c4 = q2.x; T.c5 = q2.y;                                       // v_a
            }
            if (SWEEP == SW_LIMITER) T.c0 = A.e1[i];                                         // E_a
            if (SWEEP == SW_GRADN) T.c0 = 0.0;
            if (SWEEP == SW_APPLY) { const double2 me = A.rec[2][i]; T.c0 = me.y; T.c1 = me.x; T.c2 = 4.0 * me.x; }
            if (SWEEP == SW_KGC) {
                const double2 q1 = A.rec[2][i], q2 = A.rec[3][i];
                T.c0 = A.t0[i].x;                                                            // rho_a
                T.c3 = q1.x; T.c4 = q1.y; T.c5 = q2.x;                                       // v_a
            }
        };
        if (EARLY_TARGET) load_target();
        // ---- stage the candidate records: one warp per range.  Ranges that need no periodic shift (all but those of
        //      tiles at a periodic face) are copied with cp.async (LDGSTS): no register round trip, every copy of the
        //      thread in flight at once, completion awaited just before the barrier that precedes the pair loop.
        for (int q = warp; q < (int)S.nranges; q += TILE_WARPS) {
            const uint32_t vs = S.r_vstart[q], len = S.r_vend[q] - vs, base = S.r_base[q];
            const bool shifted = (S.r_shift[q][0] | S.r_shift[q][1] | S.r_shift[q][2]) != 0;
            if (!shifted) {
                for (uint32_t k = lane; k < len; k += 32) {
#pragma unroll
                    for (int v = 0; v < NV; ++v) {
                        if (uni && ((HYD && v == 5) || (SWEEP == SW_APPLY && v == 3))) continue;
                        cp_async16(&F[v * TILE_CMAXP + base + k], &A.rec[v][vs + k]);
                    }
                    if (NRec<SWEEP>::e) cp_async8(&Ee[base + k], &A.e1[vs + k]);
                }
            } else {
                const double shx = S.r_shift[q][0] * g.L[0], shy = S.r_shift[q][1] * g.L[1], shz = S.r_shift[q][2] * g.L[2];
                for (uint32_t k = lane; k < len; k += 32) {
#pragma unroll
                    for (int v = 0; v < NV; ++v) {
                        if (uni && ((HYD && v == 5) || (SWEEP == SW_APPLY && v == 3))) continue;
                        double2 val = A.rec[v][vs + k];
                        if (v == 0) { val.x -= shx; val.y -= shy; }
                        if (v == 1) val.x -= shz;
                        F[v * TILE_CMAXP + base + k] = val;
                    }
                    if (NRec<SWEEP>::e) Ee[base + k] = A.e1[vs + k];
                }
            }
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
        if (!EARLY_TARGET) load_target();
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        __syncthreads();
        if (uni) pair_loop<SWEEP, KERNEL, true>(F, Ee, lp, wi.y, l0, l1, l2, T, A.beta, sym, acc);
        else pair_loop<SWEEP, KERNEL, false>(F, Ee, lp, wi.y, l0, l1, l2, T, A.beta, sym, acc);
        if (SWEEP == SW_DENSITY && A.ocount && active && u == 0) ngat += A.lcount[(size_t)tile * TILE_T + tgt] & 0xFFFFu;
      }
      if (pass_group) continue;
      {
        // ---- add the two half-lists of the target
        acc.a0 += __shfl_xor_sync(0xFFFFFFFFu, acc.a0, 1);
        if (SWEEP != SW_DENSITY) acc.a1 += __shfl_xor_sync(0xFFFFFFFFu, acc.a1, 1);
        if (HYD || SWEEP == SW_LIMITER || SWEEP == SW_GRADN) acc.a2 += __shfl_xor_sync(0xFFFFFFFFu, acc.a2, 1);
        if (SWEEP == SW_HYDLIM) {
#pragma unroll
            for (int e = 0; e < 3; ++e) acc.k[e] += __shfl_xor_sync(0xFFFFFFFFu, acc.k[e], 1);
        }
        if (HYD) {
            acc.a3 += __shfl_xor_sync(0xFFFFFFFFu, acc.a3, 1);
            acc.a4 += __shfl_xor_sync(0xFFFFFFFFu, acc.a4, 1);
        }
        if (SWEEP == SW_KGC) {
#pragma unroll
            for (int e = 0; e < 15; ++e) acc.k[e] += __shfl_xor_sync(0xFFFFFFFFu, acc.k[e], 1);
        }

        if (active && grp_ok && u == 0) {
            const double sc = uni ? T.fn : 1.0;                  // kFn / h_a^4 where it was hoisted out of the loop
            if (SWEEP == SW_DENSITY) {
                // self term m_a W(0; h_a) (A11)
                const double wn = wn_k<KERNEL>() * (T.hinv * T.hinv) * T.hinv;
                A.o0[ia] = wn * fma(T.c0, w0_k<KERNEL>(), acc.a0);
                if (A.ocount) A.ocount[ia] = ngat;
            } else if (HYD) {
                A.o0[ia] = -(sc * acc.a0); A.o1[ia] = -(sc * acc.a1); A.o2[ia] = -(sc * acc.a2);
                const double D = sc * acc.a3;
                A.o3[ia] = T.c0 * D - (sc * acc.a4) * T.c1;      // eq. (17) 1st term P:L129 + eq. (42)
                if (A.o4) A.o4[ia] = D;
                if (SWEEP == SW_HYDLIM) {
                    // the limiter epilogue of SW_LIMITER below, on the sums of the same pair terms
                    const double gx = T.fn * acc.k[0], gy = T.fn * acc.k[1], gz = T.fn * acc.k[2];
                    const double rk = T.rk;
                    const double gn = sqrt(gx * gx + gy * gy + gz * gz);
                    const double Rl = gn / (rk * T.e);
                    const double mu = A.c_light * (1.0 / sqrt(9.0 + Rl * Rl)) / rk;
                    A.o5[ia] = mu;
                    A.me_out[i] = make_double2(mu, T.e);
                    A.mu_sorted[i] = mu;
                    if (A.o6) { A.o6[ia] = gx; A.o6[A.n + ia] = gy; A.o6[2 * A.n + ia] = gz; }
                }
            } else if (SWEEP == SW_LIMITER) {
                // Larsen limiter, k = 2 (A20); the limiter sum always carries kFn/h_a^4 outside
                const double gx = T.fn * acc.a0, gy = T.fn * acc.a1, gz = T.fn * acc.a2;
                const double rk = A.rk_in_me ? A.me[i].x : A.t0[i].x;   // rho_a kappa_a
                const double gn = sqrt(gx * gx + gy * gy + gz * gz);
                const double Rl = gn / (rk * T.c0);
                const double mu = A.c_light * (1.0 / sqrt(9.0 + Rl * Rl)) / rk;
                A.o0[ia] = mu;
                A.me_out[i] = make_double2(mu, T.c0);
                A.mu_sorted[i] = mu;
                if (A.o1) { A.o1[ia] = gx; A.o1[A.n + ia] = gy; A.o1[2 * A.n + ia] = gz; }
            } else if (SWEEP == SW_GRADN) {
                // row N4: gradient of n_e/n_c at the particle, caller order (nullable) + the sorted records the ray kernel gathers
                const double gx = T.fn * acc.a0, gy = T.fn * acc.a1, gz = T.fn * acc.a2;
                A.g_out[0][i] = make_double2(gx, gy);
                A.g_out[1][i] = make_double2(gz, A.me[i].x);     // (G_z, kappa^ib)
                if (A.o1) { A.o1[ia] = gx; A.o1[A.n + ia] = gy; A.o1[2 * A.n + ia] = gz; }
            } else if (SWEEP == SW_KGC) {
                // M_a = -(kFn/h_a^4) sum c x (x) x (symmetric), L_a = M_a^-1 by cofactors; singular -> L_a = I (A28)
                const double fn = T.fn;
                const double m00 = -fn * acc.k[0], m01 = -fn * acc.k[1], m02 = -fn * acc.k[2];
                const double m11 = -fn * acc.k[3], m12 = -fn * acc.k[4], m22 = -fn * acc.k[5];
                const double c00 = m11 * m22 - m12 * m12, c01 = m02 * m12 - m01 * m22, c02 = m01 * m12 - m02 * m11;
                const double det = m00 * c00 + m01 * c01 + m02 * c02;
                double l00 = 1.0, l01 = 0.0, l02 = 0.0, l11 = 1.0, l12 = 0.0, l22 = 1.0;
                if (fabs(det) > 1e-12) {
                    const double id = 1.0 / det;
                    l00 = c00 * id; l01 = c01 * id; l02 = c02 * id;
                    l11 = (m00 * m22 - m02 * m02) * id; l12 = (m01 * m02 - m00 * m12) * id; l22 = (m00 * m11 - m01 * m01) * id;
                }
                const double* q = acc.k + 6;                     // q[3 i + j] = sum c dv_i x_j
                const double corr = l00 * q[0] + l11 * q[4] + l22 * q[8] + l01 * (q[1] + q[3]) + l02 * (q[2] + q[6]) + l12 * (q[5] + q[7]);
                A.o0[ia] = T.c0 * (fn * corr);
                if (A.o1) {
                    double* Lo = A.o1 + ia;
                    Lo[0] = l00; Lo[A.n] = l01; Lo[2 * A.n] = l02;
                    Lo[3 * A.n] = l01; Lo[4 * A.n] = l11; Lo[5 * A.n] = l12;
                    Lo[6 * A.n] = l02; Lo[7 * A.n] = l12; Lo[8 * A.n] = l22;
                }
                if (A.o2) A.o2[ia] = T.c0 * (fn * (q[0] + q[4] + q[8]));
            } else {
                const double yv = sc * acc.a0, lam = sc * acc.a1;
                A.o0[ia] = yv;
                if (A.o1) A.o1[ia] = lam;
                if (A.o2) A.o2[ia] = fma(-lam, T.c0, yv);        // Gamma = y - Lambda E_a  (eq. (52))
            }
        }
      }
    }
}

template <int SWEEP, int MODE>
constexpr size_t sweep_smem() {
    return sizeof(double2) * NRecM<SWEEP, MODE>::v * TILE_CMAXP + sizeof(double) * NRec<SWEEP>::e * TILE_CMAXP;
}
// The opt-in to more than 48 KB of dynamic shared memory is a per-device function attribute: set for every instantiation
// that is launched, on the current device (spray_create calls this after cudaSetDevice).
template <int SWEEP, int MODE>
static cudaError_t set_attr() {
    cudaError_t e = cudaFuncSetAttribute(k_tiled_sweep<SWEEP, 0, MODE, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sweep_smem<SWEEP, MODE>());
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_tiled_sweep<SWEEP, 1, MODE, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sweep_smem<SWEEP, MODE>());
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_tiled_sweep<SWEEP, 0, MODE, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sweep_smem<SWEEP, MODE>());
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_tiled_sweep<SWEEP, 1, MODE, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sweep_smem<SWEEP, MODE>());
    return e;
}
cudaError_t sweeps_set_attributes() {
    cudaError_t e = set_attr<SW_DENSITY, 0>();
    if (e == cudaSuccess) e = set_attr<SW_HYDRO, 0>();
    if (e == cudaSuccess) e = set_attr<SW_HYDRO, 2>();
    if (e == cudaSuccess) e = set_attr<SW_LIMITER, 0>();
    if (e == cudaSuccess) e = set_attr<SW_LIMITER, 2>();
    if (e == cudaSuccess) e = set_attr<SW_HYDLIM, 1>();
    if (e == cudaSuccess) e = set_attr<SW_GRADN, 0>();
    if (e == cudaSuccess) e = set_attr<SW_APPLY, 1>();
    if (e == cudaSuccess) e = set_attr<SW_APPLY, 2>();
    if (e == cudaSuccess) e = set_attr<SW_KGC, 0>();
    return e;
}

template <int SWEEP, int MODE>
static cudaError_t launch_m(Ctx* c, const SweepIn& a, cudaStream_t st) {
    constexpr size_t smem = sweep_smem<SWEEP, MODE>();
    CellTable ct{c->cell_start, c->cell_end, c->is_level ? c->cell_tend : c->cell_end};
    const int grid = c->tl.sms * MinBlocks<SWEEP, MODE>::v;
    if (c->kernel == SPRAY_KERNEL_WENDLAND_C2) {
        k_tiled_sweep<SWEEP, 1, MODE, false><<<grid, TILE_THREADS, smem, st>>>(c->dg, ct, a);
        k_tiled_sweep<SWEEP, 1, MODE, true><<<grid, TILE_THREADS, smem, st>>>(c->dg, ct, a);
    } else {
        k_tiled_sweep<SWEEP, 0, MODE, false><<<grid, TILE_THREADS, smem, st>>>(c->dg, ct, a);
        k_tiled_sweep<SWEEP, 0, MODE, true><<<grid, TILE_THREADS, smem, st>>>(c->dg, ct, a);
    }
    c->launches += 2;
    return cudaGetLastError();
}
template <int SWEEP>
static cudaError_t launch_t(Ctx* c, const SweepIn& a, cudaStream_t st) {
    if constexpr (SWEEP == SW_APPLY) {          // uniform-h tiles at two CTAs per SM, then whatever is left
        cudaError_t e = launch_m<SWEEP, 1>(c, a, st);
        return e != cudaSuccess ? e : launch_m<SWEEP, 2>(c, a, st);
    } else if constexpr (SWEEP == SW_HYDLIM) {  // fused sweep on the uniform-h tiles; the other tiles run the two sweeps one after the other
        cudaError_t e = launch_m<SW_HYDLIM, 1>(c, a, st);
        if (e == cudaSuccess) e = launch_m<SW_HYDRO, 2>(c, a, st);
        if (e != cudaSuccess) return e;
        SweepIn l = a;                          // limiter view of the same job: its outputs are o0 (mu), o1 (gradE)
        l.o0 = a.o5; l.o1 = a.o6; l.rk_in_me = 1;
        return launch_m<SW_LIMITER, 2>(c, l, st);
    } else {
        return launch_m<SWEEP, 0>(c, a, st);
    }
}

cudaError_t launch_tiled_sweep(Ctx* c, int sweep, const TiledArgs& t, cudaStream_t st) {
    if (c->n == 0) return cudaSuccess;
    SweepIn a{};
    const Packed& pk = c->pk;
    a.p1 = pk.p1; a.hh = pk.hh; a.t0 = pk.t0; a.me = pk.me; a.me_out = pk.me; a.mu_sorted = c->s.f[10]; a.e1 = pk.e1;
    a.perm = c->perm; a.tiles = c->tl.tiles; a.tiletab = c->tl.tiletab; a.ctr = c->tl.ctr; a.pool = c->tl.pool; a.winfo = c->tl.winfo;
    a.lcount = c->tl.lcount; a.tflags = c->tl.tflags; a.n = c->n;
    a.beta = t.beta; a.c_light = t.c_light; a.fld_sym = t.fld_sym;
    a.o0 = t.o0; a.o1 = t.o1; a.o2 = t.o2; a.o3 = t.o3; a.o4 = t.o4; a.o5 = t.o5; a.o6 = t.o6; a.ocount = t.ocount;
    a.rec[0] = pk.p0; a.rec[1] = pk.s[0];
    switch (sweep) {
        case SW_DENSITY: return launch_t<SW_DENSITY>(c, a, st);
        case SW_HYDRO:
            a.rec[2] = pk.s[1]; a.rec[3] = pk.s[2]; a.rec[4] = pk.s[3]; a.rec[5] = pk.hh;
            return launch_t<SW_HYDRO>(c, a, st);
        case SW_LIMITER: return launch_t<SW_LIMITER>(c, a, st);
        case SW_HYDLIM:
            a.rec[2] = pk.s[1]; a.rec[3] = pk.s[2]; a.rec[4] = pk.s[3]; a.rec[5] = pk.hh;
            return launch_t<SW_HYDLIM>(c, a, st);
        case SW_GRADN:
            a.g_out[0] = pk.s[1]; a.g_out[1] = pk.s[2];
            return launch_t<SW_GRADN>(c, a, st);
        case SW_APPLY:
            a.rec[2] = pk.me; a.rec[3] = pk.hh;
            return launch_t<SW_APPLY>(c, a, st);
        case SW_KGC:
            a.rec[2] = pk.s[1]; a.rec[3] = pk.s[2];
            return launch_t<SW_KGC>(c, a, st);
    }
    return cudaErrorInvalidValue;
}

}  // namespace spray
