// sweeps_tiled.cu -- the tiled pair kernels: density (eq. (35)), hydro RHS (eqs. (11), (17), (37), (41)-(43)),
// FLD limiter pre-sweep (eq. (9)) and FLD operator apply (eqs. (16), (47), (51)-(52)) of PAPER.md.
//
// One persistent CTA per SM walks the tiles of tiles.cuh.  Per tile it stages the candidate particles' fields
// (structure-of-arrays, fp64, positions moved to the periodic image next to the tile) into shared memory, then
// every thread owns ONE target particle and runs down its prebuilt neighbour list (u16 slots, tiles.cu): no
// distance test on rejected candidates, all 32 lanes busy with accepted pairs, one reciprocal square root per pair
// (MUFU.RSQ64H seed + one third-order correction), per-particle factors hoisted into the prologue kernels.
// Results are written to caller order through the sort permutation.  No floating-point atomics: each target is
// summed by one thread in list order, so results are bitwise reproducible.
#include "spray_internal.h"
#include "tiles.cuh"

namespace spray {

// 1/sqrt(x) for normal positive x to ~1e-16 relative: hardware seed (>= 20 bits) and one third-order step
// y (1 + e/2 + 3 e^2/8), e = 1 - x y^2.
__device__ __forceinline__ double rsqrt_fast(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double t = x * y;
    const double e = fma(-t, y, 1.0);
    const double p = fma(0.375, e, 0.5);
    const double ye = y * e;
    return fma(ye, p, y);
}
// 1/x for normal positive x: hardware seed and one third-order step y (1 + e + e^2), e = 1 - x y.
__device__ __forceinline__ double rcp_fast(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x, y, 1.0);
    const double p = fma(e, e, e);
    return fma(y, p, y);
}

template <int SWEEP> struct NField;
template <> struct NField<SW_DENSITY> { static constexpr int v = 4; };    // x y z m
template <> struct NField<SW_HYDRO> { static constexpr int v = 11; };     // x y z hinv V Q m AC vx vy vz
template <> struct NField<SW_LIMITER> { static constexpr int v = 5; };    // x y z V E
template <> struct NField<SW_APPLY> { static constexpr int v = 7; };      // x y z hinv V mu E

template <int SWEEP, int KERNEL>
__global__ void __launch_bounds__(TILE_T, 1)
k_tiled_sweep(DevGrid g, CellTable ct, TiledArgs A) {
    constexpr int NF = NField<SWEEP>::v;
    extern __shared__ __align__(16) unsigned char smem[];
    __shared__ TileS S;
    double* F = reinterpret_cast<double*>(smem);                 // F[f * TILE_CMAX + slot]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t ntiles = *A.ntiles;
    const bool sym = (SWEEP == SW_HYDRO) || (SWEEP == SW_APPLY && A.fld_sym != 0);

    for (uint32_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        if (!A.tile_ok[tile]) continue;
        const TileDesc td = A.tiles[tile];
        __syncthreads();
        tile_setup(td, g, ct, S);
        const uint32_t ncand = S.ncand;
        // ---- stage candidate fields
        for (uint32_t s = tid; s < ncand; s += TILE_T) {
            const int q = tile_slot_range(S, s);
            const uint32_t gi = S.r_start[q] + (s - S.r_base[q]);
            if (gi >= S.r_vstart[q] && gi < S.r_vend[q]) {
                F[0 * TILE_CMAX + s] = A.x[gi] - S.r_shift[q][0] * g.L[0];
                F[1 * TILE_CMAX + s] = A.y[gi] - S.r_shift[q][1] * g.L[1];
                F[2 * TILE_CMAX + s] = A.z[gi] - S.r_shift[q][2] * g.L[2];
                if (SWEEP == SW_DENSITY) {
                    F[3 * TILE_CMAX + s] = A.f0[gi];                                   // m
                } else if (SWEEP == SW_HYDRO) {
                    F[3 * TILE_CMAX + s] = 1.0 / A.h[gi];
                    F[4 * TILE_CMAX + s] = A.f0[gi];                                   // V = m/rho
                    F[5 * TILE_CMAX + s] = A.f1[gi];                                   // Q = V p
                    F[6 * TILE_CMAX + s] = A.f2[gi];                                   // m
                    F[7 * TILE_CMAX + s] = A.f3[gi];                                   // alpha c
                    F[8 * TILE_CMAX + s] = A.f4[gi];
                    F[9 * TILE_CMAX + s] = A.f5[gi];
                    F[10 * TILE_CMAX + s] = A.f6[gi];
                } else if (SWEEP == SW_LIMITER) {
                    F[3 * TILE_CMAX + s] = A.f0[gi];                                   // V
                    F[4 * TILE_CMAX + s] = A.f1[gi];                                   // E
                } else {
                    F[3 * TILE_CMAX + s] = 1.0 / A.h[gi];
                    F[4 * TILE_CMAX + s] = A.f0[gi];                                   // V
                    F[5 * TILE_CMAX + s] = A.f2[gi];                                   // mu
                    F[6 * TILE_CMAX + s] = A.f1[gi];                                   // E
                }
            }
        }
        // ---- this thread's target
        const bool active = tid < (int)td.nt;
        uint32_t i = 0, nloop = 0, ng = 0;
        double xa = 0, ya = 0, za = 0, hinv = 1, Wn = 0, Fn = 0;
        double a0 = 0, a1 = 0, a2 = 0, a3 = 0, a4 = 0, a5 = 0;           // per-sweep target constants
        if (active) {
            i = tile_target(td, S, tid);
            const uint32_t cnt = A.lcount[(size_t)tile * TILE_T + tid];
            ng = cnt & 0xFFFFu;
            nloop = sym ? (cnt >> 16) : ng;
            xa = A.x[i]; ya = A.y[i]; za = A.z[i];
            hinv = 1.0 / A.h[i];
            Wn = sigma<KERNEL>() * hinv * hinv * hinv;
            Fn = Wn * hinv;
            if (SWEEP == SW_DENSITY) { a0 = A.f0[i]; }
            if (SWEEP == SW_HYDRO) {
                const double rho_a = A.g0[i], p_a = A.g1[i];
                a0 = 1.0 / rho_a;                 // IA
                a1 = p_a * a0;                    // PA = p_a / rho_a
                a2 = A.f3[i];                     // alpha_a c_a
                a3 = A.f4[i]; a4 = A.f5[i]; a5 = A.f6[i];
            }
            if (SWEEP == SW_LIMITER) { a0 = A.f1[i]; }
            if (SWEEP == SW_APPLY) { a0 = A.f1[i]; a1 = A.f2[i]; }
        }
        uint32_t nmax = nloop;
#pragma unroll
        for (int o = 16; o; o >>= 1) nmax = max(nmax, __shfl_xor_sync(0xFFFFFFFFu, nmax, o));
        __syncthreads();

        double acc0 = 0, acc1 = 0, acc2 = 0, acc3 = 0, acc4 = 0;
        const uint2* lp = A.lists + list_block_u2(tile, warp) + lane;
        uint2 cur = nmax ? lp[0] : make_uint2(0u, 0u);
        for (uint32_t k0 = 0; k0 < nmax; k0 += 4) {
            const uint2 nxt = (k0 + 4 < nmax) ? lp[(size_t)(k0 / 4 + 1) * 32] : make_uint2(0u, 0u);
            const uint32_t ee[4] = {cur.x & 0xFFFFu, cur.x >> 16, cur.y & 0xFFFFu, cur.y >> 16};
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                if (k0 + j < nloop) {
                    const uint32_t s = ee[j] & 0x7FFFu;
                    const double dx = xa - F[0 * TILE_CMAX + s];
                    const double dy = ya - F[1 * TILE_CMAX + s];
                    const double dz = za - F[2 * TILE_CMAX + s];
                    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
                    const double rinv = r2 > 0.0 ? rsqrt_fast(r2) : 0.0;
                    const double r = r2 * rinv;
                    if (SWEEP == SW_DENSITY) {
                        // eq. (35)
                        acc0 = fma(F[3 * TILE_CMAX + s], shape_w<KERNEL>(r * hinv), acc0);
                    } else if (SWEEP == SW_HYDRO) {
                        const double hbinv = F[3 * TILE_CMAX + s];
                        const double hb2 = hbinv * hbinv;
                        const double Fa = Fn * shape_f<KERNEL>(r * hinv);
                        const double Fb = (sigma<KERNEL>() * (hb2 * hb2)) * shape_f<KERNEL>(r * hbinv);
                        const double Vb = F[4 * TILE_CMAX + s], Qb = F[5 * TILE_CMAX + s];
                        const double w = ((a3 - F[8 * TILE_CMAX + s]) * dx + (a4 - F[9 * TILE_CMAX + s]) * dy +
                                          (a5 - F[10 * TILE_CMAX + s]) * dz) * rinv;
                        const double VFa = Vb * Fa;
                        // eq. (11) P:L98 with the sign of eq. (5) (A3): -(m_b/(rho_a rho_b)) (p_a F_a + p_b F_b)
                        double coef = -fma(VFa, a1, (Qb * a0) * Fb);
                        if (w < 0.0) {               // eqs. (41)-(43) P:L236-L242 (A6, A7, A8)
                            const double mb = F[6 * TILE_CMAX + s];
                            const double aw = -w;
                            const double vsa = fma(A.beta, aw, a2);
                            const double vsb = fma(A.beta, aw, F[7 * TILE_CMAX + s]);
                            const double mFa = mb * Fa;
                            coef = fma(0.5 * w, fma(mFa * a0, vsa, (Vb * Fb) * vsb), coef);
                            acc4 = fma(0.5 * (w * w), mFa * vsa, acc4);
                        }
                        const double cr = coef * rinv;
                        acc0 = fma(cr, dx, acc0); acc1 = fma(cr, dy, acc1); acc2 = fma(cr, dz, acc2);
                        acc3 = fma(VFa, w, acc3);    // eq. (37)
                    } else if (SWEEP == SW_LIMITER) {
                        // eq. (9) phi = 1 with f = E (A19)
                        const double cc = (F[3 * TILE_CMAX + s] * (F[4 * TILE_CMAX + s] - a0)) * ((Fn * shape_f<KERNEL>(r * hinv)) * rinv);
                        acc0 = fma(cc, dx, acc0); acc1 = fma(cc, dy, acc1); acc2 = fma(cc, dz, acc2);
                    } else {
                        // eq. (47) first term P:L270 on eq. (16); Fbar as P:L134 (A17)
                        double Fbar = Fn * shape_f<KERNEL>(r * hinv);
                        if (sym) {
                            const double hbinv = F[3 * TILE_CMAX + s];
                            const double hb2 = hbinv * hbinv;
                            Fbar = 0.5 * fma(sigma<KERNEL>() * (hb2 * hb2), shape_f<KERNEL>(r * hbinv), Fbar);
                        }
                        const double mu_b = F[5 * TILE_CMAX + s], E_b = F[6 * TILE_CMAX + s];
                        const double hm = (4.0 * a1) * mu_b * rcp_fast(a1 + mu_b);
                        const double cab = (F[4 * TILE_CMAX + s] * hm) * (Fbar * rinv);
                        acc0 = fma(cab, a0 - E_b, acc0);
                        acc1 += cab;
                        acc2 = fma(-cab, E_b, acc2);
                    }
                }
            }
            cur = nxt;
        }

        if (active) {
            const uint32_t ia = A.perm[i];
            if (SWEEP == SW_DENSITY) {
                A.o0[ia] = Wn * (acc0 + a0);         // self term m_a W(0; h_a): both shape functions are 1 at q = 0 (A11)
                if (A.ocount) A.ocount[ia] = ng;
            } else if (SWEEP == SW_HYDRO) {
                A.o0[ia] = acc0; A.o1[ia] = acc1; A.o2[ia] = acc2;
                A.o3[ia] = a1 * acc3 - acc4 * a0;    // eq. (17) 1st term P:L129 + eq. (42)
                if (A.o4) A.o4[ia] = acc3;
            } else if (SWEEP == SW_LIMITER) {
                // Larsen limiter, k = 2 (A20)
                const double rk = A.g0[i] * A.g1[i];
                const double gn = sqrt(acc0 * acc0 + acc1 * acc1 + acc2 * acc2);
                const double R = gn / (rk * a0);
                const double mu = A.c_light * (1.0 / sqrt(9.0 + R * R)) / rk;
                A.o0[ia] = mu;
                A.mu_sorted[i] = mu;
                if (A.o1) { A.o1[ia] = acc0; A.o1[A.n + ia] = acc1; A.o1[2 * A.n + ia] = acc2; }
            } else {
                A.o0[ia] = acc0;
                if (A.o1) A.o1[ia] = acc1;
                if (A.o2) A.o2[ia] = acc2;
            }
        }
    }
}

template <int SWEEP>
static cudaError_t launch_t(Ctx* c, const TiledArgs& a, cudaStream_t st) {
    constexpr size_t smem = sizeof(double) * NField<SWEEP>::v * TILE_CMAX;
    static bool attr_done = false;
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(k_tiled_sweep<SWEEP, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_tiled_sweep<SWEEP, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr_done = true;
    }
    CellTable ct{c->cell_start, c->cell_end};
    const int per_sm = (int)((220 * 1024) / (smem + sizeof(TileS) + 1024));
    const int grid = c->tl.sms * (per_sm < 1 ? 1 : (per_sm > 4 ? 4 : per_sm));
    if (c->kernel == SPRAY_KERNEL_WENDLAND_C2) k_tiled_sweep<SWEEP, 1><<<grid, TILE_T, smem, st>>>(c->dg, ct, a);
    else k_tiled_sweep<SWEEP, 0><<<grid, TILE_T, smem, st>>>(c->dg, ct, a);
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_tiled_sweep(Ctx* c, int sweep, TiledArgs a, cudaStream_t st) {
    if (c->n == 0) return cudaSuccess;
    a.tiles = c->tl.tiles; a.ntiles = c->tl.ntiles; a.lists = c->tl.lists; a.lcount = c->tl.lcount; a.tile_ok = c->tl.tile_ok;
    a.perm = c->perm; a.n = c->n;
    a.x = c->s.x; a.y = c->s.y; a.z = c->s.z; a.h = c->s.h;
    switch (sweep) {
        case SW_DENSITY: return launch_t<SW_DENSITY>(c, a, st);
        case SW_HYDRO: return launch_t<SW_HYDRO>(c, a, st);
        case SW_LIMITER: return launch_t<SW_LIMITER>(c, a, st);
        case SW_APPLY: return launch_t<SW_APPLY>(c, a, st);
    }
    return cudaErrorInvalidValue;
}

}  // namespace spray
