// common.cuh -- device-side helpers shared by the CUDA kernels of libspray_b200 (sm_100a).
// Not shared with oracle/: the oracle is an independent C translation unit.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace spray {

struct DevGrid {
    double lo[3];
    double inv[3];    // ncell_d / L_d  (one fp64 division on the host, same as the contract O1)
    double L[3];      // hi_d - lo_d
    double halfL[3];  // 0.5 * L_d
    double edge[3];   // L_d / ncell_d: cell edge (tile geometry only, never in a set decision)
    int nc[3];
    int per[3];
};

enum SweepId { SW_DENSITY = 0, SW_HYDRO = 1, SW_LIMITER = 2, SW_APPLY = 3, SW_HSEARCH = 4, SW_COUNT = 5, SW_LIST = 6, SW_DIGEST = 7, SW_KGC = 8, SW_GRADN = 9, SW_HYDLIM = 10 };

constexpr double kPi = 3.14159265358979323846264338327950288;
constexpr double kSigmaCubic = 1.0 / kPi;            // M4 cubic spline, 3-D (A1)
constexpr double kSigmaWend = 21.0 / (16.0 * kPi);   // Wendland C2, 3-D, eq. (3)

// The tiled kernels evaluate the kernels through rescaled shape functions (sweeps_tiled.cu):
//   cubic:    W = kWnCubic / h^3 * (t2^3 - t1^3),  t2 = 2 - q, t1 = cbrt(4) (1 - q)_+ ;  F = kFnCubic / h^4 * (s1^2 - t2^2), s1 = (2 - 2q)_+
//   Wendland: W = kWnWend / h^3 * t^4 (2q + 1),    t = (1 - q/2)_+ ;                     F = kFnWend / h^4 * q t^3
constexpr double kWnCubic = 0.25 * kSigmaCubic;
constexpr double kFnCubic = 0.75 * kSigmaCubic;
constexpr double kWnWend = kSigmaWend;
constexpr double kFnWend = -5.0 * kSigmaWend;

__device__ __forceinline__ double dmax0(double a) { return a > 0.0 ? a : 0.0; }
// max(a, 0) without the FP64 pipe: clamp the (signed) high word at 0.  A negative a becomes a denormal < 2.2e-308
// (its low word survives), which is 0 at any tolerance; -0.0 and NaN handling do not matter to the callers.
__device__ __forceinline__ double dmax0_fast(double a) {
    const int hi = __double2hiint(a), lo = __double2loint(a);
    return __hiloint2double(max(hi, 0), lo);
}

// ---- kernel shape functions of q = r/h, clamped so that they vanish identically for q >= 2 ("0 for q >= 2").
// W(r;h) = sigma/h^3 * w(q);  F(r;h) = dW/dr = sigma/h^4 * f(q)
template <int KERNEL>
__device__ __forceinline__ double shape_w(double q) {
    if (KERNEL == 1) {                       // Wendland C2: (1-q/2)^4 (2q+1)
        double t = dmax0(1.0 - 0.5 * q);
        double t2 = t * t;
        return t2 * t2 * (2.0 * q + 1.0);
    } else {                                 // cubic spline: 1/4 (2-q)^3 - (1-q)^3  [second term only for q < 1]
        double t2 = dmax0(2.0 - q), t1 = dmax0(1.0 - q);
        return 0.25 * t2 * t2 * t2 - t1 * t1 * t1;
    }
}
template <int KERNEL>
__device__ __forceinline__ double shape_f(double q) {
    if (KERNEL == 1) {                       // d/dq: -5 q (1-q/2)^3
        double t = dmax0(1.0 - 0.5 * q);
        return -5.0 * q * (t * t * t);
    } else {                                 // d/dq: -3/4 (2-q)^2 + 3 (1-q)^2
        double t2 = dmax0(2.0 - q), t1 = dmax0(1.0 - q);
        return 3.0 * t1 * t1 - 0.75 * t2 * t2;
    }
}
template <int KERNEL>
__device__ __forceinline__ double sigma() { return KERNEL == 1 ? kSigmaWend : kSigmaCubic; }

// ---- the neighbour predicate pieces, bit-for-bit the contract expression (O2/A12):
//   dx = x_a - x_b;  periodic: if (dx > L/2) dx -= L; else if (dx < -L/2) dx += L;
//   r2 = fma(dz,dz, fma(dy,dy, dx*dx));   b in N(a)  <=>  r2 < 4*(h*h)
__device__ __forceinline__ double min_image(double d, int per, double L, double halfL) {
    if (per) {
        if (d > halfL) d = __dsub_rn(d, L);
        else if (d < -halfL) d = __dadd_rn(d, L);
    }
    return d;
}
__device__ __forceinline__ double r2_exact(double dx, double dy, double dz) {
    return __fma_rn(dz, dz, __fma_rn(dy, dy, __dmul_rn(dx, dx)));
}
__device__ __forceinline__ double support2(double h) { return __dmul_rn(4.0, __dmul_rn(h, h)); }

__device__ __forceinline__ uint64_t mix64(uint64_t x) {   // splitmix64 finaliser (digest export only)
    x += 0x9E3779B97F4A7C15ull;
    x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
    x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
    return x ^ (x >> 31);
}

}  // namespace spray
