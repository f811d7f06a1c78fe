// rad.cu -- row N1: the per-particle part of the implicit radiation step, section 2.3.
// The pair work of every Jacobi iteration is the FLD operator apply (sweeps_tiled.cu, eqs. (51)-(52)); what is left per
// particle is the quartic eq. (57) for chi (eq. (56)), then u by eq. (56) and E by eq. (55), and the residual of eq. (49)
// of the iterate that entered the iteration.
#include "spray_internal.h"

namespace spray {

// positive root of x^4 + b x + c = 0, b > 0, c < 0: Newton from the upper bound min((-c)^(1/4), -c/b); f is convex and
// increasing on x > 0, so the iterates fall monotonically to the root; the bound is within a factor 2 of it and 7 steps
// reach rounding error over the whole range (6 suffice on a 14-decade sweep of (b, c)).  The paper's closed form, eqs.
// (58)-(60), is the same number but cancels catastrophically when the root is small (A25).
__device__ __forceinline__ double quartic_positive_root(double b, double c) {
    double x = fmin(sqrt(sqrt(-c)), -c / b);
#pragma unroll
    for (int it = 0; it < 7; ++it) {
        const double x2 = x * x, x3 = x2 * x;
        const double f = fma(x3, x, fma(b, x, c)), fp = fma(4.0, x3, b);
        x -= f / fp;
    }
    return x;
}

__global__ void __launch_bounds__(256)
k_rad_update(RadArgs A, const uint32_t* __restrict__ perm, int64_t n) {
    double rmax = 0.0;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const uint32_t ia = perm[i];                 // sorted slot i <-> caller index ia
        const double rho = A.rho[ia], kp = A.kappa_p[ia], En = A.E_n[ia], un = A.u_n[ia], Tn = A.T_n[ia], dTdu = A.dTdu[ia];
        const double lam = A.lam[ia], gam = A.gam[ia];
        const double K = A.dt * A.c_light * kp;      // denominator of eq. (55)
        const double X = A.dt * rho * A.c_light * kp;
        if (!A.first && A.resid) {                   // both sides of eq. (49) for the iterate that enters this iteration
            const double Ecur = A.E[ia], chi0 = A.chi[ia];
            const double c2 = chi0 * chi0;
            const double rhs = En + A.dt * (lam * Ecur + gam) + X * (A.a_rad * (c2 * c2) - Ecur);
            rmax = fmax(rmax, fabs(Ecur - rhs) / fabs(Ecur));
        }
        const double D = 1.0 - A.dt * lam;
        const double Bq = (D + X) / K / dTdu;        // coefficient of chi in eq. (57)
        const double Aq = D * A.a_rad;
        const double Cq = En + A.dt * gam + Bq * Tn;
        const double chi = quartic_positive_root(Bq / Aq, -Cq / Aq);
        const double unew = un + (chi - Tn) / dTdu;  // eq. (56)
        const double ch2 = chi * chi;
        const double Enew = (unew - un) / K + A.a_rad * (ch2 * ch2);     // eq. (55)
        A.E[ia] = Enew; A.u[ia] = unew; A.chi[ia] = chi;
        A.me[i].y = Enew;                            // the next apply reads the iterate from the sorted records
        A.sE[i] = Enew;
    }
    if (A.resid) {                                   // max is exact and order independent: deterministic
        for (int o = 16; o; o >>= 1) rmax = fmax(rmax, __shfl_xor_sync(0xFFFFFFFFu, rmax, o));
        if ((threadIdx.x & 31) == 0 && rmax > 0.0)
            atomicMax((unsigned long long*)A.resid, (unsigned long long)__double_as_longlong(rmax));
    }
}

// N2: dudt_a = y_a / rho_a (the 1/rho_a prefactor of the conduction term, eqs. (17)/(18) P:L129-L132)
__global__ void k_div_by_rho(double* __restrict__ y, const double* __restrict__ rho, int64_t n) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) y[i] = y[i] / rho[i];
}
cudaError_t launch_div_by_rho(Ctx* c, double* y, const double* rho, cudaStream_t st) {
    if (c->n == 0) return cudaSuccess;
    const int64_t want = (c->n + 255) / 256;
    k_div_by_rho<<<(int)(want < 148 * 32 ? want : 148 * 32), 256, 0, st>>>(y, rho, c->n);
    c->launches += 1;
    return cudaGetLastError();
}

// N2, implicit two-temperature system: per-particle parts of eqs. (28)-(34)
__global__ void k_cond_form(CondArgs a, int64_t n) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const double gi = a.tau_i[i] * a.u_i[i], ge = a.tau_e[i] * a.u_e[i];
        a.g_i[i] = a.rhs ? a.T_i[i] - gi : gi;
        a.g_e[i] = a.rhs ? a.T_e[i] - ge : ge;
    }
}
__global__ void k_cond_combine(CondArgs a, int64_t n) {
    const double sdt = a.rhs ? a.dt : -a.dt;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const double rinv = 1.0 / a.rho[i];
        const double X = a.kei[i] * (a.g_e[i] - a.g_i[i]);       // exchange term of eqs. (26)/(27) on g
        a.out_i[i] = fma(sdt, fma(a.y_i[i], rinv, X), a.u_i[i]);
        a.out_e[i] = fma(sdt, fma(a.y_e[i], rinv, -X), a.u_e[i]);
    }
}
static int cond_blocks(int64_t n) { const int64_t want = (n + 255) / 256; return (int)(want < 148 * 32 ? want : 148 * 32); }
cudaError_t launch_cond_form(Ctx* c, const CondArgs& a, cudaStream_t st) {
    if (c->n == 0) return cudaSuccess;
    k_cond_form<<<cond_blocks(c->n), 256, 0, st>>>(a, c->n);
    c->launches += 1;
    return cudaGetLastError();
}
cudaError_t launch_cond_combine(Ctx* c, const CondArgs& a, cudaStream_t st) {
    if (c->n == 0) return cudaSuccess;
    k_cond_combine<<<cond_blocks(c->n), 256, 0, st>>>(a, c->n);
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_rad_update(Ctx* c, const RadArgs& a, cudaStream_t st) {
    if (c->n == 0) return cudaSuccess;
    const int64_t want = (c->n + 255) / 256;
    const int blocks = (int)(want < 148 * 32 ? want : 148 * 32);
    k_rad_update<<<blocks, 256, 0, st>>>(a, c->perm, c->n);
    c->launches += 1;
    return cudaGetLastError();
}

}  // namespace spray
