// probe.cu -- FP64 FMA throughput probe (measurement aid): 8 independent DFMA chains per thread.
// The roofline of the pair pass is the plain FP64 pipe; MEASURED_PEAKS.json has no FP64 entry, so bench.py measures
// the sustained DFMA rate with this kernel in the same job and quotes the pass against it.
#include "spray_internal.h"

namespace spray {

__global__ void __launch_bounds__(256) k_fp64_probe(int64_t iters, double* __restrict__ out) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    double a0 = 1.0 + t * 1e-9, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
    const double m = 1.0 - 1e-12, c = 1e-13;
#pragma unroll 1
    for (int64_t i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            a0 = __fma_rn(a0, m, c); a1 = __fma_rn(a1, m, c); a2 = __fma_rn(a2, m, c); a3 = __fma_rn(a3, m, c);
            a4 = __fma_rn(a4, m, c); a5 = __fma_rn(a5, m, c); a6 = __fma_rn(a6, m, c); a7 = __fma_rn(a7, m, c);
        }
    }
    out[t] = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
}

// one launch executes blocks*threads*iters*64 DFMA = 128*blocks*threads*iters flop
cudaError_t launch_fp64_probe(int blocks, int threads, int64_t iters, double* out, cudaStream_t st) {
    k_fp64_probe<<<blocks, threads, 0, st>>>(iters, out);
    return cudaGetLastError();
}

}  // namespace spray
