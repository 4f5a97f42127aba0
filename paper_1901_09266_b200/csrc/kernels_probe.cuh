// FP32 FFMA peak probe ("FP32 peak is not in MEASURED_PEAKS.json: builder must measure an FFMA peak").
// bench.py divides the FFMA-bound kernels' achieved TFLOP/s by this number instead of the nominal
// 148 SMs x 128 lanes x 2 x f_SM.  Not on the SPGD path.
#pragma once
#include <cuda_runtime.h>

namespace dode {

constexpr int kProbeChains = 8;       // independent FFMA chains per thread (FFMA latency 4 cycles x 4 schedulers' issue rate)
constexpr int kProbeInner = 64;       // FFMAs per chain per outer iteration (fully unrolled)

// 2 * kProbeChains * kProbeInner * outer flops per thread; operands come from memory so that nothing folds
__global__ void __launch_bounds__(1024, 2)
ffma_peak_probe(const float* __restrict__ in, float* __restrict__ out, int outer) {
    float a[kProbeChains];
    const float m = in[0], c = in[1];
#pragma unroll
    for (int j = 0; j < kProbeChains; ++j) a[j] = in[2] + (float)(threadIdx.x + j);
    for (int it = 0; it < outer; ++it) {
#pragma unroll
        for (int u = 0; u < kProbeInner; ++u)
#pragma unroll
            for (int j = 0; j < kProbeChains; ++j) a[j] = fmaf(a[j], m, c);
    }
    float s = 0.f;
#pragma unroll
    for (int j = 0; j < kProbeChains; ++j) s += a[j];
    if (s == 12345.678f) out[blockIdx.x * blockDim.x + threadIdx.x] = s;      // never true in practice: keeps the chains live
}

}  // namespace dode
