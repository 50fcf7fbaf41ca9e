// FP32 throughput micro-benchmark behind chime_bf_measure_fp32_peak: the denominator of the roofline bench.py reports
// ("the FFT flops at FP32 peak"), measured on the device instead of derived from unit counts and clocks.
#pragma once
#include <cuda_runtime.h>

namespace chime_peak {

// 16 independent accumulator chains per thread, 256 fused multiply-adds per thread and iteration; PACKED uses the
// fp32x2 instructions of sm_100 (two lanes per instruction).
template <bool PACKED>
__global__ void __launch_bounds__(512) fp32_peak_kernel(const int n_iter, float *sink) {
    float2 a[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) a[i] = make_float2(1.0f + 0.001f * (float)(threadIdx.x + i), 0.5f + 0.002f * (float)i);
    const float2 m = make_float2(0.999f, 1.001f), c = make_float2(1e-3f, -1e-3f);
#pragma unroll 1
    for (int it = 0; it < n_iter; ++it) {
#pragma unroll
        for (int r = 0; r < 16; ++r)
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                if constexpr (PACKED) a[i] = __ffma2_rn(a[i], m, c);
                else {
                    a[i].x = fmaf(a[i].x, m.x, c.x);
                    a[i].y = fmaf(a[i].y, m.y, c.y);
                }
            }
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += a[i].x + a[i].y;
    if (s == 123.456f) sink[threadIdx.x] = s;   // keeps the loops alive
}

}  // namespace chime_peak
