// Register-resident radix-2 DIF FFTs with compile-time twiddles (forward transform, exp(-2 pi i ...)).
// Complex values live in aligned register pairs and all arithmetic is written with the packed
// fp32x2 intrinsics (FADD2 / FMUL2 / FFMA2 on sm_100): ptxas folds the (y, x) swaps, per-half negations
// and scalar broadcasts into operand modifiers, so a complex add is one instruction and a complex
// multiply two -- half the issue slots of scalar code at the same fp32 pipe throughput.
// After fft_dif<N>(a), a[i] holds output bin bitrev<N>(i).  All loops unroll fully, so register
// indices, twiddle constants and the trivial-twiddle shortcuts are resolved at compile time.
#pragma once
#include <cuda_runtime.h>

namespace chime {

// cos(2 pi k / 64), k = 0..16 (quarter wave); everything else by symmetry.
__device__ constexpr float kCos64[17] = {
    1.0f,
    0.99518472667219688624f,
    0.98078528040323044913f,
    0.95694033573220886494f,
    0.92387953251128675613f,
    0.88192126434835502971f,
    0.83146961230254523708f,
    0.77301045336273696081f,
    0.70710678118654752440f,
    0.63439328416364549822f,
    0.55557023301960222474f,
    0.47139673682599764856f,
    0.38268343236508977173f,
    0.29028467725446236764f,
    0.19509032201612826785f,
    0.09801714032956060199f,
    0.0f};

__device__ __forceinline__ constexpr float cos64(int t) {
    t &= 63;
    return t <= 16 ? kCos64[t] : t <= 32 ? -kCos64[32 - t] : t <= 48 ? -kCos64[t - 32] : kCos64[64 - t];
}
__device__ __forceinline__ constexpr float sin64(int t) { return cos64(t - 16); }

__host__ __device__ __forceinline__ constexpr int bitrev(int i, int bits) {
    int r = 0;
    for (int b = 0; b < bits; ++b) r |= ((i >> b) & 1) << (bits - 1 - b);
    return r;
}

__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return __fadd2_rn(a, make_float2(-b.x, -b.y)); }

// a * b = a (b.x, b.x) + (a.y, a.x) (-b.y, b.y)
__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
    const float2 t = __fmul2_rn(make_float2(a.y, a.x), make_float2(-b.y, b.y));
    return __ffma2_rn(a, make_float2(b.x, b.x), t);
}

// d * exp(-2 pi i t / 64) with the trivial cases folded.
template <int T64>
__device__ __forceinline__ float2 twiddle64(float2 d) {
    if constexpr (T64 == 0) {
        return d;
    } else if constexpr (T64 == 16) {  // -i
        return make_float2(d.y, -d.x);
    } else if constexpr (T64 == 32) {  // -1
        return make_float2(-d.x, -d.y);
    } else if constexpr (T64 == 48) {  // +i
        return make_float2(-d.y, d.x);
    } else if constexpr (T64 == 8) {  // (1 - i)/sqrt2 : ((x + y) h, (y - x) h)
        constexpr float h = 0.70710678118654752440f;
        return __fmul2_rn(__fadd2_rn(d, make_float2(d.y, -d.x)), make_float2(h, h));
    } else if constexpr (T64 == 24) {  // (-1 - i)/sqrt2 : ((y - x) h, -(x + y) h)
        constexpr float h = 0.70710678118654752440f;
        return __fmul2_rn(__fadd2_rn(make_float2(d.y, -d.x), make_float2(-d.x, -d.y)), make_float2(h, h));
    } else {
        constexpr float c = cos64(T64), s = sin64(T64);  // multiply by (c - i s): d (c, c) + (d.y, d.x) (s, -s)
        const float2 t = __fmul2_rn(make_float2(d.y, d.x), make_float2(s, -s));
        return __ffma2_rn(d, make_float2(c, c), t);
    }
}

template <int N, int S, int BLK, int K>
__device__ __forceinline__ void bfly(float2 (&a)[N]) {
    constexpr int i = BLK + K, j = i + S;
    const float2 u = a[i], v = a[j];
    a[i] = cadd(u, v);
    a[j] = twiddle64<K*(32 / S)>(csub(u, v));
}

template <int N, int S, int IDX>
__device__ __forceinline__ void stage(float2 (&a)[N]) {
    // IDX enumerates the N/2 butterflies of the stage with half-span S
    if constexpr (IDX < N / 2) {
        constexpr int blk = (IDX / S) * 2 * S, k = IDX % S;
        bfly<N, S, blk, k>(a);
        stage<N, S, IDX + 1>(a);
    }
}

template <int N, int S>
__device__ __forceinline__ void stages(float2 (&a)[N]) {
    if constexpr (S >= 1) {
        stage<N, S, 0>(a);
        stages<N, S / 2>(a);
    }
}

template <int N>
__device__ __forceinline__ void fft_dif(float2 (&a)[N]) {
    static_assert(N == 2 || N == 4 || N == 8 || N == 16 || N == 32 || N == 64, "N");
    stages<N, N / 2>(a);
}

template <int N>
__host__ __device__ __forceinline__ constexpr int log2c() {
    int b = 0;
    for (int n = N; n > 1; n >>= 1) ++b;
    return b;
}

}  // namespace chime
