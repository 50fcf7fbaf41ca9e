// Packed integer butterflies of the time transform's first stage and the 128-point twiddle table.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace chime4 {

__constant__ float2 c_tw128[128];  // exp(-2 pi i k / 128), uploaded at plan creation
__constant__ float2 c_twr[8][16];  // [rho][u'] = exp(-2 pi i rho u' / 128): the same values in the order the time stage reads them
__constant__ float2 c_twr256[8][32];  // upchan 256: [rho][u'] = exp(-2 pi i rho u' / 256)
__constant__ float2 c_w32[16];        // upchan 256: exp(-2 pi i u / 32)

// a1: byte = ((re + 8) << 4) | (im + 8): the offset-binary real and imaginary parts of four inputs
// packed in one register, split by nibble masks into one value per byte.  This is THE decode of the hot path
// (int_bfly4 below) and what chime_bf_debug_unpack exposes for the bit-exact check.
__device__ __forceinline__ void split_nibbles(uint32_t w, uint32_t &re_off, uint32_t &im_off) {
    re_off = (w >> 4) & 0x0F0F0F0Fu;
    im_off = w & 0x0F0F0F0Fu;
}

// chime_bf_debug_unpack: byte -> (re, im) int8 through split_nibbles, four bytes per thread and step (the tail bytes of
// a length that is not a multiple of 4 are padded into a word).
__global__ void unpack_debug_kernel(const uint8_t *__restrict__ in, size_t n, int8_t *__restrict__ out) {
    const size_t nw = (n + 3) / 4, stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nw; i += stride) {
        uint32_t w = 0;
        const size_t nb = n - 4 * i < 4 ? n - 4 * i : 4;
        for (size_t b = 0; b < nb; ++b) w |= (uint32_t)in[4 * i + b] << (8 * b);
        uint32_t re_off, im_off;
        split_nibbles(w, re_off, im_off);
        for (size_t b = 0; b < nb; ++b) {
            out[2 * (4 * i + b)] = (int8_t)((int)((re_off >> (8 * b)) & 255u) - 8);
            out[2 * (4 * i + b) + 1] = (int8_t)((int)((im_off >> (8 * b)) & 255u) - 8);
        }
    }
}

// w[k] = 4 inputs' bytes of tap k (4 taps), summed with (-i)^{RHO4 k}: per output byte, value + 32 with
// value = sum_k x_k (-i)^{RHO4 k} (exact; |value| <= 32).
template <int RHO4>
__device__ __forceinline__ void int_bfly4(uint32_t w0, uint32_t w1, uint32_t w2, uint32_t w3,
                                          uint32_t &zr, uint32_t &zi) {
    constexpr uint32_t BIAS = 0x20202020u;
    uint32_t R0, I0, R1, I1, R2, I2, R3, I3;
    split_nibbles(w0, R0, I0);
    split_nibbles(w1, R1, I1);
    split_nibbles(w2, R2, I2);
    split_nibbles(w3, R3, I3);
    if constexpr (RHO4 == 0) {
        zr = R0 + R1 + R2 + R3;
        zi = I0 + I1 + I2 + I3;
    } else if constexpr (RHO4 == 1) {
        zr = (R0 + I1 + BIAS) - (R2 + I3);
        zi = (I0 + R3 + BIAS) - (R1 + I2);
    } else if constexpr (RHO4 == 2) {
        zr = (R0 + R2 + BIAS) - (R1 + R3);
        zi = (I0 + I2 + BIAS) - (I1 + I3);
    } else {
        zr = (R0 + I3 + BIAS) - (R2 + I1);
        zi = (I0 + R1 + BIAS) - (I2 + R3);
    }
}

}  // namespace chime4
