// Second-generation fused CHIME/FRB beamformer kernel for sm_100a (zero_pad = 512, upchan_len = 128).
// Steps a1-a10 of include/chime_bf.h in one launch; HBM sees the packed input once and the output once.
//
// Work decomposition: one CTA (512 threads, 1 CTA/SM) per (coarse channel c, output frame R, E-W beam
// pair ep).  For each of the 3 blocks of U = 128 samples and each polarisation it
//   stage    copies the raw 4+4-bit block [128 t][4 cyl][256 B] (128 KiB) into XOR-swizzled shared
//            memory once; it is then re-read 8 times from there, never from L2/HBM,
// and loops over the 8 residues rho of a decimation-in-frequency split of the 128-point time transform
//     S[8 q' + rho] = sum_{u'<16} W_16^{q'u'} { W_128^{rho u'} sum_{k<8} Z[u' + 16 k] W_8^{rho k} } :
//   phase A  (thread <-> MMA fragment lane): the 8-tap butterfly runs on the raw integers, packed four
//            feeds per register (exact; the 1/sqrt2 of odd rho is deferred to fp32).  The results are
//            turned into fp16 pairs (exact) and contracted with the folded gain x E-W weights on the
//            tensor cores: per feed n a 16 x 8 x 8 mma.sync (rows = time, k = cyl x re/im, cols = beam
//            x re/im) with the weights split hi + lo in fp16, fp32 accumulation  -> tile[u'][e][n]
//   phase B  (warp <-> row, half-warp <-> even/odd bins): zero-padded 512-point N-S transform as two
//            radix-16x16 FFT-256 with all twiddles in registers; the even half exchanges through the
//            row's own storage, the odd half through a 2 KiB per-warp buffer; selected bins are
//            written back in place as tile[u'][e][slot]
//   phase C  (thread <-> (beam, slot)): 16-point time FFT in registers, |.|^2, accumulation over
//            (block, pol, rho) in 16 registers (output q' <-> fine channel (q'+8) mod 16)
// epilogue: normalise, quantise (cvt.rni + saturate), 16-byte store per beam.
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "fft_regs.cuh"

namespace chime2 {

using chime::bitrev;
using chime::cmul;
using chime::fft_dif;

constexpr int kThreads = 512;
constexpr int kWarps = kThreads / 32;
constexpr int kRowsT = 16;                       // u' rows per sub-tile
constexpr int kTileRows = kRowsT * 2;            // x 2 beams of the pair
constexpr int kRawBytes = 128 * 4 * 256;         // one (block, pol): 128 KiB
constexpr int kTileBytes = kTileRows * 256 * 8;  // 64 KiB
constexpr int kExchBytes = kWarps * 256 * 8;     // 32 KiB
constexpr int kSmemBytes = kRawBytes + kTileBytes + kExchBytes + 512 * 2 + 256 * 2 + 16;
constexpr int kTmemCols = 256;                   // 4 warps per lane quarter x 64 fp32 columns

struct Params {
    const uint8_t *in;        // [C][T][2048]
    uint8_t *out_u8;          // [C][R][4][256][16]
    float *out_f32;           // same layout, or nullptr
    const uint2 *bfrag;       // [C][pol 2][ep 2][n 256][16] (hi, lo) half2 bit patterns, B fragments
    const int16_t *slot;      // [C][512] bin -> slot or -1
    const int16_t *slot_of_m; // [C][256] beam -> slot
    const float2 *tw_np;      // [512] exp(-2 pi i k / 512)
    int n_time;
    int n_frames;
    int chan0;                // first channel this launch processes
    int frame0, n_frames_launch;   // frame range of this launch within each channel
    uint8_t *const *peer_out;      // beam-major exchange (see chime::beam_major_dst), nullptr = off
    int n_peers, chan_global0;
    float norm, qscale, qoffset;
};

__constant__ float2 c_tw128[128];  // exp(-2 pi i k / 128), uploaded at plan creation

// physical float2 index of logical element idx of tile row r (XOR swizzle of 16-byte chunks)
__device__ __forceinline__ int tile_idx(int r, int idx) {
    return r * 256 + (idx & ~15) + (((((idx >> 1) & 7) ^ (r & 7))) << 1) + (idx & 1);
}

// ---- packed integer butterflies ---------------------------------------------------------------
// w[k] = 4 feeds' bytes of tap k (4 taps).  Per byte: value + 32, value = sum_k x_k (-i)^{RHO4 k}.
template <int RHO4>
__device__ __forceinline__ void int_bfly4(uint32_t w0, uint32_t w1, uint32_t w2, uint32_t w3,
                                          uint32_t &zr, uint32_t &zi) {
    constexpr uint32_t M = 0x0F0F0F0Fu, BIAS = 0x20202020u;
    const uint32_t R0 = (w0 >> 4) & M, I0 = w0 & M, R1 = (w1 >> 4) & M, I1 = w1 & M;
    const uint32_t R2 = (w2 >> 4) & M, I2 = w2 & M, R3 = (w3 >> 4) & M, I3 = w3 & M;
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

// O' = c_RHO * O on biased bytes (in: value + 32 per byte), c_RHO = W_8^RHO without its 1/sqrt2:
// 1, 1-i, -i, -1-i, -1, -1+i, i, 1+i.  Output biases are rot_bias_r/i<RHO>() (all bytes stay < 128).
template <int RHO>
__device__ __forceinline__ void rot8(uint32_t br, uint32_t bi, uint32_t &pr, uint32_t &pi) {
    constexpr uint32_t H40 = 0x40404040u, H7F = 0x7F7F7F7Fu;
    if constexpr (RHO == 0) { pr = br; pi = bi; }
    else if constexpr (RHO == 1) { pr = br + bi; pi = (bi + H40) - br; }
    else if constexpr (RHO == 2) { pr = bi; pi = H40 - br; }
    else if constexpr (RHO == 3) { pr = (bi + H40) - br; pi = H7F - (br + bi); }
    else if constexpr (RHO == 4) { pr = H40 - br; pi = H40 - bi; }
    else if constexpr (RHO == 5) { pr = H7F - (br + bi); pi = (br + H40) - bi; }
    else if constexpr (RHO == 6) { pr = H40 - bi; pi = br; }
    else { pr = (br + H40) - bi; pi = br + bi; }
}
template <int RHO> __host__ __device__ constexpr int rot_bias_r() {
    return (RHO == 0 || RHO == 2 || RHO == 4 || RHO == 6) ? 32 : (RHO == 5 ? 63 : 64);
}
template <int RHO> __host__ __device__ constexpr int rot_bias_i() {
    return (RHO == 0 || RHO == 2 || RHO == 4 || RHO == 6) ? 32 : (RHO == 3 ? 63 : 64);
}

// bytes B of zr / zi (each < 128) -> half2 (re, im) = ((byte - bias) * 2^-9), exact: the bytes are read
// as fp16 subnormals (byte * 2^-24), scaled by 2^15 and shifted in one fused multiply-add.
template <int B>
__device__ __forceinline__ uint32_t bytes_to_half2(uint32_t zr, uint32_t zi, __half2 negbias) {
    // selector: byte0 = zr.B, byte1 = sign(zr.B) = 0, byte2 = zi.B, byte3 = sign(zi.B) = 0
    constexpr uint32_t sel = (uint32_t)B | ((8u | B) << 4) | ((4u + B) << 8) | ((8u | (4u + B)) << 12);
    uint32_t u;  // raw prmt: selector bit 3 replicates the byte's sign bit (0 here), which __byte_perm masks off
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(u) : "r"(zr), "r"(zi), "r"(sel));
    const __half2 s = __halves2half2(__ushort_as_half(0x7800), __ushort_as_half(0x7800));  // 2^15
    const __half2 v = __hfma2(*reinterpret_cast<const __half2 *>(&u), s, negbias);
    return *reinterpret_cast<const uint32_t *>(&v);
}

__device__ __forceinline__ void mma_m16n8k8(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t b) {
    asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5}, {%6}, {%0,%1,%2,%3};\n"
                 : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
                 : "r"(a0), "r"(a1), "r"(b));
}

// ---- tensor memory as a per-thread parking lot (32x32b shape: lane i of the warp <-> TMEM lane base + i) ----
__device__ __forceinline__ void tmem_st8(uint32_t taddr, float a0, float a1, float a2, float a3, float a4,
                                         float a5, float a6, float a7) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                 :: "r"(taddr), "f"(a0), "f"(a1), "f"(a2), "f"(a3), "f"(a4), "f"(a5), "f"(a6), "f"(a7) : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, float *v) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 "
                 "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,"
                 "%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
                 : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[4]), "=f"(v[5]), "=f"(v[6]), "=f"(v[7]),
                   "=f"(v[8]), "=f"(v[9]), "=f"(v[10]), "=f"(v[11]), "=f"(v[12]), "=f"(v[13]), "=f"(v[14]), "=f"(v[15]),
                   "=f"(v[16]), "=f"(v[17]), "=f"(v[18]), "=f"(v[19]), "=f"(v[20]), "=f"(v[21]), "=f"(v[22]), "=f"(v[23]),
                   "=f"(v[24]), "=f"(v[25]), "=f"(v[26]), "=f"(v[27]), "=f"(v[28]), "=f"(v[29]), "=f"(v[30]), "=f"(v[31])
                 : "r"(taddr) : "memory");
}

// ---- phase A ---------------------------------------------------------------------------------------
// Warp w owns feeds n = 16 w .. 16 w + 15; lane = 4 g + tq is the mma fragment lane: time rows u' = g and
// g + 8, cylinder tq.  raw: [piece p = 4 t + cyl][256 B], 8-byte units XOR-swizzled with (p & 15).
template <int RHO>
__device__ __forceinline__ void phase_a(const unsigned char *raw, float2 *tile, const uint2 *bfrag_cpe,
                                        const int warp, const int lane, const uint32_t taddr) {
    constexpr bool ODD = (RHO & 1) != 0;
    const int g = lane >> 2, tq = lane & 3;
    const __half2 nbE = __floats2half2_rn(-32.0f / 512.0f, -32.0f / 512.0f);
    const __half2 nbO = __floats2half2_rn(-(float)rot_bias_r<RHO>() / 512.0f, -(float)rot_bias_i<RHO>() / 512.0f);
    const bool has_b = g < 4;               // B columns 4..7 are zero
    const bool stores = tq < 2;             // C columns 0..3 = (e' = tq, re/im)
    const int r0 = g * 2 + tq;              // tile row of (u' = g, e' = tq); u' = g + 8 -> r0 + 16

    // raw address of (u' = g + 8 hr, tap k): piece p = 4 (g + 8 hr + 16 k) + tq, and p & 15 = 4 (g & 3) + tq
    // for every (hr, k), so the swizzled unit is a per-thread constant and (hr, k) are immediate offsets.
    const int pz = 4 * (g & 3) + tq;
    const unsigned char *raw_t = raw + (4 * g + tq) * 256;
    // tile address of (row r0 [+16], feed n): n >> 1 = 8 warp + 4 hh + i / 2, so the swizzled 16-byte chunk is
    // ((4 hh + i / 2) ^ (r0 & 7)); byte offset = row + line(n >> 4 = warp) * 128 + chunk * 16.
    unsigned char *tile_t = reinterpret_cast<unsigned char *>(tile) + r0 * 2048 + warp * 128;
    const int rx16 = (r0 & 7) << 4;

#pragma unroll
    for (int hh = 0; hh < 2; ++hh) {        // 8 feeds at a time
        uint32_t aE[2][8], aO[2][8];
        const unsigned char *raw_h = raw_t + (((2 * warp + hh) ^ pz) << 3);
#pragma unroll
        for (int hr = 0; hr < 2; ++hr) {
            uint2 q[8];
#pragma unroll
            for (int k = 0; k < 8; ++k)
                q[k] = *reinterpret_cast<const uint2 *>(raw_h + (32 * hr + 64 * k) * 256);
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                uint32_t er, ei, orr, oi, pr, pi;
                if (j == 0) {
                    int_bfly4<RHO & 3>(q[0].x, q[2].x, q[4].x, q[6].x, er, ei);
                    int_bfly4<RHO & 3>(q[1].x, q[3].x, q[5].x, q[7].x, orr, oi);
                } else {
                    int_bfly4<RHO & 3>(q[0].y, q[2].y, q[4].y, q[6].y, er, ei);
                    int_bfly4<RHO & 3>(q[1].y, q[3].y, q[5].y, q[7].y, orr, oi);
                }
                rot8<RHO>(orr, oi, pr, pi);
                aE[hr][4 * j + 0] = bytes_to_half2<0>(er, ei, nbE);
                aE[hr][4 * j + 1] = bytes_to_half2<1>(er, ei, nbE);
                aE[hr][4 * j + 2] = bytes_to_half2<2>(er, ei, nbE);
                aE[hr][4 * j + 3] = bytes_to_half2<3>(er, ei, nbE);
                aO[hr][4 * j + 0] = bytes_to_half2<0>(pr, pi, nbO);
                aO[hr][4 * j + 1] = bytes_to_half2<1>(pr, pi, nbO);
                aO[hr][4 * j + 2] = bytes_to_half2<2>(pr, pi, nbO);
                aO[hr][4 * j + 3] = bytes_to_half2<3>(pr, pi, nbO);
            }
        }
        const int n0 = 16 * warp + 8 * hh;
        uint2 bw[8];
#pragma unroll
        for (int i = 0; i < 8; ++i)
            bw[i] = has_b ? __ldg(bfrag_cpe + (size_t)(n0 + i) * 16 + lane) : make_uint2(0u, 0u);
#pragma unroll
        for (int i = 0; i < 8; i += 2) {
            float z[2][4], zh[2][4];
#pragma unroll
            for (int ii = 0; ii < 2; ++ii) {
                float pacc[4] = {0.f, 0.f, 0.f, 0.f}, qacc[4] = {0.f, 0.f, 0.f, 0.f};
                mma_m16n8k8(pacc, aE[0][i + ii], aE[1][i + ii], bw[i + ii].x);
                mma_m16n8k8(pacc, aE[0][i + ii], aE[1][i + ii], bw[i + ii].y);
                mma_m16n8k8(qacc, aO[0][i + ii], aO[1][i + ii], bw[i + ii].x);
                mma_m16n8k8(qacc, aO[0][i + ii], aO[1][i + ii], bw[i + ii].y);
                constexpr float s = ODD ? 0.70710678118654752440f : 1.0f;
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    z[ii][c] = fmaf(s, qacc[c], pacc[c]);    // residue RHO:      E + W_8^RHO O
                    zh[ii][c] = fmaf(-s, qacc[c], pacc[c]);  // residue RHO + 4:  E - W_8^RHO O
                }
            }
            if (stores) {
                unsigned char *dst = tile_t + (rx16 ^ ((4 * hh + i / 2) << 4));
                *reinterpret_cast<float4 *>(dst) = make_float4(z[0][0], z[0][1], z[1][0], z[1][1]);
                *reinterpret_cast<float4 *>(dst + 16 * 2048) = make_float4(z[0][2], z[0][3], z[1][2], z[1][3]);
            }
            // stash the RHO + 4 tile values in this thread's tensor-memory lane (32 columns per hh)
            tmem_st8(taddr + 32 * hh + 4 * i, zh[0][0], zh[0][1], zh[1][0], zh[1][1], zh[0][2], zh[0][3], zh[1][2], zh[1][3]);
        }
    }
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}

// Phase A of residue RHO + 4: the tile values were computed with residue RHO (same integer butterflies,
// same tensor-core products, opposite sign of the odd-tap half) and parked in tensor memory.
__device__ __forceinline__ void phase_a_from_tmem(float2 *tile, const uint32_t taddr, const int warp, const int lane) {
    const int g = lane >> 2, tq = lane & 3;
    const int r0 = g * 2 + tq;
    unsigned char *tile_t = reinterpret_cast<unsigned char *>(tile) + r0 * 2048 + warp * 128;
    const int rx16 = (r0 & 7) << 4;
    float v[64];
    tmem_ld32(taddr, v);
    tmem_ld32(taddr + 32, v + 32);
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
    if (tq < 2) {
#pragma unroll
        for (int hh = 0; hh < 2; ++hh)
#pragma unroll
            for (int i = 0; i < 8; i += 2) {
                const float *w = v + 32 * hh + 4 * i;
                unsigned char *dst = tile_t + (rx16 ^ ((4 * hh + i / 2) << 4));
                *reinterpret_cast<float4 *>(dst) = make_float4(w[0], w[1], w[2], w[3]);
                *reinterpret_cast<float4 *>(dst + 16 * 2048) = make_float4(w[4], w[5], w[6], w[7]);
            }
    }
}

// ---- phase B: one tile row (256 feeds of one (u', e')) -> its selected N-S bins, in place ------------
// Half-warp h computes the bins of parity h: FFT-256 of a[n] W_512^{h n}.  twc[j2] = W_512^{l (2 j2 + h)}
// merges the inter-stage twiddle W_256^{l j2} with the lane part W_512^{h l} of the pre-twiddle; the
// rest of the pre-twiddle, W_32^{h k}, has compile-time arguments.
// All shared-memory addresses are (per-thread constant) XOR (immediate) + immediate:
//   row read      row + 128 k + rd,            rd = (((l>>1) ^ rx) << 4) | ((l&1) << 3)
//   exch write    ex + 128 j2 + (wr ^ ((j2&7) << 4)),  wr = (((l>>1) ^ x) << 4) | ((l&1) << 3)
//   exch read     ex + (er ^ (i << 4)),        er = 128 l | (((l&7) ^ x) << 4)
// with rx = r & 7 (the row's swizzle; identical for the warp's two rows r and r + 16), x = rx (even half,
// exchanging through the row) or 0 (odd half, private buffer).
// s_sel[(16 h + l) * 16 + i] = 8 * slot of bin 2 (16 bitrev(i) + l) + h, or 0x8000 (not selected).
// a[k] *= W_32^k (the compile-time part of the odd-bin pre-twiddle W_512^{l + 16 k})
__device__ __forceinline__ void w32_pretwiddle(float2 (&a)[16]) {
    a[1] = chime::twiddle64<2>(a[1]);   a[2] = chime::twiddle64<4>(a[2]);   a[3] = chime::twiddle64<6>(a[3]);
    a[4] = chime::twiddle64<8>(a[4]);   a[5] = chime::twiddle64<10>(a[5]);  a[6] = chime::twiddle64<12>(a[6]);
    a[7] = chime::twiddle64<14>(a[7]);  a[8] = chime::twiddle64<16>(a[8]);  a[9] = chime::twiddle64<18>(a[9]);
    a[10] = chime::twiddle64<20>(a[10]); a[11] = chime::twiddle64<22>(a[11]); a[12] = chime::twiddle64<24>(a[12]);
    a[13] = chime::twiddle64<26>(a[13]); a[14] = chime::twiddle64<28>(a[14]); a[15] = chime::twiddle64<30>(a[15]);
}

__device__ __forceinline__ void phase_b_row(unsigned char *S, const int rowofs, const int exofs, const int h,
                                            const int rd, const int wr, const int er,
                                            const uint4 sel0, const uint4 sel1, const float2 (&twc)[16]) {
    float2 a[16];
    const int ra = rowofs + rd;
#pragma unroll
    for (int k = 0; k < 16; ++k) a[k] = *reinterpret_cast<const float2 *>(S + (ra + 128 * k));
    if (h) {
        a[1] = chime::twiddle64<2>(a[1]);   a[2] = chime::twiddle64<4>(a[2]);   a[3] = chime::twiddle64<6>(a[3]);
        a[4] = chime::twiddle64<8>(a[4]);   a[5] = chime::twiddle64<10>(a[5]);  a[6] = chime::twiddle64<12>(a[6]);
        a[7] = chime::twiddle64<14>(a[7]);  a[8] = chime::twiddle64<16>(a[8]);  a[9] = chime::twiddle64<18>(a[9]);
        a[10] = chime::twiddle64<20>(a[10]); a[11] = chime::twiddle64<22>(a[11]); a[12] = chime::twiddle64<24>(a[12]);
        a[13] = chime::twiddle64<26>(a[13]); a[14] = chime::twiddle64<28>(a[14]); a[15] = chime::twiddle64<30>(a[15]);
    }
    fft_dif<16>(a);
    __syncwarp();  // every lane has read the row before the even half overwrites it
    const int wa = exofs + wr, ea = exofs + er;
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const int j2 = bitrev(i, 4);
        *reinterpret_cast<float2 *>(S + ((wa ^ ((j2 & 7) << 4)) + 128 * j2)) = cmul(a[i], twc[j2]);
    }
    __syncwarp();
    float2 b[16];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const float4 v = *reinterpret_cast<const float4 *>(S + (ea ^ (i << 4)));
        b[2 * i] = make_float2(v.x, v.y);
        b[2 * i + 1] = make_float2(v.z, v.w);
    }
    fft_dif<16>(b);
    __syncwarp();  // all exchange reads done before slots are written into the row
    // sel: per output i a 16-bit byte offset of its slot inside the row (slot * 8, row swizzle already applied
    // by the caller) or 0x8000 if the bin is not selected
    const uint32_t sw[8] = {sel0.x, sel0.y, sel0.z, sel0.w, sel1.x, sel1.y, sel1.z, sel1.w};
    unsigned char *rowp = S + rowofs;
#pragma unroll
    for (int i = 0; i < 16; i += 2) {
        const uint32_t w = sw[i >> 1];
        if (!(w & 0x8000u)) *reinterpret_cast<float2 *>(rowp + (w & 0xFFFFu)) = b[i];
        if ((int)w >= 0) *reinterpret_cast<float2 *>(rowp + (w >> 16)) = b[i + 1];
    }
}

// a[u] *= exp(-2 pi i RHO u / 128), u = U..15: even RHO u are compile-time twiddle64 arguments, odd ones
// come from the 128-point table in constant memory (compile-time index -> constant-bank operand).
template <int RHO, int U>
__device__ __forceinline__ void time_pretwiddle(float2 (&a)[16]) {
    if constexpr (U < 16) {
        if constexpr (((RHO * U) & 1) == 0) a[U] = chime::twiddle64<((RHO * U) / 2) & 63>(a[U]);
        else a[U] = cmul(a[U], c_tw128[(RHO * U) & 127]);
        time_pretwiddle<RHO, U + 1>(a);
    }
}

// ---- phase C: thread <-> (e', slot): 16-point time FFT, detect, accumulate ---------------------------
// col = byte offset of (row e', slot) with the row-independent part of the swizzle applied; row 2 u + e'
// adds 4096 u and XORs the 16-byte chunk index with 2 (u & 3).
template <int RHO>
__device__ __forceinline__ void phase_c(const unsigned char *S, const int col, float (&acc)[16]) {
    float2 a[16];
#pragma unroll
    for (int u = 0; u < 16; ++u)
        a[u] = *reinterpret_cast<const float2 *>(S + ((col ^ ((2 * (u & 3)) << 4)) + 4096 * u));
    if constexpr (RHO != 0) time_pretwiddle<RHO, 1>(a);
    fft_dif<16>(a);
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const int g = (bitrev(i, 4) + 8) & 15;
        acc[g] = fmaf(a[i].x, a[i].x, fmaf(a[i].y, a[i].y, acc[g]));
    }
}


__global__ void __launch_bounds__(kThreads, 1) beamform_mma_kernel(const Params prm) {
    extern __shared__ __align__(1024) unsigned char smem[];
    unsigned char *const S = smem;
    unsigned char *raw = smem;                                                   // 128 KiB
    float2 *tile = reinterpret_cast<float2 *>(smem + kRawBytes);                 // [32][256], swizzled
    constexpr int kTileOfs = kRawBytes, kExchOfs = kRawBytes + kTileBytes;
    int16_t *s_sel = reinterpret_cast<int16_t *>(smem + kRawBytes + kTileBytes + kExchBytes);  // [32][16]
    int16_t *s_slot_of_m = s_sel + 512;                                          // [256]
    uint32_t *s_tmem = reinterpret_cast<uint32_t *>(s_slot_of_m + 256);          // TMEM base address

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int ep = blockIdx.x & 1;
    const int cell = blockIdx.x >> 1;
    // a launch covers frames [frame0, frame0 + n_frames_launch) of channels chan0 ... (execute_host pipelines)
    const int Rf = prm.frame0 + cell % prm.n_frames_launch;
    const int c = prm.chan0 + cell / prm.n_frames_launch;

    {   // s_sel[(16 h + l) * 16 + i] = slot of bin 2 (16 bitrev(i) + l) + h
        const int i = tid & 15, hl = tid >> 4;
        const int sl0 = prm.slot[(size_t)c * 512 + 2 * (16 * bitrev(i, 4) + (hl & 15)) + (hl >> 4)];
        s_sel[tid] = (int16_t)(sl0 < 0 ? 0x8000 : sl0 * 8);
    }
    if (tid < 256) s_slot_of_m[tid] = prm.slot_of_m[(size_t)c * 256 + tid];
    if (warp == 0) {   // one warp allocates 256 columns of tensor memory (1 CTA per SM: no contention)
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;"
                     :: "r"((uint32_t)__cvta_generic_to_shared(s_tmem)), "n"(kTmemCols) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_base = *s_tmem;
    // a warp may touch only TMEM lanes 32 (warp % 4) .. +31; the 4 warps of a lane quarter take 64 columns each
    const uint32_t taddr = tmem_base + ((uint32_t)(32 * (warp & 3)) << 16) + 64u * (uint32_t)(warp >> 2);

    // phase B per-thread constants (rows warp and warp + 16 share the swizzle rx = warp & 7)
    const int h = lane >> 4, l = lane & 15;
    const int rx = warp & 7, xx = h ? 0 : rx;
    const int rd = (((l >> 1) ^ rx) << 4) | ((l & 1) << 3);
    const int wr = (((l >> 1) ^ xx) << 4) | ((l & 1) << 3);
    const int er = (128 * l) | (((l & 7) ^ xx) << 4);
    const int row0 = kTileOfs + warp * 2048, row1 = row0 + 16 * 2048;
    const int exw = kExchOfs + warp * 2048;
    float2 twc[16];
#pragma unroll
    for (int j2 = 0; j2 < 16; ++j2) twc[j2] = __ldg(prm.tw_np + ((l * (2 * j2 + h)) & 511));

    float acc[16];
#pragma unroll
    for (int g = 0; g < 16; ++g) acc[g] = 0.f;

    // phase C per-thread constants
    const int e1 = tid >> 8, sl = tid & 255;
    const int col = kTileOfs + e1 * 2048 + (sl >> 4) * 128 + ((((sl >> 1) & 7) ^ e1) << 4) + (sl & 1) * 8;
    const uint8_t *in_c = prm.in + (size_t)c * prm.n_time * 2048;

#pragma unroll 1
    for (int blk = 0; blk < 6; ++blk) {
        const int r3 = blk >> 1, pol = blk & 1;
        const int t0 = (Rf * 3 + r3) * 128;
        __syncthreads();  // covers the table initialisation; raw is free (last phase A ended 2 barriers ago)
        // ---- stage the raw block: 8192 16-byte chunks, 16 per thread, coalesced 512 B per warp ----
#pragma unroll
        for (int j0 = 0; j0 < 16; j0 += 4) {
            uint4 v[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int idx = (j0 + j) * kThreads + tid;
                const int ch = idx & 15, cyl = (idx >> 4) & 3, t = idx >> 6;
                v[j] = __ldg(reinterpret_cast<const uint4 *>(in_c + (size_t)(t0 + t) * 2048 + pol * 1024 + cyl * 256 + ch * 16));
            }
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int idx = (j0 + j) * kThreads + tid;
                const int ch = idx & 15, p = idx >> 4;   // p = 4 t + cyl
                const int xs = p & 15;
                uint4 w = v[j];
                if (xs & 1) w = make_uint4(v[j].z, v[j].w, v[j].x, v[j].y);
                *reinterpret_cast<uint4 *>(raw + p * 256 + ((ch ^ (xs >> 1)) << 4)) = w;
            }
        }
        __syncthreads();
        const uint2 *bf = prm.bfrag + ((((size_t)c * 2 + pol) * 2 + ep) * 256) * 16;

#pragma unroll 1
        for (int it = 0; it < 8; ++it) {
            // residues in the order 0, 4, 1, 5, 2, 6, 3, 7: RHO + 4 reuses the work of RHO (tensor-memory stash)
            const int rho = (it >> 1) + 4 * (it & 1);
            switch (rho) {
                case 0: phase_a<0>(raw, tile, bf, warp, lane, taddr); break;
                case 1: phase_a<1>(raw, tile, bf, warp, lane, taddr); break;
                case 2: phase_a<2>(raw, tile, bf, warp, lane, taddr); break;
                case 3: phase_a<3>(raw, tile, bf, warp, lane, taddr); break;
                default: phase_a_from_tmem(tile, taddr, warp, lane); break;
            }
            __syncthreads();
            {
                // slot byte offsets of this lane's 16 outputs, with the rows' chunk swizzle (rx << 4) applied
                const uint32_t xr = (uint32_t)(rx << 4) * 0x00010001u;
                uint4 sel0 = *reinterpret_cast<const uint4 *>(s_sel + lane * 16);
                uint4 sel1 = *reinterpret_cast<const uint4 *>(s_sel + lane * 16 + 8);
                sel0 = make_uint4(sel0.x ^ xr, sel0.y ^ xr, sel0.z ^ xr, sel0.w ^ xr);
                sel1 = make_uint4(sel1.x ^ xr, sel1.y ^ xr, sel1.z ^ xr, sel1.w ^ xr);
                phase_b_row(S, row0, h ? exw : row0, h, rd, wr, er, sel0, sel1, twc);
                phase_b_row(S, row1, h ? exw : row1, h, rd, wr, er, sel0, sel1, twc);
            }
            __syncthreads();
            switch (rho) {
                case 0: phase_c<0>(S, col, acc); break;
                case 1: phase_c<1>(S, col, acc); break;
                case 2: phase_c<2>(S, col, acc); break;
                case 3: phase_c<3>(S, col, acc); break;
                case 4: phase_c<4>(S, col, acc); break;
                case 5: phase_c<5>(S, col, acc); break;
                case 6: phase_c<6>(S, col, acc); break;
                default: phase_c<7>(S, col, acc); break;
            }
            __syncthreads();
        }
    }
    // tensor memory is released by the warp that allocated it, after every warp's last tcgen05.ld
    if (warp == 0)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem_base), "n"(kTmemCols));

    // ---- epilogue: thread <-> (e', slot) -> beam m ----
    const int e = 2 * ep + e1;
    const size_t out_base = ((((size_t)c * prm.n_frames + Rf) * 4 + e) * 256) * 16;
    if (prm.out_f32 != nullptr) {
        float *fb = reinterpret_cast<float *>(smem);  // [512][17]
#pragma unroll
        for (int g = 0; g < 16; ++g) fb[tid * 17 + g] = acc[g] * prm.norm;
        __syncthreads();
        const int s = s_slot_of_m[sl] + 256 * e1;
        float4 *dst = reinterpret_cast<float4 *>(prm.out_f32 + out_base + (size_t)sl * 16);
#pragma unroll
        for (int k = 0; k < 4; ++k)
            dst[k] = make_float4(fb[s * 17 + 4 * k], fb[s * 17 + 4 * k + 1], fb[s * 17 + 4 * k + 2], fb[s * 17 + 4 * k + 3]);
    } else {
        uint32_t q[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            uint32_t word = 0;
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                const float v = fmaf(acc[4 * k + b], prm.qscale, prm.qoffset);
                const int iv = __float2int_rn(fminf(fmaxf(v, 0.f), 255.f));
                word |= (uint32_t)iv << (8 * b);
            }
            q[k] = word;
        }
        uint4 *qb = reinterpret_cast<uint4 *>(smem);
        qb[tid] = make_uint4(q[0], q[1], q[2], q[3]);
        __syncthreads();
        const int s = s_slot_of_m[sl] + 256 * e1;
        reinterpret_cast<uint4 *>(prm.out_u8 + out_base)[sl] = qb[s];
    }
}

}  // namespace chime2
