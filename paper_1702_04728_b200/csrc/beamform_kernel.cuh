// Fused CHIME/FRB beamformer kernel for sm_100a: steps a1-a10 of include/chime_bf.h in ONE launch,
// touching HBM only for the packed input and the final output (PAPER.md:51-53 describes three
// kernels with two HBM round trips; here the corner turn stays in shared memory).
//
// Work decomposition: one CTA (256 threads) per (coarse channel c, output frame R, E-W beam e).
// It loops over the n_int = 3 blocks of U samples, the 2 polarisations and the RAD = U/32 residues
// rho of a decimation-in-frequency split of the U-point time transform:
//     S[RAD q' + rho] = sum_{u'<32} W_32^{q'u'} { W_U^{rho u'} sum_{k<RAD} Z[u' + 32k] W_RAD^{rho k} }
// All operators before |.|^2 are linear and act on different axes, so the radix-RAD time butterfly is
// applied to the raw 4-bit integers (exact, packed SIMD-in-register), which shrinks the on-chip tile to
// 32 rows x 256 beams x 8 B = 64 KiB per iteration:
//   phase A  (thread <-> 4 feeds, 8 rows): load raw words, integer radix-RAD time butterfly, int->fp32,
//            E-W phasing with the gains folded into the weights (B = sum_cyl W'[cyl][n] z[cyl][n]),
//            times W_U^{rho u'}  -> tile[u'][n]
//   phase B  (warp <-> row): zero-padded N-S transform as P = NP/256 radix-16x16 FFT-256s of
//            B[n] W_NP^{n c}; the selected bins are written back IN PLACE as tile[u'][slot]
//   phase C  (thread <-> slot): 32-point time FFT in registers, |.|^2, fine-channel grouping,
//            accumulation over (block, pol, rho) in 16 registers
// epilogue: normalise, quantise (cvt.rni + saturate), 16-byte store per beam.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "fft_regs.cuh"

namespace chime {

constexpr int kFeeds = 256;
constexpr int kRows = 32;         // time sub-transform length (rows of the tile)
constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
constexpr int kExchStride = 18;   // float2 per exchange row (16 + 2 pad: conflict-free LDS.128)
constexpr int kExchElems = 16 * kExchStride;

struct KernelParams {
    const uint32_t *in;      // [C][T][2048] bytes viewed as words
    uint8_t *out_u8;         // [C][R][4][256][16]
    float *out_f32;          // same layout, or nullptr
    const float2 *wp;        // [C][2][4][4][256]  folded gain x E-W weights  (pol, e, cyl, feed)
    const int16_t *slot;     // [C][NP]   bin -> slot or -1
    const int16_t *slot_of_m;// [C][256]  beam -> slot
    const float2 *tw_np;     // [NP]  exp(-2 pi i k / NP)
    const float2 *tw_u;      // [U]   exp(-2 pi i k / U)
    int n_time;              // T
    int n_frames;            // R
    int chan0;               // first channel this launch processes (grid covers n_chan channels from here)
    int frame0, n_frames_launch;   // frame range of this launch within each channel
    // beam-major exchange (chime_bf_execute_beam_major): peer_out[d] = receive buffer of rank d,
    // [C_total][R][1024 / n_peers][16]; this launch's channel c is global channel chan_global0 + c.  nullptr = off.
    uint8_t *const *peer_out;
    int n_peers, chan_global0;
    float norm;              // 1/(N N_c U)
    float qscale;            // norm * scale
    float qoffset;
};

// Beam-major exchange addressing: beam b = ew * 256 + ns of (global channel cg, frame Rf) goes to rank
// d = b / (1024 / n_peers), at [cg][Rf][b - d * 1024 / n_peers][16 fine] of that rank's receive buffer: the
// all-to-all corner turn (channel-sharded -> beam-sharded) is the epilogue's 16-byte store itself; with peer-mapped
// pointers the store crosses NVLink.
__device__ __forceinline__ uint4 *beam_major_dst(uint8_t *const *peer_out, const int n_peers, const int cg,
                                                 const int n_frames, const int Rf, const int b) {
    const int bpr = 1024 / n_peers, d = b / bpr;
    return reinterpret_cast<uint4 *>(peer_out[d] + (((size_t)cg * n_frames + Rf) * bpr + (b - d * bpr)) * 16);
}

template <int P>
__host__ __device__ constexpr int exch_bufs_per_warp() { return P <= 2 ? 2 : P; }

template <int P>
__host__ __device__ constexpr size_t smem_bytes() {
    return sizeof(float2) * (kRows * kFeeds)                               // tile
           + sizeof(float2) * (kWarps * exch_bufs_per_warp<P>() * kExchElems) // FFT exchange
           + sizeof(float2) * (256 * P)                                    // tw_np
           + sizeof(float2) * 256                                          // tw_u (U <= 256)
           + sizeof(int16_t) * (256 * P)                                   // slot
           + sizeof(int16_t) * 256;                                        // slot_of_m
}

// ---- phase A helpers ------------------------------------------------------------------------------
// Packed radix-4 time butterfly on offset nibbles.  w[k] holds 4 feeds' bytes of time sample k.
// Returns per-byte (value + 32), value = sum_k x_k (-i)^{rho4 k}, in zr / zi.
__device__ __forceinline__ void int_bfly4(const uint32_t w0, const uint32_t w1, const uint32_t w2,
                                          const uint32_t w3, const int rho4, uint32_t &zr, uint32_t &zi) {
    constexpr uint32_t M = 0x0F0F0F0Fu, BIAS = 0x20202020u;
    const uint32_t R0 = (w0 >> 4) & M, I0 = w0 & M, R1 = (w1 >> 4) & M, I1 = w1 & M;
    const uint32_t R2 = (w2 >> 4) & M, I2 = w2 & M, R3 = (w3 >> 4) & M, I3 = w3 & M;
    if (rho4 == 0) {
        zr = R0 + R1 + R2 + R3;
        zi = I0 + I1 + I2 + I3;
    } else if (rho4 == 1) {
        zr = (R0 + I1 + BIAS) - (R2 + I3);
        zi = (I0 + R3 + BIAS) - (R1 + I2);
    } else if (rho4 == 2) {
        zr = (R0 + R2 + BIAS) - (R1 + R3);
        zi = (I0 + I2 + BIAS) - (I1 + I3);
    } else {
        zr = (R0 + I3 + BIAS) - (R2 + I1);
        zi = (I0 + R1 + BIAS) - (I2 + R3);
    }
}

// byte i of z (a biased small integer) -> exact float (byte - 32) via the 2^23 magic number.
template <int I>
__device__ __forceinline__ float biased_byte_to_float(uint32_t z) {
    return __uint_as_float(__byte_perm(z, 0x4B000000u, 0x7540 | I)) - 8388640.0f;
}

template <int P, int RAD>
__global__ void __launch_bounds__(kThreads, (P <= 2) ? 2 : 1)
beamform_fused_kernel(const KernelParams prm) {
    constexpr int NP = 256 * P;
    constexpr int U = 32 * RAD;
    constexpr int NBUF = exch_bufs_per_warp<P>();

    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *tile = reinterpret_cast<float2 *>(smem_raw);                 // [32][256]
    float2 *exch = tile + kRows * kFeeds;                                // [warp][NBUF][16*18]
    float2 *s_twnp = exch + kWarps * NBUF * kExchElems;                  // [NP]
    float2 *s_twu = s_twnp + NP;                                         // [256]
    int16_t *s_slot = reinterpret_cast<int16_t *>(s_twu + 256);          // [NP]
    int16_t *s_slot_of_m = s_slot + NP;                                  // [256]

    const int tid = threadIdx.x;
    const int lane = tid & 31, warp = tid >> 5;
    const int e = blockIdx.x & 3;
    const int cell = blockIdx.x >> 2;
    // a launch covers frames [frame0, frame0 + n_frames_launch) of channels chan0 ... (execute_host pipelines)
    const int Rf = prm.frame0 + cell % prm.n_frames_launch;
    const int c = prm.chan0 + cell / prm.n_frames_launch;

    for (int i = tid; i < NP; i += kThreads) {
        s_twnp[i] = prm.tw_np[i];
        s_slot[i] = prm.slot[(size_t)c * NP + i];
    }
    s_twu[tid] = (tid < U) ? prm.tw_u[tid] : make_float2(0.f, 0.f);
    s_slot_of_m[tid] = prm.slot_of_m[(size_t)c * 256 + tid];
    __syncthreads();

    float acc[16];
#pragma unroll
    for (int g = 0; g < 16; ++g) acc[g] = 0.f;

    // phase A mapping
    const int nq = tid & 63;   // feeds 4nq .. 4nq+3
    const int ug = tid >> 6;   // rows ug, ug+4, ...
    // phase B mapping
    const int h = lane >> 4, l = lane & 15;

    const size_t chan_word0 = (size_t)c * prm.n_time * 512;  // words per sample = 2048/4

    for (int r = 0; r < 3; ++r) {
        const int t0 = (Rf * 3 + r) * U;
        for (int p = 0; p < 2; ++p) {
            // folded weights W'[cyl][feed] for this (c, p, e)
            float2 w[4][4];
            {
                const float4 *wsrc = reinterpret_cast<const float4 *>(
                    prm.wp + ((((size_t)c * 2 + p) * 4 + e) * 4) * kFeeds + 4 * nq);
#pragma unroll
                for (int cy = 0; cy < 4; ++cy) {
                    const float4 a = __ldg(wsrc + cy * (kFeeds / 2));
                    const float4 b = __ldg(wsrc + cy * (kFeeds / 2) + 1);
                    w[cy][0] = make_float2(a.x, a.y);
                    w[cy][1] = make_float2(a.z, a.w);
                    w[cy][2] = make_float2(b.x, b.y);
                    w[cy][3] = make_float2(b.z, b.w);
                }
            }
            const uint32_t *inp = prm.in + chan_word0 + (size_t)p * 256 + nq;

            for (int rho = 0; rho < RAD; ++rho) {
                const int rho4 = rho & 3;
                // ---------------- phase A ----------------
                float2 w8 = make_float2(1.f, 0.f);
                if constexpr (RAD == 8) w8 = s_twu[(rho * (U / 8)) & (U - 1)];  // W_8^rho
#pragma unroll 2
                for (int uu = ug; uu < kRows; uu += 4) {
                    float br[4], bi[4];
#pragma unroll
                    for (int i = 0; i < 4; ++i) br[i] = bi[i] = 0.f;
#pragma unroll
                    for (int cy = 0; cy < 4; ++cy) {
                        uint32_t raw[RAD];
#pragma unroll
                        for (int k = 0; k < RAD; ++k)
                            raw[k] = __ldg(inp + (size_t)(t0 + uu + 32 * k) * 512 + cy * 64);
                        float zr[4], zi[4];
                        if constexpr (RAD == 4) {
                            uint32_t pr, pi;
                            int_bfly4(raw[0], raw[1], raw[2], raw[3], rho4, pr, pi);
                            zr[0] = biased_byte_to_float<0>(pr); zi[0] = biased_byte_to_float<0>(pi);
                            zr[1] = biased_byte_to_float<1>(pr); zi[1] = biased_byte_to_float<1>(pi);
                            zr[2] = biased_byte_to_float<2>(pr); zi[2] = biased_byte_to_float<2>(pi);
                            zr[3] = biased_byte_to_float<3>(pr); zi[3] = biased_byte_to_float<3>(pi);
                        } else {
                            uint32_t er, ei, orr, oi;
                            int_bfly4(raw[0], raw[2], raw[4], raw[6], rho4, er, ei);
                            int_bfly4(raw[1], raw[3], raw[5], raw[7], rho4, orr, oi);
                            float fe_r[4], fe_i[4], fo_r[4], fo_i[4];
                            fe_r[0] = biased_byte_to_float<0>(er); fe_i[0] = biased_byte_to_float<0>(ei);
                            fe_r[1] = biased_byte_to_float<1>(er); fe_i[1] = biased_byte_to_float<1>(ei);
                            fe_r[2] = biased_byte_to_float<2>(er); fe_i[2] = biased_byte_to_float<2>(ei);
                            fe_r[3] = biased_byte_to_float<3>(er); fe_i[3] = biased_byte_to_float<3>(ei);
                            fo_r[0] = biased_byte_to_float<0>(orr); fo_i[0] = biased_byte_to_float<0>(oi);
                            fo_r[1] = biased_byte_to_float<1>(orr); fo_i[1] = biased_byte_to_float<1>(oi);
                            fo_r[2] = biased_byte_to_float<2>(orr); fo_i[2] = biased_byte_to_float<2>(oi);
                            fo_r[3] = biased_byte_to_float<3>(orr); fo_i[3] = biased_byte_to_float<3>(oi);
#pragma unroll
                            for (int i = 0; i < 4; ++i) {  // E + W_8^rho O
                                zr[i] = fmaf(w8.x, fo_r[i], fmaf(-w8.y, fo_i[i], fe_r[i]));
                                zi[i] = fmaf(w8.x, fo_i[i], fmaf(w8.y, fo_r[i], fe_i[i]));
                            }
                        }
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            br[i] = fmaf(w[cy][i].x, zr[i], fmaf(-w[cy][i].y, zi[i], br[i]));
                            bi[i] = fmaf(w[cy][i].x, zi[i], fmaf(w[cy][i].y, zr[i], bi[i]));
                        }
                    }
                    const float2 tw = s_twu[(rho * uu) & (U - 1)];  // W_U^{rho u'}
                    float4 o0, o1;
                    o0.x = fmaf(br[0], tw.x, -bi[0] * tw.y); o0.y = fmaf(br[0], tw.y, bi[0] * tw.x);
                    o0.z = fmaf(br[1], tw.x, -bi[1] * tw.y); o0.w = fmaf(br[1], tw.y, bi[1] * tw.x);
                    o1.x = fmaf(br[2], tw.x, -bi[2] * tw.y); o1.y = fmaf(br[2], tw.y, bi[2] * tw.x);
                    o1.z = fmaf(br[3], tw.x, -bi[3] * tw.y); o1.w = fmaf(br[3], tw.y, bi[3] * tw.x);
                    float4 *dst = reinterpret_cast<float4 *>(tile + uu * kFeeds + 4 * nq);
                    dst[0] = o0;
                    dst[1] = o1;
                }
                __syncthreads();

                // ---------------- phase B: N-S transform, in place ----------------
                {
                    float2 *ex = exch + (warp * NBUF) * kExchElems;
                    constexpr int ROWS_PER_ITER = (P == 1) ? 2 : 1;
                    constexpr int NJ = (P <= 2) ? 1 : P / 2;  // jobs per half-warp per iteration
                    for (int it = 0; it < kRows / (kWarps * ROWS_PER_ITER); ++it) {
                        const int row = (P == 1) ? 2 * (warp + kWarps * it) + h : warp + kWarps * it;
                        float2 *trow = tile + row * kFeeds;
#pragma unroll
                        for (int j = 0; j < NJ; ++j) {
                            const int cc = (P == 1) ? 0 : h + 2 * j;  // sub-transform: bins P*k + cc
                            float2 *exb = ex + (h + 2 * j) * kExchElems;
                            float2 a[16];
#pragma unroll
                            for (int k = 0; k < 16; ++k) a[k] = trow[l + 16 * k];
                            if (P > 1 && cc != 0) {
#pragma unroll
                                for (int k = 0; k < 16; ++k)
                                    a[k] = cmul(a[k], s_twnp[(cc * (l + 16 * k)) & (NP - 1)]);
                            }
                            fft_dif<16>(a);
#pragma unroll
                            for (int i = 0; i < 16; ++i) {
                                const int j2 = bitrev(i, 4);
                                float2 v = a[i];
                                if (j2 != 0) v = cmul(v, s_twnp[P * ((l * j2) & 255)]);
                                exb[j2 * kExchStride + l] = v;
                            }
                        }
                        __syncwarp();
#pragma unroll
                        for (int j = 0; j < NJ; ++j) {
                            const int cc = (P == 1) ? 0 : h + 2 * j;
                            const float2 *exb = ex + (h + 2 * j) * kExchElems;
                            float2 b[16];
                            const float4 *src = reinterpret_cast<const float4 *>(exb + l * kExchStride);
#pragma unroll
                            for (int k = 0; k < 8; ++k) {
                                const float4 v = src[k];
                                b[2 * k] = make_float2(v.x, v.y);
                                b[2 * k + 1] = make_float2(v.z, v.w);
                            }
                            fft_dif<16>(b);
#pragma unroll
                            for (int i = 0; i < 16; ++i) {
                                const int j1 = bitrev(i, 4);
                                const int bin = P * (16 * j1 + l) + cc;
                                const int s = s_slot[bin];
                                if (s >= 0) trow[s] = b[i];
                            }
                        }
                        __syncwarp();
                    }
                }
                __syncthreads();

                // ---------------- phase C: 32-point time FFT, detect, group ----------------
                {
                    float2 a[32];
#pragma unroll
                    for (int u = 0; u < 32; ++u) a[u] = tile[u * kFeeds + tid];
                    fft_dif<32>(a);
#pragma unroll
                    for (int i = 0; i < 32; ++i) {
                        const int qp = bitrev(i, 5);
                        const int g = ((qp + 16) & 31) >> 1;
                        acc[g] = fmaf(a[i].x, a[i].x, fmaf(a[i].y, a[i].y, acc[g]));
                    }
                }
                __syncthreads();
            }
        }
    }

    // ---------------- epilogue: thread <-> slot  ->  beam m ----------------
    const size_t out_base = ((((size_t)c * prm.n_frames + Rf) * 4 + e) * 256) * 16;
    if (prm.out_f32 != nullptr) {
        float *fb = reinterpret_cast<float *>(tile);  // [slot][16] with +1 float4 pad per 8 slots not needed
#pragma unroll
        for (int g = 0; g < 16; ++g) fb[tid * 17 + g] = acc[g] * prm.norm;
        __syncthreads();
        const int s = s_slot_of_m[tid];
        float4 *dst = reinterpret_cast<float4 *>(prm.out_f32 + out_base + (size_t)tid * 16);
#pragma unroll
        for (int k = 0; k < 4; ++k)
            dst[k] = make_float4(fb[s * 17 + 4 * k], fb[s * 17 + 4 * k + 1], fb[s * 17 + 4 * k + 2],
                                 fb[s * 17 + 4 * k + 3]);
    } else {
        uint32_t q[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            uint32_t word = 0;
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                const float v = fmaf(acc[4 * k + b], prm.qscale, prm.qoffset);
                int iv = __float2int_rn(fminf(fmaxf(v, 0.f), 255.f));
                word |= (uint32_t)iv << (8 * b);
            }
            q[k] = word;
        }
        uint4 *qb = reinterpret_cast<uint4 *>(tile);
        qb[tid] = make_uint4(q[0], q[1], q[2], q[3]);
        __syncthreads();
        const int s = s_slot_of_m[tid];
        if (prm.peer_out != nullptr) {
            *beam_major_dst(prm.peer_out, prm.n_peers, prm.chan_global0 + c, prm.n_frames, Rf, e * 256 + tid) = qb[s];
        } else {
            reinterpret_cast<uint4 *>(prm.out_u8 + out_base)[tid] = qb[s];
        }
    }
}

}  // namespace chime
