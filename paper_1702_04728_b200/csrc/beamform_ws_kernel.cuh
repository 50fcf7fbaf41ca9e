// Warp-specialised version of the fused beamformer kernel (zero_pad = 512, upchan_len = 128).
// Same mathematics and building blocks as beamform_mma_kernel.cuh; what changes is who runs what, when:
//
//   warps 8..15  PRODUCERS  stage the raw block, run phase A (packed integer radix-8 time butterfly on the
//                ALU pipe, fp16 conversion, mma.sync E-W contraction on the tensor cores) for a PAIR of
//                residues (rho, rho + 4) at once and park the two resulting tiles in TENSOR MEMORY
//                (tcgen05.st; 128 columns per thread and stage, two stages = all 512 columns).
//   warps 0..7   CONSUMERS  copy one residue's tile from tensor memory to shared memory (tcgen05.ld),
//                then run phase B (N-S FFT-256 x 2 per row, FP32 pipe) and phase C (time FFT-16, detect).
//
// Phase A is bound by the half-rate integer ALU pipe, phases B and C by the FP32 pipe; as separate
// instruction streams they overlap instead of alternating behind block-wide barriers.  Hand-over is by
// named barriers (full/empty per TMEM stage); producers and consumers each keep a private barrier.
// A consumer warp cw reads exactly the TMEM lanes its partner producer warp cw + 8 wrote (a warp can touch
// only lanes 32 (warp % 4) .. +31, and 8 = 0 mod 4).  mma columns 4..7 repeat the weights of columns 0..3,
// so lanes tq >= 2 produce the rho + 4 values (same products, opposite sign of the odd-tap part) and no
// lane is idle.
#pragma once
#include "beamform_mma_kernel.cuh"

namespace chime3 {

using namespace chime2;

constexpr int kConsumerWarps = 8, kProducerWarps = 8;
constexpr int kCThreads = 32 * kConsumerWarps, kPThreads = 32 * kProducerWarps;
constexpr int kExchBytesWs = kConsumerWarps * 2 * 2048;   // 32 KiB: two rows in flight per consumer warp
constexpr int kSmemBytesWs = kRawBytes + kTileBytes + kExchBytesWs + 512 * 2 + 256 * 2 + 16;

// named barriers (0 is __syncthreads)
enum { BAR_FULL0 = 1, BAR_FULL1 = 2, BAR_EMPTY0 = 3, BAR_EMPTY1 = 4, BAR_CONS = 5, BAR_PROD = 6 };

__device__ __forceinline__ void bar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" :: "r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void bar_arrive(int id, int n) { asm volatile("bar.arrive %0, %1;" :: "r"(id), "r"(n) : "memory"); }

// ---- producer: phase A for residues RHO and RHO + 4, feeds 32 pw + 8 hh .. + 7, into TMEM ----------------
template <int RHO>
__device__ __forceinline__ void produce_chunk(const unsigned char *raw, const uint2 *bfrag_cpe, const int pw,
                                              const int lane, const uint32_t taddr, const int hh) {
    constexpr bool ODD = (RHO & 1) != 0;
    const int g = lane >> 2, tq = lane & 3;
    const __half2 nbE = __floats2half2_rn(-32.0f / 512.0f, -32.0f / 512.0f);
    const __half2 nbO = __floats2half2_rn(-(float)rot_bias_r<RHO>() / 512.0f, -(float)rot_bias_i<RHO>() / 512.0f);
    const int pz = 4 * (g & 3) + tq;
    const unsigned char *raw_t = raw + (4 * g + tq) * 256;
    // lanes tq < 2: residue RHO (E + W_8^RHO O); lanes tq >= 2: residue RHO + 4 (E - W_8^RHO O)
    const float ss = (tq < 2 ? 1.0f : -1.0f) * (ODD ? 0.70710678118654752440f : 1.0f);
    const uint2 *bf_l = bfrag_cpe + (size_t)(32 * pw) * 16 + (lane & 15);

    {                                        // 8 feeds at a time
        uint32_t aE[2][8], aO[2][8];
        const unsigned char *raw_h = raw_t + (((4 * pw + hh) ^ pz) << 3);
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
        uint2 bw[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) bw[i] = __ldg(bf_l + (8 * hh + i) * 16);
#pragma unroll
        for (int i = 0; i < 8; i += 2) {
            float z[2][4];
#pragma unroll
            for (int ii = 0; ii < 2; ++ii) {
                float pacc[4] = {0.f, 0.f, 0.f, 0.f}, qacc[4] = {0.f, 0.f, 0.f, 0.f};
                mma_m16n8k8(pacc, aE[0][i + ii], aE[1][i + ii], bw[i + ii].x);
                mma_m16n8k8(pacc, aE[0][i + ii], aE[1][i + ii], bw[i + ii].y);
                mma_m16n8k8(qacc, aO[0][i + ii], aO[1][i + ii], bw[i + ii].x);
                mma_m16n8k8(qacc, aO[0][i + ii], aO[1][i + ii], bw[i + ii].y);
#pragma unroll
                for (int c = 0; c < 4; ++c) z[ii][c] = fmaf(ss, qacc[c], pacc[c]);
            }
            // 8 columns: row g: (n, n+1) re/im, then row g+8: (n, n+1) re/im
            tmem_st8(taddr + 32 * hh + 4 * i, z[0][0], z[0][1], z[1][0], z[1][1], z[0][2], z[0][3], z[1][2], z[1][3]);
        }
    }
}

// all 32 feeds of producer warp pw (four chunks)
template <int RHO>
__device__ __forceinline__ void produce_pair(const unsigned char *raw, const uint2 *bfrag_cpe, const int pw,
                                             const int lane, const uint32_t taddr) {
#pragma unroll 1
    for (int hh = 0; hh < 4; ++hh) produce_chunk<RHO>(raw, bfrag_cpe, pw, lane, taddr, hh);
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}

// ---- consumer: one residue's tile values of this warp's partner producer, TMEM -> swizzled smem tile ----
// half = 0: residue RHO (held by lanes tq < 2), half = 1: residue RHO + 4 (lanes tq >= 2).  All lanes take
// part in the (warp-collective) tcgen05.ld; only the half's lanes store.
__device__ __forceinline__ void tile_from_tmem(unsigned char *S, const int tile_ofs, const uint32_t taddr,
                                               const int cw, const int lane, const int half) {
    const int g = lane >> 2, tq = lane & 3;
    const int r0 = g * 2 + (tq & 1);
    const bool mine = (tq >> 1) == half;
    unsigned char *tile_t = S + tile_ofs + r0 * 2048 + (2 * cw) * 128;
    const int rx16 = (r0 & 7) << 4;
#pragma unroll
    for (int hh = 0; hh < 4; ++hh) {
        float v[32];
        tmem_ld32(taddr + 32 * hh, v);
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
        if (mine) {
#pragma unroll
            for (int i = 0; i < 8; i += 2) {
                // feed n = 32 cw + 8 hh + i: line (n >> 4) = 2 cw + (hh >> 1), chunk (n >> 1) & 7 = 4 (hh & 1) + i / 2
                unsigned char *dst = tile_t + (hh >> 1) * 128 + (rx16 ^ ((4 * (hh & 1) + i / 2) << 4));
                const float *w = v + 4 * i;
                *reinterpret_cast<float4 *>(dst) = make_float4(w[0], w[1], w[2], w[3]);
                *reinterpret_cast<float4 *>(dst + 16 * 2048) = make_float4(w[4], w[5], w[6], w[7]);
            }
        }
    }
}

// ---- consumer phase B on TWO tile rows at once (same lane constants; independent instruction streams
// give the two consumer warps of an SM sub-partition the instruction-level parallelism of four) -----------
__device__ __forceinline__ void phase_b_2rows(unsigned char *S, const int rowA, const int rowB, const int exA,
                                              const int exB, const int h, const int rd, const int wr, const int er,
                                              const uint4 sel0, const uint4 sel1, const float2 (&twc)[16]) {
    float2 a0[16], a1[16];
    const int ra0 = rowA + rd, ra1 = rowB + rd;
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        a0[k] = *reinterpret_cast<const float2 *>(S + (ra0 + 128 * k));
        a1[k] = *reinterpret_cast<const float2 *>(S + (ra1 + 128 * k));
    }
    // The two rows run half a phase apart: each shared-memory round trip of one row (exchange store -> load -> use)
    // is issued before, and lands under, an FFT of the other row; a0 / a1 are re-used as the landing registers.
    const int wa0 = exA + wr, wa1 = exB + wr, ea0 = exA + er, ea1 = exB + er;
    if (h) w32_pretwiddle(a0);
    fft_dif<16>(a0);
#pragma unroll
    for (int i = 0; i < 16; ++i) a0[i] = cmul(a0[i], twc[bitrev(i, 4)]);
    __syncwarp();  // every lane has read both rows before the even half overwrites them
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const int j2 = bitrev(i, 4);
        *reinterpret_cast<float2 *>(S + ((wa0 ^ ((j2 & 7) << 4)) + 128 * j2)) = a0[i];
    }
    __syncwarp();
#pragma unroll
    for (int i = 0; i < 8; ++i) {   // row A, second stage inputs: in flight during row B's first FFT
        const float4 v = *reinterpret_cast<const float4 *>(S + (ea0 ^ (i << 4)));
        a0[2 * i] = make_float2(v.x, v.y);
        a0[2 * i + 1] = make_float2(v.z, v.w);
    }
    if (h) w32_pretwiddle(a1);
    fft_dif<16>(a1);
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const int j2 = bitrev(i, 4);
        *reinterpret_cast<float2 *>(S + ((wa1 ^ ((j2 & 7) << 4)) + 128 * j2)) = cmul(a1[i], twc[j2]);
    }
    __syncwarp();  // exchange B complete; every lane's exchange reads of row A are done as well
#pragma unroll
    for (int i = 0; i < 8; ++i) {   // row B, second stage inputs: in flight during row A's second FFT
        const float4 w = *reinterpret_cast<const float4 *>(S + (ea1 ^ (i << 4)));
        a1[2 * i] = make_float2(w.x, w.y);
        a1[2 * i + 1] = make_float2(w.z, w.w);
    }
    fft_dif<16>(a0);
    const uint32_t sw[8] = {sel0.x, sel0.y, sel0.z, sel0.w, sel1.x, sel1.y, sel1.z, sel1.w};
    unsigned char *rp0 = S + rowA, *rp1 = S + rowB;
#pragma unroll
    for (int i = 0; i < 16; i += 2) {
        const uint32_t w = sw[i >> 1];
        if (!(w & 0x8000u)) *reinterpret_cast<float2 *>(rp0 + (w & 0xFFFFu)) = a0[i];
        if ((int)w >= 0) *reinterpret_cast<float2 *>(rp0 + (w >> 16)) = a0[i + 1];
    }
    fft_dif<16>(a1);
    __syncwarp();  // all exchange reads of row B done before its slots are written into the row
#pragma unroll
    for (int i = 0; i < 16; i += 2) {
        const uint32_t w = sw[i >> 1];
        if (!(w & 0x8000u)) *reinterpret_cast<float2 *>(rp1 + (w & 0xFFFFu)) = a1[i];
        if ((int)w >= 0) *reinterpret_cast<float2 *>(rp1 + (w >> 16)) = a1[i + 1];
    }
}

// ---- consumer phase C on the thread's two columns (beams e' = 0, 1 of one slot) at once ------------------
template <int RHO>
__device__ __forceinline__ void phase_c2(const unsigned char *S, const int col0, const int col1, float (&acc0)[16],
                                         float (&acc1)[16]) {
    float2 a0[16], a1[16];
#pragma unroll
    for (int u = 0; u < 16; ++u) {
        a0[u] = *reinterpret_cast<const float2 *>(S + ((col0 ^ ((2 * (u & 3)) << 4)) + 4096 * u));
        a1[u] = *reinterpret_cast<const float2 *>(S + ((col1 ^ ((2 * (u & 3)) << 4)) + 4096 * u));
    }
    if constexpr (RHO != 0) {
        time_pretwiddle<RHO, 1>(a0);
        time_pretwiddle<RHO, 1>(a1);
    }
    fft_dif<16>(a0);
    fft_dif<16>(a1);
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const int g = (bitrev(i, 4) + 8) & 15;
        acc0[g] = fmaf(a0[i].x, a0[i].x, fmaf(a0[i].y, a0[i].y, acc0[g]));
        acc1[g] = fmaf(a1[i].x, a1[i].x, fmaf(a1[i].y, a1[i].y, acc1[g]));
    }
}

// P1 = true: zero_pad 256 (see the consumer set-up); a template parameter so that the default instantiation's
// register allocation is untouched.
template <bool P1>
__global__ void __launch_bounds__(kThreads, 1) beamform_ws_kernel(const Params prm) {
    extern __shared__ __align__(1024) unsigned char smem[];
    unsigned char *const S = smem;
    unsigned char *raw = smem;                                                   // 128 KiB
    constexpr int kTileOfs = kRawBytes, kExchOfs = kRawBytes + kTileBytes;
    int16_t *s_sel = reinterpret_cast<int16_t *>(smem + kRawBytes + kTileBytes + kExchBytesWs);  // [32][16]
    int16_t *s_slot_of_m = s_sel + 512;                                          // [256]
    uint32_t *s_tmem = reinterpret_cast<uint32_t *>(s_slot_of_m + 256);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int ep = blockIdx.x & 1;
    const int cell = blockIdx.x >> 1;
    // a launch covers frames [frame0, frame0 + n_frames_launch) of channels chan0 ... (execute_host pipelines)
    const int Rf = prm.frame0 + cell % prm.n_frames_launch;
    const int c = prm.chan0 + cell / prm.n_frames_launch;

    {   // s_sel[(16 h + l) * 16 + i] = 8 * slot of bin 2 (16 bitrev(i) + l) + h, or 0x8000
        const int i = tid & 15, hl = tid >> 4;
        const int sl0 = prm.slot[(size_t)c * 512 + 2 * (16 * bitrev(i, 4) + (hl & 15)) + (hl >> 4)];
        s_sel[tid] = (int16_t)(sl0 < 0 ? 0x8000 : sl0 * 8);
    }
    if (tid < 256) s_slot_of_m[tid] = prm.slot_of_m[(size_t)c * 256 + tid];
    if (warp == 0) {   // all 512 columns of tensor memory: 2 stages x 2 producer warps per lane quarter x 128
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;"
                     :: "r"((uint32_t)__cvta_generic_to_shared(s_tmem)), "n"(512) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_base = *s_tmem;
    const int rw = warp & 7;   // role-local warp index; consumer rw pairs with producer rw
    // stage s of role warp rw: lanes 32 (rw & 3) .. +31, columns 256 (rw >> 2) + 128 s .. +127
    const uint32_t taddr0 = tmem_base + ((uint32_t)(32 * (rw & 3)) << 16) + 256u * (uint32_t)(rw >> 2);
    const uint8_t *in_c = prm.in + (size_t)c * prm.n_time * 2048;

    if (warp >= kConsumerWarps) {
        // ======================================= PRODUCERS =======================================
        asm volatile("setmaxnreg.dec.sync.aligned.u32 80;");
        const int ptid = tid - kCThreads;
#pragma unroll 1
        for (int blk = 0; blk < 6; ++blk) {
            const int r3 = blk >> 1, pol = blk & 1;
            const int t0 = (Rf * 3 + r3) * 128;
            bar_sync(BAR_PROD, kPThreads);   // every producer is done reading the previous raw block
#pragma unroll 1
            for (int j0 = 0; j0 < 32; j0 += 4) {   // 8192 16-byte chunks, 32 per producer thread
                uint4 v[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int idx = (j0 + j) * kPThreads + ptid;
                    const int ch = idx & 15, cyl = (idx >> 4) & 3, t = idx >> 6;
                    v[j] = __ldg(reinterpret_cast<const uint4 *>(in_c + (size_t)(t0 + t) * 2048 + pol * 1024 + cyl * 256 + ch * 16));
                }
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int idx = (j0 + j) * kPThreads + ptid;
                    const int ch = idx & 15, p = idx >> 4;   // p = 4 t + cyl
                    const int xs = p & 15;
                    uint4 w = v[j];
                    if (xs & 1) w = make_uint4(v[j].z, v[j].w, v[j].x, v[j].y);
                    *reinterpret_cast<uint4 *>(raw + p * 256 + ((ch ^ (xs >> 1)) << 4)) = w;
                }
            }
            bar_sync(BAR_PROD, kPThreads);
            const uint2 *bf = prm.bfrag + ((((size_t)c * 2 + pol) * 2 + ep) * 256) * 16;
#pragma unroll 1
            for (int pr = 0; pr < 4; ++pr) {
                const int pp = blk * 4 + pr, st = pp & 1;
                if (pp >= 2) {   // wait until the consumers have drained this TMEM stage (pair pp - 2)
                    bar_sync(st ? BAR_EMPTY1 : BAR_EMPTY0, kThreads);
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                }
                const uint32_t ta = taddr0 + 128u * (uint32_t)st;
                switch (pr) {
                    case 0: produce_pair<0>(raw, bf, rw, lane, ta); break;
                    case 1: produce_pair<1>(raw, bf, rw, lane, ta); break;
                    case 2: produce_pair<2>(raw, bf, rw, lane, ta); break;
                    default: produce_pair<3>(raw, bf, rw, lane, ta); break;
                }
                asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                bar_arrive(st ? BAR_FULL1 : BAR_FULL0, kThreads);
            }
        }
    } else {
        // ======================================= CONSUMERS =======================================
        asm volatile("setmaxnreg.inc.sync.aligned.u32 176;");
        // P1 (zero_pad 256): only the even bins of the 512-point transform exist, so the two half-warps do not
        // split the bin parities but the ROWS: lanes 0..15 take rows rw, rw + 16, lanes 16..31 rows rw + 8, rw + 24,
        // every lane on the even-parity path (hp = 0) -- one phase-B call per residue instead of two.
        const int hl = lane >> 4, l = lane & 15;
        const int h = P1 ? 0 : hl;
        const int rx = rw & 7, xx = h ? 0 : rx;   // rows rw, rw + 8, rw + 16, rw + 24 share the swizzle
        const int rd = (((l >> 1) ^ rx) << 4) | ((l & 1) << 3);
        const int wr = (((l >> 1) ^ xx) << 4) | ((l & 1) << 3);
        const int er = (128 * l) | (((l & 7) ^ xx) << 4);
        const int row0 = kTileOfs + rw * 2048;
        const int exw = kExchOfs + rw * 4096;
        float2 twc[16];
#pragma unroll
        for (int j2 = 0; j2 < 16; ++j2) twc[j2] = __ldg(prm.tw_np + ((l * (2 * j2 + h)) & 511));
        float acc0[16], acc1[16];
#pragma unroll
        for (int g = 0; g < 16; ++g) acc0[g] = acc1[g] = 0.f;
        const int sl = tid;   // slot of this thread's two columns (e' = 0, 1)
        const int col0 = kTileOfs + (sl >> 4) * 128 + (((sl >> 1) & 7) << 4) + (sl & 1) * 8;
        const int col1 = kTileOfs + 2048 + (sl >> 4) * 128 + ((((sl >> 1) & 7) ^ 1) << 4) + (sl & 1) * 8;

#pragma unroll 1
        for (int pp = 0; pp < 24; ++pp) {
            const int st = pp & 1, pr = pp & 3;
            bar_sync(st ? BAR_FULL1 : BAR_FULL0, kThreads);
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            const uint32_t ta = taddr0 + 128u * (uint32_t)st;
#pragma unroll 1
            for (int half = 0; half < 2; ++half) {
                // this lane's selected-bin slots: read now, so that the load lands during the copy and the barrier
                const uint32_t xr = (uint32_t)(rx << 4) * 0x00010001u;
                uint4 sel0 = *reinterpret_cast<const uint4 *>(s_sel + (16 * h + l) * 16);
                uint4 sel1 = *reinterpret_cast<const uint4 *>(s_sel + (16 * h + l) * 16 + 8);
                sel0 = make_uint4(sel0.x ^ xr, sel0.y ^ xr, sel0.z ^ xr, sel0.w ^ xr);
                sel1 = make_uint4(sel1.x ^ xr, sel1.y ^ xr, sel1.z ^ xr, sel1.w ^ xr);
                tile_from_tmem(S, kTileOfs, ta, rw, lane, half);
                if (half == 1 && pp < 22) {   // stage drained: hand it back (the last two pairs have no successor)
                    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                    bar_arrive(st ? BAR_EMPTY1 : BAR_EMPTY0, kThreads);
                }
                bar_sync(BAR_CONS, kCThreads);
                {
                    if constexpr (P1) {
                        const int rowA = row0 + hl * 8 * 2048, rowB = rowA + 16 * 2048;
                        phase_b_2rows(S, rowA, rowB, rowA, rowB, 0, rd, wr, er, sel0, sel1, twc);
                    } else {
#pragma unroll 1
                        for (int rr = 0; rr < 4; rr += 2) {
                            const int rowA = row0 + rr * 8 * 2048, rowB = rowA + 8 * 2048;
                            phase_b_2rows(S, rowA, rowB, h ? exw : rowA, h ? exw + 2048 : rowB, h, rd, wr, er, sel0, sel1, twc);
                        }
                    }
                }
                bar_sync(BAR_CONS, kCThreads);
                switch (pr + 4 * half) {
                    case 0: phase_c2<0>(S, col0, col1, acc0, acc1); break;
                    case 1: phase_c2<1>(S, col0, col1, acc0, acc1); break;
                    case 2: phase_c2<2>(S, col0, col1, acc0, acc1); break;
                    case 3: phase_c2<3>(S, col0, col1, acc0, acc1); break;
                    case 4: phase_c2<4>(S, col0, col1, acc0, acc1); break;
                    case 5: phase_c2<5>(S, col0, col1, acc0, acc1); break;
                    case 6: phase_c2<6>(S, col0, col1, acc0, acc1); break;
                    default: phase_c2<7>(S, col0, col1, acc0, acc1); break;
                }
                bar_sync(BAR_CONS, kCThreads);
            }
        }

        // ---- epilogue (consumers only): thread <-> slot, both beams of the pair -> beam m ----
        float *fb = reinterpret_cast<float *>(smem + kTileOfs);   // tile is free; raw may still be in use
#pragma unroll
        for (int e1 = 0; e1 < 2; ++e1) {
            const float (&acc)[16] = e1 ? acc1 : acc0;
            const int e = 2 * ep + e1;
            const size_t out_base = ((((size_t)c * prm.n_frames + Rf) * 4 + e) * 256) * 16;
            if (prm.out_f32 != nullptr) {
#pragma unroll
                for (int g = 0; g < 16; ++g) fb[sl * 17 + g] = acc[g] * prm.norm;
                bar_sync(BAR_CONS, kCThreads);
                const int s = s_slot_of_m[sl];   // < 0: beam sl belongs to the other pass (zero_pad 1024 runs two)
                float4 *dst = reinterpret_cast<float4 *>(prm.out_f32 + out_base + (size_t)sl * 16);
                if (s >= 0) {
#pragma unroll
                    for (int k = 0; k < 4; ++k)
                        dst[k] = make_float4(fb[s * 17 + 4 * k], fb[s * 17 + 4 * k + 1], fb[s * 17 + 4 * k + 2], fb[s * 17 + 4 * k + 3]);
                }
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
                uint4 *qb = reinterpret_cast<uint4 *>(fb);
                qb[sl] = make_uint4(q[0], q[1], q[2], q[3]);
                bar_sync(BAR_CONS, kCThreads);
                const int s = s_slot_of_m[sl];
                if (s >= 0) {
                    if (prm.peer_out != nullptr)
                        *chime::beam_major_dst(prm.peer_out, prm.n_peers, prm.chan_global0 + c, prm.n_frames, Rf, e * 256 + sl) = qb[s];
                    else
                        reinterpret_cast<uint4 *>(prm.out_u8 + out_base)[sl] = qb[s];
                }
            }
            bar_sync(BAR_CONS, kCThreads);
        }
    }
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem_base), "n"(512));
}

}  // namespace chime3
