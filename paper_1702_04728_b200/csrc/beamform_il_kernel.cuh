// Interleaved version of the fused beamformer kernel (zero_pad = 512, upchan_len = 128).
// Same mathematics and building blocks as beamform_mma_kernel.cuh.  What changes is the schedule:
//
//  * Phase A (packed integer radix-8 time butterfly on the half-rate ALU pipe, fp16 conversion, mma.sync
//    E-W contraction) no longer writes the shared-memory tile.  Each warp computes, for its 16 feeds, the
//    tile values of a PAIR of residues (rho, rho + 4) -- mma columns 4..7 repeat the weights of columns
//    0..3, so lanes tq >= 2 hold the rho + 4 values (same products, opposite sign of the odd-tap part) --
//    and parks them in its own TENSOR-MEMORY lanes (tcgen05.st; 64 columns per pair, two stages).
//  * Because phase A touches neither the tile nor another warp's data, it needs no barrier: the two halves
//    (8 feeds each) of phase A for pair p + 1 are executed inside the two phase-B intervals of pair p, the
//    even warps before their FFT rows and the odd warps after them.  At any moment about half of the warps
//    issue integer/tensor work and half issue FP32 work, so the ALU pipe and the FP32 pipe overlap instead
//    of alternating behind block-wide barriers -- with all 16 warps still sharing phase B (2 rows each).
//  * The raw block of the next (block, pol) is fetched with cp.async during a phase-C interval.
//
// Per residue: barrier; tile <- TMEM (own lanes); barrier; {phase A half | phase B}; barrier; phase C.
#pragma once
#include "beamform_mma_kernel.cuh"

namespace chime4 {

using namespace chime2;

// ---- phase A for residues RHO and RHO + 4, feeds 16 warp + 8 hh .. + 7, into this warp's TMEM lanes ----
template <int RHO>
__device__ __forceinline__ void phase_a_half(const unsigned char *raw, const uint2 *bfrag_cpe, const int warp,
                                             const int lane, const uint32_t taddr, const int hh) {
    constexpr bool ODD = (RHO & 1) != 0;
    const int g = lane >> 2, tq = lane & 3;
    const __half2 nbE = __floats2half2_rn(-32.0f / 512.0f, -32.0f / 512.0f);
    const __half2 nbO = __floats2half2_rn(-(float)rot_bias_r<RHO>() / 512.0f, -(float)rot_bias_i<RHO>() / 512.0f);
    const int pz = 4 * (g & 3) + tq;
    // lanes tq < 2: residue RHO (E + W_8^RHO O); lanes tq >= 2: residue RHO + 4 (E - W_8^RHO O)
    const float ss = (tq < 2 ? 1.0f : -1.0f) * (ODD ? 0.70710678118654752440f : 1.0f);
    const uint2 *bf_l = bfrag_cpe + (size_t)(16 * warp + 8 * hh) * 16 + (lane & 15);
    const unsigned char *raw_h = raw + (4 * g + tq) * 256 + (((2 * warp + hh) ^ pz) << 3);

    uint2 bw[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) bw[i] = __ldg(bf_l + i * 16);
    uint32_t aE[2][8], aO[2][8];
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
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}

template <int DUMMY = 0>
__device__ __forceinline__ void phase_a_half_pr(const int pr, const unsigned char *raw, const uint2 *bf, const int warp,
                                                const int lane, const uint32_t taddr, const int hh) {
    switch (pr) {
        case 0: phase_a_half<0>(raw, bf, warp, lane, taddr, hh); break;
        case 1: phase_a_half<1>(raw, bf, warp, lane, taddr, hh); break;
        case 2: phase_a_half<2>(raw, bf, warp, lane, taddr, hh); break;
        default: phase_a_half<3>(raw, bf, warp, lane, taddr, hh); break;
    }
}

// ---- one residue's tile values of this warp's 16 feeds, own TMEM lanes -> swizzled smem tile ----------
// half = 0: residue RHO (held by lanes tq < 2), half = 1: residue RHO + 4 (lanes tq >= 2).
__device__ __forceinline__ void tile_from_tmem(unsigned char *S, const int tile_ofs, const uint32_t taddr,
                                               const int warp, const int lane, const int half) {
    const int g = lane >> 2, tq = lane & 3;
    const int r0 = g * 2 + (tq & 1);
    const bool mine = (tq >> 1) == half;
    unsigned char *tile_t = S + tile_ofs + r0 * 2048 + warp * 128;
    const int rx16 = (r0 & 7) << 4;
    float v[64];
    tmem_ld32(taddr, v);
    tmem_ld32(taddr + 32, v + 32);
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
    if (mine) {
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

__device__ __forceinline__ void cp_async8(void *smem_dst, const void *gsrc) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" :: "r"((uint32_t)__cvta_generic_to_shared(smem_dst)), "l"(gsrc) : "memory");
}

// raw block [128 t][4 cyl][256 B] -> smem, 8-byte units XOR-swizzled by (4 t + cyl) & 15 (asynchronous)
__device__ __forceinline__ void stage_raw_async(unsigned char *raw, const uint8_t *src_block, const int pol, const int tid) {
#pragma unroll 4
    for (int j = 0; j < 32; ++j) {   // 16384 units, 32 per thread; a warp reads 256 contiguous bytes
        const int idx = j * kThreads + tid;
        const int u = idx & 31, p = idx >> 5;     // p = 4 t + cyl
        cp_async8(raw + p * 256 + ((u ^ (p & 15)) << 3),
                  src_block + (size_t)(p >> 2) * 2048 + pol * 1024 + (p & 3) * 256 + u * 8);
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
}

__global__ void __launch_bounds__(kThreads, 1) beamform_il_kernel(const Params prm) {
    extern __shared__ __align__(1024) unsigned char smem[];
    unsigned char *const S = smem;
    unsigned char *raw = smem;                                                   // 128 KiB
    constexpr int kTileOfs = kRawBytes, kExchOfs = kRawBytes + kTileBytes;
    int16_t *s_sel = reinterpret_cast<int16_t *>(smem + kRawBytes + kTileBytes + kExchBytes);  // [32][16]
    int16_t *s_slot_of_m = s_sel + 512;                                          // [256]
    uint32_t *s_tmem = reinterpret_cast<uint32_t *>(s_slot_of_m + 256);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int ep = blockIdx.x & 1;
    const int cell = blockIdx.x >> 1;
    const int Rf = cell % prm.n_frames;
    const int c = cell / prm.n_frames;
    const uint8_t *in_c = prm.in + (size_t)c * prm.n_time * 2048;
    const uint8_t *in_f = in_c + (size_t)(Rf * 3) * 128 * 2048;   // first sample of this output frame

    stage_raw_async(raw, in_f, 0, tid);   // block 0 = (r3 = 0, pol = 0)
    {   // s_sel[(16 h + l) * 16 + i] = 8 * slot of bin 2 (16 bitrev(i) + l) + h, or 0x8000
        const int i = tid & 15, hl = tid >> 4;
        const int sl0 = prm.slot[(size_t)c * 512 + 2 * (16 * bitrev(i, 4) + (hl & 15)) + (hl >> 4)];
        s_sel[tid] = (int16_t)(sl0 < 0 ? 0x8000 : sl0 * 8);
    }
    if (tid < 256) s_slot_of_m[tid] = prm.slot_of_m[(size_t)c * 256 + tid];
    if (warp == 0) {   // all 512 columns: 4 warps per lane quarter x 2 stages x 64 columns
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;"
                     :: "r"((uint32_t)__cvta_generic_to_shared(s_tmem)), "n"(512) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("cp.async.wait_all;" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_base = *s_tmem;
    // a warp touches only TMEM lanes 32 (warp % 4) .. +31; stage s of warp w: columns 128 (w >> 2) + 64 s .. +63
    const uint32_t taddr0 = tmem_base + ((uint32_t)(32 * (warp & 3)) << 16) + 128u * (uint32_t)(warp >> 2);

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
    const int e1 = tid >> 8, sl = tid & 255;
    const int col = kTileOfs + e1 * 2048 + (sl >> 4) * 128 + ((((sl >> 1) & 7) ^ e1) << 4) + (sl & 1) * 8;
    const bool a_first = ((warp >> 2) & 1) == 0;   // per SM sub-partition (warp % 4) two warps run phase A first, two run their FFT rows first

    // prologue: phase A of pair 0 (block 0, residues 0 and 4) into stage 0
    {
        const uint2 *bf0 = prm.bfrag + ((((size_t)c * 2 + 0) * 2 + ep) * 256) * 16;
        phase_a_half<0>(raw, bf0, warp, lane, taddr0, 0);
        phase_a_half<0>(raw, bf0, warp, lane, taddr0, 1);
    }

#pragma unroll 1
    for (int pp = 0; pp < 24; ++pp) {
        const int st = pp & 1, pr = pp & 3;
        const int np = pp + 1, npr = np & 3, npol = (np >> 2) & 1;    // the pair phase A works on meanwhile
        const uint2 *nbf = prm.bfrag + ((((size_t)c * 2 + npol) * 2 + ep) * 256) * 16;
        const uint32_t ta = taddr0 + 64u * (uint32_t)st, nta = taddr0 + 64u * (uint32_t)(st ^ 1);
#pragma unroll 1
        for (int half = 0; half < 2; ++half) {
            __syncthreads();   // tile free: every thread finished phase C of the previous residue
            tile_from_tmem(S, kTileOfs, ta, warp, lane, half);
            __syncthreads();   // tile complete (and, at the right moments, the next raw block has landed)
            const uint32_t xr = (uint32_t)(rx << 4) * 0x00010001u;
            uint4 sel0 = *reinterpret_cast<const uint4 *>(s_sel + lane * 16);
            uint4 sel1 = *reinterpret_cast<const uint4 *>(s_sel + lane * 16 + 8);
            sel0 = make_uint4(sel0.x ^ xr, sel0.y ^ xr, sel0.z ^ xr, sel0.w ^ xr);
            sel1 = make_uint4(sel1.x ^ xr, sel1.y ^ xr, sel1.z ^ xr, sel1.w ^ xr);
#pragma unroll 1
            for (int step = 0; step < 2; ++step) {
                if ((step == 0) == a_first) {
                    if (np < 24) phase_a_half_pr(npr, raw, nbf, warp, lane, nta, half);
                } else {
                    phase_b_row(S, row0, h ? exw : row0, h, rd, wr, er, sel0, sel1, twc);
                    phase_b_row(S, row1, h ? exw : row1, h, rd, wr, er, sel0, sel1, twc);
                }
            }
            __syncthreads();   // all rows transformed; raw no longer needed by this interval's phase A
            // the raw block of the NEXT (block, pol) is needed from pair 4 b + 4 on, whose phase A starts in
            // the intervals of pair 4 b + 3; the last reader of the current block is phase A of pair 4 b + 3,
            // which ran in the two intervals of pair 4 b + 2.  So fetch it now, under phase C.
            if (pr == 2 && half == 1 && pp < 20) {
                const int nb = (pp >> 2) + 1;
                stage_raw_async(raw, in_f + (size_t)(nb >> 1) * 128 * 2048, nb & 1, tid);
            }
            switch (pr + 4 * half) {
                case 0: phase_c<0>(S, col, acc); break;
                case 1: phase_c<1>(S, col, acc); break;
                case 2: phase_c<2>(S, col, acc); break;
                case 3: phase_c<3>(S, col, acc); break;
                case 4: phase_c<4>(S, col, acc); break;
                case 5: phase_c<5>(S, col, acc); break;
                case 6: phase_c<6>(S, col, acc); break;
                default: phase_c<7>(S, col, acc); break;
            }
            asm volatile("cp.async.wait_all;" ::: "memory");
        }
    }
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem_base), "n"(512));

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

}  // namespace chime4
