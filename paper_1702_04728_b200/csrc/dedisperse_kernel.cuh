// Incoherent dedispersion of the beamformer output to one nominal DM (the paper's proposed fourth kernel,
// "a fourth kernel which will incoherently dedisperse the post-upchannelized data to a high
// nominal DM").  Reading F1 in DESIGN.md:
//     D[b][r] = sum_c sum_g  I[c][r + delay[c][g]][b][g],      r = 0 .. n_out - 1,
// I = uint8 intensity codes [C][R][1024 beams][16 fine], delay[c][g] >= 0 in output frames, D exact in uint32
// (at most 1024 * 16 * 255 < 2^32).  HBM-bound: every input byte is needed exactly once.
//
// Mapping: thread <-> (beam, quad of 4 fine channels) loads one 32-bit word per (frame, beam, quad): a warp
// reads 8 beams x 16 bytes = one 128-byte line per frame.  A CTA of 128 threads owns 32 beams x TR output
// samples; its accumulators acc[TR] live in registers (static indices).  Each line is read once per distinct
// delay of the quad (usually one) and once more by the neighbouring time tiles that overlap it by the delay
// spread inside one coarse channel (from L2); DRAM sees each byte once.  When beams x time tiles alone
// would not fill the 148 SMs (long sweeps leave few output samples), the channels are split over blockIdx.z
// and the partial sums meet in the output with integer atomicAdd (exact, order-independent).
#pragma once
#include <cstdint>

namespace chime_dd {

constexpr int kTR = 32;          // output samples per thread
constexpr int kBeamsPerCta = 32; // 128 threads = 32 beams x 4 quads
constexpr int kThreads = 128;

struct Params {
    const uint32_t *in;      // [C][R][n_beams][4] words (4 fine channels per word, little endian)
    const int32_t *delay;    // [C][16]
    uint32_t *out;           // [n_beams][n_out]
    int C, R, n_out;
    int n_beams;             // beams in the array (1024, or 1024 / W after the beam-major exchange); multiple of 32
    int c_per_split;         // channels per blockIdx.z slice; > 1 slice: out is pre-zeroed and summed with atomicAdd (exact)
};

// NB = beams in the array as a compile-time constant (1024: the full array), or 0 = p.n_beams at run time (beam shards).
// With a constant the 32 loads of a pass are one base register + immediate offsets; with a run-time stride each load
// needs its own 64-bit address (100 registers instead of 90, 0.203 ms instead of 0.156 ms on the bench workload).
// TR = output samples per thread: 32 (TR), or 16 for short outputs, where 32-sample tiles would leave most of the SMs
// idle or force a deep channel split (twice the CTAs, 8 resident per SM instead of 5).
template <int NB, int TR>
__global__ void __launch_bounds__(kThreads, (TR == 32 ? 4 : 8)) dedisperse_kernel(const Params p) {
    const int tid = threadIdx.x;
    const int q = tid & 3;
    const int b = blockIdx.x * kBeamsPerCta + (tid >> 2);
    const int r0 = blockIdx.y * TR;
    uint32_t acc[TR];
#pragma unroll
    for (int r = 0; r < TR; ++r) acc[r] = 0u;
    const int n_valid = min(TR, p.n_out - r0);      // ragged last tile
    const size_t frame_words = NB ? (size_t)NB * 4 : (size_t)p.n_beams * 4;
    const int c_lo = blockIdx.z * p.c_per_split, c_hi = min(p.C, c_lo + p.c_per_split);
    int4 dl_next = *reinterpret_cast<const int4 *>(p.delay + c_lo * 16 + 4 * q);
#pragma unroll 1
    for (int c = c_lo; c < c_hi; ++c) {
        const int4 dl = dl_next;   // the next channel's delays are fetched under this channel's loads (one dependent latency less per channel)
        if (c + 1 < c_hi) dl_next = *reinterpret_cast<const int4 *>(p.delay + (c + 1) * 16 + 4 * q);
        const uint32_t *base = p.in + (size_t)c * p.R * frame_words + (size_t)b * 4 + q;
        // One pass per delay value v of the quad: the lane adds the bytes whose delay is v with dp4a against a
        // 0/1 byte mask -- every word is loaded once per distinct delay of its quad (once, for most quads),
        // not once per fine channel.
        const int v_lo = min(min(dl.x, dl.y), min(dl.z, dl.w)), v_hi = max(max(dl.x, dl.y), max(dl.z, dl.w));
#pragma unroll 1
        for (int v = v_lo; v <= v_hi; ++v) {
            const uint32_t mask = (dl.x == v ? 0x01u : 0u) | (dl.y == v ? 0x0100u : 0u) | (dl.z == v ? 0x010000u : 0u) |
                                  (dl.w == v ? 0x01000000u : 0u);
            if (mask == 0u) continue;
            const uint32_t *src = base + (size_t)(r0 + v) * frame_words;
            uint32_t w[TR];   // all TR loads are issued before the first use: 32 x 128 B per warp in flight
#pragma unroll
            for (int r = 0; r < TR; ++r) w[r] = (r < n_valid) ? __ldg(src + (size_t)r * frame_words) : 0u;
#pragma unroll
            for (int r = 0; r < TR; ++r) acc[r] = __dp4a(w[r], mask, acc[r]);
        }
    }
    // sum the 4 quads of a beam (lanes 4k .. 4k+3), then lane q == 0 .. 3 stores every 4th sample
#pragma unroll
    for (int r = 0; r < TR; ++r) {
        acc[r] += __shfl_xor_sync(0xFFFFFFFFu, acc[r], 1);
        acc[r] += __shfl_xor_sync(0xFFFFFFFFu, acc[r], 2);
    }
    uint32_t *dst = p.out + (size_t)b * p.n_out + r0;
    // Split channel loop: the output is cleared by zero_kernel, the launch before this one in the stream.  This kernel
    // is launched with programmatic stream serialization, so it starts (and does all of its loads) while the clearing
    // still runs; only here, before the first atomic, does it wait for that grid to be complete and visible.
    if (gridDim.z > 1) asm volatile("griddepcontrol.wait;" ::: "memory");
#pragma unroll
    for (int r = 0; r < TR; ++r)
        if ((r & 3) == q && r < n_valid) {
            if (gridDim.z == 1) dst[r] = acc[r];
            else atomicAdd(dst + r, acc[r]);
        }
}

// Clears the output of a split launch (instead of a memset node: a kernel can be the primary of a programmatic
// dependent launch).  Lets the dependent grid start at once.
__global__ void __launch_bounds__(256) zero_kernel(uint4 *out, size_t n16, uint32_t *tail, int n_tail) {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += stride) out[i] = make_uint4(0u, 0u, 0u, 0u);
    if (blockIdx.x == 0 && threadIdx.x < n_tail) tail[threadIdx.x] = 0u;
}

// ---- streaming form: sweeps longer than one execute buffer (PAPER.md:86 asks for a HIGH nominal DM) ------------------
// A plan-owned ring of partial sums ring[n_beams][L], L >= D + R (D = largest delay).  Buffer number k holds frames
// t0 .. t0 + R - 1 of the stream (t0 = k R).  With rel = 0 .. D + R - 1 and r = t0 - D + rel the dedispersed sample a
// ring column stands for, the buffer contributes
//     ring[b][(t0 + rel) mod L] += sum_{c, g : 0 <= rel - D + delay[c][g] < R} I[c][rel - D + delay[c][g]][b][g];
// afterwards the columns rel < R are complete (every frame they need has been seen): emit_kernel hands them out and
// clears them for re-use.  Same thread mapping and one-load-per-distinct-delay scheme as dedisperse_kernel; every
// input byte is still read once.
struct StreamParams {
    const uint32_t *in;      // [C][R][n_beams][4] words
    const int32_t *delay;    // [C][16]
    uint32_t *ring;          // [n_beams][L]
    uint32_t *out;           // [n_beams][R] (emit_kernel)
    int C, R, D, L, n_beams;
    long long t0;            // first frame of this buffer in the stream
    int c_per_split;
};

template <int NB>
__global__ void __launch_bounds__(kThreads, 4) dedisperse_stream_kernel(const StreamParams p) {
    const int tid = threadIdx.x;
    const int q = tid & 3;
    const int b = blockIdx.x * kBeamsPerCta + (tid >> 2);
    const int rel0 = blockIdx.y * kTR;
    uint32_t acc[kTR];
#pragma unroll
    for (int r = 0; r < kTR; ++r) acc[r] = 0u;
    const size_t frame_words = NB ? (size_t)NB * 4 : (size_t)p.n_beams * 4;
    const int c_lo = blockIdx.z * p.c_per_split, c_hi = min(p.C, c_lo + p.c_per_split);
#pragma unroll 1
    for (int c = c_lo; c < c_hi; ++c) {
        const int4 dl = *reinterpret_cast<const int4 *>(p.delay + c * 16 + 4 * q);
        const uint32_t *base = p.in + (size_t)c * p.R * frame_words + (size_t)b * 4 + q;
        const int v_lo = min(min(dl.x, dl.y), min(dl.z, dl.w)), v_hi = max(max(dl.x, dl.y), max(dl.z, dl.w));
#pragma unroll 1
        for (int v = v_lo; v <= v_hi; ++v) {
            const uint32_t mask = (dl.x == v ? 0x01u : 0u) | (dl.y == v ? 0x0100u : 0u) | (dl.z == v ? 0x010000u : 0u) |
                                  (dl.w == v ? 0x01000000u : 0u);
            const int f0 = rel0 - p.D + v;                         // frame (inside this buffer) of the tile's first sample
            if (mask == 0u || f0 + kTR <= 0 || f0 >= p.R) continue;  // the whole tile lies in another buffer
            const uint32_t *src = base + (ptrdiff_t)f0 * (ptrdiff_t)frame_words;
            uint32_t w[kTR];
#pragma unroll
            for (int r = 0; r < kTR; ++r) w[r] = ((unsigned)(f0 + r) < (unsigned)p.R) ? __ldg(src + (size_t)r * frame_words) : 0u;
#pragma unroll
            for (int r = 0; r < kTR; ++r) acc[r] = __dp4a(w[r], mask, acc[r]);
        }
    }
#pragma unroll
    for (int r = 0; r < kTR; ++r) {
        acc[r] += __shfl_xor_sync(0xFFFFFFFFu, acc[r], 1);
        acc[r] += __shfl_xor_sync(0xFFFFFFFFu, acc[r], 2);
    }
    uint32_t *row = p.ring + (size_t)b * p.L;
#pragma unroll
    for (int r = 0; r < kTR; ++r)
        if ((r & 3) == q && rel0 + r < p.D + p.R && acc[r] != 0u) {
            const int col = (int)((p.t0 + rel0 + r) % p.L);
            if (gridDim.z == 1) row[col] += acc[r];
            else atomicAdd(row + col, acc[r]);
        }
}

// out[b][s] = the completed sample r = t0 - D + s (0 where r < 0: before the start of the stream); its ring column is cleared.
__global__ void __launch_bounds__(256) dedisperse_emit_kernel(const StreamParams p) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x, b = blockIdx.y;
    if (s >= p.R) return;
    uint32_t *cell = p.ring + (size_t)b * p.L + (int)((p.t0 + s) % p.L);
    p.out[(size_t)b * p.R + s] = (p.t0 + s >= p.D) ? *cell : 0u;
    *cell = 0u;
}

}  // namespace chime_dd
