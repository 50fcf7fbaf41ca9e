/*
 * chime_bf.h -- C-ABI boundary of the B200-native CHIME/FRB hybrid beamformer hot path.
 *
 * What the library computes (arXiv:1702.04728; line numbers are /root/reference/PAPER.md):
 *   input   4+4-bit complex baseband, 2048 inputs (2 pol x 4 cylinders x 256 N-S feeds) per
 *           390 kHz coarse channel at 2.56 us cadence            (Table 1; sec. 2, :47)
 *   a1-a2   unpack, per-input complex gain                        (:40-41, :47; gains: BASELINE.json)
 *   a3-a4   zero-padded N-S spatial DFT (256 -> NP bins) and selection of the 256 bins nearest
 *           the desired pointings                                 (sec. 3.1, :59-61; eq. (1),(2), :67-78)
 *   a5      exact phasing of the 4 cylinders into 4 E-W beams     (:18, :51, :80)
 *   a6      corner turn time-slowest -> time-fastest              (the paper's 2nd kernel, :51)
 *   a7      U-point DFT over every U consecutive time samples     (sec. 3.2, :51, :84-86)
 *   a8-a10  |.|^2, sum 2 polarisations, sum U/16 adjacent fine channels, sum 3 blocks,
 *           rescale to 8-bit integers                             (:37-42, :53)
 *   output  1024 beams (4 E-W x 256 N-S) x 16 fine channels per coarse channel every
 *           3*U samples (0.983 ms for U = 128), uint8.
 * The conventions the paper leaves open (nibble order, sign of the DFTs, grouping of fine channels,
 * normalisation, rounding of the index table) are the readings A1-A16 listed in DESIGN.md.
 *
 * Every step runs in hand-written sm_100a CUDA kernels; there is no CPU fallback.  All entry points
 * are thread-compatible (one thread per plan at a time).  Pointers are marked HOST or DEVICE.
 */
#ifndef CHIME_BF_H
#define CHIME_BF_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CHIME_BF_N_FEED 256   /* N-S feeds per cylinder */
#define CHIME_BF_N_CYL 4      /* cylinders */
#define CHIME_BF_N_POL 2      /* polarisations */
#define CHIME_BF_N_INPUT 2048 /* input index i = (pol*4 + cyl)*256 + feed */
#define CHIME_BF_N_EW 4       /* E-W formed beams */
#define CHIME_BF_N_BEAM 1024  /* beam index b = ew*256 + ns */
#define CHIME_BF_N_FINE 16    /* fine channels per coarse channel in the output */
#define CHIME_BF_N_INT 3      /* U-sample blocks integrated per output frame */

/* return codes of the int-returning calls */
#define CHIME_BF_OK 0
#define CHIME_BF_E_INVALID_ARG (-1)
#define CHIME_BF_E_ALIGNMENT (-2)
#define CHIME_BF_E_CUDA (-3)
#define CHIME_BF_E_UNSUPPORTED (-4)

typedef struct chime_bf_plan chime_bf_plan; /* opaque; owns its device tables */

/*
 * Plan creation, north-star form.  Channel k has centre frequency 800 - k*0.390625 MHz;
 * n_time = 49152 samples per execute; f_ref = 600 MHz; scale 1/64, offset 128; feed spacing
 * 0.3048 m; cylinder spacing 22 m.
 *   n_coarse    number of coarse channels C (>= 1)
 *   gains       HOST, [C][2048][2] float (re, im), copied; NULL = unit gains.  Zero = flagged input.
 *   ew_angles   HOST, [4] double, E-W beam angles in degrees, copied
 *   zero_pad    NP, padded N-S transform length: 256, 512 or 1024
 *   upchan_len  U, up-channelisation length: 128 or 256 (fine channels out = 16, D = U/16)
 * Returns NULL on error; chime_bf_last_error() tells why.  Binds to the current CUDA device.
 */
chime_bf_plan *chime_bf_plan_create(int n_coarse, const float *gains, const double *ew_angles,
                                    int zero_pad, int upchan_len);

/* Extended form: everything the five BASELINE.json configurations vary. */
typedef struct {
    int n_coarse;                /* C */
    const double *freq_mhz;      /* HOST [C] centre frequencies in MHz; NULL = 800 - k*0.390625 */
    const float *gains;          /* HOST [C][2048][2] or NULL */
    const double *ew_angles_deg; /* HOST [4] */
    int zero_pad;                /* NP in {256, 512, 1024} */
    int upchan_len;              /* U in {128, 256} */
    int n_time;                  /* samples per execute; multiple of 3*U */
    double f_ref_mhz;            /* reference frequency of the desired pointings (A2); <= 0 -> 600 */
    const double *ns_sin_theta;  /* HOST [256] explicit desired pointings sin(theta_m), or NULL */
    float scale, offset;         /* u8 = sat(rne(I*scale + offset)); scale <= 0 -> 1/64, 128 */
    double feed_spacing_m;       /* <= 0 -> 0.3048 */
    double cyl_spacing_m;        /* <= 0 -> 22 */
    int exact_pointing;          /* 0: nearest bin of the zero-padded transform.
                                    1: exact chromatic alignment ("beam interpolation"): beam m is phased
                                    to its desired pointing itself, exp(-2 pi i n f d sin(theta_m) / c0); zero_pad then
                                    only defines the index table that chime_bf_get_ns_index reports (the tensor-core
                                    N-S transform takes any steering vector). */
} chime_bf_params;

chime_bf_plan *chime_bf_plan_create_ex(const chime_bf_params *params);

/*
 * One pass of the whole hot path (a1-a10) over [C][n_time] samples, asynchronous on `cuda_stream`
 * (a cudaStream_t / CUstream passed as void*; NULL = legacy default stream).  Never synchronises,
 * never allocates.
 *   in_u8    DEVICE, [C][n_time][2048] bytes, byte = ((re+8) << 4) | (im+8); 16-byte aligned;
 *            caller-owned, read-only
 *   out_u8   DEVICE, [C][n_time/(3U)][4][256][16] bytes; 16-byte aligned; caller-owned
 * Returns CHIME_BF_OK or a negative code.
 */
int chime_bf_execute(chime_bf_plan *plan, void *cuda_stream, const uint8_t *in_u8, uint8_t *out_u8);

/* Same pass, but writes the pre-quantisation float intensities I (a9) in the same layout. */
int chime_bf_execute_f32(chime_bf_plan *plan, void *cuda_stream, const uint8_t *in_u8,
                         float *out_f32);

/* Convenience: HOST buffers (ideally pinned) in and out; the library stages them through device memory
 * (allocated on first use, owned by the plan) and pipelines by channel group: a plan-owned copy stream
 * uploads chunk k+1 while `cuda_stream` beamforms chunk k and downloads its output (up to 8 chunks: channel
 * groups, or frame ranges of each channel when there are fewer than 8 channels; one kernel launch each).  Ordered after the work already enqueued on `cuda_stream`; synchronises it. */
int chime_bf_execute_host(chime_bf_plan *plan, void *cuda_stream, const uint8_t *in_u8_host,
                          uint8_t *out_u8_host);

/*
 * Re-plannable tables (sec. 3.1: "The extent of the N-S horizon coverage is tunable, and we
 * have the flexibility to form denser or sparser beam tilings.  ... the E-W formed beams can be configured
 * as static or tracking"; gains: BASELINE.json).  Each call recomputes the affected host tables in double
 * precision exactly as plan creation does and copies them into the plan's existing device allocations,
 * ordered on `cuda_stream`: executes enqueued on that stream after the call see the new tables, executes
 * enqueued before it the old ones.  The caller must not have executes of this plan in flight on OTHER
 * streams.  No allocation, no plan rebuild.  The host-side copies (what chime_bf_get_ns_index reports) change
 * with the call and are put back if it fails; the small tables are copied from pageable host memory, so the call may
 * block the host until earlier work on `cuda_stream` has drained.  Return CHIME_BF_OK or a negative code.
 *   update_gains       gains: HOST [C][2048][2] float, copied; NULL = unit gains
 *   update_ew_angles   ew_angles_deg: HOST [4] double (tracking E-W beams: call once per pointing update)
 *   update_pointings   ns_sin_theta: HOST [256] double explicit pointings sin(theta_m) in [-1, 1], or NULL
 *                      to use the native 256-point grid at f_ref_mhz (<= 0 keeps the current f_ref).
 *                      Rebuilds the clamped index table J (eq. (1),(2)) and the N-S weights on the device.
 */
int chime_bf_update_gains(chime_bf_plan *plan, void *cuda_stream, const float *gains);
int chime_bf_update_ew_angles(chime_bf_plan *plan, void *cuda_stream, const double *ew_angles_deg);
int chime_bf_update_pointings(chime_bf_plan *plan, void *cuda_stream, double f_ref_mhz,
                              const double *ns_sin_theta);

/*
 * Incoherent dedispersion of the beamformer's uint8 output to one nominal DM -- the fourth kernel the paper
 * proposes (sec. 3.2: "a fourth kernel which will incoherently dedisperse the post-upchannelized
 * data to a high nominal DM").  Reading F1: with fine-channel frequencies
 * f(c,g) = f_c + (g - 7.5)*0.390625/16 MHz and output frames of 3*U*2.56 us,
 *     delay[c][g] = floor( 4148.808 * dm * (f(c,g)^-2 - f_ref^-2) / (3*U*2.56e-6) + 0.5 )   frames,
 *     D[b][r] = sum_c sum_g beams_u8[c][r + delay[c][g]][b][g],   r = 0 .. n_out-1,  n_out = n_frames - max delay
 * (exact in uint32; b = ew*256 + ns).
 *   dm          dispersion measure in pc/cm^3, >= 0
 *   f_ref_mhz   reference (zero-delay) frequency; <= 0 selects the highest fine-channel frequency of the plan.
 *               A reference below any fine channel (negative delay) is an error.
 * chime_bf_dedisp_delays: HOST host_out [C][16] int32 (may be NULL) and HOST *n_out (may be NULL).
 * chime_bf_dedisperse:    DEVICE beams_u8 [C][n_frames][1024][16] (the layout execute writes), 16-byte aligned;
 *                         DEVICE out_u32 [1024][n_out]; n_out must be the value dedisp_delays reports (>= 1).
 *                         Asynchronous on cuda_stream; one kernel launch, preceded by a small clearing kernel when
 *                         the channel loop is split over CTAs, and by the upload of the delay table unless the
 *                         calling thread's previous call left the same table in the same place on the same stream;
 *                         uses a plan-owned 64*C-byte table, so one dedisperse call per plan may be in flight at a time.
 */
int chime_bf_dedisp_delays(const chime_bf_plan *plan, double dm, double f_ref_mhz, int32_t *host_out,
                           int *n_out);
int chime_bf_dedisperse(chime_bf_plan *plan, void *cuda_stream, const uint8_t *beams_u8, double dm,
                        double f_ref_mhz, uint32_t *out_u32, int n_out);

/*
 * Beam-major exchange fused into the beamformer (the formed beams leave the X-engine
 * node "to a FRB backend" per beam): with the coarse channels sharded over W GPUs (one plan per GPU, no collective
 * inside the beamformer), the consumer of the beams wants all channels of a SUBSET of beams.  This call runs the
 * same pass as chime_bf_execute but its epilogue stores each beam's 16 bytes straight into the receive buffer of
 * the rank that owns the beam: beam b = ew*256 + ns of (global channel cg, frame r) goes to rank d = b / (1024/W),
 * at peer_out[d][cg][r][b - d*1024/W][16].  With peer-mapped pointers (CUDA IPC / symmetric memory over NVLink) the
 * all-to-all IS the kernel's store; with W = 1 or local pointers it is a plain re-layout.  No NCCL call, no staging.
 *   peer_out      HOST array of n_peers DEVICE pointers (copied to a plan-owned device table on `cuda_stream`);
 *                 buffer d has shape [C_total][n_frames][1024/n_peers][16], 16-byte aligned, caller-owned.
 *   n_peers       W; must divide 1024, <= 64
 *   chan_global0  global index of this plan's channel 0 (channels chan_global0 .. + n_coarse - 1 are written)
 * The caller synchronises the ranks (all writers done) before any rank reads its receive buffer.
 */
int chime_bf_execute_beam_major(chime_bf_plan *plan, void *cuda_stream, const uint8_t *in_u8,
                                uint8_t *const *peer_out, int n_peers, int chan_global0);

/* chime_bf_dedisperse on a beam subset, e.g. a rank's receive buffer after the beam-major exchange: DEVICE beams_u8
 * [n_coarse][n_frames][n_beams][16], n_beams a multiple of 32; HOST freq_mhz[n_coarse]; DEVICE delay_scratch
 * [n_coarse*16] int32 (caller-owned); DEVICE out_u32 [n_beams][n_out], n_out = n_frames - max delay.  Same formula,
 * same kernel as chime_bf_dedisperse; needs no plan. */
int chime_bf_dedisp_delays_ex(const double *freq_mhz, int n_coarse, int upchan_len, double dm, double f_ref_mhz,
                              int32_t *host_out /* [n_coarse][16] or NULL */, int *max_delay /* HOST, or NULL */);
int chime_bf_dedisperse_beams(void *cuda_stream, const uint8_t *beams_u8, int n_coarse, const double *freq_mhz,
                              int n_frames, int n_beams, int upchan_len, double dm, double f_ref_mhz,
                              int32_t *delay_scratch, uint32_t *out_u32, int n_out);

/*
 * chime_bf_dedisperse_beams for callers that cannot allocate device memory (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc): the same kernel and formula (reading F1), but the
 * kernel's scratch -- the delay table [n_coarse][16] int32 -- lives in a file-scope device array of the library
 * instead of a caller-owned buffer.  Limit: n_coarse <= CHIME_BF_NOALLOC_MAX_COARSE (1024 = the full band; the array is
 * 64 KiB and every GPU that loads the library holds it until exit); a larger n_coarse is CHIME_BF_E_INVALID_ARG with a
 * message.  The call allocates nothing on the device and frees nothing (no cudaMalloc / cudaFree / allocating library
 * routine; on the host two thread-local tables are sized on a thread's first calls).  Arguments as
 * chime_bf_dedisperse_beams without delay_scratch: beams_u8, out_u32 DEVICE and caller-owned; freq_mhz HOST.
 * Every call on a device shares the one array and finds the previous call's table in it: each call rewrites the
 * n_coarse*16 entries it uses on `cuda_stream` before its kernel reads them (left out only when the calling thread's
 * previous call wrote exactly this table, on this stream, and no other call has written the array since; out_u32 is
 * cleared when the channel loop is split), so calls that follow each other on one stream are safe; calls that OVERLAP
 * on the GPU (different streams without an event between them) race on the table.
 */
#define CHIME_BF_NOALLOC_MAX_COARSE 1024
int chime_bf_dedisperse_beams_noalloc(void *cuda_stream, const uint8_t *beams_u8, int n_coarse, const double *freq_mhz,
                                      int n_frames, int n_beams, int upchan_len, double dm, double f_ref_mhz,
                                      uint32_t *out_u32, int n_out);

/*
 * chime_bf_execute with the packetiser's per-packet rescale ("rescaled to 8-bit integers ... in a custom
 * UDP packet format"; the paper gives no formula -- reading F4 of DESIGN.md): a packet is the 32 consecutive N-S beams
 * x 16 fine channels (512 intensities) of one (channel, frame, E-W beam); its scale and offset follow from its own
 * data, scale = 16 / sigma (1 if sigma = 0), offset = 128 - mean * scale, u8 = sat(rne(I * scale + offset)), so that
 * I ~ (u8 - offset) / scale.  Statistics in fp32.
 *   out_u8        DEVICE, as chime_bf_execute
 *   scale_offset  DEVICE, [C][n_frames][4][8][2] float (scale, offset) per packet, 8-byte aligned, caller-owned
 */
int chime_bf_execute_packets(chime_bf_plan *plan, void *cuda_stream, const uint8_t *in_u8, uint8_t *out_u8,
                             float *scale_offset);

/*
 * Dedispersion ACROSS execute buffers (PAPER.md:86 asks for "a high nominal DM": at DM 500 the sweep over the band is
 * 9.7 s, ten execute buffers of configs[2]).  _begin fixes DM and reference (as chime_bf_dedisp_delays), allocates /
 * clears a plan-owned ring of partial sums [1024][max delay + n_frames] uint32 and restarts the stream at frame 0
 * (synchronises `cuda_stream`); *max_delay (may be NULL) = largest delay in frames.  Every _push adds one more buffer
 * of uint8 beams [C][n_frames][1024][16] (frames t0 .. t0 + n_frames - 1 of the stream, t0 = n_frames x the number of
 * earlier pushes) and hands out the n_frames dedispersed samples that are complete with it:
 *   out_u32       DEVICE, [1024][n_frames]: out[b][s] = D[b][*first_sample + s], D[b][r] = sum_c sum_g I[c][r + delay[c][g]][b][g]
 *                 over the whole stream; samples with a negative index (before the stream starts) are 0
 *   first_sample  HOST (may be NULL): t0 - max delay
 * Asynchronous on `cuda_stream` (two kernels), exact in uint32.
 */
int chime_bf_dedisperse_stream_begin(chime_bf_plan *plan, void *cuda_stream, double dm, double f_ref_mhz, int *max_delay);
int chime_bf_dedisperse_stream_push(chime_bf_plan *plan, void *cuda_stream, const uint8_t *beams_u8, uint32_t *out_u32,
                                    long long *first_sample);

/* Copy of the clamped N-S bin index table J (eq. (1),(2)): HOST out, [C][256] int32. */
int chime_bf_get_ns_index(const chime_bf_plan *plan, int32_t *host_out);

/* Step a1 alone: DEVICE in_u8 [n_bytes] -> DEVICE out_re_im [n_bytes][2] int8 (re, im). */
int chime_bf_debug_unpack(chime_bf_plan *plan, void *cuda_stream, const uint8_t *in_u8,
                          size_t n_bytes, int8_t *out_re_im);

/* Shape queries (so bindings need not re-derive them). */
int chime_bf_n_frames(const chime_bf_plan *plan);       /* n_time / (3U) */
size_t chime_bf_in_bytes(const chime_bf_plan *plan);    /* C * n_time * 2048 */
size_t chime_bf_out_elems(const chime_bf_plan *plan);   /* C * n_frames * 1024 * 16 */
int chime_bf_launches_per_execute(const chime_bf_plan *plan); /* kernels launched by one execute */

/*
 * 0 while every kernel of the plan has run its pipeline to the end; non-zero once a hand-over inside the tensor-core
 * kernel timed out (a protocol bug: the kernel then stops itself with a trap instead of hanging the device, and the
 * CUDA context reports the launch failure).  Reads a host-mapped word, no CUDA call.
 */
int chime_bf_kernel_status(const chime_bf_plan *plan);

/*
 * The roofline denominator, measured: FP32 throughput of this device ("the FFT flops at FP32 peak").
 * Runs two register-resident loops (scalar FFMA, packed FFMA2) on every SM for ~n_iter iterations of 256 operations
 * per thread, timed with CUDA events on `cuda_stream` (synchronises that stream).
 *   tflops_out  HOST [2]: scalar FFMA, packed FFMA2, in TFLOP/s (2 flop per lane and FMA)
 */
int chime_bf_measure_fp32_peak(void *cuda_stream, int n_iter, double *tflops_out);

void chime_bf_destroy(chime_bf_plan *plan); /* NULL-safe */

const char *chime_bf_last_error(void); /* thread-local, never NULL */

#ifdef __cplusplus
}
#endif
#endif /* CHIME_BF_H */
