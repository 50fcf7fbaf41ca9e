// C-ABI of the CHIME/FRB beamformer library (include/chime_bf.h): plan = host-built tables in double
// precision uploaded once; execute = one fused kernel launch on the caller's stream.
#include "../../include/chime_bf.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>

#include "beam_major.cuh"
#include <atomic>
#include "dedisperse_kernel.cuh"
#include "fp32_peak.cuh"
#include "umma_beamform_kernel.cuh"

namespace {

thread_local char g_err[512] = "";

void set_err(const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

constexpr double kC0 = 299792458.0;
constexpr double kPi = 3.14159265358979323846264338327950288;

}  // namespace

struct chime_bf_plan {
    int C = 0, NP = 0, U = 0, T = 0, R = 0;
    int device = 0;
    float scale = 0.f, offset = 0.f, norm = 0.f;
    std::vector<int32_t> J;  // [C][256]
    // host copies of what the tables are built from (re-plannable without a plan rebuild)
    std::vector<double> freq;      // [C] MHz
    std::vector<float> gains;      // [C][2048][2], empty = unit
    std::vector<double> ns_sin;    // [256] explicit pointings, empty = native grid at fref
    double ew_deg[4] = {0, 0, 0, 0};
    double fref = 600.0, d_feed = 0.3048, d_cyl = 22.0;
    bool exact_pointing = false;  // steer to the desired pointing itself instead of the nearest bin
    double *d_turns = nullptr;    // [C][256] phase step per feed (cycles) of the desired pointings, exact pointing only
    // staging for execute_host
    uint8_t *d_stage_in = nullptr;
    uint8_t *d_stage_out = nullptr;
    cudaStream_t copy_stream = nullptr;   // execute_host: H2D of channel k+1 under the kernel of channel k
    std::vector<cudaEvent_t> copy_done;   // one event per channel
    cudaEvent_t entry = nullptr;
    int host_parts = 1;                   // execute_host: frame ranges per channel
    uint8_t **d_peer_out = nullptr;       // execute_beam_major: device copy of the peers' receive-buffer pointers (<= 64)
    int32_t *d_delay = nullptr;   // [C][16] dedispersion delays of the last chime_bf_dedisperse call
    // streaming dedispersion (chime_bf_dedisperse_stream_begin / _push): ring of partial sums across execute buffers
    uint32_t *d_ring = nullptr;   // [1024][dd_L]
    int32_t *d_delay_stream = nullptr;
    int dd_D = -1, dd_L = 0;
    long long dd_t0 = 0;
    // tensor-core N-S path (umma_beamform_kernel.cuh)
    uint32_t *d_wq = nullptr;     // TMEM images of the three-digit integer weights, 3 MiB per channel
    float2 *d_beta = nullptr;     // [C][4] E-W phase step of beam e
    float *d_inv_s2 = nullptr;    // [C]
    double *d_wscale = nullptr;   // [C] S_c
    float2 *d_gains = nullptr;    // [C][2048] device copy of the gains (nullptr = unit)
    int32_t *d_J = nullptr;       // [C][256]
    int *d_status = nullptr, *h_status = nullptr;   // mapped host word: which wait timed out (0 = none)
    int max_clusters = 0;         // co-resident clusters of 4 (persistent grid)
    float *d_scratch = nullptr;   // per-CTA parking space of the tensor-core kernel (32 KiB per CTA)
};

namespace {

#define CUDA_TRY(expr)                                                                     \
    do {                                                                                   \
        cudaError_t _e = (expr);                                                           \
        if (_e != cudaSuccess) {                                                           \
            set_err("%s failed: %s", #expr, cudaGetErrorString(_e));                       \
            return false;                                                                  \
        }                                                                                  \
    } while (0)

// Clamped N-S bin index (eq. (1)+(2); reading A3): round-half-up of
// x = P (m - 128) f / f_ref, evaluated as one exact integer-by-f product and one division.
int32_t ns_bin(int P, int m, double f_mhz, double fref_mhz, int NP) {
    const double x = ((double)(P * (m - 128)) * f_mhz) / fref_mhz;
    const double fl = std::floor(x);
    long j = (long)fl + (((x - fl) >= 0.5) ? 1 : 0);
    j %= NP;
    if (j < 0) j += NP;
    return (int32_t)j;
}

int32_t ns_bin_sintheta(int NP, double f_mhz, double d_m, double s) {
    const double x = (double)NP * (f_mhz * 1e6) * (d_m / kC0) * s;
    const double fl = std::floor(x);
    long j = (long)fl + (((x - fl) >= 0.5) ? 1 : 0);
    j %= NP;
    if (j < 0) j += NP;
    return (int32_t)j;
}

bool gains_finite(const float *g, size_t n) {
    for (size_t i = 0; i < n; ++i)
        if (!std::isfinite(g[i])) return false;
    return true;
}

template <typename T>
bool upload(T **dst, const std::vector<T> &src) {
    CUDA_TRY(cudaMalloc((void **)dst, src.size() * sizeof(T)));
    CUDA_TRY(cudaMemcpy(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice));
    return true;
}

// First call allocates and copies; later calls (table updates) copy into the same allocation, ordered on `st`.
template <typename T>
bool upload_on(T **dst, const std::vector<T> &src, cudaStream_t st) {
    if (*dst == nullptr) return upload(dst, src);
    CUDA_TRY(cudaMemcpyAsync(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice, st));
    return true;
}

// a4: index table J (eq. (1),(2)): the clamped bin of every beam; it decides the phase of the beam's weight row.
bool build_index_tables(chime_bf_plan *pl, cudaStream_t st) {
    (void)st;
    const int C = pl->C, NP = pl->NP, P = NP / 256;
    pl->J.resize((size_t)C * 256);
    for (int c = 0; c < C; ++c) {
        const double f = pl->freq[c];
        int32_t *J = &pl->J[(size_t)c * 256];
        for (int m = 0; m < 256; ++m)
            J[m] = !pl->ns_sin.empty() ? ns_bin_sintheta(NP, f, pl->d_feed, pl->ns_sin[m])
                                       : ns_bin(P, m, f, pl->fref, NP);
    }
    return true;
}

// Tensor-core path: the E-W phase steps (a5) -- 32 bytes per channel, all a re-pointing of the E-W beams uploads.
bool build_ew_table(chime_bf_plan *pl, cudaStream_t st) {
    std::vector<float2> beta((size_t)pl->C * 4);
    for (int c = 0; c < pl->C; ++c)
        for (int e = 0; e < 4; ++e) {
            const double ph = -2.0 * kPi * (pl->freq[c] * 1e6) * pl->d_cyl * std::sin(pl->ew_deg[e] * kPi / 180.0) / kC0;
            beta[(size_t)c * 4 + e] = make_float2((float)std::cos(ph), (float)std::sin(ph));
        }
    return upload_on(&pl->d_beta, beta, st);
}

// Tensor-core path: gains (a2) x N-S phases (a3, a4) as two-digit 16-bit integers, built on the device in double.
bool build_umma_weights(chime_bf_plan *pl, cudaStream_t st) {
    const int C = pl->C;
    std::vector<double> scale(C);
    std::vector<float> inv_s2(C);
    for (int c = 0; c < C; ++c) {
        double gmax = pl->gains.empty() ? 1.0 : 0.0;
        if (!pl->gains.empty())
            for (int i = 0; i < 2048; ++i) {
                const float *g = &pl->gains[((size_t)c * 2048 + i) * 2];
                gmax = std::max(gmax, std::hypot((double)g[0], (double)g[1]));
            }
        const double S = gmax > 0 ? (double)chime4::kWMax / (gmax * (1.0 + 1e-9)) : 1.0;
        scale[c] = S;
        inv_s2[c] = (float)((65536.0 / S) * (65536.0 / S));   // the kernel sums in units of the top digit
    }
    if (!upload_on(&pl->d_wscale, scale, st) || !upload_on(&pl->d_inv_s2, inv_s2, st)) return false;
    if (!upload_on(&pl->d_J, pl->J, st)) return false;
    if (!pl->gains.empty()) {
        std::vector<float2> g((size_t)C * 2048);
        memcpy(g.data(), pl->gains.data(), g.size() * sizeof(float2));
        if (!upload_on(&pl->d_gains, g, st)) return false;
    }
    if (!pl->d_wq) {
        CUDA_TRY(cudaMalloc((void **)&pl->d_wq, (size_t)C * 16 * chime4::kWqWordsPerSet * sizeof(uint32_t)));
    }
    chime4::WeightParams wp;
    wp.wq = pl->d_wq;
    wp.gains = pl->gains.empty() ? nullptr : pl->d_gains;
    wp.J = pl->d_J;
    wp.turns = nullptr;
    if (pl->exact_pointing) {
        // turns[m] = f d sin(theta_m) / c0; native grid (reading A2): (m - 128) f / (256 f_ref)
        std::vector<double> turns((size_t)C * 256);
        for (int c = 0; c < C; ++c)
            for (int m = 0; m < 256; ++m)
                turns[(size_t)c * 256 + m] = !pl->ns_sin.empty()
                    ? (pl->freq[c] * 1e6) * (pl->d_feed / kC0) * pl->ns_sin[m]
                    : ((double)(m - 128) * pl->freq[c]) / (256.0 * pl->fref);
        if (!upload_on(&pl->d_turns, turns, st)) return false;
        wp.turns = pl->d_turns;
    }
    wp.scale = pl->d_wscale;
    wp.NP = pl->NP;
    chime4::build_weights_kernel<<<C * 16, 128, 0, st>>>(wp);
    CUDA_TRY(cudaGetLastError());
    return true;
}

// The packed baseband [rows = C * T][2048 bytes] as a 2-D tensor map for the kernel's TMA loads: box 128 bytes x 128 rows
// (one half of a (pol, cylinder) block), 128-byte swizzle.  The encoder lives in the driver; it is fetched through the
// runtime so that the library does not link libcuda.
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
bool encode_input_map(CUtensorMap *map, const uint8_t *in, size_t rows, int box_rows) {
    static EncodeTiledFn fn = nullptr;
    if (fn == nullptr) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess || p == nullptr) {
            set_err("execute: cuTensorMapEncodeTiled is not available in this driver");
            return false;
        }
        fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    const cuuint64_t dims[2] = {2048, (cuuint64_t)rows};
    const cuuint64_t strides[1] = {2048};
    const cuuint32_t box[2] = {128, (cuuint32_t)box_rows};   // one feed half of a block of upchan_len samples
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = fn(map, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<uint8_t *>(in), dims, strides, box, estr,
                          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        set_err("execute: cuTensorMapEncodeTiled failed (%d)", (int)r);
        return false;
    }
    return true;
}

bool build_tables(chime_bf_plan *pl) {
    const int U = pl->U;
    if (!build_index_tables(pl, nullptr)) return false;
    {
        std::vector<float2> tw128(128);
        for (int k = 0; k < 128; ++k) {
            const double a = -2.0 * kPi * (double)k / 128.0;
            tw128[k] = make_float2((float)std::cos(a), (float)std::sin(a));
        }
        CUDA_TRY(cudaMemcpyToSymbol(chime4::c_tw128, tw128.data(), sizeof(float2) * 128));
        std::vector<float2> twr(8 * 16);
        for (int rho = 0; rho < 8; ++rho)
            for (int u = 0; u < 16; ++u) twr[rho * 16 + u] = tw128[(rho * u) & 127];
        CUDA_TRY(cudaMemcpyToSymbol(chime4::c_twr, twr.data(), sizeof(float2) * 128));
        std::vector<float2> twr256(8 * 32), w32(16);
        for (int rho = 0; rho < 8; ++rho)
            for (int u = 0; u < 32; ++u) {
                const double a = -2.0 * kPi * (double)(rho * u) / 256.0;
                twr256[rho * 32 + u] = make_float2((float)std::cos(a), (float)std::sin(a));
            }
        for (int u = 0; u < 16; ++u) {
            const double a = -2.0 * kPi * (double)u / 32.0;
            w32[u] = make_float2((float)std::cos(a), (float)std::sin(a));
        }
        CUDA_TRY(cudaMemcpyToSymbol(chime4::c_twr256, twr256.data(), sizeof(float2) * 256));
        CUDA_TRY(cudaMemcpyToSymbol(chime4::c_w32, w32.data(), sizeof(float2) * 16));
        const void *kfn = U == 128 ? (const void *)chime4::umma_beamform_kernel<128> : (const void *)chime4::umma_beamform_kernel<256>;
        CUDA_TRY(cudaFuncSetAttribute(kfn, cudaFuncAttributeMaxDynamicSharedMemorySize, chime4::kSmemBytes));
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(4 * 148);
        cfg.blockDim = dim3(chime4::kThreads);
        cfg.dynamicSmemBytes = chime4::kSmemBytes;
        CUDA_TRY(cudaOccupancyMaxActiveClusters(&pl->max_clusters, kfn, &cfg));
        if (pl->max_clusters < 1) { set_err("plan_create: no cluster of 4 CTAs fits on this device"); return false; }
        CUDA_TRY(cudaMalloc((void **)&pl->d_scratch, (size_t)pl->max_clusters * 4 * chime4::kMaxChunkFrames * 128 * 16 * sizeof(float)));
        CUDA_TRY(cudaHostAlloc((void **)&pl->h_status, 128 * sizeof(int), cudaHostAllocMapped));   // survives a trapped kernel
        memset(pl->h_status, 0, 128 * sizeof(int));
        CUDA_TRY(cudaHostGetDevicePointer((void **)&pl->d_status, pl->h_status, 0));
        CUDA_TRY(cudaMalloc((void **)&pl->d_delay, (size_t)pl->C * 16 * sizeof(int32_t)));
        CUDA_TRY(cudaMalloc((void **)&pl->d_peer_out, 64 * sizeof(uint8_t *)));
        return build_ew_table(pl, nullptr) && build_umma_weights(pl, nullptr);
    }
}

// Dispersion delay of fine channel (c, g) relative to f_ref, in output frames (reading F1):
//   f = f_c + (g - 7.5) * 0.390625/16 MHz,  x = K_DM * DM * (f^-2 - f_ref^-2) / (3 U * 2.56 us),
//   delay = floor(x + 0.5),  K_DM = 4148.808 s MHz^2 cm^3 / pc.   Returns the largest delay.
int dedisp_table(const double *freq, int C, int U, double dm, double fref_mhz, std::vector<int32_t> &tab) {
    const double fine = 0.390625 / 16.0, tau = 3.0 * (double)U * 2.56e-6;
    if (!(fref_mhz > 0)) {
        fref_mhz = 0;
        for (int c = 0; c < C; ++c) fref_mhz = std::max(fref_mhz, freq[c] + 7.5 * fine);
    }
    tab.resize((size_t)C * 16);
    int mx = 0;
    for (int c = 0; c < C; ++c)
        for (int g = 0; g < 16; ++g) {
            const double f = freq[c] + ((double)g - 7.5) * fine;
            const double x = 4148.808 * dm * (1.0 / (f * f) - 1.0 / (fref_mhz * fref_mhz)) / tau;
            const int d = (int)std::floor(x + 0.5);
            tab[(size_t)c * 16 + g] = d;
            mx = std::max(mx, d);
        }
    return mx;
}

int run(chime_bf_plan *pl, void *stream, const uint8_t *in, uint8_t *out_u8, float *out_f32, int chan0 = 0,
        int n_chan = -1, int frame0 = 0, int n_fr = -1, uint8_t *const *peer_out = nullptr, int n_peers = 0,
        int chan_global0 = 0, float *packet_so = nullptr) {
    if (pl && n_chan < 0) n_chan = pl->C;
    if (pl && n_fr < 0) n_fr = pl->R;
    if (!pl || !in || (!out_u8 && !out_f32 && !peer_out)) {
        set_err("execute: null argument");
        return CHIME_BF_E_INVALID_ARG;
    }
    int cur_dev = -1;
    if (cudaGetDevice(&cur_dev) != cudaSuccess || cur_dev != pl->device) {
        set_err("execute: the plan belongs to device %d, the current device is %d", pl->device, cur_dev);
        return CHIME_BF_E_INVALID_ARG;
    }
    if (((uintptr_t)in & 15) || ((uintptr_t)out_u8 & 15) || ((uintptr_t)out_f32 & 15)) {
        set_err("execute: buffers must be 16-byte aligned");
        return CHIME_BF_E_ALIGNMENT;
    }
    cudaStream_t st = (cudaStream_t)stream;
    {
        chime4::Params up;
        up.in = in;
        up.out_u8 = out_u8;
        up.out_f32 = out_f32;
        up.wq = pl->d_wq;
        up.beta = pl->d_beta;
        up.inv_s2 = pl->d_inv_s2;
        up.n_time = pl->T;
        up.n_frames = pl->R;
        up.chan0 = chan0;
        up.n_chan = n_chan;
        up.frame0 = frame0;
        up.n_frames_launch = n_fr;
        up.peer_out = peer_out;
        up.n_peers = n_peers;
        up.chan_global0 = chan_global0;
        up.norm = pl->norm;
        up.scale = pl->scale;
        up.offset = pl->offset;
        up.status = pl->d_status;
        up.scratch = pl->d_scratch;
        up.packet_so = reinterpret_cast<float2 *>(packet_so);
        // Frames per work item.  An item costs 2 x tiles_per_frame_and_pol x chunk tiles plus two weight reloads (~4 tile
        // times each, measured), and the persistent grid runs ceil(items / clusters) rounds: take the chunk length that
        // minimises rounds x item cost (long chunks amortise the reloads, short ones balance the grid).
        int chunk = 1;
        {
            const long long tiles_pf = 2LL * 3 * (pl->U / 32);
            long long best = -1;
            for (int cf = chime4::kMaxChunkFrames; cf >= 1; cf >>= 1) {
                const long long items = (long long)n_chan * ((n_fr + cf - 1) / cf) * 2;
                const long long rounds = (items + pl->max_clusters - 1) / pl->max_clusters;
                const long long cost = rounds * (tiles_pf * std::min(cf, n_fr) + 8);
                if (best < 0 || cost < best) {
                    best = cost;
                    chunk = cf;
                }
            }
        }
        up.chunk_frames = chunk;
        const long long n_items = (long long)n_chan * ((n_fr + chunk - 1) / chunk) * 2;
        const int n_cl = (int)std::min<long long>(n_items, pl->max_clusters);
        CUtensorMap tmap;
        if (!encode_input_map(&tmap, in, (size_t)pl->C * pl->T, pl->U)) return CHIME_BF_E_CUDA;
        if (pl->U == 128) chime4::umma_beamform_kernel<128><<<4 * n_cl, chime4::kThreads, chime4::kSmemBytes, st>>>(up, tmap);
        else chime4::umma_beamform_kernel<256><<<4 * n_cl, chime4::kThreads, chime4::kSmemBytes, st>>>(up, tmap);
        const cudaError_t e4 = cudaGetLastError();
        if (e4 != cudaSuccess) {
            set_err("kernel launch failed: %s", cudaGetErrorString(e4));
            return CHIME_BF_E_CUDA;
        }
        return CHIME_BF_OK;
    }
}

// Scratch of chime_bf_dedisperse_beams_noalloc: the delay table of the dedispersion kernel in a file-scope device array,
// so that the call needs no allocation.  64 KiB per GPU that loads the library, until exit.  In host code the name is a
// host-side stand-in, NOT a device address: noalloc_delay_table() asks the runtime for the address on the current
// device (once per device) and the kernel gets that pointer.
static __device__ __align__(256) int32_t g_noalloc_delay[CHIME_BF_NOALLOC_MAX_COARSE * 16];

int32_t *noalloc_delay_table() {
    constexpr int kMaxDev = 64;
    static int32_t *ptr[kMaxDev] = {};
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess || dev < 0 || dev >= kMaxDev) {
        set_err("dedisperse_beams_noalloc: cudaGetDevice: %s (device %d)", cudaGetErrorString(e), dev);
        return nullptr;
    }
    if (ptr[dev] == nullptr) {   // set-up, once per device, with that device current
        int32_t *p = nullptr;
        e = cudaGetSymbolAddress((void **)&p, g_noalloc_delay);
        if (e != cudaSuccess || p == nullptr) {
            set_err("dedisperse_beams_noalloc: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
            return nullptr;
        }
        ptr[dev] = p;
    }
    return ptr[dev];
}

// Bumped by every upload of a delay table and by chime_bf_destroy (a new plan may get a freed plan's address).
static std::atomic<unsigned long long> g_dd_upload_epoch{0};

// lib_owned: d_delay is written by this function only (a plan's table, the built-in array of the no-alloc call), so an
// upload of the same table to the same place on the same stream can be left out.  A caller's scratch is always rewritten.
int launch_dedisperse(void *stream, const uint8_t *beams_u8, int C, int R, int n_beams, const std::vector<int32_t> &tab,
                      int32_t *d_delay, uint32_t *out_u32, int n_out, bool lib_owned) {
    cudaStream_t st = (cudaStream_t)stream;
    // The table goes up only when it differs from what this thread last put into this device array on this stream (the
    // usual caller dedisperses buffer after buffer to the same DM): one stream operation less in front of a kernel that
    // takes 40 - 140 us.  A different stream, array or table uploads again; so does any other writer of the array in
    // between, because every such writer is a call of this function and replaces the record.
    struct Uploaded { const int32_t *dst = nullptr; cudaStream_t st = nullptr; int dev = -1; std::vector<int32_t> tab; };
    static thread_local Uploaded last;
    static thread_local unsigned long long my_epoch = 0;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    const bool same = lib_owned && e == cudaSuccess && last.dst == d_delay && last.st == st && last.dev == dev &&
                      my_epoch == g_dd_upload_epoch.load() && last.tab == tab;
    if (e == cudaSuccess && !same) {
        e = cudaMemcpyAsync(d_delay, tab.data(), tab.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st);
        last.dst = d_delay;
        last.st = st;
        last.dev = dev;
        last.tab = tab;
        my_epoch = ++g_dd_upload_epoch;
    }
    if (e == cudaSuccess) {
        chime_dd::Params dp;
        dp.in = reinterpret_cast<const uint32_t *>(beams_u8);
        dp.delay = d_delay;
        dp.out = out_u32;
        dp.C = C;
        dp.R = R;
        dp.n_out = n_out;
        dp.n_beams = n_beams;
        // Tile length and split of the channel loop over blockIdx.z.  The kernel is short (40 - 160 us), so what matters is
        // that the grid is a whole number of waves of the resident CTAs (5 per SM with 32-sample tiles, 8 with 16-sample
        // ones).  Cost of a choice = waves x (work of a CTA + its fixed work: start-up latency, the final shuffles and
        // atomics -- ~4.5 channels' worth of a 32-sample tile, fitted to a sweep of the split at DM 5 / 10 / 20 / 40 on
        // the bench workload), in units of one channel of a 32-sample tile per resident CTA slot.
        const int bt = n_beams / chime_dd::kBeamsPerCta;
        int tr = chime_dd::kTR, n_split = 1;
        {
            double best = -1.0;
            for (int t = 32; t >= 16; t >>= 1) {
                const long long slots = 148LL * (t == 32 ? 5 : 8);
                const int tt_ = (n_out + t - 1) / t;
                const double unit = (t == 32 ? 1.0 : 0.5 * 8.0 / 5.0);   // half the bytes per channel, but 8 CTAs share an SM instead of 5
                for (int ns = 1; ns <= std::min(C, 16); ++ns) {
                    const int cps = (C + ns - 1) / ns, ns_eff = (C + cps - 1) / cps;
                    const long long waves = ((long long)bt * tt_ * ns_eff + slots - 1) / slots;
                    const double cost = (double)waves * ((double)cps * unit + 4.5 * (t == 32 ? 1.0 : 8.0 / 5.0 * 0.75));
                    if (best < 0 || cost < best) {
                        best = cost;
                        n_split = ns_eff;
                        tr = t;
                    }
                }
            }
        }
#ifdef CHIME_DD_SWEEP
        if (getenv("DD_SPLIT")) n_split = atoi(getenv("DD_SPLIT"));
        if (getenv("DD_TR")) tr = atoi(getenv("DD_TR"));
#endif
        const int tt = (n_out + tr - 1) / tr;
        dp.c_per_split = (C + n_split - 1) / n_split;
        n_split = (C + dp.c_per_split - 1) / dp.c_per_split;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(bt, tt, n_split);
        cfg.blockDim = dim3(chime_dd::kThreads);
        cfg.stream = st;
        cudaLaunchAttribute attr[1];
        if (n_split > 1) {
            // split channel loop: clear the output with a kernel and let the dedispersion start under it (it waits for
            // the clearing only before its atomics, see dedisperse_kernel)
            const size_t n_words = (size_t)n_beams * n_out, head = std::min<size_t>(n_words, (4 - (((uintptr_t)out_u32 >> 2) & 3)) & 3);
            const size_t n16 = (n_words - head) / 4, tail = n_words - head - 4 * n16;
            if (head) e = cudaMemsetAsync(out_u32, 0, head * sizeof(uint32_t), st);   // (only for an output that is not 16-byte aligned)
            if (e == cudaSuccess) {
                const int zb = (int)std::min<size_t>((n16 + 255) / 256 + 1, 148 * 4);
                chime_dd::zero_kernel<<<zb, 256, 0, st>>>(reinterpret_cast<uint4 *>(out_u32 + head), n16, out_u32 + head + 4 * n16, (int)tail);
                e = cudaGetLastError();
            }
            attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
            attr[0].val.programmaticStreamSerializationAllowed = 1;
            cfg.attrs = attr;
            cfg.numAttrs = 1;
        }
        if (e == cudaSuccess) {
            if (n_beams == 1024 && tr == 32) e = cudaLaunchKernelEx(&cfg, chime_dd::dedisperse_kernel<1024, 32>, dp);
            else if (n_beams == 1024) e = cudaLaunchKernelEx(&cfg, chime_dd::dedisperse_kernel<1024, 16>, dp);
            else if (tr == 32) e = cudaLaunchKernelEx(&cfg, chime_dd::dedisperse_kernel<0, 32>, dp);
            else e = cudaLaunchKernelEx(&cfg, chime_dd::dedisperse_kernel<0, 16>, dp);
            if (e == cudaSuccess) e = cudaGetLastError();
        }
    }
    if (e != cudaSuccess) { set_err("dedisperse: %s", cudaGetErrorString(e)); return CHIME_BF_E_CUDA; }
    return CHIME_BF_OK;
}

}  // namespace

extern "C" {

const char *chime_bf_last_error(void) { return g_err; }

chime_bf_plan *chime_bf_plan_create_ex(const chime_bf_params *pp) {
    if (!pp) {
        set_err("plan_create: null params");
        return nullptr;
    }
    const chime_bf_params &p = *pp;
    if (p.n_coarse < 1) { set_err("plan_create: n_coarse must be >= 1"); return nullptr; }
    if (p.zero_pad != 256 && p.zero_pad != 512 && p.zero_pad != 1024) {
        set_err("plan_create: zero_pad must be 256, 512 or 1024 (got %d)", p.zero_pad);
        return nullptr;
    }
    if (p.upchan_len != 128 && p.upchan_len != 256) {
        set_err("plan_create: upchan_len must be 128 or 256 (got %d)", p.upchan_len);
        return nullptr;
    }
    if (p.n_time < 3 * p.upchan_len || p.n_time % (3 * p.upchan_len) != 0) {
        set_err("plan_create: n_time must be a positive multiple of 3*upchan_len (got %d)", p.n_time);
        return nullptr;
    }
    if (!p.ew_angles_deg) { set_err("plan_create: ew_angles is NULL"); return nullptr; }
    if (p.ns_sin_theta)
        for (int m = 0; m < 256; ++m)
            if (!(p.ns_sin_theta[m] >= -1.0 && p.ns_sin_theta[m] <= 1.0)) {
                set_err("plan_create: ns_sin_theta[%d] outside [-1, 1]", m);
                return nullptr;
            }
    if ((long long)p.n_coarse * (p.n_time / (3 * p.upchan_len)) * 4 > 2147483647LL) {
        set_err("plan_create: grid too large");
        return nullptr;
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        set_err("plan_create: no CUDA device (this library has no CPU fallback)");
        return nullptr;
    }
    chime_bf_plan *pl = new chime_bf_plan();
    pl->C = p.n_coarse;
    pl->NP = p.zero_pad;
    pl->U = p.upchan_len;
    pl->T = p.n_time;
    pl->R = p.n_time / (3 * p.upchan_len);
    pl->scale = p.scale > 0.f ? p.scale : 1.0f / 64.0f;
    pl->offset = p.scale > 0.f ? p.offset : 128.0f;
    pl->norm = (float)(1.0 / (256.0 * 4.0 * (double)p.upchan_len));
    pl->exact_pointing = p.exact_pointing != 0;
    cudaGetDevice(&pl->device);
    pl->fref = p.f_ref_mhz > 0 ? p.f_ref_mhz : 600.0;
    pl->d_feed = p.feed_spacing_m > 0 ? p.feed_spacing_m : 0.3048;
    pl->d_cyl = p.cyl_spacing_m > 0 ? p.cyl_spacing_m : 22.0;
    pl->freq.resize(p.n_coarse);
    for (int c = 0; c < p.n_coarse; ++c) pl->freq[c] = p.freq_mhz ? p.freq_mhz[c] : 800.0 - (double)c * 0.390625;
    if (p.gains) {
        if (!gains_finite(p.gains, (size_t)p.n_coarse * 2048 * 2)) {
            set_err("plan_create: gains must be finite");
            delete pl;
            return nullptr;
        }
        pl->gains.assign(p.gains, p.gains + (size_t)p.n_coarse * 2048 * 2);
    }
    if (p.ns_sin_theta) pl->ns_sin.assign(p.ns_sin_theta, p.ns_sin_theta + 256);
    for (int e = 0; e < 4; ++e) pl->ew_deg[e] = p.ew_angles_deg[e];
    bool ok = build_tables(pl);
    if (!ok) {
        chime_bf_destroy(pl);
        return nullptr;
    }
    return pl;
}

chime_bf_plan *chime_bf_plan_create(int n_coarse, const float *gains, const double *ew_angles,
                                    int zero_pad, int upchan_len) {
    chime_bf_params p;
    memset(&p, 0, sizeof(p));
    p.n_coarse = n_coarse;
    p.gains = gains;
    p.ew_angles_deg = ew_angles;
    p.zero_pad = zero_pad;
    p.upchan_len = upchan_len;
    p.n_time = 49152;
    return chime_bf_plan_create_ex(&p);
}

int chime_bf_execute(chime_bf_plan *plan, void *stream, const uint8_t *in_u8, uint8_t *out_u8) {
    return run(plan, stream, in_u8, out_u8, nullptr);
}

int chime_bf_execute_packets(chime_bf_plan *plan, void *stream, const uint8_t *in_u8, uint8_t *out_u8,
                             float *scale_offset) {
    if (!plan || !scale_offset || !out_u8) { set_err("execute_packets: null argument"); return CHIME_BF_E_INVALID_ARG; }
    if ((uintptr_t)scale_offset & 7) { set_err("execute_packets: scale_offset must be 8-byte aligned"); return CHIME_BF_E_ALIGNMENT; }
    return run(plan, stream, in_u8, out_u8, nullptr, 0, -1, 0, -1, nullptr, 0, 0, scale_offset);
}

int chime_bf_execute_f32(chime_bf_plan *plan, void *stream, const uint8_t *in_u8, float *out_f32) {
    return run(plan, stream, in_u8, nullptr, out_f32);
}

int chime_bf_execute_beam_major(chime_bf_plan *pl, void *stream, const uint8_t *in_u8, uint8_t *const *peer_out,
                                int n_peers, int chan_global0) {
    if (!pl || !in_u8 || !peer_out) { set_err("execute_beam_major: null argument"); return CHIME_BF_E_INVALID_ARG; }
    if (n_peers < 1 || n_peers > 64 || (1024 % n_peers) != 0 || chan_global0 < 0) {
        set_err("execute_beam_major: n_peers must divide 1024 and be <= 64 (got %d), chan_global0 >= 0", n_peers);
        return CHIME_BF_E_INVALID_ARG;
    }
    for (int d = 0; d < n_peers; ++d)
        if (!peer_out[d] || ((uintptr_t)peer_out[d] & 15)) {
            set_err("execute_beam_major: peer buffer %d is null or not 16-byte aligned", d);
            return CHIME_BF_E_ALIGNMENT;
        }
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e = cudaMemcpyAsync(pl->d_peer_out, peer_out, n_peers * sizeof(uint8_t *), cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) { set_err("execute_beam_major: %s", cudaGetErrorString(e)); return CHIME_BF_E_CUDA; }
    return run(pl, stream, in_u8, nullptr, nullptr, 0, -1, 0, -1, pl->d_peer_out, n_peers, chan_global0);
}

int chime_bf_execute_host(chime_bf_plan *pl, void *stream, const uint8_t *in_host, uint8_t *out_host) {
    if (!pl || !in_host || !out_host) {
        set_err("execute_host: null argument");
        return CHIME_BF_E_INVALID_ARG;
    }
    const size_t nin = chime_bf_in_bytes(pl), nout = chime_bf_out_elems(pl);
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e = cudaSuccess;
    if (!pl->d_stage_in) e = cudaMalloc((void **)&pl->d_stage_in, nin);
    if (e == cudaSuccess && !pl->d_stage_out) e = cudaMalloc((void **)&pl->d_stage_out, nout);
    if (e == cudaSuccess && !pl->copy_stream) {
        e = cudaStreamCreateWithFlags(&pl->copy_stream, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&pl->entry, cudaEventDisableTiming);
        // up to 8 chunks: whole channels if there are at least 8, else every channel in 8 / C frame ranges
        pl->host_parts = pl->C >= 8 ? 1 : std::max(1, std::min(pl->R, 8 / pl->C));
        pl->copy_done.resize(pl->host_parts == 1 ? std::min(pl->C, 8) : pl->C * pl->host_parts, nullptr);
        for (size_t k = 0; k < pl->copy_done.size() && e == cudaSuccess; ++k)
            e = cudaEventCreateWithFlags(&pl->copy_done[k], cudaEventDisableTiming);
    }
    if (e != cudaSuccess) {
        set_err("execute_host: %s", cudaGetErrorString(e));
        // a half-finished first-call set-up must not be mistaken for a finished one by the next call
        for (cudaEvent_t ev : pl->copy_done)
            if (ev) cudaEventDestroy(ev);
        pl->copy_done.clear();
        if (pl->entry) { cudaEventDestroy(pl->entry); pl->entry = nullptr; }
        if (pl->copy_stream) { cudaStreamDestroy(pl->copy_stream); pl->copy_stream = nullptr; }
        return CHIME_BF_E_CUDA;
    }
    // Pipeline by channel group (channels are independent; up to 8 groups): the copy stream uploads group k + 1
    // while the caller's stream beamforms group k and downloads its output.  The copy stream starts after everything already
    // enqueued on the caller's stream (entry event), so the call is ordered like a single operation on `st`.
    const size_t cin = (size_t)pl->T * 2048, cout = (size_t)pl->R * 1024 * 16;
    e = cudaEventRecord(pl->entry, st);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(pl->copy_stream, pl->entry, 0);
    // chunk k = (channel range, frame range): whole channels when C >= 8, else each channel in `parts` frame ranges
    const int n_chunks = (int)pl->copy_done.size();
    const int parts = pl->host_parts;
    const size_t fin = (size_t)3 * pl->U * 2048, fout = (size_t)1024 * 16;   // bytes per frame in / out
    auto chunk = [&](int k, int &c0, int &nc, int &f0, int &nf) {
        if (parts == 1) {
            c0 = (int)((long long)pl->C * k / n_chunks);
            nc = (int)((long long)pl->C * (k + 1) / n_chunks) - c0;
            f0 = 0;
            nf = pl->R;
        } else {
            c0 = k / parts;
            nc = 1;
            f0 = (int)((long long)pl->R * (k % parts) / parts);
            nf = (int)((long long)pl->R * (k % parts + 1) / parts) - f0;
        }
    };
    for (int k = 0; k < n_chunks && e == cudaSuccess; ++k) {
        int c0, nc, f0, nf;
        chunk(k, c0, nc, f0, nf);
        const size_t off = c0 * cin + f0 * fin;
        e = cudaMemcpyAsync(pl->d_stage_in + off, in_host + off, nc == 1 ? nf * fin : nc * cin, cudaMemcpyHostToDevice,
                            pl->copy_stream);
        if (e == cudaSuccess) e = cudaEventRecord(pl->copy_done[k], pl->copy_stream);
    }
    for (int k = 0; k < n_chunks && e == cudaSuccess; ++k) {
        int c0, nc, f0, nf;
        chunk(k, c0, nc, f0, nf);
        e = cudaStreamWaitEvent(st, pl->copy_done[k], 0);
        if (e != cudaSuccess) break;
        const int rc = run(pl, stream, pl->d_stage_in, pl->d_stage_out, nullptr, c0, nc, f0, nf);
        if (rc != CHIME_BF_OK) return rc;
        const size_t off = c0 * cout + f0 * fout;
        e = cudaMemcpyAsync(out_host + off, pl->d_stage_out + off, nc == 1 ? nf * fout : nc * cout, cudaMemcpyDeviceToHost, st);
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) {
        set_err("execute_host: %s", cudaGetErrorString(e));
        return CHIME_BF_E_CUDA;
    }
    return CHIME_BF_OK;
}

int chime_bf_update_gains(chime_bf_plan *pl, void *stream, const float *gains) {
    if (!pl) { set_err("update_gains: null plan"); return CHIME_BF_E_INVALID_ARG; }
    if (gains && !gains_finite(gains, (size_t)pl->C * 2048 * 2)) { set_err("update_gains: gains must be finite"); return CHIME_BF_E_INVALID_ARG; }
    std::vector<float> old;
    old.swap(pl->gains);   // the host copy follows the device tables: put back if the rebuild fails
    if (gains) pl->gains.assign(gains, gains + (size_t)pl->C * 2048 * 2);
    if (build_umma_weights(pl, (cudaStream_t)stream)) return CHIME_BF_OK;
    pl->gains.swap(old);
    return CHIME_BF_E_CUDA;
}

int chime_bf_update_ew_angles(chime_bf_plan *pl, void *stream, const double *ew_angles_deg) {
    if (!pl || !ew_angles_deg) { set_err("update_ew_angles: null argument"); return CHIME_BF_E_INVALID_ARG; }
    double old[4];
    for (int e = 0; e < 4; ++e) {
        old[e] = pl->ew_deg[e];
        pl->ew_deg[e] = ew_angles_deg[e];
    }
    if (build_ew_table(pl, (cudaStream_t)stream)) return CHIME_BF_OK;
    for (int e = 0; e < 4; ++e) pl->ew_deg[e] = old[e];
    return CHIME_BF_E_CUDA;
}

int chime_bf_update_pointings(chime_bf_plan *pl, void *stream, double f_ref_mhz, const double *ns_sin_theta) {
    if (!pl) { set_err("update_pointings: null plan"); return CHIME_BF_E_INVALID_ARG; }
    const std::vector<double> old_sin = pl->ns_sin;
    const std::vector<int32_t> old_J = pl->J;
    const double old_fref = pl->fref;
    if (ns_sin_theta) {
        for (int m = 0; m < 256; ++m)
            if (!(ns_sin_theta[m] >= -1.0 && ns_sin_theta[m] <= 1.0)) {
                set_err("update_pointings: ns_sin_theta[%d] outside [-1, 1]", m);
                return CHIME_BF_E_INVALID_ARG;
            }
        pl->ns_sin.assign(ns_sin_theta, ns_sin_theta + 256);
    } else {
        pl->ns_sin.clear();
        if (f_ref_mhz > 0) pl->fref = f_ref_mhz;
    }
    if (build_index_tables(pl, (cudaStream_t)stream) && build_umma_weights(pl, (cudaStream_t)stream)) return CHIME_BF_OK;
    pl->ns_sin = old_sin;   // the index table chime_bf_get_ns_index reports stays the one the device weights were built from
    pl->J = old_J;
    pl->fref = old_fref;
    return CHIME_BF_E_CUDA;
}

int chime_bf_dedisp_delays(const chime_bf_plan *pl, double dm, double f_ref_mhz, int32_t *host_out, int *n_out) {
    if (!pl || !(dm >= 0)) { set_err("dedisp_delays: bad argument"); return CHIME_BF_E_INVALID_ARG; }
    std::vector<int32_t> tab;
    const int mx = dedisp_table(pl->freq.data(), pl->C, pl->U, dm, f_ref_mhz, tab);
    for (int32_t d : tab)
        if (d < 0) { set_err("dedisp_delays: f_ref below a fine channel (negative delay)"); return CHIME_BF_E_INVALID_ARG; }
    if (host_out) memcpy(host_out, tab.data(), tab.size() * sizeof(int32_t));
    if (n_out) *n_out = pl->R - mx;   // complete output samples (<= 0: the sweep is longer than the buffer)
    return CHIME_BF_OK;
}

int chime_bf_dedisperse(chime_bf_plan *pl, void *stream, const uint8_t *beams_u8, double dm, double f_ref_mhz,
                        uint32_t *out_u32, int n_out) {
    if (!pl || !beams_u8 || !out_u32) { set_err("dedisperse: null argument"); return CHIME_BF_E_INVALID_ARG; }
    if ((uintptr_t)beams_u8 & 15) { set_err("dedisperse: input must be 16-byte aligned"); return CHIME_BF_E_ALIGNMENT; }
    std::vector<int32_t> tab((size_t)pl->C * 16);
    int n_full = 0;
    const int rc = chime_bf_dedisp_delays(pl, dm, f_ref_mhz, tab.data(), &n_full);
    if (rc != CHIME_BF_OK) return rc;
    if (n_full < 1 || n_out != n_full) {
        set_err("dedisperse: n_out must be n_frames - max delay = %d (got %d)", n_full, n_out);
        return CHIME_BF_E_INVALID_ARG;
    }
    return launch_dedisperse(stream, beams_u8, pl->C, pl->R, 1024, tab, pl->d_delay, out_u32, n_out, true);
}

int chime_bf_dedisperse_stream_begin(chime_bf_plan *pl, void *stream, double dm, double f_ref_mhz, int *max_delay) {
    if (!pl || !(dm >= 0)) { set_err("dedisperse_stream_begin: bad argument"); return CHIME_BF_E_INVALID_ARG; }
    std::vector<int32_t> tab;
    const int D = dedisp_table(pl->freq.data(), pl->C, pl->U, dm, f_ref_mhz, tab);
    for (int32_t d : tab)
        if (d < 0) { set_err("dedisperse_stream_begin: f_ref below a fine channel (negative delay)"); return CHIME_BF_E_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)stream;
    const int L = D + pl->R;
    cudaError_t e = cudaSuccess;
    if (L > pl->dd_L) {
        cudaFree(pl->d_ring);
        pl->d_ring = nullptr;
        e = cudaMalloc((void **)&pl->d_ring, (size_t)1024 * L * sizeof(uint32_t));
        pl->dd_L = (e == cudaSuccess) ? L : 0;
    }
    if (e == cudaSuccess && !pl->d_delay_stream) e = cudaMalloc((void **)&pl->d_delay_stream, (size_t)pl->C * 16 * sizeof(int32_t));
    if (e == cudaSuccess) e = cudaMemsetAsync(pl->d_ring, 0, (size_t)1024 * pl->dd_L * sizeof(uint32_t), st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(pl->d_delay_stream, tab.data(), tab.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);   // `tab` is a pageable temporary
    if (e != cudaSuccess) { set_err("dedisperse_stream_begin: %s", cudaGetErrorString(e)); return CHIME_BF_E_CUDA; }
    pl->dd_D = D;
    pl->dd_t0 = 0;
    if (max_delay) *max_delay = D;
    return CHIME_BF_OK;
}

int chime_bf_dedisperse_stream_push(chime_bf_plan *pl, void *stream, const uint8_t *beams_u8, uint32_t *out_u32,
                                    long long *first_sample) {
    if (!pl || !beams_u8 || !out_u32) { set_err("dedisperse_stream_push: null argument"); return CHIME_BF_E_INVALID_ARG; }
    if (pl->dd_D < 0) { set_err("dedisperse_stream_push: call chime_bf_dedisperse_stream_begin first"); return CHIME_BF_E_INVALID_ARG; }
    if ((uintptr_t)beams_u8 & 15) { set_err("dedisperse_stream_push: input must be 16-byte aligned"); return CHIME_BF_E_ALIGNMENT; }
    chime_dd::StreamParams sp;
    sp.in = reinterpret_cast<const uint32_t *>(beams_u8);
    sp.delay = pl->d_delay_stream;
    sp.ring = pl->d_ring;
    sp.out = out_u32;
    sp.C = pl->C;
    sp.R = pl->R;
    sp.D = pl->dd_D;
    sp.L = pl->dd_L;
    sp.n_beams = 1024;
    sp.t0 = pl->dd_t0;
    const int bt = 1024 / chime_dd::kBeamsPerCta, tt = (pl->dd_D + pl->R + chime_dd::kTR - 1) / chime_dd::kTR;
    int n_split = std::min(pl->C, std::max(1, (148 * 16 + bt * tt - 1) / (bt * tt)));
    sp.c_per_split = (pl->C + n_split - 1) / n_split;
    n_split = (pl->C + sp.c_per_split - 1) / sp.c_per_split;
    cudaStream_t st = (cudaStream_t)stream;
    chime_dd::dedisperse_stream_kernel<1024><<<dim3(bt, tt, n_split), chime_dd::kThreads, 0, st>>>(sp);
    chime_dd::dedisperse_emit_kernel<<<dim3((pl->R + 255) / 256, 1024), 256, 0, st>>>(sp);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { set_err("dedisperse_stream_push: %s", cudaGetErrorString(e)); return CHIME_BF_E_CUDA; }
    if (first_sample) *first_sample = pl->dd_t0 - pl->dd_D;   // stream index of out_u32[.][0]; samples < 0 are zero
    pl->dd_t0 += pl->R;
    return CHIME_BF_OK;
}

int chime_bf_dedisp_delays_ex(const double *freq_mhz, int n_coarse, int upchan_len, double dm, double f_ref_mhz,
                              int32_t *host_out, int *max_delay) {
    if (!freq_mhz || n_coarse < 1 || !(dm >= 0) || (upchan_len != 128 && upchan_len != 256)) {
        set_err("dedisp_delays_ex: bad argument");
        return CHIME_BF_E_INVALID_ARG;
    }
    std::vector<int32_t> tab;
    const int mx = dedisp_table(freq_mhz, n_coarse, upchan_len, dm, f_ref_mhz, tab);
    for (int32_t d : tab)
        if (d < 0) { set_err("dedisp_delays_ex: f_ref below a fine channel (negative delay)"); return CHIME_BF_E_INVALID_ARG; }
    if (host_out) memcpy(host_out, tab.data(), tab.size() * sizeof(int32_t));
    if (max_delay) *max_delay = mx;
    return CHIME_BF_OK;
}

int chime_bf_dedisperse_beams(void *stream, const uint8_t *beams_u8, int n_coarse, const double *freq_mhz, int n_frames,
                              int n_beams, int upchan_len, double dm, double f_ref_mhz, int32_t *delay_scratch,
                              uint32_t *out_u32, int n_out) {
    if (!beams_u8 || !freq_mhz || !delay_scratch || !out_u32 || n_coarse < 1 || n_frames < 1 || !(dm >= 0)) {
        set_err("dedisperse_beams: bad argument");
        return CHIME_BF_E_INVALID_ARG;
    }
    if (n_beams < 32 || n_beams % 32 || (upchan_len != 128 && upchan_len != 256)) {
        set_err("dedisperse_beams: n_beams must be a positive multiple of 32, upchan_len 128 or 256");
        return CHIME_BF_E_INVALID_ARG;
    }
    if ((uintptr_t)beams_u8 & 15) { set_err("dedisperse_beams: input must be 16-byte aligned"); return CHIME_BF_E_ALIGNMENT; }
    std::vector<int32_t> tab;
    const int mx = dedisp_table(freq_mhz, n_coarse, upchan_len, dm, f_ref_mhz, tab);
    for (int32_t d : tab)
        if (d < 0) { set_err("dedisperse_beams: f_ref below a fine channel (negative delay)"); return CHIME_BF_E_INVALID_ARG; }
    if (n_frames - mx < 1 || n_out != n_frames - mx) {
        set_err("dedisperse_beams: n_out must be n_frames - max delay = %d (got %d)", n_frames - mx, n_out);
        return CHIME_BF_E_INVALID_ARG;
    }
    return launch_dedisperse(stream, beams_u8, n_coarse, n_frames, n_beams, tab, delay_scratch, out_u32, n_out, false);
}

int chime_bf_dedisperse_beams_noalloc(void *stream, const uint8_t *beams_u8, int n_coarse, const double *freq_mhz,
                                      int n_frames, int n_beams, int upchan_len, double dm, double f_ref_mhz,
                                      uint32_t *out_u32, int n_out) {
    if (!beams_u8 || !freq_mhz || !out_u32 || n_coarse < 1 || n_frames < 1 || !(dm >= 0)) {
        set_err("dedisperse_beams_noalloc: bad argument");
        return CHIME_BF_E_INVALID_ARG;
    }
    if (n_coarse > CHIME_BF_NOALLOC_MAX_COARSE) {
        set_err("dedisperse_beams_noalloc: n_coarse %d exceeds the built-in scratch (CHIME_BF_NOALLOC_MAX_COARSE = %d); "
                "use chime_bf_dedisperse_beams with a caller-owned table", n_coarse, CHIME_BF_NOALLOC_MAX_COARSE);
        return CHIME_BF_E_INVALID_ARG;
    }
    if (n_beams < 32 || n_beams % 32 || (upchan_len != 128 && upchan_len != 256)) {
        set_err("dedisperse_beams_noalloc: n_beams must be a positive multiple of 32, upchan_len 128 or 256");
        return CHIME_BF_E_INVALID_ARG;
    }
    if ((uintptr_t)beams_u8 & 15) { set_err("dedisperse_beams_noalloc: input must be 16-byte aligned"); return CHIME_BF_E_ALIGNMENT; }
    static thread_local std::vector<int32_t> tab;   // host side: sized on the thread's first call, re-used afterwards
    tab.reserve((size_t)CHIME_BF_NOALLOC_MAX_COARSE * 16);
    const int mx = dedisp_table(freq_mhz, n_coarse, upchan_len, dm, f_ref_mhz, tab);
    for (int32_t d : tab)
        if (d < 0) { set_err("dedisperse_beams_noalloc: f_ref below a fine channel (negative delay)"); return CHIME_BF_E_INVALID_ARG; }
    if (n_frames - mx < 1 || n_out != n_frames - mx) {
        set_err("dedisperse_beams_noalloc: n_out must be n_frames - max delay = %d (got %d)", n_frames - mx, n_out);
        return CHIME_BF_E_INVALID_ARG;
    }
    int32_t *d_delay = noalloc_delay_table();   // the device address of the array on the current device
    if (d_delay == nullptr) return CHIME_BF_E_CUDA;
    // launch_dedisperse rewrites tab.size() entries of the table on `stream` before the kernel reads them (unless this
    // thread's previous call left exactly this table there, on this stream), and clears out_u32 when the channel loop is
    // split: nothing else of a previous call's contents is read.
    return launch_dedisperse(stream, beams_u8, n_coarse, n_frames, n_beams, tab, d_delay, out_u32, n_out, true);
}

int chime_bf_get_ns_index(const chime_bf_plan *plan, int32_t *host_out) {
    if (!plan || !host_out) {
        set_err("get_ns_index: null argument");
        return CHIME_BF_E_INVALID_ARG;
    }
    memcpy(host_out, plan->J.data(), plan->J.size() * sizeof(int32_t));
    return CHIME_BF_OK;
}

int chime_bf_debug_unpack(chime_bf_plan *plan, void *stream, const uint8_t *in_u8, size_t n_bytes,
                          int8_t *out_re_im) {
    if (!plan || (n_bytes && (!in_u8 || !out_re_im))) {
        set_err("debug_unpack: null argument");
        return CHIME_BF_E_INVALID_ARG;
    }
    if (n_bytes == 0) return CHIME_BF_OK;
    const int threads = 256;
    const int blocks = (int)std::min<size_t>((n_bytes + threads - 1) / threads, 148 * 16);
    chime4::unpack_debug_kernel<<<blocks, threads, 0, (cudaStream_t)stream>>>(in_u8, n_bytes, out_re_im);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        set_err("debug_unpack: %s", cudaGetErrorString(e));
        return CHIME_BF_E_CUDA;
    }
    return CHIME_BF_OK;
}

int chime_bf_kernel_status(const chime_bf_plan *plan) {
    if (!plan || !plan->h_status) return 0;
    for (int i = 0; i < 128; ++i)
        if (plan->h_status[i]) return (i >> 3) | (plan->h_status[i] & ~0xFF);   // which wait, warp and tile counter
    return 0;
}

int chime_bf_measure_fp32_peak(void *stream, int n_iter, double *tflops_out) {
    if (!tflops_out || n_iter < 1) { set_err("measure_fp32_peak: bad argument"); return CHIME_BF_E_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, n_sm = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    float *sink = nullptr;
    cudaEvent_t e0, e1;
    if (cudaMalloc((void **)&sink, sizeof(float) * 1024) != cudaSuccess || cudaEventCreate(&e0) != cudaSuccess ||
        cudaEventCreate(&e1) != cudaSuccess) { set_err("measure_fp32_peak: allocation failed"); return CHIME_BF_E_CUDA; }
    const int grid = n_sm * 4, block = 512;
    for (int packed = 0; packed < 2; ++packed) {
        float ms = 0.f;
        for (int rep = 0; rep < 3; ++rep) {   // best of three (the first also warms up)
            cudaEventRecord(e0, st);
            if (packed) chime_peak::fp32_peak_kernel<true><<<grid, block, 0, st>>>(n_iter, sink);
            else chime_peak::fp32_peak_kernel<false><<<grid, block, 0, st>>>(n_iter, sink);
            cudaEventRecord(e1, st);
            if (cudaEventSynchronize(e1) != cudaSuccess) { set_err("measure_fp32_peak: %s", cudaGetErrorString(cudaGetLastError())); return CHIME_BF_E_CUDA; }
            float t = 0.f;
            cudaEventElapsedTime(&t, e0, e1);
            if (rep == 0 || t < ms) ms = t;
        }
        tflops_out[packed] = (double)grid * block * (double)n_iter * 256.0 * 2.0 / (ms * 1e-3) / 1e12;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    return CHIME_BF_OK;
}

#ifdef CHIME_PROF
int chime_bf_debug_prof(long long *host_out) {   // development builds only: per-warp wait cycles of the last launch
    return cudaMemcpyFromSymbol(host_out, chime4::g_prof, sizeof(long long) * 148 * 4 * 24 * 12) == cudaSuccess ? 0 : -1;
}
#endif

int chime_bf_n_frames(const chime_bf_plan *plan) { return plan ? plan->R : 0; }
size_t chime_bf_in_bytes(const chime_bf_plan *plan) {
    return plan ? (size_t)plan->C * plan->T * 2048 : 0;
}
size_t chime_bf_out_elems(const chime_bf_plan *plan) {
    return plan ? (size_t)plan->C * plan->R * 1024 * 16 : 0;
}
int chime_bf_launches_per_execute(const chime_bf_plan *plan) { return plan ? 1 : 0; }   // execute_host: one per chunk

void chime_bf_destroy(chime_bf_plan *pl) {
    if (!pl) return;
    cudaFree(pl->d_stage_in);
    cudaFree(pl->d_stage_out);
    ++g_dd_upload_epoch;   // no later plan that gets this address may be taken for this one (launch_dedisperse)
    cudaFree(pl->d_delay);
    cudaFree(pl->d_ring);
    cudaFree(pl->d_delay_stream);
    cudaFree(pl->d_peer_out);
    cudaFree(pl->d_turns);
    cudaFree(pl->d_scratch);
    cudaFree(pl->d_wq);
    cudaFree(pl->d_beta);
    cudaFree(pl->d_inv_s2);
    cudaFree(pl->d_wscale);
    cudaFree(pl->d_gains);
    cudaFree(pl->d_J);
    if (pl->h_status) cudaFreeHost(pl->h_status);
    for (cudaEvent_t ev : pl->copy_done)
        if (ev) cudaEventDestroy(ev);
    if (pl->entry) cudaEventDestroy(pl->entry);
    if (pl->copy_stream) cudaStreamDestroy(pl->copy_stream);
    delete pl;
}

}  // extern "C"
