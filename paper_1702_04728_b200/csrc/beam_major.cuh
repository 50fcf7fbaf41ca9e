// Beam-major exchange addressing (chime_bf_execute_beam_major, the corner turn from
// channel-sharded beamformer nodes to beam-sharded search nodes).
#pragma once
#include <stdint.h>
#include <cuda_runtime.h>

namespace chime {

// Beam b = ew * 256 + ns of (global channel cg, frame Rf) goes to rank d = b / (1024 / n_peers), at
// [cg][Rf][b - d * 1024 / n_peers][16 fine] of that rank's receive buffer: the all-to-all corner turn is the
// epilogue's 16-byte store itself; with peer-mapped pointers the store crosses NVLink.
__device__ __forceinline__ uint4 *beam_major_dst(uint8_t *const *peer_out, const int n_peers, const int cg,
                                                 const int n_frames, const int Rf, const int b) {
    const int bpr = 1024 / n_peers, d = b / bpr;
    return reinterpret_cast<uint4 *>(peer_out[d] + (((size_t)cg * n_frames + Rf) * bpr + (b - d * bpr)) * 16);
}

}  // namespace chime
