"""Seeded synthetic CHIME-shaped inputs (stand-ins for telescope data, which is not available).

This module serves both the tests' oracle side and the CUDA side and therefore holds NONE of the
beamformer's arithmetic: it only draws packed 4+4-bit baseband bytes, gains and frequency lists.
Whatever it emits, *the byte buffer is the test vector*: both sides read the same bytes.

Recipe (BASELINE.json configs; PAPER.md:32-47 for shapes and rates):
  * counter-based generator: splitmix64 of (seed, global byte index) -> 64 random bits per byte,
    high 32 bits drive the real nibble, low 32 bits the imaginary nibble.  Integer only, so CPU and
    CUDA tensors hold identical bytes, and any sub-block can be generated on its own.
  * noise: each nibble value k in [-7, 7] with probability Phi((k+1/2)/sigma) - Phi((k-1/2)/sigma),
    tails lumped into +-7 (round(N(0, sigma)) clipped), via a 14-entry uint32 CDF table.
  * byte = ((re + 8) << 4) | (im + 8)   (offset binary, high nibble real; reading A1).
"""
import math

import numpy as np
import torch

BASE_SEED = 170204728
N_INPUT = 2048  # 2 pol x 4 cyl x 256 feeds; input index i = (pol*4 + cyl)*256 + feed
C0 = 299792458.0

_M64 = (1 << 64) - 1


def _s64(v):
    """Python int (mod 2^64) -> the same bits as a signed int64 value."""
    v &= _M64
    return v - (1 << 64) if v >= (1 << 63) else v


def _lsr(x, s):
    """Logical shift right of an int64 tensor."""
    return (x >> s) & ((1 << (64 - s)) - 1)


def splitmix64(idx, seed):
    """idx: int64 tensor of counters.  Returns int64 tensor of 64 mixed bits (wrapping arithmetic)."""
    z = idx + _s64(seed * 0x9E3779B97F4A7C15 + 0x9E3779B97F4A7C15)
    z = (z ^ _lsr(z, 30)) * _s64(0xBF58476D1CE4E5B9)
    z = (z ^ _lsr(z, 27)) * _s64(0x94D049BB133111EB)
    return z ^ _lsr(z, 31)


def _cdf_thresholds(sigma):
    """14 thresholds T_k = floor(2^32 Phi((k+1/2)/sigma)), k = -7..6."""
    t = []
    for k in range(-7, 7):
        phi = 0.5 * (1.0 + math.erf((k + 0.5) / (sigma * math.sqrt(2.0))))
        t.append(int(math.floor(phi * 4294967296.0)))
    return t


def _nibbles_from_bits(bits, thr):
    """bits: int64 tensor holding a uint32 in [0, 2^32). -> offset nibble (value + 8) in [1, 15]."""
    return torch.bucketize(bits, thr, right=True) + 1


def noise_bytes(seed, n_chan, n_time, sigma=2.5, device="cpu", chan0=0, time0=0, n_time_total=None,
                chunk=1 << 24):
    """Packed Gaussian-noise baseband [n_chan][n_time][2048] uint8.  The counter of a byte is its
    index in the full [.. n_chan_total ..][n_time_total][2048] array, so sub-blocks (chan0, time0)
    reproduce the same bytes as the corresponding slice of a full generation."""
    n_time_total = n_time if n_time_total is None else n_time_total
    thr = torch.tensor(_cdf_thresholds(sigma), dtype=torch.int64, device=device)
    out = torch.empty((n_chan, n_time, N_INPUT), dtype=torch.uint8, device=device)
    flat = out.view(n_chan, -1)
    per_chan = n_time * N_INPUT
    for c in range(n_chan):
        base = ((chan0 + c) * n_time_total + time0) * N_INPUT
        for s in range(0, per_chan, chunk):
            e = min(per_chan, s + chunk)
            idx = torch.arange(base + s, base + e, dtype=torch.int64, device=device)
            h = splitmix64(idx, seed)
            re = _nibbles_from_bits(_lsr(h, 32), thr)
            im = _nibbles_from_bits(h & 0xFFFFFFFF, thr)
            flat[c, s:e] = ((re << 4) | im).to(torch.uint8)
    return out


def uniform01(seed, n, stream, device="cpu"):
    """n float64 uniforms in [0,1) from counter stream `stream` (independent of the byte streams)."""
    idx = torch.arange(n, dtype=torch.int64, device=device) + _s64((stream + 1) << 40)
    h = splitmix64(idx, seed ^ 0x5DEECE66D)
    return _lsr(h, 11).to(torch.float64) * (1.0 / 9007199254740992.0)


def gaussian(seed, shape, stream, device="cpu"):
    """float64 standard normals (Box-Muller on two counter streams)."""
    n = int(np.prod(shape))
    u1 = uniform01(seed, n, 2 * stream + 100, device)
    u2 = uniform01(seed, n, 2 * stream + 101, device)
    r = torch.sqrt(-2.0 * torch.log(1.0 - u1))
    return (r * torch.cos(2.0 * math.pi * u2)).reshape(shape)


def pack_voltage(v_re, v_im):
    """round-half-even, clip to [-7, 7], offset-binary pack.  v_*: float tensors, same shape."""
    re = torch.clamp(torch.round(v_re), -7, 7).to(torch.int64) + 8
    im = torch.clamp(torch.round(v_im), -7, 7).to(torch.int64) + 8
    return ((re << 4) | im).to(torch.uint8)


def tone_bytes(seed, f_mhz, n_time, sin_theta=0.2, sin_phi=0.0, q0=37, U=128, amp=3.0, sigma=2.5,
               feed_spacing_m=0.3048, cyl_spacing_m=22.0, device="cpu"):
    """cfg0: noise + one point-source tone, added before rounding/clipping.
    Plane wave exp(+2 pi i f (n d sin_theta + x_cyl sin_phi)/c0) exp(+2 pi i q0 t/U) on both pols.
    Returns [1][n_time][2048] uint8."""
    shape = (n_time, 2, 4, 256)
    nr = gaussian(seed, shape, 0, device) * sigma
    ni = gaussian(seed, shape, 1, device) * sigma
    t = torch.arange(n_time, dtype=torch.float64, device=device).view(-1, 1, 1, 1)
    cyl = torch.arange(4, dtype=torch.float64, device=device).view(1, 1, 4, 1)
    n = torch.arange(256, dtype=torch.float64, device=device).view(1, 1, 1, 256)
    ph = 2.0 * math.pi * ((f_mhz * 1e6 / C0) * (n * feed_spacing_m * sin_theta
                                                + cyl * cyl_spacing_m * sin_phi) + q0 * t / U)
    b = pack_voltage(nr + amp * torch.cos(ph), ni + amp * torch.sin(ph))
    return b.reshape(1, n_time, N_INPUT)


def gains(seed, n_chan, flagged_frac=0.02, amp_lo=0.8, amp_hi=1.2):
    """Per-input complex gains [n_chan][2048][2] float32: |g| ~ U(lo,hi), arg ~ U(0,2pi);
    a fraction `flagged_frac` of inputs has g = 0 (flagged)."""
    n = n_chan * N_INPUT
    a = amp_lo + (amp_hi - amp_lo) * uniform01(seed, n, 10)
    ph = 2.0 * math.pi * uniform01(seed, n, 11)
    keep = (uniform01(seed, n, 12) >= flagged_frac).to(torch.float64)
    g = torch.stack([a * torch.cos(ph) * keep, a * torch.sin(ph) * keep], dim=-1)
    return g.to(torch.float32).reshape(n_chan, N_INPUT, 2).numpy()


def saturate_bursts(b, seed, frac=0.05, burst=64, inplace=False):
    """cfg4 RFI: a fraction `frac` of time samples, in bursts of `burst` consecutive samples, have
    every input's re and im set to +-7 with random signs.  b: [C][T][2048] uint8 (a modified copy is
    returned unless inplace=True: the 51 GB buffer of cfg4 is not cloned).
    Returns (bytes, burst_mask [C][T] bool)."""
    C, T, _ = b.shape
    dev = b.device
    nb = (T + burst - 1) // burst
    u = uniform01(seed, C * nb, 20, dev).reshape(C, nb)
    mask = (u < frac).repeat_interleave(burst, dim=1)[:, :T]
    out = b if inplace else b.clone()
    for c in range(C):
        ts = torch.nonzero(mask[c]).flatten()
        if ts.numel() == 0:
            continue
        idx = (c * T + ts).view(-1, 1) * N_INPUT + torch.arange(N_INPUT, dtype=torch.int64, device=dev)
        h = splitmix64(idx, seed ^ 0xABCDEF)
        re = torch.where((h & 1) == 0, 15, 1)   # +7 -> nibble 15, -7 -> nibble 1
        im = torch.where((h & 2) == 0, 15, 1)
        out[c, ts] = ((re << 4) | im).to(torch.uint8)
    return out, mask


K_DM_MS = 4.148808          # dispersion constant: delay = K_DM_MS ms * DM * (f/GHz)^-2
SAMPLE_S = 2.56e-6          # PAPER.md:37 (Table 1)


def pulse_centres(freqs_mhz, n_time, dm=500.0, t0_samples=1000.0, f_top_mhz=800.0):
    """cfg2: arrival time (in samples, float64) of a dispersed pulse in each coarse channel,
    t0 + K_DM*DM*(f^-2 - f_top^-2), wrapped modulo the n_time window so that every channel contains
    the pulse (the 9.7 s sweep of DM 500 over 400-800 MHz is longer than the 1 s buffer)."""
    f = np.asarray(freqs_mhz, dtype=np.float64) / 1e3
    delay_s = K_DM_MS * 1e-3 * dm * (f ** -2 - (f_top_mhz / 1e3) ** -2)
    return np.mod(t0_samples + delay_s / SAMPLE_S, float(n_time))


def pulse_amplitude_var(snr=20.0, width_samples=390.625, sigma_in2=12.556, n_inputs_per_pol=1024):
    """Peak per-input variance p0 of the pulse voltage such that the matched-filter S/N of the
    16-fine-channel-summed intensity of the on-source beam is `snr` in one coarse channel:
      signal = 2 pol * N*N_c * sum_t p(t) = 2*1024 * 1.0645 p0 w      (Gaussian envelope, FWHM w)
      noise  = sigma_in^2 * sqrt(2 pol * w)                          (|.|^2 of Gaussian noise, w samples)
    sigma_in2 = variance of one complex noise sample (re + im) of round(N(0, 2.5)) clipped."""
    w = width_samples
    return snr * sigma_in2 * math.sqrt(2.0 * w) / (2.0 * n_inputs_per_pol * 1.0645 * w)


def add_pulse(b, seed, freqs_mhz, gains=None, sin_theta=0.0, sin_phi=0.0, dm=500.0, snr=20.0,
              width_s=1e-3, sigma=2.5, t0_samples=1000.0, feed_spacing_m=0.3048, cyl_spacing_m=22.0,
              half_window=640):
    """cfg2: adds a dispersed, noise-like (FRB-like) pulse from direction (sin_theta, sin_phi) to the
    packed baseband b [C][T][2048] IN PLACE and returns the per-channel pulse centres (samples).

    Inside a window of +-half_window samples around each channel's arrival time the samples are redrawn
    as  pack(round(clip( N(0, sigma) noise + h_i * a(t) s(t) * geometric phase ))), i.e. the pulse is added
    BEFORE the 4-bit quantisation.  s(t) is one complex Gaussian series common to all inputs, a(t) a
    Gaussian envelope of FWHM width_s, h_i = 1/g_i the instrumental response that the plan's calibration
    gain g_i undoes (flagged inputs, g = 0, carry noise only).  The intra-channel dispersion chirp is
    omitted (flagged simplification).  Windows that would cross the buffer ends are clipped."""
    C, T, _ = b.shape
    dev = b.device
    w = width_s / SAMPLE_S
    centres = pulse_centres(freqs_mhz, T, dm, t0_samples)
    p0 = pulse_amplitude_var(snr, w)
    n = torch.arange(256, dtype=torch.float64, device=dev).view(1, 1, 1, 256)
    cyl = torch.arange(4, dtype=torch.float64, device=dev).view(1, 1, 4, 1)
    for c in range(C):
        lo = max(0, int(centres[c]) - half_window)
        hi = min(T, int(centres[c]) + half_window)
        L = hi - lo
        shape = (L, 2, 4, 256)
        nr = gaussian(seed + 7919 * (c + 1), shape, 0, dev) * sigma
        ni = gaussian(seed + 7919 * (c + 1), shape, 1, dev) * sigma
        t = torch.arange(lo, hi, dtype=torch.float64, device=dev)
        env = torch.sqrt(p0 / 2.0 * torch.exp(-4.0 * math.log(2.0) * ((t - centres[c]) / w) ** 2))
        sr = gaussian(seed + 7919 * (c + 1), (L,), 2, dev) * env
        si = gaussian(seed + 7919 * (c + 1), (L,), 3, dev) * env
        ph = 2.0 * math.pi * (float(freqs_mhz[c]) * 1e6 / C0) * (n * feed_spacing_m * sin_theta
                                                                 + cyl * cyl_spacing_m * sin_phi)
        hr, hi_ = torch.cos(ph), torch.sin(ph)                      # geometric phase [1][1][4][256]
        if gains is not None:                                       # h = 1/g = conj(g)/|g|^2
            g = torch.as_tensor(gains[c], dtype=torch.float64, device=dev).reshape(1, 2, 4, 256, 2)
            g2 = g[..., 0] ** 2 + g[..., 1] ** 2
            inv = torch.where(g2 > 0, 1.0 / torch.where(g2 > 0, g2, torch.ones_like(g2)), torch.zeros_like(g2))
            ir, ii = g[..., 0] * inv, -g[..., 1] * inv
            hr, hi_ = hr * ir - hi_ * ii, hr * ii + hi_ * ir
        sr4, si4 = sr.view(L, 1, 1, 1), si.view(L, 1, 1, 1)
        vr = nr + (hr * sr4 - hi_ * si4)
        vi = ni + (hr * si4 + hi_ * sr4)
        b[c, lo:hi] = pack_voltage(vr, vi).reshape(L, N_INPUT)
    return centres


def chime_freqs_mhz(n_coarse, step=1, k0=0):
    """f_k = 800 - (k0 + step*k) * 0.390625 MHz (1024 channels over 400-800 MHz)."""
    return np.array([800.0 - (k0 + step * k) * 0.390625 for k in range(n_coarse)], dtype=np.float64)


# The five BASELINE.json configurations (shapes only; see DESIGN.md for what is compared).
CONFIGS = {
    0: dict(name="tiny", n_coarse=1, freqs=[600.0], n_time=768, gains=False),
    1: dict(name="single_node_load", n_coarse=4, step=1, n_time=49152, gains=True, flagged=0.02),
    2: dict(name="pulse", n_coarse=64, step=16, n_time=390528, gains=True, flagged=0.0),
    3: dict(name="full_band", n_coarse=1024, step=1, n_time=49152, gains=False, group=128),
    4: dict(name="stress", n_coarse=256, step=4, n_time=98304, gains=True, flagged=0.10),
}


def config_freqs(cfg_id):
    c = CONFIGS[cfg_id]
    if "freqs" in c:
        return np.array(c["freqs"], dtype=np.float64)
    return chime_freqs_mhz(c["n_coarse"], c["step"])


def config_seed(cfg_id):
    return BASE_SEED + cfg_id
