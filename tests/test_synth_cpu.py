"""The seeded input generators (synth/): reproducibility of sub-blocks, the cfg2 dispersed-pulse recipe
(DESIGN.md "Input recipe"), checked through the oracle: the pulse must land in the injected beam."""
import numpy as np
import torch

import synth


def test_noise_subblock_reproduces_full_generation():
    full = synth.noise_bytes(5, 3, 40)
    sub = synth.noise_bytes(5, 1, 8, chan0=2, time0=16, n_time_total=40)
    assert torch.equal(full[2:3, 16:24], sub)
    v = (full.to(torch.int64) >> 4) - 8
    assert int(v.min()) >= -7 and int(v.max()) <= 7          # nibble 0 (-8) is never emitted


def test_pulse_centres_follow_cold_plasma_dispersion():
    f = synth.config_freqs(2)
    assert len(f) == 64 and f[0] == 800.0 and f[-1] == 800.0 - 63 * 16 * 0.390625
    c = synth.pulse_centres(f, 10 ** 9, dm=500.0, t0_samples=1000.0)       # no wrap in a huge window
    assert abs(c[0] - 1000.0) < 1e-9
    d = (c - 1000.0) * synth.SAMPLE_S                                      # seconds
    expect = 4.148808e-3 * 500.0 * ((f / 1e3) ** -2 - 0.8 ** -2)
    assert np.allclose(d, expect, rtol=1e-12, atol=1e-9)
    assert 9.0 < d[-1] < 9.8                                               # ~9.7 s sweep down to 406 MHz
    w = synth.pulse_centres(f, 390528)
    assert np.all((w >= 0) & (w < 390528))


def test_saturate_bursts_inplace_equals_copy():
    b = synth.noise_bytes(9, 2, 512)
    out, mask = synth.saturate_bursts(b, 9, frac=0.2)
    b2 = b.clone()
    out2, mask2 = synth.saturate_bursts(b2, 9, frac=0.2, inplace=True)
    assert out2.data_ptr() == b2.data_ptr() and torch.equal(out, out2) and torch.equal(mask, mask2)
    sat = out[mask]
    assert sat.numel() > 0 and bool((((sat >> 4) == 15) | ((sat >> 4) == 1)).all())
    assert torch.equal(out[~mask], b[~mask])


def test_pulse_lands_in_injected_beam(orc):
    """One channel, three frames: the noise-like pulse injected from (N-S beam 140, E-W beam 2), with the
    instrumental response 1/g on every input, must be the arg-max beam of the oracle's intensity in the
    frames it covers, at a matched S/N of the order of the 20 the recipe asks for."""
    f = np.array([600.0])
    T = 3 * 384
    seed = synth.config_seed(2)
    g = synth.gains(seed, 1, flagged_frac=0.0)
    b = synth.noise_bytes(seed, 1, T)
    m0, e0 = 140, 2
    s0 = (m0 - 128) * synth.C0 / (256 * 0.3048 * 600e6)
    sphi = np.sin(np.deg2rad(0.2))
    centres = synth.add_pulse(b, seed, f, gains=g, sin_theta=s0, sin_phi=sphi)
    assert 0 <= centres[0] < T
    hb = b.numpy()
    I = np.array([orc.cell(hb[0, 384 * R:384 * (R + 1)], 600.0, gains=g[0])[0].sum(-1) for R in range(3)])
    R0 = int(centres[0]) // 384
    e, m = np.unravel_index(I[R0].argmax(), I[R0].shape)
    assert (e, m) == (e0, m0)
    off = np.delete(I[R0].ravel(), e0 * 256 + m0)
    snr = (I[:, e0, m0].sum() - 3 * off.mean()) / (np.sqrt(3) * off.std())
    assert 8.0 < snr < 40.0, snr
