"""Exact chromatic alignment (section 4 "beam interpolation"): with exact_pointing the N-S
weights steer beam m to its desired pointing itself instead of the nearest bin of the zero-padded transform.
Expected values: oracle.cell_exact (direct sums at the exact phase), same tolerances as the nearest-bin path."""
import numpy as np
import pytest
import torch

import synth

pytestmark = pytest.mark.gpu

REL_TOL = 1e-4
U8_FRAC = 1e-3


@pytest.fixture(scope="module")
def bf():
    import __graft_entry__ as g
    g.build()
    import paper_1702_04728_b200 as bf
    return bf


def _check(orc, out_f32, out_u8, cells, hb, freqs, gains, **kw):
    worst, n_diff, n_tot = 0.0, 0, 0
    for (c, R) in cells:
        I = orc.cell_exact(hb[c, 384 * R:384 * (R + 1)], float(freqs[c]), gains=None if gains is None else gains[c], **kw)
        err = np.abs(out_f32[c, R] - I).max(axis=-1) / I.mean(axis=-1)
        worst = max(worst, float(err.max()))
        d = np.abs(out_u8[c, R].astype(int) - orc.quantize(I).astype(int))
        assert d.max() <= 1
        n_diff += int((d != 0).sum())
        n_tot += d.size
    assert worst <= REL_TOL, worst
    assert n_diff <= U8_FRAC * n_tot
    return worst


def test_exact_pointing_matches_oracle(bf, orc):
    C, T = 3, 2 * 384
    freqs = np.array([800.0, 611.71875, 400.390625])
    seed = synth.config_seed(4) + 7
    gains = synth.gains(seed, C, flagged_frac=0.05)
    b = synth.noise_bytes(seed, C, T)
    plan = bf.plan_create_ex(C, freq_mhz=freqs, gains=gains, n_time=T, exact_pointing=True)
    out_f32 = plan.execute_f32(b.cuda()).cpu().numpy()
    out_u8 = plan.execute(b.cuda()).cpu().numpy()
    worst = _check(orc, out_f32, out_u8, [(0, 0), (1, 1), (2, 0)], b.numpy(), freqs, gains)
    print(f"exact pointing: worst rel err {worst:.2e}")
    # and it is NOT the nearest-bin result away from f_ref (the two differ by the pointing loss)
    near = bf.plan_create_ex(C, freq_mhz=freqs, gains=gains, n_time=T)
    diff = np.abs(near.execute_f32(b.cuda()).cpu().numpy() - out_f32).max() / out_f32.mean()
    assert diff > 1e-2
    plan.destroy()
    near.destroy()


def test_exact_pointing_tone_peaks_with_full_gain(bf, orc):
    """cfg0's tone (sin theta = 0.2 at 600 MHz) moved to 710 MHz: with exact pointing the brightest N-S beam is the one
    whose desired pointing is nearest to the source, as for the oracle."""
    f = 710.15625
    b = synth.tone_bytes(synth.config_seed(0), f, 768)
    plan = bf.plan_create_ex(1, freq_mhz=[f], n_time=768, exact_pointing=True)
    out_f32 = plan.execute_f32(b.cuda()).cpu().numpy()
    out_u8 = plan.execute(b.cuda()).cpu().numpy()
    _check(orc, out_f32, out_u8, [(0, 0), (0, 1)], b.numpy(), [f], None)
    I = orc.cell_exact(b.numpy()[0, :384], f)
    assert np.unravel_index(out_f32[0, 0].argmax(), out_f32[0, 0].shape)[1] == np.unravel_index(I.argmax(), I.shape)[1]
    plan.destroy()


def test_exact_pointing_explicit_grid_and_repointing(bf, orc):
    """An explicit sin(theta) grid (denser tiling), then a re-pointing on the live plan."""
    f = 523.4375
    s1 = np.linspace(-0.35, 0.35, 256)
    s2 = np.linspace(-0.8, 0.6, 256)
    b = synth.noise_bytes(12, 1, 384)
    plan = bf.plan_create_ex(1, freq_mhz=[f], n_time=384, ns_sin_theta=s1, exact_pointing=True)
    for s in (s1, s2):
        if s is s2:
            plan.update_pointings(ns_sin_theta=s2)
        out_f32 = plan.execute_f32(b.cuda()).cpu().numpy()
        out_u8 = plan.execute(b.cuda()).cpu().numpy()
        _check(orc, out_f32, out_u8, [(0, 0)], b.numpy(), [f], None, sin_theta=s)
    plan.destroy()


def test_exact_pointing_upchan_256(bf, orc):
    """The tensor-core N-S transform serves both up-channelisation lengths, so exact pointing does too."""
    C, U = 2, 256
    T = 2 * 3 * U
    freqs = np.array([779.296875, 433.984375])
    seed = synth.config_seed(4) + 19
    gains = synth.gains(seed, C, flagged_frac=0.05)
    b = synth.noise_bytes(seed, C, T)
    plan = bf.plan_create_ex(C, freq_mhz=freqs, gains=gains, n_time=T, upchan_len=U, exact_pointing=True)
    out_f32 = plan.execute_f32(b.cuda()).cpu().numpy()
    out_u8 = plan.execute(b.cuda()).cpu().numpy()
    hb = b.numpy()
    worst = 0.0
    for (c, R) in [(0, 1), (1, 0)]:
        I = orc.cell_exact(hb[c, 3 * U * R:3 * U * (R + 1)], float(freqs[c]), gains=gains[c], U=U)
        worst = max(worst, float((np.abs(out_f32[c, R] - I).max(axis=-1) / I.mean(axis=-1)).max()))
        d = np.abs(out_u8[c, R].astype(int) - orc.quantize(I).astype(int))
        assert d.max() <= 1 and (d != 0).mean() <= U8_FRAC
    assert worst <= REL_TOL, worst
    plan.destroy()
