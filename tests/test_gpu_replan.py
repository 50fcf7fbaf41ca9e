"""Re-plannable tables ("tunable" N-S extent, "static or tracking" E-W beams):
chime_bf_update_gains / _ew_angles / _pointings change a live plan; after each update the CUDA path must
match the oracle evaluated with the new parameters, and be bit-identical to a freshly created plan."""
import numpy as np
import pytest
import torch

import synth

pytestmark = pytest.mark.gpu

REL_TOL, U8_FRAC = 1e-4, 1e-3


@pytest.fixture(scope="module")
def bf():
    import __graft_entry__ as g
    g.build()
    import paper_1702_04728_b200 as bf
    return bf


def _check(orc, plan, d_in, hb, freqs, gains, cells, NP, U, ew_deg, fref=600.0, sin_theta=None):
    frame = 3 * U
    out_f32 = plan.execute_f32(d_in)
    out_u8 = plan.execute(d_in)
    torch.cuda.synchronize()
    J = plan.get_ns_index()
    worst, n_diff, n_tot = 0.0, 0, 0
    for (c, R) in cells:
        f = float(freqs[c])
        Jo = orc.ns_index(f, NP, 256, fref) if sin_theta is None else orc.ns_index_sintheta(f, sin_theta, NP)
        assert np.array_equal(J[c], Jo)
        I = orc.cell_from_u8(hb[c, frame * R:frame * (R + 1)], None if gains is None else gains[c], Jo,
                             orc.ew_weights(f, ew_deg), NP, U)
        got = out_f32[c, R].cpu().numpy()
        mean = I.mean(axis=-1, keepdims=True)
        worst = max(worst, float((np.abs(got - I) / np.where(mean > 0, mean, 1.0)).max()))
        d = np.abs(out_u8[c, R].cpu().numpy().astype(int) - orc.quantize(I).astype(int))
        assert d.max() <= 1
        n_diff += int((d != 0).sum())
        n_tot += d.size
    assert worst <= REL_TOL and n_diff <= U8_FRAC * n_tot, (worst, n_diff, n_tot)
    return out_u8


@pytest.mark.parametrize("NP,U", [(512, 128), (1024, 128), (256, 128), (1024, 256)])
def test_update_tables_match_oracle_and_fresh_plan(bf, orc, NP, U):
    C, T = 2, 2 * 3 * U
    seed = synth.config_seed(1) + 17
    freqs = np.array([717.96875, 455.078125])
    b = synth.noise_bytes(seed, C, T)
    hb, d_in = b.numpy(), b.cuda()
    cells = [(0, 0), (1, 1)]
    ew0 = bf.EW_ANGLES_DEG
    plan = bf.plan_create_ex(C, freq_mhz=freqs, zero_pad=NP, upchan_len=U, n_time=T)
    _check(orc, plan, d_in, hb, freqs, None, cells, NP, U, ew0)

    # 1. new gains (5 % flagged) on the live plan
    gains = synth.gains(seed, C, flagged_frac=0.05)
    plan.update_gains(gains)
    out = _check(orc, plan, d_in, hb, freqs, gains, cells, NP, U, ew0)
    fresh = bf.plan_create_ex(C, freq_mhz=freqs, gains=gains, zero_pad=NP, upchan_len=U, n_time=T)
    assert torch.equal(out, fresh.execute(d_in))
    fresh.destroy()

    # 2. tracking E-W beams: re-point them, gains kept
    ew1 = (-0.45, -0.05, 0.35, 0.75)
    plan.update_ew_angles(ew1)
    out = _check(orc, plan, d_in, hb, freqs, gains, cells, NP, U, ew1)
    fresh = bf.plan_create_ex(C, freq_mhz=freqs, gains=gains, ew_angles=ew1, zero_pad=NP, upchan_len=U, n_time=T)
    assert torch.equal(out, fresh.execute(d_in))
    fresh.destroy()

    # 3. N-S extent: native grid at another reference frequency (wider tiling: f_ref 450 MHz)
    plan.update_pointings(f_ref_mhz=450.0)
    _check(orc, plan, d_in, hb, freqs, gains, cells, NP, U, ew1, fref=450.0)

    # 4. explicit, denser tiling: 256 pointings uniform in sin(theta) over +-0.5
    s = np.linspace(-0.5, 0.5, 256)
    plan.update_pointings(ns_sin_theta=s)
    out = _check(orc, plan, d_in, hb, freqs, gains, cells, NP, U, ew1, sin_theta=s)
    fresh = bf.plan_create_ex(C, freq_mhz=freqs, gains=gains, ew_angles=ew1, zero_pad=NP, upchan_len=U, n_time=T,
                              ns_sin_theta=s)
    assert torch.equal(out, fresh.execute(d_in))
    fresh.destroy()

    # 5. back to unit gains and the default grid: identical to the very first plan state
    plan.update_gains(None)
    plan.update_ew_angles(ew0)
    plan.update_pointings(f_ref_mhz=600.0)
    _check(orc, plan, d_in, hb, freqs, None, cells, NP, U, ew0)
    with pytest.raises(bf.ChimeBfError):
        plan.update_pointings(ns_sin_theta=np.full(256, 1.5))
    plan.destroy()


def test_repointing_the_ew_beams_is_cheap_at_full_band(bf):
    """Tracking E-W beams: on the tensor-core path a re-pointing uploads 32 bytes per channel (the E-W phase
    steps), not the folded weight tables: well under a millisecond of stream time for all 1024 channels."""
    import time
    plan = bf.plan_create_ex(1024, n_time=384)
    torch.cuda.synchronize()
    plan.update_ew_angles((-0.5, -0.1, 0.3, 0.7))
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for k in range(20):
        plan.update_ew_angles((-0.5 + 0.01 * k, -0.1, 0.3, 0.7))
    torch.cuda.synchronize()
    dt = (time.perf_counter() - t0) / 20
    assert dt < 1e-3, dt
    plan.destroy()
