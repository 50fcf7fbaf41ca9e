"""GPU parity at BASELINE.json's FULL sizes for configs 2, 3 and 4 (config 0 and 1 are in test_gpu_parity.py).
The oracle checks a seeded sample of output cells plus every cell that holds injected structure (pulse
track, RFI bursts); cells are exactly independent (no state crosses a frame boundary), so a
sample exercises every code path.  Inputs are generated on the device by the counter-based generators of
synth/; the bytes the oracle reads are copied back from the device buffer (the byte buffer is the test
vector) or, for config 3 whose buffers are recycled, regenerated on the CPU from the same counters."""
import numpy as np
import pytest
import torch

import synth
from test_gpu_parity import compare_cells

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def bf():
    import __graft_entry__ as g
    g.build()
    import paper_1702_04728_b200 as bf
    assert torch.cuda.is_available()
    return bf


def _free():
    import gc
    gc.collect()
    torch.cuda.empty_cache()


def test_cfg2_pulse_full_size(bf, orc):
    """64 channels x 390528 samples (51.2 GB): noise + dispersed FRB-like pulse (DM 500, 1 ms, S/N 20 per
    channel) from the direction of beam (E-W 2, N-S 140), random gains.  Oracle on the pulse track +-2 frames
    in every channel and on 128 random cells; the arg-max beam of the track-summed intensity must agree."""
    cfg = synth.CONFIGS[2]
    C, T = cfg["n_coarse"], cfg["n_time"]
    R_tot = T // 384
    seed = synth.config_seed(2)
    freqs = synth.config_freqs(2)
    gains = synth.gains(seed, C, flagged_frac=cfg["flagged"])
    m0, e0 = 140, 2
    s0 = (m0 - 128) * synth.C0 / (256 * 0.3048 * 600e6)          # centre of N-S beam 140 (reading A2)
    sphi = float(np.sin(np.deg2rad(0.2)))                         # centre of E-W beam 2
    d_in = synth.noise_bytes(seed, C, T, device="cuda")
    centres = synth.add_pulse(d_in, seed, freqs, gains=gains, sin_theta=s0, sin_phi=sphi)
    plan = bf.plan_create_ex(C, freq_mhz=freqs, gains=gains, n_time=T)
    out_f32 = plan.execute_f32(d_in)
    out_u8 = plan.execute(d_in)
    torch.cuda.synchronize()

    track = [(c, int(centres[c]) // 384) for c in range(C)]
    cells = set()
    for c, R0 in track:
        for dR in range(-2, 3):
            if 0 <= R0 + dR < R_tot:
                cells.add((c, R0 + dR))
    rng = np.random.default_rng(seed)
    cells |= {(int(rng.integers(C)), int(rng.integers(R_tot))) for _ in range(128)}
    cells |= {(0, 0), (C - 1, R_tot - 1)}
    cells = sorted(cells)

    cache = {}

    def host_bytes(c, R):
        return d_in[c, 384 * R:384 * (R + 1)].cpu().numpy()

    # compare_cells computes the oracle cell by cell; keep the oracle's intensities of the track cells
    orig_cell = orc.cell

    def caching_cell(blk, f, **kw):
        I, J = orig_cell(blk, f, **kw)
        cache[len(cache)] = I
        return I, J

    orc_proxy = type("O", (), {"cell": staticmethod(caching_cell), "quantize": staticmethod(orc.quantize)})
    worst, frac = compare_cells(orc_proxy, plan, d_in, host_bytes, freqs, gains, cells, 512, 128,
                                out_f32=out_f32, out_u8=out_u8)
    by_cell = {cell: cache[i] for i, cell in enumerate(cells)}

    # beam localisation: intensity summed over the fine channels and over the pulse-track cells of all channels
    acc_o = np.zeros((4, 256))
    acc_g = np.zeros((4, 256))
    for c, R0 in track:
        for dR in (-1, 0, 1):
            if (c, R0 + dR) in by_cell:
                acc_o += by_cell[(c, R0 + dR)].sum(-1)
                acc_g += out_f32[c, R0 + dR].sum(-1).double().cpu().numpy()
    peak_o = np.unravel_index(acc_o.argmax(), acc_o.shape)
    peak_g = np.unravel_index(acc_g.argmax(), acc_g.shape)
    assert tuple(peak_o) == (e0, m0), f"oracle localises the pulse in beam {peak_o}"
    assert tuple(peak_g) == tuple(peak_o), f"GPU localises the pulse in {peak_g}, oracle in {peak_o}"
    off = np.delete(acc_o.ravel(), e0 * 256 + m0)
    print(f"cfg2: {len(cells)} cells, worst rel err {worst:.2e}, u8 diff frac {frac:.2e}, "
          f"pulse beam (ew,ns)={tuple(int(x) for x in peak_g)}, band-summed S/N "
          f"{(acc_o[e0, m0] - off.mean()) / off.std():.0f}")
    plan.destroy()
    del d_in, out_f32, out_u8
    _free()


def test_cfg3_full_band_streaming(bf, orc):
    """1024 channels x 49152 samples as 8 channel groups of 128 (12.9 GB each) through two device buffers on
    two streams; 64 random cells against the oracle (their bytes regenerated on the CPU from the counters)."""
    from paper_1702_04728_b200.streaming import FullBandStreamer
    cfg = synth.CONFIGS[3]
    C, T, G = cfg["n_coarse"], cfg["n_time"], cfg["group"]
    seed = synth.config_seed(3)
    freqs = synth.config_freqs(3)
    st = FullBandStreamer(C, G, T, freq_mhz=freqs)
    assert st.n_groups == 8 and st.group_in_bytes == 128 * 49152 * 2048

    def fill(g, buf):
        buf.copy_(synth.noise_bytes(seed, G, T, device="cuda", chan0=g * G))

    out_f32 = [torch.empty(st.group_out_shape, dtype=torch.float32, device="cuda") for _ in range(st.n_groups)]
    out_u8 = st.run_chunk(fill, out_f32=out_f32)
    st.synchronize()
    torch.cuda.synchronize()
    assert st.launches == 16

    rng = np.random.default_rng(seed)
    cells = [(0, 0), (C - 1, T // 384 - 1)] + [(int(rng.integers(C)), int(rng.integers(T // 384)))
                                               for _ in range(62)]
    worst, n_diff, n_tot = 0.0, 0, 0
    for (c, R) in cells:
        blk = synth.noise_bytes(seed, 1, 384, chan0=c, time0=384 * R, n_time_total=T).numpy()[0]
        I, Jo = orc.cell(blk, float(freqs[c]))
        g, cl = divmod(c, G)
        assert np.array_equal(st.plans[g].get_ns_index()[cl], Jo)
        got = out_f32[g][cl, R].cpu().numpy()
        worst = max(worst, float((np.abs(got - I) / I.mean(axis=-1, keepdims=True)).max()))
        d = np.abs(out_u8[g][cl, R].cpu().numpy().astype(int) - orc.quantize(I).astype(int))
        assert d.max() <= 1
        n_diff += int((d != 0).sum())
        n_tot += d.size
    assert worst <= 1e-4 and n_diff <= 1e-3 * n_tot
    print(f"cfg3: {len(cells)} cells over 1024 channels, worst rel err {worst:.2e}, u8 diff frac {n_diff / n_tot:.2e}")
    st.destroy()
    del out_f32, out_u8, st
    _free()


@pytest.fixture(scope="module")
def cfg4_input():
    cfg = synth.CONFIGS[4]
    C, T = cfg["n_coarse"], cfg["n_time"]
    seed = synth.config_seed(4)
    d_in = synth.noise_bytes(seed, C, T, device="cuda")
    d_in, mask = synth.saturate_bursts(d_in, seed, frac=0.05, burst=64, inplace=True)
    yield d_in, mask.cpu().numpy()
    del d_in
    _free()


@pytest.mark.parametrize("NP,U", [(256, 128), (512, 128), (1024, 128), (256, 256), (512, 256), (1024, 256)])
def test_cfg4_stress_full_size(bf, orc, cfg4_input, NP, U):
    """256 channels x 98304 samples (51.5 GB), 5 % of samples saturated at +-7 in bursts of 64, 10 % of inputs
    zero-weighted; every zero_pad x upchan setting: index table in full, 64 random cells + 32 cells that contain
    a burst against the oracle."""
    d_in, mask = cfg4_input
    cfg = synth.CONFIGS[4]
    C, T = cfg["n_coarse"], cfg["n_time"]
    seed = synth.config_seed(4)
    freqs = synth.config_freqs(4)
    gains = synth.gains(seed, C, flagged_frac=cfg["flagged"])
    assert abs(float((np.abs(gains).sum(-1) == 0).mean()) - 0.10) < 0.01
    assert abs(float(mask.mean()) - 0.05) < 0.01
    frame = 3 * U
    R_tot = T // frame
    plan = bf.plan_create_ex(C, freq_mhz=freqs, gains=gains, zero_pad=NP, upchan_len=U, n_time=T)
    J = plan.get_ns_index()
    for c in range(C):
        assert np.array_equal(J[c], orc.ns_index(freqs[c], NP)), (NP, c)
    rng = np.random.default_rng(seed + NP + U)
    cells = {(int(rng.integers(C)), int(rng.integers(R_tot))) for _ in range(64)}
    has_burst = mask.reshape(C, R_tot, frame).any(-1)
    bc, bR = np.nonzero(has_burst)
    pick = rng.choice(len(bc), size=32, replace=False)
    cells |= {(int(bc[i]), int(bR[i])) for i in pick}
    cells = sorted(cells)
    worst, frac = compare_cells(orc, plan, d_in, lambda c, R: d_in[c, frame * R:frame * (R + 1)].cpu().numpy(),
                                freqs, gains, cells, NP, U)
    print(f"cfg4 NP={NP} U={U}: {len(cells)} cells, worst rel err {worst:.2e}, u8 diff frac {frac:.2e}")
    plan.destroy()
    _free()
