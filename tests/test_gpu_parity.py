"""GPU parity: the CUDA path (through the C-ABI) against the oracle, element by element, on the same
seeded bytes.  Tolerances are BASELINE.json's: float intensities within 1e-4 of the beam's mean power;
uint8 bit-exact except +-1 LSB on at most 0.1 % of entries; index table and unpack bit-exact."""
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
    assert torch.cuda.is_available()
    return bf


def compare_cells(orc, plan, d_in, host_bytes_fn, freqs, gains, cells, np_, U, out_f32=None, out_u8=None):
    """cells: list of (c, R).  host_bytes_fn(c, R) -> [3U][2048] uint8 numpy."""
    if out_f32 is None:
        out_f32 = plan.execute_f32(d_in)
    if out_u8 is None:
        out_u8 = plan.execute(d_in)
    torch.cuda.synchronize()
    J = plan.get_ns_index()
    worst, n_diff, n_tot = 0.0, 0, 0
    for (c, R) in cells:
        g = None if gains is None else gains[c]
        I, Jo = orc.cell(host_bytes_fn(c, R), float(freqs[c]), gains=g, np_=np_, U=U)
        assert np.array_equal(J[c], Jo), f"index table differs for channel {c}"
        got = out_f32[c, R].cpu().numpy()
        mean = I.mean(axis=-1, keepdims=True)
        mean = np.where(mean > 0, mean, 1.0)
        err = np.abs(got - I) / mean
        worst = max(worst, float(err.max()))
        q = orc.quantize(I)
        d = np.abs(out_u8[c, R].cpu().numpy().astype(int) - q.astype(int))
        assert d.max() <= 1, f"uint8 differs by {d.max()} LSB in cell {(c, R)}"
        n_diff += int((d != 0).sum())
        n_tot += d.size
    assert worst <= REL_TOL, f"float intensities off by {worst:.3e} of the beam mean power"
    assert n_diff <= U8_FRAC * n_tot, f"{n_diff}/{n_tot} uint8 entries differ"
    return worst, n_diff / n_tot


def test_cfg0_tiny_full(bf, orc):
    f = 600.0
    b = synth.tone_bytes(synth.config_seed(0), f, 768)
    plan = bf.plan_create_ex(1, freq_mhz=[f], n_time=768)
    d_in = b.cuda()
    hb = b.numpy()
    worst, frac = compare_cells(orc, plan, d_in, lambda c, R: hb[c, 384 * R:384 * (R + 1)], [f], None,
                                [(0, 0), (0, 1)], 512, 128)
    out = plan.execute_f32(d_in).cpu().numpy()
    e, m, g = np.unravel_index(out[0, 0].argmax(), out[0, 0].shape)
    assert m == 159 and g == 12 and e in (1, 2)
    print(f"cfg0: worst rel err {worst:.2e}, u8 diff frac {frac:.2e}")


def test_unpack_bit_exact(bf, orc):
    plan = bf.plan_create_ex(1, n_time=384)
    b = torch.arange(256, dtype=torch.uint8).repeat(37)[:9001].contiguous()   # ragged length
    got = plan.debug_unpack(b.cuda()).cpu().numpy()
    assert np.array_equal(got, orc.unpack(b.numpy()))
    empty = plan.debug_unpack(torch.empty(0, dtype=torch.uint8, device="cuda"))
    assert empty.numel() == 0


def test_index_table_bit_exact_full_band(bf, orc):
    freqs = synth.chime_freqs_mhz(1024)
    for NP in (256, 512, 1024):
        plan = bf.plan_create_ex(1024, zero_pad=NP, n_time=384)
        J = plan.get_ns_index()
        for k in range(1024):
            assert np.array_equal(J[k], orc.ns_index(freqs[k], NP)), (NP, k)
        plan.destroy()


@pytest.mark.parametrize("NP,U", [(256, 128), (512, 128), (1024, 128), (256, 256), (512, 256), (1024, 256)])
def test_variants_small(bf, orc, NP, U):
    """cfg4-style sweep at a size the oracle finishes in seconds: 3 channels x 2 frames, random gains
    with 10 % flagged inputs, 5 % saturated samples."""
    C, frame = 3, 3 * U
    T = 2 * frame
    seed = synth.config_seed(4)
    freqs = np.array([800.0, 611.71875, 400.390625])
    gains = synth.gains(seed, C, flagged_frac=0.10)
    b = synth.noise_bytes(seed, C, T)
    b, _ = synth.saturate_bursts(b, seed)
    plan = bf.plan_create_ex(C, freq_mhz=freqs, gains=gains, zero_pad=NP, upchan_len=U, n_time=T)
    hb = b.numpy()
    cells = [(c, R) for c in range(C) for R in range(2)]
    worst, frac = compare_cells(orc, plan, b.cuda(), lambda c, R: hb[c, frame * R:frame * (R + 1)], freqs,
                                gains, cells, NP, U)
    print(f"NP={NP} U={U}: worst rel err {worst:.2e}, u8 diff frac {frac:.2e}")


def test_degenerate_inputs(bf, orc):
    plan = bf.plan_create_ex(1, freq_mhz=[612.5], n_time=384)
    z = torch.full((1, 384, 2048), 0x88, dtype=torch.uint8, device="cuda")
    assert torch.all(plan.execute_f32(z) == 0)
    assert torch.all(plan.execute(z) == 128)
    # all gains zero
    g0 = np.zeros((1, 2048, 2), dtype=np.float32)
    plan0 = bf.plan_create_ex(1, freq_mhz=[612.5], gains=g0, n_time=384)
    nb = synth.noise_bytes(3, 1, 384).cuda()
    assert torch.all(plan0.execute(nb) == 128)
    # saturation of the quantiser: every sample at +7+7i on every input -> huge zenith power -> 255
    s = torch.full((1, 384, 2048), 0xFF, dtype=torch.uint8, device="cuda")
    q = plan.execute(s)
    assert int(q.max()) == 255 and int(q.min()) == 128


@pytest.mark.parametrize("C,frames,NP,U", [(2, 2, 512, 128), (3, 5, 1024, 128), (9, 2, 1024, 256), (1, 1, 256, 128),
                                            (13, 3, 512, 128)])
def test_execute_host_matches_device(bf, C, frames, NP, U):
    """execute_host pipelines H2D / kernels / D2H over up to 8 chunks (channel groups, or frame ranges of each
    channel when there are fewer than 8 channels): the result must be the device path's, bit for bit."""
    T = frames * 3 * U
    plan = bf.plan_create_ex(C, zero_pad=NP, upchan_len=U, n_time=T, gains=synth.gains(5, C))
    b = synth.noise_bytes(11, C, T)
    ref = plan.execute(b.cuda()).cpu()
    out = plan.execute_host(b.pin_memory())
    assert torch.equal(ref, out.reshape(ref.shape))
    out2 = plan.execute_host(b.pin_memory())          # second call re-uses the staging buffers and events
    assert torch.equal(ref, out2.reshape(ref.shape))
    plan.destroy()


def test_cfg1_full_size_sampled(bf, orc):
    """BASELINE config 1 at full size, in the launch configuration bench.py times; the oracle checks a
    seeded sample of cells (cells are independent)."""
    cfg = synth.CONFIGS[1]
    C, T = cfg["n_coarse"], cfg["n_time"]
    seed = synth.config_seed(1)
    freqs = synth.config_freqs(1)
    gains = synth.gains(seed, C, flagged_frac=cfg["flagged"])
    d_in = synth.noise_bytes(seed, C, T, device="cuda")
    plan = bf.plan_create(C, gains=gains)          # north-star form: default freqs, n_time 49152
    rng = np.random.default_rng(seed)
    cells = [(0, 0), (C - 1, T // 384 - 1)] + [(int(rng.integers(C)), int(rng.integers(T // 384))) for _ in range(10)]

    def host_bytes(c, R):
        blk = d_in[c, 384 * R:384 * (R + 1)].cpu().numpy()
        # the generator is counter-based: the same block drawn on the CPU must be identical
        if R == 0:
            assert np.array_equal(blk, synth.noise_bytes(seed, 1, 384, chan0=c, time0=0, n_time_total=T).numpy()[0])
        return blk

    worst, frac = compare_cells(orc, plan, d_in, host_bytes, freqs, gains, cells, 512, 128)
    print(f"cfg1: worst rel err {worst:.2e}, u8 diff frac {frac:.2e}")


@pytest.mark.parametrize("NP,U", [(512, 128), (256, 128), (1024, 128), (512, 256)])
def test_repeated_executes_are_bit_identical(bf, NP, U):
    """The kernels hand tiles between warps through shared and tensor memory behind named barriers; a missing
    barrier would show as run-to-run differences.  30 executes of the same input (6 channels x 10 frames, so that
    several CTAs share every SM and the waves overlap) must give identical bytes and identical floats."""
    C, T = 6, 10 * 3 * U
    plan = bf.plan_create_ex(C, zero_pad=NP, upchan_len=U, n_time=T, gains=synth.gains(3, C))
    d_in = synth.noise_bytes(77, C, T, device="cuda")
    ref_u8 = plan.execute(d_in).clone()
    ref_f32 = plan.execute_f32(d_in).clone()
    for _ in range(30):
        assert torch.equal(plan.execute(d_in), ref_u8)
    for _ in range(5):
        assert torch.equal(plan.execute_f32(d_in), ref_f32)
    plan.destroy()


@pytest.mark.parametrize("NP", [256, 512, 1024])
def test_every_byte_value_including_minus_eight(bf, orc, NP):
    """The generators never emit nibble 0 (= -8, reading A1); the packed integer butterflies of the hot path must
    handle it all the same: bytes uniform over 0..255, plus all-0x00 and mixed 0x00 / 0xFF blocks."""
    C, U, frame = 2, 128, 384
    T = 2 * frame
    freqs = np.array([800.0, 523.4375])
    rng = np.random.default_rng(1702)
    hb = rng.integers(0, 256, size=(C, T, 2048), dtype=np.uint8)
    hb[1, frame:frame + 128] = 0x00
    hb[1, frame + 128:frame + 256, ::2] = 0x00
    hb[1, frame + 128:frame + 256, 1::2] = 0xFF
    gains = synth.gains(9, C, flagged_frac=0.0)
    plan = bf.plan_create_ex(C, freq_mhz=freqs, gains=gains, zero_pad=NP, n_time=T)
    b = torch.from_numpy(hb)
    # the intensities of full-range bytes are ~4 x those of the sigma 2.5 noise: still inside the uint8 range / 64
    cells = [(0, 0), (1, 1)]
    worst, frac = compare_cells(orc, plan, b.cuda(), lambda c, R: hb[c, frame * R:frame * (R + 1)], freqs, gains, cells, NP, U)
    print(f"NP={NP} all byte values: worst rel err {worst:.2e}, u8 diff frac {frac:.2e}")
    plan.destroy()


@pytest.mark.parametrize("NP,U", [(512, 128), (1024, 256)])
def test_accumulator_range_limit(bf, orc, NP, U):
    """Largest accumulators the tensor-core path can see: every input at -8 - 8i (nibble 0, |x| largest) for whole
    blocks, coherent over the feeds, unit gains, f = f_ref (beam 128 has the all-ones weight row).  The digit sums reach
    their bound K x 128 x 64 < 2^22 there, on which the integer recombination 256 a2 + a1 (31 bits) of the drain
    relies; the last block of each frame is noise so that every beam has a mean power to compare against."""
    frame = 3 * U
    T = 2 * frame
    freqs = np.array([600.0])
    hb = np.zeros((1, T, 2048), dtype=np.uint8)                      # 0x00 = -8 - 8i
    noise = synth.noise_bytes(77, 1, T).numpy()
    hb[0, frame - U:frame] = noise[0, :U]                            # frame 0: blocks 0, 1 coherent, block 2 noise
    hb[0, frame:frame + U] = 0xFF                                    # frame 1: +7 + 7i, then -8 - 8i, then noise
    hb[0, T - U:] = noise[0, U:2 * U]
    plan = bf.plan_create_ex(1, freq_mhz=freqs, zero_pad=NP, upchan_len=U, n_time=T)
    d_in = torch.from_numpy(hb).cuda()
    out_f32 = plan.execute_f32(d_in)
    torch.cuda.synchronize()
    worst = 0.0
    for R in range(2):
        I, _ = orc.cell(hb[0, frame * R:frame * (R + 1)], 600.0, gains=None, np_=NP, U=U)
        got = out_f32[0, R].cpu().numpy()
        mean = I.mean(axis=-1, keepdims=True)
        assert mean.min() > 0
        worst = max(worst, float((np.abs(got - I) / mean).max()))
    # the zenith beam holds the coherent power: (2 blocks x U samples) x |2048 x 8 sqrt2|^2 / (1024 U) spread over nothing
    assert float(out_f32[0, 0, :, 128].max()) > 1e5
    assert worst <= REL_TOL, f"float intensities off by {worst:.3e} of the beam mean power"
    print(f"NP={NP} U={U} accumulator range limit: worst rel err {worst:.2e}")
    plan.destroy()


@pytest.mark.parametrize("amp", [1e-4, 1.0, 1e3])
def test_gain_range(bf, orc, amp):
    """Gains far from unity (the weights are scaled per channel, so only the RATIO of gains inside a channel costs
    precision): the float intensities must stay within tolerance; the uint8 scale is chosen to keep the output in
    range."""
    C, frame = 1, 384
    freqs = np.array([650.0])
    gains = synth.gains(21, C, flagged_frac=0.02) * np.float32(amp)
    b = synth.noise_bytes(5, C, frame)
    plan = bf.plan_create_ex(C, freq_mhz=freqs, gains=gains, n_time=frame, scale=float(1.0 / (64.0 * amp * amp)), offset=128.0)
    out = plan.execute_f32(b.cuda()).cpu().numpy()
    I, _ = orc.cell(b.numpy()[0], 650.0, gains=gains[0])
    err = np.abs(out[0, 0] - I).max(axis=-1) / I.mean(axis=-1)
    assert err.max() <= REL_TOL, err.max()
    q = orc.quantize(I, scale=1.0 / (64.0 * amp * amp), offset=128.0)
    d = np.abs(plan.execute(b.cuda()).cpu().numpy()[0, 0].astype(int) - q.astype(int))
    assert d.max() <= 1 and (d != 0).mean() <= U8_FRAC
    plan.destroy()


def test_non_finite_gains_are_rejected(bf):
    g = np.ones((1, 2048, 2), dtype=np.float32)
    g[0, 17, 1] = np.inf
    with pytest.raises(bf.ChimeBfError):
        bf.plan_create_ex(1, gains=g, n_time=384)
    plan = bf.plan_create_ex(1, n_time=384)
    g[0, 17, 1] = np.nan
    with pytest.raises(bf.ChimeBfError):
        plan.update_gains(g)
    plan.destroy()
