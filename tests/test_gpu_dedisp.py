"""GPU parity of the dedispersion kernel (chime_bf_dedisperse; reading F1): delay table and uint32
sums bit-exact against the oracle on seeded random uint8 beams, ragged tiles included; and the whole chain
baseband -> beams -> dedispersed series against the oracle chain on a small dispersed pulse."""
import numpy as np
import pytest
import torch

import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def bf():
    import __graft_entry__ as g
    g.build()
    import paper_1702_04728_b200 as bf
    return bf


@pytest.mark.parametrize("C,R,U,dm,step", [(5, 200, 128, 6.0, 100), (3, 77, 256, 9.0, 300), (64, 1017, 128, 40.0, 16),
                                            (2, 40, 128, 0.0, 1)])
def test_dedisperse_bit_exact(bf, orc, C, R, U, dm, step):
    freqs = synth.chime_freqs_mhz(C, step)
    plan = bf.plan_create_ex(C, freq_mhz=freqs, upchan_len=U, n_time=R * 3 * U)
    tab, n_out = plan.dedisp_delays(dm)
    want_tab, mx = orc.dedisp_delays(freqs, dm, U=U)
    assert np.array_equal(tab, want_tab) and n_out == R - mx and n_out >= 1
    g = torch.Generator(device="cuda").manual_seed(synth.BASE_SEED + C)
    beams = torch.randint(0, 256, (C, R, 4, 256, 16), dtype=torch.uint8, device="cuda", generator=g)
    got = plan.dedisperse(beams, dm).cpu().numpy()
    hb = beams.cpu().numpy().reshape(C, R, 1024, 16)
    if C * R > 2000:     # the full cfg2-sized array: oracle on a sample of beams (columns are independent)
        sel = np.random.default_rng(1).choice(1024, size=48, replace=False)
        sel[:2] = (0, 1023)
        want = orc.dedisperse(hb[:, :, sel, :], want_tab)
        assert np.array_equal(got[sel].astype(np.int64), want)
    else:
        assert np.array_equal(got.astype(np.int64), orc.dedisperse(hb, want_tab))
    if dm > 0:
        with pytest.raises(bf.ChimeBfError):
            plan.dedisp_delays(dm, f_ref_mhz=float(freqs.min()))  # reference below the band: negative delays
    plan.destroy()


def test_repeated_calls_reuse_the_uploaded_table_and_stay_exact(bf, orc):
    """A call leaves the delay-table upload out when the calling thread's previous call put the same table into the same
    library-owned array on the same stream.  Sequences that must all stay bit-exact against the oracle: the same DM twice
    (second upload left out), another DM (uploaded), the first one again; the no-alloc array the same way, with a call
    on ANOTHER stream and a call of another shape in between; a plan destroyed and re-created (possibly at the same address)."""
    C, R, U = 6, 120, 128
    freqs = synth.chime_freqs_mhz(C, 100)
    g = torch.Generator(device="cuda").manual_seed(synth.BASE_SEED + 99)
    beams = torch.randint(0, 256, (C, R, 4, 256, 16), dtype=torch.uint8, device="cuda", generator=g)
    hb = beams.cpu().numpy().reshape(C, R, 1024, 16)[:, :, ::37, :]        # 28 of the 1024 beams for the oracle
    want = {}
    for dm in (5.0, 8.0):
        tab, _ = orc.dedisp_delays(freqs, dm, U=U)
        want[dm] = orc.dedisperse(hb, tab)

    def check(out, dm):
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy()[::37].astype(np.int64), want[dm]), dm

    for rep in range(2):      # second round: a new plan, maybe at the freed plan's addresses
        plan = bf.plan_create_ex(C, freq_mhz=freqs, upchan_len=U, n_time=R * 3 * U)
        for dm in (5.0, 5.0, 8.0, 5.0, 5.0):
            check(plan.dedisperse(beams, dm), dm)
        plan.destroy()
    b4 = beams.reshape(C, R, 1024, 16)
    side = torch.cuda.Stream()
    for dm, stream in ((5.0, None), (5.0, None), (8.0, None), (8.0, side), (8.0, None), (5.0, side), (5.0, side)):
        _, mx = bf.dedisp_delays_ex(freqs, dm)
        out = torch.full((1024, R - mx), -7, dtype=torch.int32, device="cuda")
        torch.cuda.synchronize()
        bf.dedisperse_beams_noalloc(b4, freqs, dm, out, stream=stream)
        check(out, dm)
        if dm == 8.0 and stream is None:      # another shape through the same array in between
            small = torch.randint(0, 256, (3, 40, 32, 16), dtype=torch.uint8, device="cuda")
            o2 = torch.empty((32, 40), dtype=torch.int32, device="cuda")
            bf.dedisperse_beams_noalloc(small, synth.chime_freqs_mhz(3, 7), 0.0, o2)
            torch.cuda.synchronize()
            assert torch.equal(o2, small.to(torch.int32).sum(dim=(0, 3)).transpose(0, 1).contiguous())


def test_sweep_longer_than_buffer_is_an_error(bf):
    plan = bf.plan_create_ex(2, freq_mhz=[800.0, 400.390625], n_time=10 * 384)
    _, n_out = plan.dedisp_delays(500.0)
    assert n_out < 1
    with pytest.raises(bf.ChimeBfError):
        plan.dedisperse(torch.zeros((2, 10, 4, 256, 16), dtype=torch.uint8, device="cuda"), 500.0)


def test_chain_baseband_to_dedispersed_pulse(bf, orc):
    """8 channels 800 -> 625 MHz, 24 frames, a DM 3 pulse (S/N 20 per channel) from beam (E-W 1, N-S 100):
    oracle chain (all 192 cells -> uint8 -> dedisperse) vs CUDA chain (execute -> dedisperse)."""
    C, R, dm = 8, 24, 3.0
    T = R * 384
    seed = synth.config_seed(2) + 5
    freqs = synth.chime_freqs_mhz(C, 64)
    gains = synth.gains(seed, C, flagged_frac=0.02)
    m0, e0 = 100, 1
    s0 = (m0 - 128) * synth.C0 / (256 * 0.3048 * 600e6)
    b = synth.noise_bytes(seed, C, T)
    centres = synth.add_pulse(b, seed, freqs, gains=gains, sin_theta=s0, sin_phi=float(np.sin(np.deg2rad(-0.2))),
                              dm=dm, t0_samples=1000.0)
    assert centres.max() < T - 640
    hb = b.numpy()
    q = np.zeros((C, R, 1024, 16), dtype=np.uint8)
    for c in range(C):
        for r in range(R):
            I, _ = orc.cell(hb[c, 384 * r:384 * (r + 1)], float(freqs[c]), gains=gains[c])
            q[c, r] = orc.quantize(I).reshape(1024, 16)
    tab, _ = orc.dedisp_delays(freqs, dm)
    want = orc.dedisperse(q, tab)

    plan = bf.plan_create_ex(C, freq_mhz=freqs, gains=gains, n_time=T)
    beams = plan.execute(b.cuda())
    got = plan.dedisperse(beams, dm).cpu().numpy().astype(np.int64)
    assert got.shape == want.shape
    # the uint8 codes may differ by 1 LSB on <= 0.1 % of entries (A15): a sum of 128 codes moves by a few at most
    assert np.abs(got - want).max() <= 2 and (got != want).mean() < 0.05
    bpk, rpk = np.unravel_index(want.argmax(), want.shape)
    assert (bpk // 256, bpk % 256) == (e0, m0) and rpk == int(centres[0]) // 384
    assert np.unravel_index(got.argmax(), got.shape) == (bpk, rpk)
    # dedispersion is what makes it stand out: the plain band sum (DM 0) has a lower peak
    plain = orc.dedisperse(q, np.zeros_like(tab))
    assert want.max() > plain.max()
    plan.destroy()


@pytest.mark.parametrize("dm,R,U", [(60.0, 24, 128), (500.0, 40, 128), (3.0, 16, 256)])
def test_streaming_dedispersion_across_buffers(bf, orc, dm, R, U):
    """Sweeps longer than one buffer ("a high nominal DM"): the stream of K buffers pushed one at a time
    must give, sample for sample, the oracle's dedispersion of the concatenated stream.  DM 500 on this shortened band
    (8 channels from 800 to 400 MHz) sweeps 9892 frames = 247 buffers of 40 frames; 12 buffers are pushed for DM 60."""
    C = 8
    freqs = np.linspace(800.0, 400.390625, C)
    plan = bf.plan_create_ex(C, freq_mhz=freqs, upchan_len=U, n_time=R * 3 * U)
    D = plan.dedisperse_stream_begin(dm)
    delays, mx = orc.dedisp_delays(freqs, dm, U=U)
    assert D == mx
    K = int(np.ceil((D + 3 * R) / R)) + 1
    rng = np.random.default_rng(int(dm))
    # few beams carry data (the rest zero): the oracle's quadruple sum over 1024 beams x K R frames stays cheap
    stream = np.zeros((C, K * R, 1024, 16), dtype=np.uint8)
    bsel = [0, 5, 513, 1023]
    stream[:, :, bsel, :] = rng.integers(0, 256, size=(C, K * R, len(bsel), 16), dtype=np.uint8)
    want = orc.dedisperse(stream[:, :, bsel, :], delays)            # [4][K R - D]
    got = np.zeros((1024, K * R), dtype=np.int64)
    for k in range(K):
        out, first = plan.dedisperse_stream_push(torch.from_numpy(stream[:, k * R:(k + 1) * R].copy()).cuda())
        assert first == k * R - D
        o = out.cpu().numpy().astype(np.int64)
        for s in range(R):
            r = first + s
            if r >= 0:
                got[:, r] = o[:, s]
            else:
                assert not o[:, s].any()
    n = K * R - D - R       # samples completed by the pushes so far: r < K R - D, minus nothing; compare what both have
    n = min(want.shape[1], (K - 0) * R - D)
    assert n > R
    assert np.array_equal(got[bsel, :n], want[:, :n])
    assert not got[[1, 2, 700], :n].any()
    # a second stream on the same plan starts clean
    plan.dedisperse_stream_begin(dm / 2)
    out, first = plan.dedisperse_stream_push(torch.from_numpy(stream[:, :R].copy()).cuda())
    d2, mx2 = orc.dedisp_delays(freqs, dm / 2, U=U)
    assert first == -mx2
    plan.destroy()
