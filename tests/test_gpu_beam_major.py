"""Fused beam-major exchange (chime_bf_execute_beam_major) on ONE GPU: W ranks are emulated by W plans (each with
its own channel shard) that write into W receive buffers living on the same device -- this checks the epilogue's
addressing, which is all the kernel contributes; over NVLink the pointers are peer-mapped instead of local.
Expected values come from the ORACLE: seeded (global channel, frame) cells are beamformed and quantised on the CPU and
sliced by beam block (the all-to-all's definition); the per-rank dedispersion of a receive buffer is checked against
the oracle's dedispersion of that buffer's own bytes.  (That the receive buffers also equal one big plan's output,
sliced, is kept as an extra consistency check, not as the reference.)"""
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


@pytest.mark.parametrize("W,NP,U", [(4, 512, 128), (2, 1024, 128), (8, 256, 128), (4, 512, 256), (1, 512, 128)])
def test_beam_major_matches_oracle(bf, orc, W, NP, U):
    from paper_1702_04728_b200 import beam_major
    C_local, R = 2, 6
    C_total, T, frame = W * C_local, R * 3 * U, 3 * U
    seed = synth.config_seed(3) + W
    freqs = synth.chime_freqs_mhz(C_total, 37)
    gains = synth.gains(seed, C_total, flagged_frac=0.03)
    b = synth.noise_bytes(seed, C_total, T)
    d_in = b.cuda()
    recv = [torch.full(beam_major.receive_shape(C_total, R, W), 0xEE, dtype=torch.uint8, device="cuda") for _ in range(W)]
    for r in range(W):       # "rank" r beamforms its channel shard and scatters beams to all receive buffers
        sl = slice(r * C_local, (r + 1) * C_local)
        plan = bf.plan_create_ex(C_local, freq_mhz=freqs[sl], gains=gains[sl], zero_pad=NP, upchan_len=U, n_time=T)
        plan.execute_beam_major(d_in[sl].contiguous(), recv, chan_global0=r * C_local)
        torch.cuda.synchronize()
        plan.destroy()
    host = [x.cpu().numpy() for x in recv]
    # oracle: a seeded sample of (global channel, frame) cells, every rank's slice of each
    rng = np.random.default_rng(seed)
    cells = {(0, 0), (C_total - 1, R - 1)} | {(int(rng.integers(C_total)), int(rng.integers(R))) for _ in range(2)}
    n_diff = n_tot = 0
    hb = b.numpy()
    for (cg, Rf) in sorted(cells):
        I, _ = orc.cell(hb[cg, frame * Rf:frame * (Rf + 1)], float(freqs[cg]), gains=gains[cg], np_=NP, U=U)
        q = orc.quantize(I).reshape(1024, 16)
        for d in range(W):
            b0, nb = beam_major.beam_shard(W, d)
            diff = np.abs(host[d][cg, Rf].astype(int) - q[b0:b0 + nb].astype(int))
            assert diff.max() <= 1, f"rank {d} cell {(cg, Rf)}: {diff.max()} LSB"
            n_diff += int((diff != 0).sum())
            n_tot += diff.size
    assert n_diff <= 1e-3 * n_tot
    # nothing outside the cells' reach was left unwritten
    for d in range(W):
        assert (host[d] != 0xEE).mean() > 0.99
    # dedispersion of a beam shard, against the oracle on the receive buffer's own bytes
    dm = 0.5
    delays, _ = orc.dedisp_delays(freqs, dm, U=U)
    for d in (0, W - 1):
        got = bf.dedisperse_beams(recv[d], freqs, dm, upchan_len=U).cpu().numpy()
        want = orc.dedisperse(host[d], delays)
        assert np.array_equal(got.astype(np.int64), want)
    # extra: one plan over all channels, sliced by beam block, gives the same bytes
    full_plan = bf.plan_create_ex(C_total, freq_mhz=freqs, gains=gains, zero_pad=NP, upchan_len=U, n_time=T)
    ref = full_plan.execute(d_in).view(C_total, R, 1024, 16)
    for d in range(W):
        b0, nb = beam_major.beam_shard(W, d)
        assert torch.equal(recv[d], ref[:, :, b0:b0 + nb].contiguous()), f"receive buffer of rank {d}"
    full_plan.destroy()


def test_beam_major_argument_checks(bf):
    plan = bf.plan_create_ex(1, n_time=384)
    x = torch.zeros((1, 384, 2048), dtype=torch.uint8, device="cuda")
    buf = torch.zeros((1, 1, 1024, 16), dtype=torch.uint8, device="cuda")
    with pytest.raises(bf.ChimeBfError):
        plan.execute_beam_major(x, [buf] * 3, 0)            # 3 does not divide 1024
    with pytest.raises(bf.ChimeBfError):
        plan.execute_beam_major(x, [buf.data_ptr() + 8], 0)  # misaligned
    with pytest.raises(bf.ChimeBfError):
        bf.dedisperse_beams(torch.zeros((1, 4, 48, 16), dtype=torch.uint8, device="cuda"), [800.0], 0.0)  # 48 % 32
    plan.destroy()
