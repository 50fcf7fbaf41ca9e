"""Fused beam-major exchange (chime_bf_execute_beam_major) on ONE GPU: W ranks are emulated by W plans (each with
its own channel shard) that write into W receive buffers living on the same device -- this checks the epilogue's
addressing, which is all the kernel contributes; over NVLink the pointers are peer-mapped instead of local.
Reference: one plan over all channels (chime_bf_execute) sliced by beam block, i.e. the all-to-all's definition.
Then the per-rank dedispersion of a receive buffer against the slice of the full dedispersion."""
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
def test_beam_major_matches_sliced_reference(bf, W, NP, U):
    from paper_1702_04728_b200 import beam_major
    C_local, R = 2, 6
    C_total, T = W * C_local, R * 3 * U
    seed = synth.config_seed(3) + W
    freqs = synth.chime_freqs_mhz(C_total, 37)
    gains = synth.gains(seed, C_total, flagged_frac=0.03)
    d_in = synth.noise_bytes(seed, C_total, T, device="cuda")
    full_plan = bf.plan_create_ex(C_total, freq_mhz=freqs, gains=gains, zero_pad=NP, upchan_len=U, n_time=T)
    ref = full_plan.execute(d_in).view(C_total, R, 1024, 16)
    recv = [torch.full(beam_major.receive_shape(C_total, R, W), 0xEE, dtype=torch.uint8, device="cuda") for _ in range(W)]
    for r in range(W):       # "rank" r beamforms its channel shard and scatters beams to all receive buffers
        sl = slice(r * C_local, (r + 1) * C_local)
        plan = bf.plan_create_ex(C_local, freq_mhz=freqs[sl], gains=gains[sl], zero_pad=NP, upchan_len=U, n_time=T)
        plan.execute_beam_major(d_in[sl].contiguous(), recv, chan_global0=r * C_local)
        torch.cuda.synchronize()
        plan.destroy()
    for d in range(W):
        b0, nb = beam_major.beam_shard(W, d)
        assert torch.equal(recv[d], ref[:, :, b0:b0 + nb].contiguous()), f"receive buffer of rank {d}"
    # dedispersion of a beam shard = the shard of the dedispersion
    dm = 0.5
    want = full_plan.dedisperse(ref.view(full_plan.out_shape), dm)
    for d in (0, W - 1):
        b0, nb = beam_major.beam_shard(W, d)
        got = bf.dedisperse_beams(recv[d], freqs, dm, upchan_len=U)
        assert torch.equal(got, want[b0:b0 + nb])
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
