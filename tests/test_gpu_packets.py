"""chime_bf_execute_packets (second half: the packetiser's per-packet scale / offset)
against oracle.packet_quantize applied to the oracle's intensities."""
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


@pytest.mark.parametrize("NP", [512, 1024])
def test_packets_match_oracle(bf, orc, NP):
    C, T = 2, 3 * 384
    freqs = np.array([744.140625, 466.40625])
    seed = synth.config_seed(4) + 11
    gains = synth.gains(seed, C, flagged_frac=0.05)
    b = synth.noise_bytes(seed, C, T)
    b, _ = synth.saturate_bursts(b, seed)
    plan = bf.plan_create_ex(C, freq_mhz=freqs, gains=gains, zero_pad=NP, n_time=T)
    u8, so = plan.execute_packets(b.cuda())
    u8, so = u8.cpu().numpy(), so.cpu().numpy()
    hb = b.numpy()
    n_diff = n_tot = 0
    for (c, R) in [(0, 0), (0, 2), (1, 1)]:
        I, _ = orc.cell(hb[c, 384 * R:384 * (R + 1)], float(freqs[c]), gains=gains[c], np_=NP)
        q, so_ref = orc.packet_quantize(I)
        assert np.allclose(so[c, R], so_ref, rtol=2e-5, atol=1e-3), np.abs(so[c, R] - so_ref).max()
        d = np.abs(u8[c, R].astype(int) - q.astype(int))
        assert d.max() <= 1
        n_diff += int((d != 0).sum())
        n_tot += d.size
    assert n_diff <= 1e-3 * n_tot, (n_diff, n_tot)
    # the bytes of a packet have mean 128 and 16 counts per sigma, whatever the gains
    P = u8.reshape(C, 3, 4, 8, 512).astype(float)
    assert np.abs(P.mean(axis=-1) - 128).max() < 0.6 and np.abs(P.std(axis=-1) - 16).max() < 0.6
    plan.destroy()


def test_packets_zero_input(bf):
    plan = bf.plan_create_ex(1, n_time=384)
    z = torch.full((1, 384, 2048), 0x88, dtype=torch.uint8, device="cuda")
    u8, so = plan.execute_packets(z)
    assert torch.all(u8 == 128) and torch.all(so[..., 0] == 1.0) and torch.all(so[..., 1] == 128.0)
    plan.destroy()


def test_packets_upchan_256(bf, orc):
    C, U = 1, 256
    T = 2 * 3 * U
    freqs = np.array([650.390625])
    seed = synth.config_seed(4) + 23
    gains = synth.gains(seed, C, flagged_frac=0.05)
    b = synth.noise_bytes(seed, C, T)
    plan = bf.plan_create_ex(C, freq_mhz=freqs, gains=gains, n_time=T, upchan_len=U)
    u8, so = plan.execute_packets(b.cuda())
    u8, so = u8.cpu().numpy(), so.cpu().numpy()
    I, _ = orc.cell(b.numpy()[0, 3 * U:6 * U], float(freqs[0]), gains=gains[0], U=U)
    q, so_ref = orc.packet_quantize(I)
    assert np.allclose(so[0, 1], so_ref, rtol=2e-5, atol=1e-3)
    d = np.abs(u8[0, 1].astype(int) - q.astype(int))
    assert d.max() <= 1 and (d != 0).mean() <= 1e-3
    plan.destroy()
