"""Pins of oracle.packet_quantize (the packetiser's per-packet scale / offset, reading F4).  The paper
prints no formula, so the CONVENTION (16 counts per sigma around 128, 32 beams per packet) is unpinned; what is pinned
is that the function does what the convention says: hand values, the invariances the definition implies and the
statistics of its output."""
import numpy as np

import oracle


def test_hand_values():
    # one packet of 2 beams x 2 fine channels: values 0, 2, 4, 6 -> mean 3, sigma sqrt(5)
    I = np.array([[[0.0, 2.0], [4.0, 6.0]]])
    q, so = oracle.packet_quantize(I, beams_per_packet=2)
    s = 16.0 / np.sqrt(5.0)
    assert np.allclose(so[0, 0], [s, 128.0 - 3.0 * s])
    want = np.rint(np.array([0.0, 2.0, 4.0, 6.0]) * s + 128.0 - 3.0 * s)      # 106.5 -> 106 (half to even), 121, 135, 149.5 -> 150
    assert list(q.ravel()) == [int(v) for v in want]


def test_constant_packet_and_zero():
    q, so = oracle.packet_quantize(np.zeros((4, 256, 16)))
    assert np.all(q == 128) and np.all(so[..., 0] == 1.0) and np.all(so[..., 1] == 128.0)
    q, so = oracle.packet_quantize(np.full((1, 32, 16), 777.0))
    assert np.all(q == 128) and so[0, 0, 0] == 1.0 and so[0, 0, 1] == 128.0 - 777.0


def test_scaling_the_intensities_leaves_the_bytes_unchanged():
    rng = np.random.default_rng(4)
    I = rng.exponential(500.0, size=(4, 256, 16))
    q1, so1 = oracle.packet_quantize(I)
    q2, so2 = oracle.packet_quantize(I * 7.25)
    assert np.array_equal(q1, q2)
    assert np.allclose(so2[..., 0] * 7.25, so1[..., 0]) and np.allclose(so2[..., 1], so1[..., 1])
    # an added constant moves only the offset
    q3, so3 = oracle.packet_quantize(I + 1000.0)
    assert np.array_equal(q1, q3) and np.allclose(so3[..., 0], so1[..., 0])


def test_output_statistics_and_reconstruction():
    rng = np.random.default_rng(5)
    I = rng.normal(600.0, 40.0, size=(4, 256, 16))
    q, so = oracle.packet_quantize(I)
    P = q.reshape(4, 8, 512).astype(float)
    assert np.abs(P.mean(axis=-1) - 128.0).max() < 0.1
    assert np.abs(P.std(axis=-1) - 16.0).max() < 0.1
    rec = (P - so[..., 1:2]) / so[..., 0:1]
    assert np.abs(rec - I.reshape(4, 8, 512)).max() <= 0.5 / so[..., 0].min() + 1e-9     # half a count
    assert (q == 0).mean() + (q == 255).mean() < 1e-3                                   # +-8 sigma range
