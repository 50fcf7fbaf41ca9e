"""Pins of the dedispersion oracle (oracle.dedisp_delays / oracle.dedisperse; reading F1)."""
import json
import os

import numpy as np

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "dispersion.json")))


def test_delay_closed_forms(orc):
    # DM 1 between 1 GHz and infinity = 4.148808 ms: one coarse "channel" whose fine channel 8 - 0.5 ... use n_fine=1
    d, mx = orc.dedisp_delays([1000.0], 1.0, U=128, fref_mhz=1e9, n_fine=1)
    assert d[0, 0] == int(np.floor(GOLD["dm1_at_1ghz_ms"] * 1e-3 / GOLD["frame_s_u128"] + 0.5)) == 4 == mx
    # DM 500, 800 -> 400 MHz: 9.72376875 s (hand arithmetic in the golden file) = 9891.53 frames of 0.98304 ms
    d, _ = orc.dedisp_delays([400.0], 500.0, U=128, fref_mhz=800.0, n_fine=1)
    assert d[0, 0] == int(np.floor(GOLD["dm500_400_to_800_mhz_s"] / GOLD["frame_s_u128"] + 0.5)) == 9892
    # U = 256 halves the frame count; DM 0 -> no delay; delay falls with frequency and is 0 at the reference
    d2, _ = orc.dedisp_delays([400.0], 500.0, U=256, fref_mhz=800.0, n_fine=1)
    assert d2[0, 0] == 4946
    f = 800.0 - 16 * 0.390625 * np.arange(64)
    d0, m0 = orc.dedisp_delays(f, 0.0)
    assert m0 == 0 and not d0.any()
    d, mx = orc.dedisp_delays(f, 40.0)
    flat = d.reshape(-1)                       # channel-major, fine ascending: frequency is NOT monotone in this order
    freq = (f[:, None] + (np.arange(16) - 7.5) * 0.390625 / 16).reshape(-1)
    order = np.argsort(-freq)
    assert np.all(np.diff(flat[order]) >= 0) and flat[order][0] == 0 and flat.max() == mx
    # within one coarse channel the highest fine channel (g = 15) arrives first (reading A9: g ascends in frequency)
    assert d[-1, 15] < d[-1, 0]


def test_dedisperse_brute_force_tiny(orc):
    rng = np.random.default_rng(7)
    C, R, B, G = 3, 12, 2, 4
    I = rng.integers(0, 256, size=(C, R, B, G), dtype=np.uint8)
    delays = rng.integers(0, 5, size=(C, G)).astype(np.int32)
    n_out = R - delays.max()
    want = np.zeros((B, n_out), dtype=np.int64)
    for b in range(B):
        for r in range(n_out):
            s = 0
            for c in range(C):
                for g in range(G):
                    s += int(I[c, r + delays[c, g], b, g])
            want[b, r] = s
    assert np.array_equal(orc.dedisperse(I, delays), want)
    # DM 0: plain band sum
    assert np.array_equal(orc.dedisperse(I, np.zeros((C, G), dtype=np.int32)), I.astype(np.int64).sum(axis=(0, 3)).T)


def test_impulse_on_the_track_collapses_to_one_sample(orc):
    f = 800.0 - 64 * 0.390625 * np.arange(8)
    delays, mx = orc.dedisp_delays(f, 12.0)
    R, r0, A = mx + 20, 7, 9
    I = np.zeros((8, R, 3, 16), dtype=np.uint8)
    for c in range(8):
        for g in range(16):
            I[c, r0 + delays[c, g], 1, g] = A
    D = orc.dedisperse(I, delays)
    assert D.shape == (3, 20) and D[1, r0] == 8 * 16 * A and D.sum() == 8 * 16 * A
    # a wrong DM smears it: no sample holds everything
    D2 = orc.dedisperse(I, orc.dedisp_delays(f, 6.0)[0])
    assert D2.max() < 8 * 16 * A
