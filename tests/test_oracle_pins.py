"""Pins of the oracle to things other than itself (CPU only).

Each test fixes the oracle to something the paper or the mathematics determines: literal-cexp
brute force on tiny arrays (P1), numpy.fft special cases (P2), the closed-form Dirichlet response
to a tone (P3), Parseval (P4), linearity (P5), zero-in/zero-out (P6), single-input impulse (P7),
Table 1 arithmetic (P8), the alias geometry printed in PAPER.md section 3.3 (P9) and index-table
invariants (P10).  A plausible slip in the oracle (dropped term, wrong sign or index, transposed
operand) fails at least one of them.
"""
import json
import os

import numpy as np
import pytest

import synth

C0 = 299792458.0
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rng(seed):
    return np.random.default_rng(seed)


def _cplx(rng, shape):
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


# ---------------------------------------------------------------- P1 brute force, tiny arrays
def _brute_cell(x, g, J, NP, f_mhz, ew_deg, cyl_sp, U, n_int, n_fine):
    """Literal triple loops with cexp, written independently of the oracle's table indexing."""
    n_t, n_pol, n_cyl, n_feed = x.shape
    n_ew, n_beam = len(ew_deg), len(J)
    D = U // n_fine
    I = np.zeros((n_ew, n_beam, n_fine))
    for e in range(n_ew):
        s = np.sin(np.deg2rad(ew_deg[e]))
        for m in range(n_beam):
            for p in range(n_pol):
                z = np.zeros(n_t, dtype=complex)
                for t in range(n_t):
                    acc = 0j
                    for c in range(n_cyl):
                        wc = np.exp(-2j * np.pi * f_mhz * 1e6 * c * cyl_sp * s / C0)
                        for n in range(n_feed):
                            acc += wc * g[p, c, n] * x[t, p, c, n] * np.exp(-2j * np.pi * J[m] * n / NP)
                    z[t] = acc
                for r in range(n_int):
                    for q in range(U):
                        S = sum(z[U * r + u] * np.exp(-2j * np.pi * q * u / U) for u in range(U))
                        I[e, m, ((q + U // 2) % U) // D] += abs(S) ** 2
    return I / (n_feed * n_cyl * U)


@pytest.mark.parametrize("n_feed,n_cyl,P,U,n_fine", [(4, 2, 2, 4, 2), (8, 2, 2, 8, 4), (6, 3, 1, 4, 4)])
def test_p1_brute_force_tiny(orc, n_feed, n_cyl, P, U, n_fine):
    rng = _rng(1)
    NP, n_int, n_pol = n_feed * P, 3, 2
    f, fref = 733.0, 600.0
    ew = [-0.6, 0.3]
    x = _cplx(rng, (n_int * U, n_pol, n_cyl, n_feed))
    g = _cplx(rng, (n_pol, n_cyl, n_feed))
    J = orc.ns_index(f, NP, n_feed, fref)
    w = orc.ew_weights(f, ew, n_cyl, 22.0)
    got = orc.cell_from_voltage(x, g, J, w, NP, U, n_int, n_fine)
    want = _brute_cell(x, g, J, NP, f, ew, 22.0, U, n_int, n_fine)
    np.testing.assert_allclose(got, want, rtol=1e-11, atol=1e-11)


def test_p1_index_table_brute_force(orc):
    """eq. (1)+(2) evaluated with exact rationals (fractions) instead of floating point."""
    from fractions import Fraction
    for NP in (256, 512, 1024):
        P = NP // 256
        for k in (0, 1, 17, 512, 683, 1023):
            f = Fraction(800) - Fraction(k * 25, 64)
            J = orc.ns_index(float(f), NP)
            for m in range(256):
                x = Fraction(P * (m - 128)) * f / Fraction(600)
                j = (x + Fraction(1, 2)).__floor__()  # floor(t_m + dt_m), eq. (1) with its +0.5
                assert J[m] == j % NP, (NP, k, m)


# ---------------------------------------------------------------- P2 library special cases
def test_p2_numpy_fft(orc):
    rng = _rng(2)
    NP, U, n_int = 512, 128, 3
    f = 647.265625
    x = _cplx(rng, (4, 2, 4, 256))
    g = _cplx(rng, (2, 4, 256))
    J = orc.ns_index(f, NP)
    w = orc.ew_weights(f)
    Z = orc.beamform(x, g, J, w, NP)
    Y = np.fft.fft(g[None] * x, n=NP, axis=-1)[..., J]            # [t][p][cyl][m]
    wc = w[..., 0] + 1j * w[..., 1]
    want = np.einsum("ec,tpcm->tpem", wc, Y)
    np.testing.assert_allclose(Z, want, rtol=1e-10, atol=1e-9)
    # at f = f_ref the selection is the even bins: a plain fftshifted 256-point FFT
    Jr = orc.ns_index(600.0, NP)
    assert np.array_equal(Jr, (2 * (np.arange(256) - 128)) % NP)
    v = _cplx(rng, 256)
    np.testing.assert_allclose(orc.ns_dft_allbins(v, NP)[Jr], np.fft.fftshift(np.fft.fft(v)),
                               rtol=1e-10, atol=1e-9)
    # time transform against numpy.fft over U-blocks
    Zt = _cplx(rng, (n_int * U, 2, 5))
    I, S = orc.upchan_detect(Zt, U, n_int, 16, norm=1.0, return_S=True)
    Sw = np.fft.fft(Zt.reshape(n_int, U, 2, 5), axis=1)
    np.testing.assert_allclose(S, Sw, rtol=1e-10, atol=1e-9)
    P = (np.abs(np.fft.fftshift(Sw, axes=1)) ** 2).sum(axis=(0, 2))   # [U][beam], fftshifted
    want_I = P.reshape(16, 8, 5).sum(axis=1).T
    np.testing.assert_allclose(I, want_I, rtol=1e-10)


# ---------------------------------------------------------------- P3 closed form, tone
def test_p3_tone_closed_form(orc):
    f, NP, U, A = 600.0, 512, 128, 1.7
    s0, phi0, q0 = 0.2, np.sin(np.deg2rad(0.2)), 37
    d, xc = 0.3048, 22.0
    n = np.arange(256)
    cyl = np.arange(4)
    t = np.arange(3 * U)
    x = A * np.exp(2j * np.pi * (f * 1e6 / C0) * (d * n[None, None, None, :] * s0
                                                 + xc * cyl[None, None, :, None] * phi0)
                   + 2j * np.pi * q0 * t[:, None, None, None] / U) * np.ones((1, 2, 1, 1))
    g = np.ones((2, 4, 256), dtype=complex)
    J = orc.ns_index(f, NP)
    w = orc.ew_weights(f)
    I = orc.cell_from_voltage(x, g, J, w, NP, U)
    # closed form: Dirichlet kernels along N-S and E-W, all time power in bin q0
    delta = f * 1e6 * d * s0 / C0 - J / NP
    ns = np.abs(np.sin(np.pi * 256 * delta) / np.sin(np.pi * delta)) ** 2
    ew = np.array([abs(sum(np.exp(2j * np.pi * f * 1e6 * xc * c * (phi0 - np.sin(np.deg2rad(a))) / C0)
                           for c in range(4))) ** 2 for a in (-0.6, -0.2, 0.2, 0.6)])
    want = np.zeros((4, 256, 16))
    gq = ((q0 + 64) % 128) // 8
    want[:, :, gq] = 3 * 2 * A ** 2 * U ** 2 * ew[:, None] * ns[None, :] / (256 * 4 * U)
    np.testing.assert_allclose(I, want, rtol=1e-9, atol=1e-6 * want.max())
    e, m, gg = np.unravel_index(I.argmax(), I.shape)
    assert (e, m, gg) == (2, 159, 12)          # beam 159 = bin 62, E-W beam at +0.2 deg


def test_p3_cfg0_tone_peaks_in_predicted_beam(orc):
    """BASELINE.json config 0 through the packed 4-bit path: peak at N-S beam 159, fine channel of q0,
    E-W beams 1 and 2 tie in expectation (source at E-W offset 0) -- either may win (reading A15)."""
    b = synth.tone_bytes(synth.config_seed(0), 600.0, 768).numpy()[0]
    for R in range(2):
        I, J = orc.cell(b[384 * R:384 * (R + 1)], 600.0)
        e, m, g = np.unravel_index(I.argmax(), I.shape)
        assert m == 159 and g == 12 and e in (1, 2)
        assert 0.9 < I[1, 159, 12] / I[2, 159, 12] < 1.1
        assert I[e, m, g] > 100 * np.median(I)


# ---------------------------------------------------------------- P4 Parseval
def test_p4_parseval(orc):
    rng = _rng(4)
    v = _cplx(rng, 256)
    for NP in (256, 512, 1024):
        Y = orc.ns_dft_allbins(v, NP)
        assert np.isclose((np.abs(Y) ** 2).sum(), NP * (np.abs(v) ** 2).sum(), rtol=1e-12)
    U = 128
    Z = _cplx(rng, (3 * U, 2, 3))
    I, S = orc.upchan_detect(Z, U, 3, 16, norm=1.0, return_S=True)
    assert np.isclose((np.abs(S) ** 2).sum(), U * (np.abs(Z) ** 2).sum(), rtol=1e-12)
    assert np.isclose(I.sum(), U * (np.abs(Z) ** 2).sum(), rtol=1e-12)   # detection keeps every bin once


# ---------------------------------------------------------------- P5 linearity / scaling
def test_p5_linearity_and_gain_scaling(orc):
    rng = _rng(5)
    NP, f = 512, 701.5625
    J, w = orc.ns_index(f, NP), orc.ew_weights(f)
    x1, x2 = _cplx(rng, (3, 2, 4, 256)), _cplx(rng, (3, 2, 4, 256))
    g = _cplx(rng, (2, 4, 256))
    a, b = 0.7 - 0.2j, -1.3 + 0.5j
    lhs = orc.beamform(a * x1 + b * x2, g, J, w, NP)
    rhs = a * orc.beamform(x1, g, J, w, NP) + b * orc.beamform(x2, g, J, w, NP)
    np.testing.assert_allclose(lhs, rhs, rtol=1e-10, atol=1e-9)
    x = _cplx(rng, (384, 2, 4, 256))
    I1 = orc.cell_from_voltage(x, g, J, w, NP, 128)
    I2 = orc.cell_from_voltage(x, (2.0 * np.exp(0.9j)) * g, J, w, NP, 128)
    np.testing.assert_allclose(I2, 4.0 * I1, rtol=1e-10)


# ---------------------------------------------------------------- P6 zero in -> zero out
def test_p6_zero_in_zero_out(orc):
    b = np.full((384, 2048), 0x88, dtype=np.uint8)
    I, _ = orc.cell(b, 612.5)
    assert np.all(I == 0.0)
    assert np.all(orc.quantize(I) == 128)
    rb = synth.noise_bytes(7, 1, 384).numpy()[0]
    g0 = np.zeros((2048, 2), dtype=np.float32)
    I0, _ = orc.cell(rb, 612.5, gains=g0)
    assert np.all(I0 == 0.0)
    # zero gain on an input == that input's data replaced by 0x88
    g = np.zeros((2048, 2), dtype=np.float32)
    g[:, 0] = 1.0
    flagged = [3, 700, 1500, 2047]
    g[flagged] = 0.0
    rb2 = rb.copy()
    rb2[:, flagged] = 0x88
    Ia, _ = orc.cell(rb, 612.5, gains=g)
    Ib, _ = orc.cell(rb2, 612.5)
    np.testing.assert_allclose(Ia, Ib, rtol=1e-12)


def test_unpack_all_bytes(orc):
    b = np.arange(256, dtype=np.uint8)
    u = orc.unpack(b)
    assert np.array_equal(u[:, 0], (np.arange(256) // 16) - 8)
    assert np.array_equal(u[:, 1], (np.arange(256) % 16) - 8)
    assert tuple(orc.unpack(np.array([0x88, 0xF1, 0x1F], dtype=np.uint8)).ravel()) == (0, 0, 7, -7, -7, 7)


# ---------------------------------------------------------------- P7 single-input impulse
def test_p7_single_input_constant(orc):
    a = 5 - 3j
    gval = 0.9 + 0.4j
    x = np.zeros((384, 2, 4, 256), dtype=complex)
    x[:, 1, 2, 77] = a
    g = np.full((2, 4, 256), gval)
    f = 523.4375
    I = orc.cell_from_voltage(x, g, orc.ns_index(f), orc.ew_weights(f), 512, 128)
    want = 3 * 128 * abs(gval * a) ** 2 / (256 * 4)
    np.testing.assert_allclose(I[:, :, 8], want, rtol=1e-10)
    mask = np.ones(16, bool)
    mask[8] = False
    assert np.abs(I[:, :, mask]).max() < 1e-9 * want


# ---------------------------------------------------------------- P8 Table 1 arithmetic
def test_p8_table1_arithmetic():
    with open(os.path.join(GOLD, "table1.json")) as fh:
        t1 = json.load(fh)
    frame = 3 * 128
    assert abs(frame * t1["in_time_res_us"] * 1e-3 - t1["out_time_res_ms"]) < 5e-4      # 0.983 ms
    assert abs(t1["in_freq_res_khz"] / 16 - t1["out_freq_res_khz"]) < 0.5               # 24 kHz
    assert t1["out_channels"] == 16 * t1["in_channels"]
    in_bytes = frame * 2048                       # one coarse channel, one output frame
    out_bytes = 1024 * 16
    assert in_bytes == 48 * out_bytes
    in_tbps = 8 * 2048 * 1024 / (t1["in_time_res_us"] * 1e-6) / 1e12
    assert abs(in_tbps / 1.024 - t1["in_rate_tbps"]) < 1e-9                              # 6.4 Tbps
    out_gbps = 8 * 1024 * 16 * 1024 / 1.024e-3 / 1e9
    assert abs(out_gbps - t1["out_rate_gbps_text"]) < 1e-6                               # 131.072 Gbps


# ---------------------------------------------------------------- P9 alias geometry (section 3.3)
def test_p9_alias_geometry(orc):
    with open(os.path.join(GOLD, "alias_sec33.json")) as fh:
        gold = json.load(fh)
    d = 0.3048
    assert abs(C0 / (2 * d) / 1e6 - gold["alias_onset_mhz"]) < 5.0            # "~490 MHz"
    s0 = np.sin(np.deg2rad(gold["source_deg"]))                                  # ~26 deg
    # alias of the source: sin(theta_a) = s0 - c/(f d); paper: smeared over roughly -88..-50 deg
    hi = np.rad2deg(np.arcsin(s0 - C0 / (800e6 * d)))
    assert abs(hi - gold["alias_range_deg"][1]) < 3.0                           # ~ -50 (we get -52.3)
    f_edge = C0 / (d * (s0 + 1.0)) / 1e6                                         # alias reaches -90 deg
    lo = np.rad2deg(np.arcsin(max(-1.0, s0 - C0 / ((f_edge + 1.0) * 1e6 * d))))
    assert lo < gold["alias_range_deg"][0] + 3.0                                # ~ -88
    # the oracle's table + DFT put the main lobe and the alias where the geometry says (sign, wrap)
    n = np.arange(256)
    for f in (800.0, 790.625):
        v = np.exp(2j * np.pi * f * 1e6 * d * n * s0 / C0)
        J = orc.ns_index(f)
        pw = np.abs(orc.ns_dft_allbins(v, 512)[J]) ** 2
        sin_m = (np.arange(256) - 128) * C0 / (256 * d * 600e6)
        m_main = np.argmin(np.abs(sin_m - s0))
        m_alias = np.argmin(np.abs(sin_m - (s0 - C0 / (f * 1e6 * d))))
        top2 = sorted(np.argsort(pw)[-2:])
        # nearest-bin clamping points each beam to within half a padded bin of its target, so the
        # strongest beam is the predicted one or its neighbour
        assert abs(top2[1] - m_main) <= 1 and abs(top2[0] - m_alias) <= 1, (f, m_main, m_alias, top2)
        assert sin_m[m_alias] < -0.75
    # below the frequency where the alias leaves the beam grid there is a single strong beam
    f = 700.0
    v = np.exp(2j * np.pi * f * 1e6 * d * n * s0 / C0)
    pw = np.abs(orc.ns_dft_allbins(v, 512)[orc.ns_index(f)]) ** 2
    order = np.argsort(pw)
    assert abs(order[-1] - np.argmin(np.abs(sin_m - s0))) <= 1
    assert pw[order[-3]] < 0.1 * pw[order[-1]]


# ---------------------------------------------------------------- P10 index-table invariants
def test_p10_index_invariants(orc):
    freqs = synth.chime_freqs_mhz(1024)
    n_ties = 0
    for NP in (256, 512, 1024):
        P = NP // 256
        for f in freqs[::7]:
            J = orc.ns_index(f, NP)
            assert J[128] == 0
            assert J.min() >= 0 and J.max() < NP
            x = P * (np.arange(256) - 128) * f / 600.0
            # nearest bin: |x - unwrapped j| <= 1/2
            ju = np.floor(x + 0.5)
            assert np.array_equal(J, ju.astype(np.int64) % NP)
            assert np.all(np.diff(ju) >= 0)                        # monotone before wrapping
            tie = np.isclose(x - np.floor(x), 0.5, atol=1e-12)
            m = np.arange(1, 256)
            anti = (NP - J[256 - m]) % NP == J[m]
            assert np.all(anti | tie[m] | tie[256 - m])            # antisymmetric except exact ties
            n_ties += int(tie.sum()) if NP == 512 else 0
    assert n_ties > 0
    # duplicates appear only through aliasing wrap at P = 2
    for f in (400.390625, 600.0):
        assert len(set(orc.ns_index(f, 512))) == 256
    assert len(set(orc.ns_index(800.0, 512))) == 256 - 64


def test_p10_tie_count_full_band(orc):
    """2126 exact .5 ties over the 1024x256 table at P = 2, f_ref = 600 MHz; all rounded up."""
    from fractions import Fraction
    ties = 0
    for k in range(1024):
        f = Fraction(800) - Fraction(k * 25, 64)
        J = None
        for m in range(256):
            x = Fraction(2 * (m - 128)) * f / 600
            if x - x.__floor__() == Fraction(1, 2):
                ties += 1
                if J is None:
                    J = orc.ns_index(float(f), 512)
                assert J[m] == (x.__floor__() + 1) % 512
    assert ties == 2126


def test_explicit_sintheta_grid_matches_default(orc):
    f = 655.859375
    s = (np.arange(256) - 128) * C0 / (256 * 0.3048 * 600e6)
    Ja, Jb = orc.ns_index(f), orc.ns_index_sintheta(f, s)
    x = 2 * (np.arange(256) - 128) * f / 600.0
    near_tie = np.abs((x - np.floor(x)) - 0.5) < 1e-9
    assert np.array_equal(Ja[~near_tie], Jb[~near_tie])


def test_quantize_rne_and_saturation(orc):
    I = np.array([0.0, 32.0, 96.0, 160.0, 64.0 * 127.0, 1e9, -1e9, 64.0 * 0.49, 64 * 0.51])
    q = orc.quantize(I, 1.0 / 64.0, 128.0)
    assert list(q) == [128, 128, 130, 130, 255, 255, 0, 128, 129]   # 128.5->128, 129.5->130, 130.5->130


def test_p14_frequency_summed_beam_width_sec31(orc):
    """P14 -- PAPER.md:80: the frequency-summed formed beam is ~0.5 deg wide (FWHM) at zenith and ~2.8 deg at 10 deg
    elevation.  Oracle N-S beamformer (direct sums, nearest-bin clamping at every frequency) on plane waves swept in
    angle, summed over 64 frequencies of the band; see tests/golden/beam_fwhm_sec31.json for the reading."""
    import json
    import os
    gold = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "beam_fwhm_sec31.json")))
    d, c0 = 0.3048, 299792458.0
    freqs = 800.0 - 0.390625 * np.arange(0, 1024, 16)
    n = np.arange(256)

    def widths(s0, span_deg, npts=321):
        th = np.arcsin(s0) + np.deg2rad(np.linspace(-span_deg, span_deg, npts))
        power = np.zeros(npts)
        for f in freqs:
            J = orc.ns_index_sintheta(f, [s0], 512)
            x = np.exp(2j * np.pi * f * 1e6 * d * np.outer(np.sin(th), n) / c0).reshape(npts, 1, 1, 256)
            w = np.zeros((1, 1, 2))
            w[0, 0, 0] = 1.0
            Z = orc.beamform(x, np.ones((1, 1, 256), dtype=complex), J, w, 512)
            power += np.abs(Z[:, 0, 0, 0]) ** 2
        out = []
        for patt in (power / power.max(), np.sqrt(power / power.max())):     # power and voltage pattern
            above = np.where(patt >= 0.5)[0]
            out.append(float(np.rad2deg(th[above[-1]] - th[above[0]])))
        return out

    p_zen, v_zen = widths(0.0, 1.0)
    p_low, v_low = widths(np.sin(np.deg2rad(80.0)), 8.0)
    ratio = gold["fwhm_10deg_elevation_deg"] / gold["fwhm_zenith_deg"]
    assert abs(p_low / p_zen - ratio) < 0.15 * ratio and abs(v_low / v_zen - ratio) < 0.15 * ratio
    assert abs(v_zen - gold["fwhm_zenith_deg"]) < 0.2 * gold["fwhm_zenith_deg"]
    assert abs(v_low - gold["fwhm_10deg_elevation_deg"]) < 0.2 * gold["fwhm_10deg_elevation_deg"]
    assert 0.28 < p_zen < 0.36          # 0.886 lambda / D at the band's power-weighted mean wavelength


# ---- exact chromatic alignment: oracle.beamform_exact / cell_exact ---------------------------------
def test_exact_pointing_brute_force_tiny():
    """P15a: literal cexp triple loop on a tiny array (3 samples, 1 pol, 2 cylinders, 5 feeds, 4 pointings)."""
    import cmath
    import oracle
    rng = np.random.default_rng(31)
    x = rng.normal(size=(3, 1, 2, 5)) + 1j * rng.normal(size=(3, 1, 2, 5))
    g = rng.normal(size=(1, 2, 5)) + 1j * rng.normal(size=(1, 2, 5))
    turns = np.array([-0.31, 0.0, 0.123456, 0.49])
    w = rng.normal(size=(2, 2)) + 1j * rng.normal(size=(2, 2))
    Z = oracle.beamform_exact(x, g, turns, np.stack([w.real, w.imag], axis=-1))
    for t in range(3):
        for e in range(2):
            for m in range(4):
                acc = 0
                for c in range(2):
                    y = sum(g[0, c, n] * x[t, 0, c, n] * cmath.exp(-2j * cmath.pi * n * turns[m]) for n in range(5))
                    acc += w[e, c] * y
                assert abs(Z[t, 0, e, m] - acc) < 1e-12


def test_exact_pointing_equals_nearest_bin_where_the_bin_is_exact():
    """P15b: at f = f_ref the desired pointings ARE bins of the padded transform (J = P (m - 128)), so the exact
    and the nearest-bin beamformers are the same sums."""
    import oracle
    rng = np.random.default_rng(32)
    x = rng.normal(size=(2, 2, 4, 256)) + 1j * rng.normal(size=(2, 2, 4, 256))
    g = np.ones((2, 4, 256), dtype=complex)
    w = oracle.ew_weights(600.0)
    J = oracle.ns_index(600.0, 512)
    Za = oracle.beamform(x, g, J, w, 512)
    Zb = oracle.beamform_exact(x, g, oracle.ns_turns(600.0), w)
    assert np.abs(Za - Zb).max() < 1e-9 * np.abs(Za).max()


def test_exact_pointing_full_gain_on_target_and_convergence_with_padding():
    """P15c: a plane wave from the desired pointing of beam m is received with the full gain N A by the exact
    beamformer (Dirichlet kernel at zero offset) at ANY frequency; the nearest-bin beamformer loses
    |sin(pi N d)/(N sin(pi d))| with d = turns - J/NP, and converges to the exact one as the padding factor grows
    (the padding trades cost against beam sensitivity)."""
    import oracle
    f, m = 437.5, 201
    turns = oracle.ns_turns(f)
    n = np.arange(256)
    x = np.zeros((1, 1, 1, 256), dtype=complex)
    x[0, 0, 0] = 2.5 * np.exp(2j * np.pi * n * turns[m])
    g = np.ones((1, 1, 256), dtype=complex)
    w = np.array([[[1.0, 0.0]]])
    Ze = oracle.beamform_exact(x, g, turns, w)[0, 0, 0]
    assert abs(abs(Ze[m]) - 256 * 2.5) < 1e-9
    assert np.argmax(np.abs(Ze)) == m
    prev = None
    for P in (1, 2, 4, 8, 32):
        J = oracle.ns_index(f, 256 * P)
        Zn = oracle.beamform(x, g, J, w, 256 * P)[0, 0, 0]
        d = turns[m] - J[m] / (256.0 * P)
        d -= np.rint(d)
        closed = 256 * 2.5 if d == 0 else 2.5 * abs(np.sin(np.pi * 256 * d) / np.sin(np.pi * d))
        assert abs(abs(Zn[m]) - closed) < 1e-8
        loss = 1.0 - abs(Zn[m]) / (256 * 2.5)
        assert loss >= -1e-12
        if prev is not None and P >= 4:
            assert loss <= prev + 1e-12
        prev = loss
    assert prev < 2e-3          # P = 32: the nearest bin is within 1/64 of a native beam spacing


def test_cell_exact_matches_cell_at_fref():
    """P15d: the packed-baseband entry point with exact pointing reduces to oracle.cell at f = f_ref."""
    import oracle
    import synth
    b = synth.noise_bytes(3, 1, 384).numpy()[0]
    Ia, _ = oracle.cell(b, 600.0)
    Ib = oracle.cell_exact(b, 600.0)
    assert np.abs(Ia - Ib).max() < 1e-9 * Ia.max()
