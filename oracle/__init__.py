"""ctypes face of oracle/chime_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It imports nothing from paper_1702_04728_b200 and shares no code with it.
Each function cites the passage of PAPER.md it follows in chime_oracle.c.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "chime_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")

# Geometry / convention defaults (BASELINE.json configs; readings A2, A6, A11)
N_FEED, N_CYL, N_POL, N_EW, N_FINE, N_INT = 256, 4, 2, 4, 16, 3
FEED_SPACING_M, CYL_SPACING_M, F_REF_MHZ = 0.3048, 22.0, 600.0
EW_ANGLES_DEG = (-0.6, -0.2, 0.2, 0.6)
C0 = 299792458.0


def build(force=False):
    """Compile the oracle with gcc (plain C, OpenMP).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c99",
                               "-ffp-contract=off", "-o", _LIB, _SRC, "-lm"])
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.oracle_max_threads.restype = ctypes.c_int
    return _lib


def _p(a, t):
    return a.ctypes.data_as(ctypes.POINTER(t))


def max_threads():
    return int(lib().oracle_max_threads())


def ns_index(f_mhz, np_=512, n_feed=N_FEED, fref_mhz=F_REF_MHZ):
    J = np.zeros(n_feed, dtype=np.int32)
    lib().oracle_ns_index(ctypes.c_int(n_feed), ctypes.c_int(np_), ctypes.c_double(f_mhz),
                          ctypes.c_double(fref_mhz), _p(J, ctypes.c_int32))
    return J


def ns_index_sintheta(f_mhz, sin_theta, np_=512, n_feed=N_FEED, feed_spacing_m=FEED_SPACING_M):
    s = np.ascontiguousarray(sin_theta, dtype=np.float64)
    J = np.zeros(s.size, dtype=np.int32)
    lib().oracle_ns_index_sintheta(ctypes.c_int(n_feed), ctypes.c_int(np_), ctypes.c_double(f_mhz),
                                   ctypes.c_double(feed_spacing_m), _p(s, ctypes.c_double),
                                   ctypes.c_int(s.size), _p(J, ctypes.c_int32))
    return J


def unpack(b):
    b = np.ascontiguousarray(b, dtype=np.uint8).ravel()
    out = np.zeros((b.size, 2), dtype=np.int8)
    lib().oracle_unpack(_p(b, ctypes.c_uint8), ctypes.c_size_t(b.size), _p(out, ctypes.c_int8))
    return out


def ew_weights(f_mhz, ew_deg=EW_ANGLES_DEG, n_cyl=N_CYL, cyl_spacing_m=CYL_SPACING_M):
    ew = np.ascontiguousarray(ew_deg, dtype=np.float64)
    w = np.zeros((ew.size, n_cyl, 2), dtype=np.float64)
    lib().oracle_ew_weights(ctypes.c_int(n_cyl), ctypes.c_int(ew.size), ctypes.c_double(f_mhz),
                            ctypes.c_double(cyl_spacing_m), _p(ew, ctypes.c_double),
                            _p(w, ctypes.c_double))
    return w


def _c2d(a):
    """complex128 array -> contiguous float64 view with trailing (re, im)."""
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return a.view(np.float64).reshape(a.shape + (2,))


def beamform(x, g, J, w_ew, np_):
    """Steps 2-4.  x [n_t][n_pol][n_cyl][n_feed] complex, g [n_pol][n_cyl][n_feed] complex,
    w_ew [n_ew][n_cyl][2] -> Z [n_t][n_pol][n_ew][n_beam] complex."""
    n_t, n_pol, n_cyl, n_feed = x.shape
    J = np.ascontiguousarray(J, dtype=np.int32)
    n_ew = w_ew.shape[0]
    xd, gd = _c2d(x), _c2d(g)
    w = np.ascontiguousarray(w_ew, dtype=np.float64)
    Z = np.zeros((n_t, n_pol, n_ew, J.size, 2), dtype=np.float64)
    i = ctypes.c_int
    lib().oracle_beamform(_p(xd, ctypes.c_double), _p(gd, ctypes.c_double), i(n_t), i(n_pol),
                          i(n_cyl), i(n_feed), i(np_), _p(J, ctypes.c_int32), i(J.size), i(n_ew),
                          _p(w, ctypes.c_double), _p(Z, ctypes.c_double))
    return Z.view(np.complex128)[..., 0]


def ns_dft_allbins(v, np_):
    vd = _c2d(v)
    Y = np.zeros((np_, 2), dtype=np.float64)
    lib().oracle_ns_dft_allbins(_p(vd, ctypes.c_double), ctypes.c_int(v.size), ctypes.c_int(np_),
                                _p(Y, ctypes.c_double))
    return Y.view(np.complex128)[..., 0]


def upchan_detect(Z, U, n_int=N_INT, n_fine=N_FINE, norm=1.0, return_S=False):
    """Steps 5-6.  Z [n_int*U][n_pol][n_beams] complex -> I [n_beams][n_fine] (and S)."""
    n_t, n_pol, n_beams = Z.shape
    assert n_t == n_int * U
    zd = _c2d(Z)
    I = np.zeros((n_beams, n_fine), dtype=np.float64)
    S = np.zeros((n_int, U, n_pol, n_beams, 2), dtype=np.float64) if return_S else None
    i = ctypes.c_int
    lib().oracle_upchan_detect(_p(zd, ctypes.c_double), i(n_int), i(U), i(n_pol), i(n_beams),
                               i(n_fine), ctypes.c_double(norm), _p(I, ctypes.c_double),
                               _p(S, ctypes.c_double) if return_S else None)
    if return_S:
        return I, S.view(np.complex128)[..., 0]
    return I


def quantize(I, scale=1.0 / 64.0, offset=128.0):
    I = np.ascontiguousarray(I, dtype=np.float64)
    out = np.zeros(I.shape, dtype=np.uint8)
    lib().oracle_quantize(_p(I, ctypes.c_double), ctypes.c_size_t(I.size), ctypes.c_double(scale),
                          ctypes.c_double(offset), _p(out, ctypes.c_uint8))
    return out


def cell_from_voltage(x, g, J, w_ew, np_, U, n_int=N_INT, n_fine=N_FINE):
    """Steps 2-6 from complex voltages x [n_int*U][n_pol][n_cyl][n_feed].
    Returns I [n_ew][n_beam][n_fine] with norm 1/(n_feed n_cyl U)."""
    n_t, n_pol, n_cyl, n_feed = x.shape
    assert n_t == n_int * U
    J = np.ascontiguousarray(J, dtype=np.int32)
    w = np.ascontiguousarray(w_ew, dtype=np.float64)
    n_ew = w.shape[0]
    xd, gd = _c2d(x), _c2d(g)
    I = np.zeros((n_ew, J.size, n_fine), dtype=np.float64)
    i = ctypes.c_int
    lib().oracle_cell_from_voltage(_p(xd, ctypes.c_double), _p(gd, ctypes.c_double), i(n_pol),
                                   i(n_cyl), i(n_feed), i(np_), _p(J, ctypes.c_int32), i(J.size),
                                   i(n_ew), _p(w, ctypes.c_double), i(U), i(n_int), i(n_fine),
                                   _p(I, ctypes.c_double))
    return I


def cell_from_u8(in_u8, gains, J, w_ew, np_, U, n_pol=N_POL, n_cyl=N_CYL, n_feed=N_FEED,
                 n_int=N_INT, n_fine=N_FINE):
    """Steps 1-6 for one output cell.  in_u8 [n_int*U][n_pol*n_cyl*n_feed] uint8;
    gains [n_pol*n_cyl*n_feed][2] float32 or None (unit)."""
    b = np.ascontiguousarray(in_u8, dtype=np.uint8)
    assert b.shape == (n_int * U, n_pol * n_cyl * n_feed), b.shape
    J = np.ascontiguousarray(J, dtype=np.int32)
    w = np.ascontiguousarray(w_ew, dtype=np.float64)
    n_ew = w.shape[0]
    gp = None
    if gains is not None:
        gains = np.ascontiguousarray(gains, dtype=np.float32)
        assert gains.shape == (n_pol * n_cyl * n_feed, 2)
        gp = _p(gains, ctypes.c_float)
    I = np.zeros((n_ew, J.size, n_fine), dtype=np.float64)
    i = ctypes.c_int
    lib().oracle_cell_from_u8(_p(b, ctypes.c_uint8), gp, i(n_pol), i(n_cyl), i(n_feed), i(np_),
                              _p(J, ctypes.c_int32), i(J.size), i(n_ew), _p(w, ctypes.c_double),
                              i(U), i(n_int), i(n_fine), _p(I, ctypes.c_double))
    return I


def cell(in_u8_cell, f_mhz, gains=None, np_=512, U=128, ew_deg=EW_ANGLES_DEG, fref_mhz=F_REF_MHZ,
         cyl_spacing_m=CYL_SPACING_M):
    """Convenience for the CHIME geometry: one (channel, output frame) cell, steps 1-6.
    Returns (I [4][256][16] float64, J [256] int32)."""
    J = ns_index(f_mhz, np_, N_FEED, fref_mhz)
    w = ew_weights(f_mhz, ew_deg, N_CYL, cyl_spacing_m)
    return cell_from_u8(in_u8_cell, gains, J, w, np_, U), J


# ---- incoherent dedispersion to a nominal DM (the paper's proposed fourth kernel) --------------
# Reading F1.  The paper gives no formula; the cold-plasma delay is the textbook one
# (t = K_DM * DM * f^-2, K_DM = 4.148808 ms GHz^2 cm^3/pc) and is pinned against that constant, not the paper.
K_DM_MS_GHZ2 = 4.148808
SAMPLE_S = 2.56e-6          # PAPER.md:37 (Table 1)
COARSE_MHZ = 0.390625       # 400 MHz / 1024 channels


def dedisp_delays(freqs_mhz, dm, U=128, fref_mhz=None, n_fine=N_FINE, n_int=N_INT):
    """delay[c][g] in output frames (of n_int*U samples): fine channel g of coarse channel c sits at
    f_c + (g - (n_fine-1)/2) * COARSE_MHZ/n_fine (reading A9: g ascends in frequency); delay relative to fref
    (default: the highest fine-channel frequency), rounded half up.  Returns (int32 [C][n_fine], max delay)."""
    f = np.asarray(freqs_mhz, dtype=np.float64)[:, None] + \
        (np.arange(n_fine, dtype=np.float64)[None, :] - (n_fine - 1) / 2.0) * (COARSE_MHZ / n_fine)
    if fref_mhz is None or fref_mhz <= 0:
        fref_mhz = f.max()
    delay_s = K_DM_MS_GHZ2 * 1e-3 * dm * ((f / 1e3) ** -2 - (fref_mhz / 1e3) ** -2)
    frames = delay_s / (n_int * U * SAMPLE_S)
    d = np.floor(frames + 0.5).astype(np.int64)
    return d.astype(np.int32), int(d.max())


def dedisperse(I, delays):
    """D[b][r] = sum_c sum_g I[c][r + delays[c][g]][b][g], r = 0 .. R - max(delays) - 1.
    I: [C][R][n_beam][n_fine] (any integer or float dtype); exact in int64 for integer input."""
    I = np.asarray(I)
    C, R, B, G = I.shape
    delays = np.asarray(delays)
    assert delays.shape == (C, G) and delays.min() >= 0
    n_out = R - int(delays.max())
    assert n_out >= 1, "the sweep is longer than the buffer"
    acc_t = np.int64 if np.issubdtype(I.dtype, np.integer) else np.float64
    D = np.zeros((B, n_out), dtype=acc_t)
    for c in range(C):
        for g in range(G):
            d = int(delays[c, g])
            D += I[c, d:d + n_out, :, g].astype(acc_t).T
    return D


# ---- exact chromatic alignment (section 4: beam interpolation) -----------------------------------
def ns_turns(f_mhz, fref_mhz=F_REF_MHZ, sin_theta=None, n_feed=N_FEED, feed_spacing_m=FEED_SPACING_M):
    """Phase step per feed, in cycles, of the 256 desired pointings at frequency f: f d sin(theta_m) / c0.
    Native grid (reading A2): sin(theta_m) = (m - N/2) c0 / (N d f_ref), i.e. turns = (m - N/2) f / (N f_ref)."""
    if sin_theta is None:
        m = np.arange(n_feed, dtype=np.float64) - n_feed // 2
        return (m * float(f_mhz)) / (float(n_feed) * float(fref_mhz))
    s = np.ascontiguousarray(sin_theta, dtype=np.float64)
    return (float(f_mhz) * 1e6) * (feed_spacing_m / C0) * s


def beamform_exact(x, g, turns, w_ew):
    """Steps 2-4 with the N-S phase of the desired pointing itself (no nearest bin).  Shapes as `beamform`."""
    n_t, n_pol, n_cyl, n_feed = x.shape
    turns = np.ascontiguousarray(turns, dtype=np.float64)
    n_ew = w_ew.shape[0]
    xd, gd = _c2d(x), _c2d(g)
    w = np.ascontiguousarray(w_ew, dtype=np.float64)
    Z = np.zeros((n_t, n_pol, n_ew, turns.size, 2), dtype=np.float64)
    i = ctypes.c_int
    lib().oracle_beamform_exact(_p(xd, ctypes.c_double), _p(gd, ctypes.c_double), i(n_t), i(n_pol), i(n_cyl),
                                i(n_feed), _p(turns, ctypes.c_double), i(turns.size), i(n_ew),
                                _p(w, ctypes.c_double), _p(Z, ctypes.c_double))
    return Z.view(np.complex128)[..., 0]


def cell_exact(in_u8_cell, f_mhz, gains=None, U=128, ew_deg=EW_ANGLES_DEG, fref_mhz=F_REF_MHZ, sin_theta=None,
               cyl_spacing_m=CYL_SPACING_M):
    """One (channel, output frame) cell with exact pointing, steps 1-6.  Returns I [4][256][16] float64."""
    b = np.ascontiguousarray(in_u8_cell, dtype=np.uint8)
    assert b.shape == (N_INT * U, N_POL * N_CYL * N_FEED), b.shape
    turns = np.ascontiguousarray(ns_turns(f_mhz, fref_mhz, sin_theta), dtype=np.float64)
    w = np.ascontiguousarray(ew_weights(f_mhz, ew_deg, N_CYL, cyl_spacing_m), dtype=np.float64)
    gp = None
    if gains is not None:
        gains = np.ascontiguousarray(gains, dtype=np.float32)
        assert gains.shape == (N_POL * N_CYL * N_FEED, 2)
        gp = _p(gains, ctypes.c_float)
    I = np.zeros((N_EW, turns.size, N_FINE), dtype=np.float64)
    i = ctypes.c_int
    lib().oracle_cell_from_u8_exact(_p(b, ctypes.c_uint8), gp, i(N_POL), i(N_CYL), i(N_FEED),
                                    _p(turns, ctypes.c_double), i(turns.size), i(N_EW), _p(w, ctypes.c_double),
                                    i(U), i(N_INT), i(N_FINE), _p(I, ctypes.c_double))
    return I


# ---- the packetiser's per-packet rescale (reading F4 of DESIGN.md -- the paper gives no formula) ------
def packet_quantize(I, beams_per_packet=32):
    """I [n_ew][n_beam][n_fine] intensities of one (channel, frame).  A packet = `beams_per_packet` consecutive N-S
    beams x all fine channels of one E-W beam; scale = 16 / sigma (1 if sigma = 0), offset = 128 - mean * scale
    (population statistics of the packet), u8 = clamp(rne(I * scale + offset), 0, 255).
    Returns (u8 like I, scale_offset [n_ew][n_beam / beams_per_packet][2])."""
    I = np.asarray(I, dtype=np.float64)
    n_ew, n_beam, n_fine = I.shape
    n_p = n_beam // beams_per_packet
    P = I.reshape(n_ew, n_p, beams_per_packet * n_fine)
    mean = P.mean(axis=-1)
    sd = np.sqrt(((P - mean[..., None]) ** 2).mean(axis=-1))
    scale = np.where(sd > 0, 16.0 / np.where(sd > 0, sd, 1.0), 1.0)
    offset = 128.0 - mean * scale
    x = P * scale[..., None] + offset[..., None]
    q = np.clip(np.rint(x), 0, 255).astype(np.uint8)        # np.rint rounds half to even, like cvt.rni
    return q.reshape(I.shape), np.stack([scale, offset], axis=-1)
