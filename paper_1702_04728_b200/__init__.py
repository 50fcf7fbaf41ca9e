"""paper_1702_04728_b200 -- thin Python binding of libchime_bf.so (include/chime_bf.h).

Argument marshalling only: every step of the beamformer runs in the CUDA kernels of csrc/.
PyTorch is used for device memory and streams.  There is no CPU fallback: if the library or a
CUDA device is missing, calls raise.
"""
import ctypes
import os

import numpy as np

from .build import LIB_PATH, build_library

N_FEED, N_CYL, N_POL, N_INPUT, N_EW, N_BEAM, N_FINE, N_INT = 256, 4, 2, 2048, 4, 1024, 16, 3
EW_ANGLES_DEG = (-0.6, -0.2, 0.2, 0.6)

EXPORTS = [
    "chime_bf_plan_create", "chime_bf_plan_create_ex", "chime_bf_execute", "chime_bf_execute_f32",
    "chime_bf_execute_host", "chime_bf_get_ns_index", "chime_bf_debug_unpack", "chime_bf_n_frames",
    "chime_bf_in_bytes", "chime_bf_out_elems", "chime_bf_launches_per_execute", "chime_bf_destroy",
    "chime_bf_last_error", "chime_bf_update_gains", "chime_bf_update_ew_angles", "chime_bf_update_pointings",
    "chime_bf_dedisp_delays", "chime_bf_dedisperse", "chime_bf_execute_beam_major", "chime_bf_dedisperse_beams",
    "chime_bf_dedisp_delays_ex", "chime_bf_kernel_status", "chime_bf_measure_fp32_peak",
    "chime_bf_execute_packets", "chime_bf_dedisperse_stream_begin", "chime_bf_dedisperse_stream_push",
    "chime_bf_dedisperse_beams_noalloc",
]


class chime_bf_params(ctypes.Structure):
    _fields_ = [
        ("n_coarse", ctypes.c_int),
        ("freq_mhz", ctypes.POINTER(ctypes.c_double)),
        ("gains", ctypes.POINTER(ctypes.c_float)),
        ("ew_angles_deg", ctypes.POINTER(ctypes.c_double)),
        ("zero_pad", ctypes.c_int),
        ("upchan_len", ctypes.c_int),
        ("n_time", ctypes.c_int),
        ("f_ref_mhz", ctypes.c_double),
        ("ns_sin_theta", ctypes.POINTER(ctypes.c_double)),
        ("scale", ctypes.c_float),
        ("offset", ctypes.c_float),
        ("feed_spacing_m", ctypes.c_double),
        ("cyl_spacing_m", ctypes.c_double),
        ("exact_pointing", ctypes.c_int),
    ]


_lib = None


def load_library():
    """dlopen the in-tree C-ABI library (must have been built: __graft_entry__.build())."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                           "(there is no fallback path)")
    lib = ctypes.CDLL(LIB_PATH)
    vp, ci = ctypes.c_void_p, ctypes.c_int
    lib.chime_bf_plan_create.restype = vp
    lib.chime_bf_plan_create.argtypes = [ci, vp, vp, ci, ci]
    lib.chime_bf_plan_create_ex.restype = vp
    lib.chime_bf_plan_create_ex.argtypes = [ctypes.POINTER(chime_bf_params)]
    lib.chime_bf_execute.restype = ci
    lib.chime_bf_execute.argtypes = [vp, vp, vp, vp]
    lib.chime_bf_execute_f32.restype = ci
    lib.chime_bf_execute_f32.argtypes = [vp, vp, vp, vp]
    lib.chime_bf_dedisperse_stream_begin.restype = ci
    lib.chime_bf_dedisperse_stream_begin.argtypes = [vp, vp, ctypes.c_double, ctypes.c_double, ctypes.POINTER(ci)]
    lib.chime_bf_dedisperse_stream_push.restype = ci
    lib.chime_bf_dedisperse_stream_push.argtypes = [vp, vp, vp, vp, ctypes.POINTER(ctypes.c_longlong)]
    lib.chime_bf_execute_packets.restype = ci
    lib.chime_bf_execute_packets.argtypes = [vp, vp, vp, vp, vp]
    lib.chime_bf_execute_host.restype = ci
    lib.chime_bf_execute_host.argtypes = [vp, vp, vp, vp]
    lib.chime_bf_get_ns_index.restype = ci
    lib.chime_bf_get_ns_index.argtypes = [vp, vp]
    lib.chime_bf_debug_unpack.restype = ci
    lib.chime_bf_debug_unpack.argtypes = [vp, vp, vp, ctypes.c_size_t, vp]
    lib.chime_bf_update_gains.restype = ci
    lib.chime_bf_update_gains.argtypes = [vp, vp, vp]
    lib.chime_bf_update_ew_angles.restype = ci
    lib.chime_bf_update_ew_angles.argtypes = [vp, vp, vp]
    lib.chime_bf_update_pointings.restype = ci
    lib.chime_bf_update_pointings.argtypes = [vp, vp, ctypes.c_double, vp]
    lib.chime_bf_dedisp_delays.restype = ci
    lib.chime_bf_dedisp_delays.argtypes = [vp, ctypes.c_double, ctypes.c_double, vp, ctypes.POINTER(ci)]
    lib.chime_bf_dedisperse.restype = ci
    lib.chime_bf_dedisperse.argtypes = [vp, vp, vp, ctypes.c_double, ctypes.c_double, vp, ci]
    lib.chime_bf_execute_beam_major.restype = ci
    lib.chime_bf_execute_beam_major.argtypes = [vp, vp, vp, vp, ci, ci]
    lib.chime_bf_dedisp_delays_ex.restype = ci
    lib.chime_bf_dedisp_delays_ex.argtypes = [vp, ci, ci, ctypes.c_double, ctypes.c_double, vp, ctypes.POINTER(ci)]
    lib.chime_bf_dedisperse_beams.restype = ci
    lib.chime_bf_dedisperse_beams.argtypes = [vp, vp, ci, vp, ci, ci, ci, ctypes.c_double, ctypes.c_double, vp, vp, ci]
    lib.chime_bf_dedisperse_beams_noalloc.restype = ci
    lib.chime_bf_dedisperse_beams_noalloc.argtypes = [vp, vp, ci, vp, ci, ci, ci, ctypes.c_double, ctypes.c_double, vp, ci]
    lib.chime_bf_kernel_status.restype = ci
    lib.chime_bf_kernel_status.argtypes = [vp]
    lib.chime_bf_measure_fp32_peak.restype = ci
    lib.chime_bf_measure_fp32_peak.argtypes = [vp, ci, vp]
    lib.chime_bf_n_frames.restype = ci
    lib.chime_bf_n_frames.argtypes = [vp]
    lib.chime_bf_in_bytes.restype = ctypes.c_size_t
    lib.chime_bf_in_bytes.argtypes = [vp]
    lib.chime_bf_out_elems.restype = ctypes.c_size_t
    lib.chime_bf_out_elems.argtypes = [vp]
    lib.chime_bf_launches_per_execute.restype = ci
    lib.chime_bf_launches_per_execute.argtypes = [vp]
    lib.chime_bf_destroy.restype = None
    lib.chime_bf_destroy.argtypes = [vp]
    lib.chime_bf_last_error.restype = ctypes.c_char_p
    lib.chime_bf_last_error.argtypes = []
    _lib = lib
    return lib


def last_error():
    return load_library().chime_bf_last_error().decode()


class ChimeBfError(RuntimeError):
    pass


def _stream_ptr(stream):
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


class Plan:
    """Owns a chime_bf_plan*.  Methods carry the C-ABI names (chime_bf_ prefix dropped)."""

    def __init__(self, handle, n_coarse, zero_pad, upchan_len, n_time):
        self._h = handle
        self.n_coarse, self.zero_pad, self.upchan_len, self.n_time = n_coarse, zero_pad, upchan_len, n_time
        lib = load_library()
        self.n_frames = lib.chime_bf_n_frames(handle)
        self.in_bytes = lib.chime_bf_in_bytes(handle)
        self.out_elems = lib.chime_bf_out_elems(handle)
        self.launches_per_execute = lib.chime_bf_launches_per_execute(handle)
        self.in_shape = (n_coarse, n_time, N_INPUT)
        self.out_shape = (n_coarse, self.n_frames, N_EW, N_FEED, N_FINE)

    def _check(self, rc):
        if rc != 0:
            raise ChimeBfError(f"chime_bf error {rc}: {last_error()}")

    def _check_in(self, in_u8):
        import torch
        if not (in_u8.is_cuda and in_u8.dtype == torch.uint8 and in_u8.is_contiguous()
                and in_u8.numel() == self.in_bytes):
            raise ValueError(f"in_u8 must be a contiguous CUDA uint8 tensor of {self.in_bytes} bytes")

    def execute(self, in_u8, out_u8=None, stream=None):
        import torch
        self._check_in(in_u8)
        if out_u8 is None:
            out_u8 = torch.empty(self.out_shape, dtype=torch.uint8, device=in_u8.device)
        assert out_u8.is_cuda and out_u8.dtype == torch.uint8 and out_u8.numel() == self.out_elems
        self._check(load_library().chime_bf_execute(self._h, _stream_ptr(stream), in_u8.data_ptr(),
                                                    out_u8.data_ptr()))
        return out_u8

    def execute_f32(self, in_u8, out_f32=None, stream=None):
        import torch
        self._check_in(in_u8)
        if out_f32 is None:
            out_f32 = torch.empty(self.out_shape, dtype=torch.float32, device=in_u8.device)
        assert out_f32.is_cuda and out_f32.dtype == torch.float32 and out_f32.numel() == self.out_elems
        self._check(load_library().chime_bf_execute_f32(self._h, _stream_ptr(stream), in_u8.data_ptr(),
                                                        out_f32.data_ptr()))
        return out_f32

    def execute_packets(self, in_u8, out_u8=None, scale_offset=None, stream=None):
        """chime_bf_execute_packets -> (uint8 beams, float32 (scale, offset) per packet [C][R][4][8][2])."""
        import torch
        self._check_in(in_u8)
        if out_u8 is None:
            out_u8 = torch.empty(self.out_shape, dtype=torch.uint8, device=in_u8.device)
        if scale_offset is None:
            scale_offset = torch.empty((self.n_coarse, self.n_frames, N_EW, 8, 2), dtype=torch.float32, device=in_u8.device)
        assert scale_offset.is_cuda and scale_offset.dtype == torch.float32 and scale_offset.numel() == self.n_coarse * self.n_frames * 64
        self._check(load_library().chime_bf_execute_packets(self._h, _stream_ptr(stream), in_u8.data_ptr(),
                                                            out_u8.data_ptr(), scale_offset.data_ptr()))
        return out_u8, scale_offset

    def execute_host(self, in_u8_host, out_u8_host=None, stream=None):
        """HOST tensors (ideally pinned) in and out; H2D, kernels and D2H all inside the call."""
        import torch
        assert (not in_u8_host.is_cuda) and in_u8_host.dtype == torch.uint8 and in_u8_host.is_contiguous()
        assert in_u8_host.numel() == self.in_bytes
        if out_u8_host is None:
            out_u8_host = torch.empty(self.out_shape, dtype=torch.uint8).pin_memory()
        assert out_u8_host.numel() == self.out_elems and out_u8_host.is_contiguous()
        self._check(load_library().chime_bf_execute_host(self._h, _stream_ptr(stream),
                                                         in_u8_host.data_ptr(), out_u8_host.data_ptr()))
        return out_u8_host

    def update_gains(self, gains, stream=None):
        """chime_bf_update_gains: new per-input gains [n_coarse][2048][2] (None = unit), no plan rebuild."""
        g = None if gains is None else np.ascontiguousarray(gains, dtype=np.float32)
        if g is not None and g.size != self.n_coarse * N_INPUT * 2:
            raise ValueError("gains must have shape [n_coarse][2048][2]")
        self._check(load_library().chime_bf_update_gains(self._h, _stream_ptr(stream),
                                                         None if g is None else g.ctypes.data))

    def update_ew_angles(self, ew_angles_deg, stream=None):
        """chime_bf_update_ew_angles: re-point the 4 E-W beams (tracking beams)."""
        ew = np.ascontiguousarray(ew_angles_deg, dtype=np.float64)
        if ew.size != N_EW:
            raise ValueError("ew_angles must have 4 entries")
        self._check(load_library().chime_bf_update_ew_angles(self._h, _stream_ptr(stream), ew.ctypes.data))

    def update_pointings(self, f_ref_mhz=0.0, ns_sin_theta=None, stream=None):
        """chime_bf_update_pointings: re-tile the 256 N-S beams (tunable extent / density)."""
        s = None if ns_sin_theta is None else np.ascontiguousarray(ns_sin_theta, dtype=np.float64)
        if s is not None and s.size != N_FEED:
            raise ValueError("ns_sin_theta must have 256 entries")
        self._check(load_library().chime_bf_update_pointings(self._h, _stream_ptr(stream), float(f_ref_mhz),
                                                             None if s is None else s.ctypes.data))

    def execute_beam_major(self, in_u8, peer_ptrs, chan_global0, stream=None):
        """chime_bf_execute_beam_major: peer_ptrs = the W receive buffers (CUDA uint8 tensors of shape
        [C_total][n_frames][1024/W][16], or raw device pointers of peer-mapped buffers)."""
        self._check_in(in_u8)
        ptrs = [p if isinstance(p, int) else p.data_ptr() for p in peer_ptrs]
        arr = (ctypes.c_void_p * len(ptrs))(*ptrs)
        self._check(load_library().chime_bf_execute_beam_major(self._h, _stream_ptr(stream), in_u8.data_ptr(), arr,
                                                               len(ptrs), int(chan_global0)))

    def dedisp_delays(self, dm, f_ref_mhz=0.0):
        """chime_bf_dedisp_delays -> (delay [n_coarse][16] int32, n_out)."""
        tab = np.zeros((self.n_coarse, N_FINE), dtype=np.int32)
        n_out = ctypes.c_int(0)
        self._check(load_library().chime_bf_dedisp_delays(self._h, float(dm), float(f_ref_mhz), tab.ctypes.data,
                                                          ctypes.byref(n_out)))
        return tab, n_out.value

    def dedisperse(self, beams_u8, dm, f_ref_mhz=0.0, out_u32=None, stream=None):
        """chime_bf_dedisperse: uint8 beams [n_coarse][n_frames][4][256][16] -> uint32 [1024][n_out]."""
        import torch
        assert beams_u8.is_cuda and beams_u8.dtype == torch.uint8 and beams_u8.is_contiguous()
        assert beams_u8.numel() == self.out_elems
        _, n_out = self.dedisp_delays(dm, f_ref_mhz)
        if n_out < 1:
            raise ChimeBfError(f"dedisperse: the DM {dm} sweep is longer than the {self.n_frames}-frame buffer")
        if out_u32 is None:
            out_u32 = torch.empty((N_BEAM, n_out), dtype=torch.int32, device=beams_u8.device)
        assert out_u32.is_cuda and out_u32.dtype == torch.int32 and out_u32.numel() == N_BEAM * n_out
        self._check(load_library().chime_bf_dedisperse(self._h, _stream_ptr(stream), beams_u8.data_ptr(),
                                                       float(dm), float(f_ref_mhz), out_u32.data_ptr(), n_out))
        return out_u32

    def dedisperse_stream_begin(self, dm, f_ref_mhz=0.0, stream=None):
        """chime_bf_dedisperse_stream_begin -> largest delay in frames."""
        mx = ctypes.c_int(0)
        self._check(load_library().chime_bf_dedisperse_stream_begin(self._h, _stream_ptr(stream), float(dm),
                                                                    float(f_ref_mhz), ctypes.byref(mx)))
        return mx.value

    def dedisperse_stream_push(self, beams_u8, out_u32=None, stream=None):
        """chime_bf_dedisperse_stream_push -> (int32 [1024][n_frames], stream index of its first sample)."""
        import torch
        assert beams_u8.is_cuda and beams_u8.dtype == torch.uint8 and beams_u8.is_contiguous()
        assert beams_u8.numel() == self.out_elems
        if out_u32 is None:
            out_u32 = torch.empty((N_BEAM, self.n_frames), dtype=torch.int32, device=beams_u8.device)
        first = ctypes.c_longlong(0)
        self._check(load_library().chime_bf_dedisperse_stream_push(self._h, _stream_ptr(stream), beams_u8.data_ptr(),
                                                                   out_u32.data_ptr(), ctypes.byref(first)))
        return out_u32, first.value

    def get_ns_index(self):
        J = np.zeros((self.n_coarse, N_FEED), dtype=np.int32)
        self._check(load_library().chime_bf_get_ns_index(self._h, J.ctypes.data))
        return J

    def debug_unpack(self, in_u8, stream=None):
        import torch
        assert in_u8.is_cuda and in_u8.dtype == torch.uint8 and in_u8.is_contiguous()
        out = torch.empty((in_u8.numel(), 2), dtype=torch.int8, device=in_u8.device)
        self._check(load_library().chime_bf_debug_unpack(self._h, _stream_ptr(stream), in_u8.data_ptr(),
                                                         in_u8.numel(), out.data_ptr()))
        return out

    def kernel_status(self):
        """chime_bf_kernel_status: 0 unless a hand-over inside the tensor-core kernel timed out."""
        return load_library().chime_bf_kernel_status(self._h)

    def destroy(self):
        if self._h:
            load_library().chime_bf_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def dedisp_delays_ex(freq_mhz, dm, upchan_len=128, f_ref_mhz=0.0):
    """chime_bf_dedisp_delays_ex -> (delay table int32 [C][16], max delay in output frames)."""
    f = np.ascontiguousarray(freq_mhz, dtype=np.float64)
    tab = np.zeros((f.size, N_FINE), dtype=np.int32)
    mx = ctypes.c_int(0)
    rc = load_library().chime_bf_dedisp_delays_ex(f.ctypes.data, int(f.size), upchan_len, float(dm), float(f_ref_mhz),
                                                  tab.ctypes.data, ctypes.byref(mx))
    if rc != 0:
        raise ChimeBfError(f"chime_bf error {rc}: {last_error()}")
    return tab, mx.value


def dedisperse_beams(beams_u8, freq_mhz, dm, upchan_len=128, f_ref_mhz=0.0, stream=None):
    """chime_bf_dedisperse_beams: uint8 beams [C][R][n_beams][16] (any beam subset) -> int32 [n_beams][n_out].
    n_out = R - max delay comes from chime_bf_dedisp_delays_ex."""
    import torch
    assert beams_u8.is_cuda and beams_u8.dtype == torch.uint8 and beams_u8.is_contiguous() and beams_u8.dim() == 4
    C, R, nb, nf = beams_u8.shape
    assert nf == N_FINE
    f = np.ascontiguousarray(freq_mhz, dtype=np.float64)
    if f.size != C:
        raise ValueError("freq_mhz must have one entry per coarse channel")
    mx = ctypes.c_int(0)
    rc = load_library().chime_bf_dedisp_delays_ex(f.ctypes.data, C, upchan_len, float(dm), float(f_ref_mhz), None,
                                                  ctypes.byref(mx))
    if rc != 0:
        raise ChimeBfError(f"chime_bf error {rc}: {last_error()}")
    n_out = R - mx.value
    if n_out < 1:
        raise ChimeBfError(f"dedisperse_beams: the DM {dm} sweep is longer than the {R}-frame buffer")
    out = torch.empty((nb, n_out), dtype=torch.int32, device=beams_u8.device)
    scratch = torch.empty(C * 16, dtype=torch.int32, device=beams_u8.device)
    if stream is not None and not isinstance(stream, int):      # the kernel runs on `stream`: keep the caching allocator
        out.record_stream(stream)                               # from re-using these blocks before it has finished
        scratch.record_stream(stream)
    rc = load_library().chime_bf_dedisperse_beams(_stream_ptr(stream), beams_u8.data_ptr(), C, f.ctypes.data, R, nb,
                                                  upchan_len, float(dm), float(f_ref_mhz), scratch.data_ptr(),
                                                  out.data_ptr(), n_out)
    if rc != 0:
        raise ChimeBfError(f"chime_bf error {rc}: {last_error()}")
    return out


NOALLOC_MAX_COARSE = 1024


def dedisperse_beams_noalloc(beams_u8, freq_mhz, dm, out, upchan_len=128, f_ref_mhz=0.0, stream=None):
    """chime_bf_dedisperse_beams_noalloc: as dedisperse_beams, but nothing is allocated on the device -- the delay table
    lives in the library's built-in device array (at most NOALLOC_MAX_COARSE channels) and the CALLER passes `out`,
    int32 [n_beams][n_out] with n_out = R - max delay (dedisp_delays_ex).  Calls that overlap on the GPU race."""
    import torch
    assert beams_u8.is_cuda and beams_u8.dtype == torch.uint8 and beams_u8.is_contiguous() and beams_u8.dim() == 4
    C, R, nb, nf = beams_u8.shape
    assert nf == N_FINE
    assert out.is_cuda and out.dtype == torch.int32 and out.is_contiguous() and out.dim() == 2 and out.shape[0] == nb
    f = np.ascontiguousarray(freq_mhz, dtype=np.float64)
    if f.size != C:
        raise ValueError("freq_mhz must have one entry per coarse channel")
    rc = load_library().chime_bf_dedisperse_beams_noalloc(_stream_ptr(stream), beams_u8.data_ptr(), C, f.ctypes.data, R,
                                                          nb, upchan_len, float(dm), float(f_ref_mhz), out.data_ptr(),
                                                          int(out.shape[1]))
    if rc != 0:
        raise ChimeBfError(f"chime_bf error {rc}: {last_error()}")
    return out


def measure_fp32_peak(n_iter=2000, stream=None):
    """chime_bf_measure_fp32_peak -> (scalar FFMA, packed FFMA2) TFLOP/s of the current device."""
    out = (ctypes.c_double * 2)()
    rc = load_library().chime_bf_measure_fp32_peak(_stream_ptr(stream), int(n_iter), out)
    if rc != 0:
        raise ChimeBfError(f"chime_bf error {rc}: {last_error()}")
    return float(out[0]), float(out[1])


def plan_create(n_coarse, gains=None, ew_angles=EW_ANGLES_DEG, zero_pad=512, upchan_len=128):
    """chime_bf_plan_create: north-star form (f_k = 800 - k*0.390625 MHz, n_time = 49152)."""
    lib = load_library()
    g = None if gains is None else np.ascontiguousarray(gains, dtype=np.float32)
    if g is not None and g.size != n_coarse * N_INPUT * 2:
        raise ValueError("gains must have shape [n_coarse][2048][2]")
    ew = np.ascontiguousarray(ew_angles, dtype=np.float64)
    if ew.size != N_EW:
        raise ValueError("ew_angles must have 4 entries")
    h = lib.chime_bf_plan_create(n_coarse, None if g is None else g.ctypes.data, ew.ctypes.data,
                                 zero_pad, upchan_len)
    if not h:
        raise ChimeBfError(last_error())
    return Plan(h, n_coarse, zero_pad, upchan_len, 49152)


def plan_create_ex(n_coarse, freq_mhz=None, gains=None, ew_angles=EW_ANGLES_DEG, zero_pad=512,
                   upchan_len=128, n_time=49152, f_ref_mhz=0.0, ns_sin_theta=None, scale=0.0, offset=0.0,
                   feed_spacing_m=0.0, cyl_spacing_m=0.0, exact_pointing=False):
    """chime_bf_plan_create_ex: every knob of chime_bf_params (zeros select the defaults)."""
    lib = load_library()
    keep = []

    def dptr(a, n, ctype, npt):
        if a is None:
            return None
        a = np.ascontiguousarray(a, dtype=npt)
        if a.size != n:
            raise ValueError(f"expected {n} elements, got {a.size}")
        keep.append(a)
        return a.ctypes.data_as(ctypes.POINTER(ctype))

    p = chime_bf_params()
    p.n_coarse = n_coarse
    p.freq_mhz = dptr(freq_mhz, n_coarse, ctypes.c_double, np.float64)
    p.gains = dptr(gains, n_coarse * N_INPUT * 2, ctypes.c_float, np.float32)
    p.ew_angles_deg = dptr(ew_angles, N_EW, ctypes.c_double, np.float64)
    p.zero_pad, p.upchan_len, p.n_time = zero_pad, upchan_len, n_time
    p.f_ref_mhz = f_ref_mhz
    p.ns_sin_theta = dptr(ns_sin_theta, N_FEED, ctypes.c_double, np.float64)
    p.scale, p.offset = scale, offset
    p.feed_spacing_m, p.cyl_spacing_m = feed_spacing_m, cyl_spacing_m
    p.exact_pointing = 1 if exact_pointing else 0
    h = lib.chime_bf_plan_create_ex(ctypes.byref(p))
    if not h:
        raise ChimeBfError(last_error())
    return Plan(h, n_coarse, zero_pad, upchan_len, n_time)
