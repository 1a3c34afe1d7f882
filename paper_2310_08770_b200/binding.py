"""Thin ctypes binding of the C-ABI library (include/cc.h): argument
marshalling only -- every step of the path runs in the CUDA kernels of
``libcc_b200.so``.  PyTorch is used for device memory and streams.

There is no CPU fallback: if the extension is missing or the device is not a
compute-capability-10.x GPU, calls raise.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# CC_B200_LIB selects another build of the same library (the schedule-fuzzing build libcc_b200_fuzz.so of build.py --fuzz)
LIB_PATH = os.environ.get("CC_B200_LIB") or os.path.join(_HERE, "libcc_b200.so")

CC_U8, CC_U16 = 0, 1
_STATUS = {0: "CC_OK", 1: "CC_ERR_INVALID_ARG", 2: "CC_ERR_UNSUPPORTED", 3: "CC_ERR_NOMEM",
           4: "CC_ERR_CUDA", 5: "CC_ERR_ARCH"}

EXPORTS = ["cc_plan_create", "cc_plan_create_weighted", "cc_track", "cc_track_static", "cc_track_debug", "cc_track_profile", "cc_track_host",
           "cc_plan_set_host_chunk", "cc_plan_destroy",
           "cc_plan_info", "cc_plan_enable_reference_update", "cc_plan_get_reference_spectrum", "cc_plan_get_reference_spectrum_f64", "cc_track_accumulate",
           "cc_plan_update_reference_from_accumulator", "cc_drift_correct", "cc_fp32_peak_probe", "cc_fp32_tile_probe", "cc_tc_gemm_probe", "cc_track_latency_probe",
           "cc_rt_open", "cc_rt_submit", "cc_rt_wait", "cc_rt_track", "cc_rt_close", "cc_rt_latency_probe", "cc_status_string", "cc_last_error"]


class CcError(RuntimeError):
    def __init__(self, status: int, detail: str):
        super().__init__("%s: %s" % (_STATUS.get(status, str(status)), detail))
        self.status = status


class PlanInfo(ctypes.Structure):
    _fields_ = [("H", ctypes.c_int), ("W", ctypes.c_int), ("upsample", ctypes.c_int), ("dtype", ctypes.c_int),
                ("grid_M", ctypes.c_int), ("cluster_size", ctypes.c_int), ("threads", ctypes.c_int),
                ("smem_bytes", ctypes.c_int), ("max_clusters", ctypes.c_int),
                ("lat_cluster_size", ctypes.c_int), ("lat_max_clusters", ctypes.c_int),
                ("scratch_bytes", ctypes.c_longlong), ("table_bytes", ctypes.c_longlong),
                ("super_blocks", ctypes.c_int), ("offsets_per_cta", ctypes.c_int),
                ("tensor_core_stage1", ctypes.c_int)]


_lib = None


def load_library() -> ctypes.CDLL:
    """dlopen libcc_b200.so (built in-tree by ``python -m paper_2310_08770_b200.build``)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("CUDA extension %s is missing: run `python -m paper_2310_08770_b200.build` "
                              "(there is no CPU fallback)" % LIB_PATH)
        lib = ctypes.CDLL(LIB_PATH)
        vp, ci = ctypes.c_void_p, ctypes.c_int
        lib.cc_plan_create.argtypes = [ctypes.POINTER(vp), ci, ci, ci, ci, vp]
        lib.cc_plan_create.restype = ci
        lib.cc_plan_create_weighted.argtypes = [ctypes.POINTER(vp), ci, ci, ci, ci, vp, ci, ctypes.c_float]
        lib.cc_plan_create_weighted.restype = ci
        lib.cc_track.argtypes = [vp, vp, ci, vp, vp, vp, vp]
        lib.cc_track.restype = ci
        lib.cc_track_static.argtypes = [vp, vp, ci, vp, vp, vp, vp]
        lib.cc_track_static.restype = ci
        lib.cc_track_debug.argtypes = [vp, vp, ci, vp, vp, vp, vp, vp, vp]
        lib.cc_track_debug.restype = ci
        lib.cc_track_profile.argtypes = [vp, vp, ci, vp, vp, vp, vp, vp]
        lib.cc_track_profile.restype = ci
        lib.cc_track_host.argtypes = [vp, vp, ci, vp, vp, vp]
        lib.cc_track_host.restype = ci
        lib.cc_plan_set_host_chunk.argtypes = [vp, ci]
        lib.cc_plan_set_host_chunk.restype = ci
        lib.cc_track_latency_probe.argtypes = [vp, vp, ci, vp, vp, vp, vp, vp]
        lib.cc_track_latency_probe.restype = ci
        lib.cc_rt_open.argtypes = [vp, ci, ctypes.POINTER(vp)]
        lib.cc_rt_open.restype = ci
        lib.cc_rt_submit.argtypes = [vp, vp]
        lib.cc_rt_submit.restype = ci
        fp = ctypes.POINTER(ctypes.c_float)
        lib.cc_rt_wait.argtypes = [vp, fp, fp, fp]
        lib.cc_rt_wait.restype = ci
        lib.cc_rt_track.argtypes = [vp, vp, fp, fp, fp]
        lib.cc_rt_track.restype = ci
        lib.cc_rt_close.argtypes = [vp]
        lib.cc_rt_close.restype = ci
        lib.cc_rt_latency_probe.argtypes = [vp, vp, ci, vp, vp, vp, vp]
        lib.cc_rt_latency_probe.restype = ci
        lib.cc_plan_enable_reference_update.argtypes = [vp, ctypes.c_double]
        lib.cc_plan_enable_reference_update.restype = ci
        lib.cc_plan_get_reference_spectrum.argtypes = [vp, vp]
        lib.cc_plan_get_reference_spectrum.restype = ci
        lib.cc_plan_get_reference_spectrum_f64.argtypes = [vp, vp]
        lib.cc_plan_get_reference_spectrum_f64.restype = ci
        lib.cc_track_accumulate.argtypes = [vp, vp, ci, vp, vp, vp, vp]
        lib.cc_track_accumulate.restype = ci
        lib.cc_plan_update_reference_from_accumulator.argtypes = [vp, vp]
        lib.cc_plan_update_reference_from_accumulator.restype = ci
        lib.cc_plan_destroy.argtypes = [vp]
        lib.cc_plan_destroy.restype = ci
        lib.cc_plan_info.argtypes = [vp, ctypes.POINTER(PlanInfo)]
        lib.cc_plan_info.restype = ci
        lib.cc_fp32_peak_probe.argtypes = [ctypes.POINTER(ctypes.c_double), vp]
        lib.cc_fp32_peak_probe.restype = ci
        lib.cc_drift_correct.argtypes = [vp, vp, ci, ctypes.c_double, ctypes.c_double, vp, vp, vp, vp]
        lib.cc_drift_correct.restype = ci
        lib.cc_fp32_tile_probe.argtypes = [ctypes.POINTER(ctypes.c_double), vp]
        lib.cc_fp32_tile_probe.restype = ci
        lib.cc_tc_gemm_probe.argtypes = [vp, vp, ci, ci, ci, ci, vp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
        lib.cc_tc_gemm_probe.restype = ci
        lib.cc_status_string.argtypes = [ci]
        lib.cc_status_string.restype = ctypes.c_char_p
        lib.cc_last_error.restype = ctypes.c_char_p
        _lib = lib
    return _lib


def _check(st: int):
    if st != 0:
        raise CcError(st, load_library().cc_last_error().decode())


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("a CUDA device is required (no CPU fallback)")
    return torch


class Plan:
    """cc_plan_create / cc_track / cc_plan_destroy (include/cc.h)."""

    def __init__(self, H: int, W: int, dtype, upsample: int, reference, method: str = "u", epsilon: float = 0.0):
        lib = load_library()
        _torch()
        dt = np.dtype(dtype)
        if dt == np.uint8:
            self.cc_dtype = CC_U8
        elif dt == np.uint16:
            self.cc_dtype = CC_U16
        else:
            raise TypeError("pixel dtype must be uint8 or uint16")
        self.np_dtype = dt
        self.H, self.W, self.upsample = int(H), int(W), int(upsample)
        ref = np.ascontiguousarray(reference, dtype=np.float32)
        if ref.shape != (self.H, self.W):
            raise ValueError("reference must be (H, W)")
        self._h = ctypes.c_void_p()
        if method not in ("u", "sn"):
            raise ValueError("method must be 'u' (CC-U) or 'sn' (CC-SN)")
        _check(lib.cc_plan_create_weighted(ctypes.byref(self._h), self.H, self.W, self.cc_dtype, self.upsample,
                                           ref.ctypes.data_as(ctypes.c_void_p), 1 if method == "sn" else 0, float(epsilon)))

    def close(self):
        if getattr(self, "_h", None):
            load_library().cc_plan_destroy(self._h)
            self._h = None

    __del__ = close

    def enable_reference_update(self, a0: float):
        """cc_plan_enable_reference_update: running reference image of PAPER.md Eq. (9); a0 = 0 switches it off."""
        _check(load_library().cc_plan_enable_reference_update(self._h, float(a0)))

    def reference_spectrum(self, f64: bool = False) -> np.ndarray:
        """cc_plan_get_reference_spectrum[_f64]: complex64 / complex128 (H, W/2 + 1), the spectrum F[E] of the plan's
        current reference image."""
        out = np.empty((self.H, self.W // 2 + 1), np.complex128 if f64 else np.complex64)
        fn = load_library().cc_plan_get_reference_spectrum_f64 if f64 else load_library().cc_plan_get_reference_spectrum
        _check(fn(self._h, out.ctypes.data_as(ctypes.c_void_p)))
        return out

    def track_accumulate(self, frames_dev, batch: int | None = None):
        """cc_track_accumulate (offline analysis, Eq. (8)): cc_track that also sums the aligned spectra."""
        torch = _torch()
        fb = self.H * self.W * self.np_dtype.itemsize
        if batch is None:
            batch = frames_dev.numel() * frames_dev.element_size() // fb
        dev = frames_dev.device
        dx = torch.empty(batch, dtype=torch.float32, device=dev)
        dy = torch.empty(batch, dtype=torch.float32, device=dev)
        pk = torch.empty(batch, dtype=torch.float32, device=dev)
        _check(load_library().cc_track_accumulate(self._h, frames_dev.data_ptr(), batch, dx.data_ptr(), dy.data_ptr(),
                                                  pk.data_ptr(), torch.cuda.current_stream(dev).cuda_stream))
        return dx, dy, pk

    def update_reference_from_accumulator(self):
        """cc_plan_update_reference_from_accumulator: the reference becomes the mean of the aligned frames."""
        torch = _torch()
        _check(load_library().cc_plan_update_reference_from_accumulator(self._h, torch.cuda.current_stream().cuda_stream))

    def info(self) -> dict:
        inf = PlanInfo()
        _check(load_library().cc_plan_info(self._h, ctypes.byref(inf)))
        return {k: getattr(inf, k) for k, _ in PlanInfo._fields_}

    def device_frames(self, frames_np):
        """Copy a (B, H, W) uint8/uint16 numpy array to the device (torch has no
        uint16 arithmetic; the tensor is only a byte container)."""
        torch = _torch()
        a = np.ascontiguousarray(frames_np, dtype=self.np_dtype)
        if a.ndim == 2:
            a = a[None]
        assert a.shape[1:] == (self.H, self.W)
        t = torch.from_numpy(a.view(np.uint8).reshape(a.shape[0], -1)).cuda()
        return t

    def track(self, frames_dev, batch: int | None = None, want_peak: bool = True, debug: bool = False,
              out=None, stream=None):
        """cc_track on a device tensor of raw frame bytes.  Returns device
        tensors (dx, dy, peak[, iy, ix]); nothing is synchronised."""
        torch = _torch()
        lib = load_library()
        fb = self.H * self.W * self.np_dtype.itemsize
        if batch is None:
            batch = frames_dev.numel() * frames_dev.element_size() // fb
        dev = frames_dev.device
        if out is None:
            dx = torch.empty(batch, dtype=torch.float32, device=dev)
            dy = torch.empty(batch, dtype=torch.float32, device=dev)
            pk = torch.empty(batch, dtype=torch.float32, device=dev) if want_peak else None
        else:
            dx, dy, pk = out
        s = (stream.cuda_stream if stream is not None else torch.cuda.current_stream(dev).cuda_stream)
        pkp = pk.data_ptr() if pk is not None else None
        if debug:
            iy = torch.empty(batch, dtype=torch.int32, device=dev)
            ix = torch.empty(batch, dtype=torch.int32, device=dev)
            _check(lib.cc_track_debug(self._h, frames_dev.data_ptr(), batch, dx.data_ptr(), dy.data_ptr(), pkp,
                                      iy.data_ptr(), ix.data_ptr(), s))
            return dx, dy, pk, iy, ix
        _check(lib.cc_track(self._h, frames_dev.data_ptr(), batch, dx.data_ptr(), dy.data_ptr(), pkp, s))
        return dx, dy, pk

    def track_static(self, frames_dev, out, batch: int | None = None, stream=None):
        """cc_track_static: cc_track without any allocation -- the global spectrum scratch (1024 x 1024 shapes) is a
        static array inside the library (include/cc.h for the limits); `out` = caller's (dx, dy, peak) device tensors."""
        torch = _torch()
        fb = self.H * self.W * self.np_dtype.itemsize
        if batch is None:
            batch = frames_dev.numel() * frames_dev.element_size() // fb
        dx, dy, pk = out
        s = (stream.cuda_stream if stream is not None else torch.cuda.current_stream(frames_dev.device).cuda_stream)
        _check(load_library().cc_track_static(self._h, frames_dev.data_ptr(), batch, dx.data_ptr(), dy.data_ptr(),
                                              pk.data_ptr() if pk is not None else None, s))
        return dx, dy, pk

    def track_profile(self, frames_dev, batch: int | None = None):
        """cc_track_profile: returns (dx, dy, peak, cycles[batch, 8]) device tensors."""
        torch = _torch()
        fb = self.H * self.W * self.np_dtype.itemsize
        if batch is None:
            batch = frames_dev.numel() * frames_dev.element_size() // fb
        dev = frames_dev.device
        dx = torch.empty(batch, dtype=torch.float32, device=dev)
        dy = torch.empty(batch, dtype=torch.float32, device=dev)
        pk = torch.empty(batch, dtype=torch.float32, device=dev)
        cyc = torch.zeros((batch, 8), dtype=torch.int64, device=dev)
        _check(load_library().cc_track_profile(self._h, frames_dev.data_ptr(), batch, dx.data_ptr(), dy.data_ptr(),
                                               pk.data_ptr(), cyc.data_ptr(), torch.cuda.current_stream(dev).cuda_stream))
        return dx, dy, pk, cyc

    def latency_probe(self, frames_dev, n: int | None = None):
        """cc_track_latency_probe: n sequential batch-1 calls timed by the library's native loop.
        Returns (dx, dy, peak) device tensors and a numpy array of per-call latencies in microseconds."""
        torch = _torch()
        fb = self.H * self.W * self.np_dtype.itemsize
        if n is None:
            n = frames_dev.numel() * frames_dev.element_size() // fb
        dev = frames_dev.device
        dx = torch.empty(n, dtype=torch.float32, device=dev)
        dy = torch.empty(n, dtype=torch.float32, device=dev)
        pk = torch.empty(n, dtype=torch.float32, device=dev)
        lat = np.empty(n, np.float64)
        _check(load_library().cc_track_latency_probe(self._h, frames_dev.data_ptr(), n, dx.data_ptr(), dy.data_ptr(),
                                                     pk.data_ptr(), lat.ctypes.data_as(ctypes.c_void_p),
                                                     torch.cuda.current_stream(dev).cuda_stream))
        return dx, dy, pk, lat

    def set_host_chunk(self, frames_per_chunk: int):
        """cc_plan_set_host_chunk: frames per host->device chunk of track_host (0: default)."""
        _check(load_library().cc_plan_set_host_chunk(self._h, int(frames_per_chunk)))

    def track_host(self, frames_np, dx=None, dy=None, peak=None):
        """cc_track_host: host numpy frames in, host numpy results out (H2D/D2H inside)."""
        lib = load_library()
        a = frames_np
        assert a.dtype == self.np_dtype and a.flags["C_CONTIGUOUS"]
        batch = a.shape[0] if a.ndim == 3 else 1
        dx = np.empty(batch, np.float32) if dx is None else dx
        dy = np.empty(batch, np.float32) if dy is None else dy
        peak = np.empty(batch, np.float32) if peak is None else peak
        _check(lib.cc_track_host(self._h, a.ctypes.data_as(ctypes.c_void_p), batch,
                                 dx.ctypes.data_as(ctypes.c_void_p), dy.ctypes.data_as(ctypes.c_void_p),
                                 peak.ctypes.data_as(ctypes.c_void_p)))
        return dx, dy, peak


class RtSession:
    """cc_rt_open / cc_rt_track / cc_rt_close (include/cc.h): a resident session kernel serves single frames.
    While a session is open, do not call device-wide synchronisation (torch.cuda.synchronize())."""

    def __init__(self, plan: Plan, idle_timeout_ms: int = 1000):
        self.plan = plan
        self._h = ctypes.c_void_p()
        _check(load_library().cc_rt_open(plan._h, int(idle_timeout_ms), ctypes.byref(self._h)))
        self._out = (ctypes.c_float * 3)()

    def track(self, frame_ptr: int):
        """One frame at device (or pinned host) address `frame_ptr`; returns (dx, dy, peak) as Python floats."""
        o = self._out
        f = ctypes.c_float
        _check(load_library().cc_rt_track(self._h, ctypes.c_void_p(frame_ptr), ctypes.cast(ctypes.byref(o, 0), ctypes.POINTER(f)),
                                          ctypes.cast(ctypes.byref(o, 4), ctypes.POINTER(f)),
                                          ctypes.cast(ctypes.byref(o, 8), ctypes.POINTER(f))))
        return o[0], o[1], o[2]

    def latency_probe(self, frames_ptr: int, n: int):
        """cc_rt_latency_probe: returns (dx, dy, peak, lat_us) numpy arrays."""
        dx, dy, pk = np.empty(n, np.float32), np.empty(n, np.float32), np.empty(n, np.float32)
        lat = np.empty(n, np.float64)
        vp = ctypes.c_void_p
        _check(load_library().cc_rt_latency_probe(self._h, vp(frames_ptr), n, dx.ctypes.data_as(vp), dy.ctypes.data_as(vp),
                                                  pk.ctypes.data_as(vp), lat.ctypes.data_as(vp)))
        return dx, dy, pk, lat

    def close(self):
        if getattr(self, "_h", None):
            load_library().cc_rt_close(self._h)
            self._h = None

    __del__ = close


def fp32_peak_probe() -> float:
    _torch()
    v = ctypes.c_double()
    _check(load_library().cc_fp32_peak_probe(ctypes.byref(v), None))
    return v.value


def fp32_tile_probe() -> float:
    _torch()
    v = ctypes.c_double()
    _check(load_library().cc_fp32_tile_probe(ctypes.byref(v), None))
    return v.value


def drift_correct(dx, dy, a0: float, max_step: float = 0.0, state=None, stream=None):
    """cc_drift_correct on device tensors dx, dy (float32).  `state` = device float64 tensor (Rx, Ry), updated in
    place (None: starts from zero).  Returns (dx', dy', state); nothing is synchronised."""
    torch = _torch()
    n = dx.numel()
    if state is None:
        state = torch.zeros(2, dtype=torch.float64, device=dx.device)
    ox, oy = torch.empty_like(dx), torch.empty_like(dy)
    s = (stream.cuda_stream if stream is not None else torch.cuda.current_stream(dx.device).cuda_stream)
    _check(load_library().cc_drift_correct(dx.data_ptr(), dy.data_ptr(), n, float(a0), float(max_step), state.data_ptr(),
                                           ox.data_ptr(), oy.data_ptr(), s))
    return ox, oy, state


def tc_gemm_probe(A, B, passes: int = 3, iters: int = 50, repeat: int = 1):
    """cc_tc_gemm_probe: D = A B (128 x K times K x 128) on the tensor cores (TF32, 1 or 3 passes).
    Returns (D, stage_cycles, mma_cycles)."""
    _torch()
    A = np.ascontiguousarray(A, dtype=np.float32)
    B = np.ascontiguousarray(B, dtype=np.float32)
    assert A.shape[0] == 128 and B.shape[1] == 128 and A.shape[1] == B.shape[0]
    D = np.empty((128, 128), np.float32)
    sc, mc = ctypes.c_double(), ctypes.c_double()
    vp = ctypes.c_void_p
    _check(load_library().cc_tc_gemm_probe(A.ctypes.data_as(vp), B.ctypes.data_as(vp), A.shape[1], int(passes), int(iters), int(repeat),
                                           D.ctypes.data_as(vp), ctypes.byref(sc), ctypes.byref(mc)))
    return D, sc.value, mc.value
