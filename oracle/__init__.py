"""CPU ORACLE -- TEST INFRASTRUCTURE, NOT A PRODUCT PATH.

ctypes binding of ``oracle/cc_oracle.c`` (plain C, float64, naive DFTs): the
slow, obviously-correct restatement of the displacement estimator of
arxiv 2310.08770 (Eq. (4); Sec. III) that the
CUDA library is checked against.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this package.  It
imports nothing from ``paper_2310_08770_b200`` and shares no code with it.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cc_oracle.c")
_HDR = os.path.join(_HERE, "cc_oracle.h")
_LIB = os.path.join(_HERE, "libcc_oracle.so")

_lib = None


def build(force: bool = False) -> str:
    """Compile cc_oracle.c with gcc (-O2 -fopenmp) into oracle/libcc_oracle.so."""
    newest = max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < newest:
        tmp = _LIB + ".tmp.%d" % os.getpid()
        cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-Wall",
               "-o", tmp, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


class _Result(ctypes.Structure):
    _fields_ = [("dy", ctypes.c_double), ("dx", ctypes.c_double),
                ("peak", ctypes.c_double),
                ("wy", ctypes.c_int), ("wx", ctypes.c_int),
                ("m", ctypes.c_int), ("n", ctypes.c_int),
                ("cc_top1", ctypes.c_double), ("cc_top2", ctypes.c_double),
                ("up_top1", ctypes.c_double), ("up_top2", ctypes.c_double)]


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int)
        lib.cco_dft2_real.argtypes = [dp, ctypes.c_int, ctypes.c_int, dp, dp]
        lib.cco_dft2_literal.argtypes = [dp, ctypes.c_int, ctypes.c_int, dp, dp]
        lib.cco_idft2.argtypes = [dp, dp, ctypes.c_int, ctypes.c_int, dp, dp]
        lib.cco_cc_direct.argtypes = [dp, dp, ctypes.c_int, ctypes.c_int, dp]
        lib.cco_cc_dft.argtypes = [dp, dp, ctypes.c_int, ctypes.c_int, dp, dp, dp]
        lib.cco_argmax.argtypes = [dp, ctypes.c_long]
        lib.cco_argmax.restype = ctypes.c_long
        lib.cco_grid_size.argtypes = [ctypes.c_int]
        lib.cco_upsampled.argtypes = [dp, dp, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                      ctypes.c_int, ctypes.c_int, dp, ip, ip, dp, dp]
        lib.cco_upsampled_literal.argtypes = [dp, dp, ctypes.c_int, ctypes.c_int,
                                              ctypes.c_int, ctypes.c_int, ctypes.c_int, dp]
        lib.cco_interp_at.argtypes = [dp, dp, ctypes.c_int, ctypes.c_int,
                                      ctypes.c_double, ctypes.c_double]
        lib.cco_interp_at.restype = ctypes.c_double
        lib.cco_track.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                  ctypes.c_int, ctypes.c_int, ctypes.POINTER(ctypes.c_float),
                                  ctypes.POINTER(_Result), ctypes.c_int]
        lib.cco_track_sn.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                     ctypes.c_int, ctypes.c_int, ctypes.POINTER(ctypes.c_float),
                                     ctypes.c_double, ctypes.POINTER(_Result), ctypes.c_int]
        lib.cco_drift_correct.argtypes = [ctypes.POINTER(ctypes.c_float), ctypes.POINTER(ctypes.c_float), ctypes.c_int,
                                          ctypes.c_double, ctypes.c_double, dp, dp, dp]
        lib.cco_track_rt.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                     ctypes.POINTER(ctypes.c_float), ctypes.c_double, ctypes.POINTER(_Result), dp, dp]
        lib.cco_iterate_reference.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                              ctypes.POINTER(ctypes.c_float), ctypes.c_int, ctypes.POINTER(_Result), dp, dp]
        lib.cco_step_from_spectrum.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, dp, dp,
                                               ctypes.c_double, ctypes.POINTER(_Result), dp, dp]
        lib.cco_track_rt_sn.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                        ctypes.POINTER(ctypes.c_float), ctypes.c_double, ctypes.c_double, ctypes.POINTER(_Result), dp, dp]
        lib.cco_iterate_reference_sn.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                                 ctypes.POINTER(ctypes.c_float), ctypes.c_double, ctypes.c_int, ctypes.POINTER(_Result), dp, dp]
        lib.cco_step_from_spectrum_sn.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, dp, dp,
                                                  ctypes.c_double, ctypes.c_double, ctypes.POINTER(_Result), dp, dp]
        lib.cco_num_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def _d(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def dft2(img, literal: bool = False):
    """O2: naive 2D DFT of a real image -> complex128 (H, W)."""
    img = _f64(img)
    H, W = img.shape
    re, im = np.empty((H, W)), np.empty((H, W))
    fn = _load().cco_dft2_literal if literal else _load().cco_dft2_real
    if fn(_d(img), H, W, _d(re), _d(im)):
        raise MemoryError("oracle dft2")
    return re + 1j * im


def idft2(P):
    """O4: naive inverse 2D DFT (1/(HW) included) -> complex128 (H, W)."""
    P = np.asarray(P, dtype=np.complex128)
    H, W = P.shape
    pr, pi = _f64(P.real), _f64(P.imag)
    re, im = np.empty((H, W)), np.empty((H, W))
    if _load().cco_idft2(_d(pr), _d(pi), H, W, _d(re), _d(im)):
        raise MemoryError("oracle idft2")
    return re + 1j * im


def cc_direct(I, E):
    """Left side of Eq. (4): brute-force circular cross-correlation."""
    I, E = _f64(I), _f64(E)
    H, W = I.shape
    cc = np.empty((H, W))
    _load().cco_cc_direct(_d(I), _d(E), H, W, _d(cc))
    return cc


def cc_dft(I, E):
    """Right side of Eq. (4): returns (cc, P) with P = F[I] conj(F[E])."""
    I, E = _f64(I), _f64(E)
    H, W = I.shape
    cc, pr, pi = np.empty((H, W)), np.empty((H, W)), np.empty((H, W))
    if _load().cco_cc_dft(_d(I), _d(E), H, W, _d(cc), _d(pr), _d(pi)):
        raise MemoryError("oracle cc_dft")
    return cc, pr + 1j * pi


def argmax(a) -> int:
    a = _f64(a).ravel()
    return int(_load().cco_argmax(_d(a), a.size))


def grid_size(u: int) -> int:
    return int(_load().cco_grid_size(int(u)))


def upsampled(P, u: int, y0: int, x0: int, want_grid: bool = True, literal: bool = False):
    """O6: upsampled CC around integer peak (y0, x0).

    Returns dict(C, m, n, top1, top2); C is None when want_grid is False."""
    P = np.asarray(P, dtype=np.complex128)
    H, W = P.shape
    pr, pi = _f64(P.real), _f64(P.imag)
    M = grid_size(u)
    lib = _load()
    if literal:
        C = np.empty((M, M))
        if lib.cco_upsampled_literal(_d(pr), _d(pi), H, W, u, y0, x0, _d(C)):
            raise MemoryError("oracle upsampled_literal")
        i = argmax(C)
        return dict(C=C, m=i // M, n=i % M, top1=float(C.ravel()[i]), top2=None)
    C = np.empty((M, M)) if want_grid else None
    m, n = ctypes.c_int(), ctypes.c_int()
    t1, t2 = ctypes.c_double(), ctypes.c_double()
    rc = lib.cco_upsampled(_d(pr), _d(pi), H, W, u, y0, x0,
                           _d(C) if C is not None else None,
                           ctypes.byref(m), ctypes.byref(n), ctypes.byref(t1), ctypes.byref(t2))
    if rc:
        raise MemoryError("oracle upsampled")
    return dict(C=C, m=m.value, n=n.value, top1=t1.value, top2=t2.value)


def interp_at(P, sy: float, sx: float) -> float:
    P = np.asarray(P, dtype=np.complex128)
    H, W = P.shape
    pr, pi = _f64(P.real), _f64(P.imag)
    return float(_load().cco_interp_at(_d(pr), _d(pi), H, W, float(sy), float(sx)))


@dataclass
class TrackResult:
    dy: np.ndarray
    dx: np.ndarray
    peak: np.ndarray
    wy: np.ndarray
    wx: np.ndarray
    m: np.ndarray
    n: np.ndarray
    cc_top1: np.ndarray
    cc_top2: np.ndarray
    up_top1: np.ndarray
    up_top2: np.ndarray


def num_threads() -> int:
    return int(_load().cco_num_threads())


def track(frames, reference, u: int, threads: int = 0, method: str = "u", epsilon: float = 0.0) -> TrackResult:
    """The whole path O1-O7 for a batch of uint8/uint16 frames (B, H, W)
    against a float32 reference (H, W).  method "u": CC-U, Eq. (4); method "sn":
    CC-SN, Eqs. (5)-(7) with offset epsilon (minimum of the weighted sum)."""
    frames = np.ascontiguousarray(frames)
    if frames.ndim == 2:
        frames = frames[None]
    if frames.dtype == np.uint8:
        dt = 0
    elif frames.dtype == np.uint16:
        dt = 1
    else:
        raise TypeError("frames must be uint8 or uint16")
    B, H, W = frames.shape
    ref = np.ascontiguousarray(reference, dtype=np.float32)
    if ref.shape != (H, W):
        raise ValueError("reference shape mismatch")
    out = (_Result * max(B, 1))()
    if method == "sn":
        rc = _load().cco_track_sn(frames.ctypes.data_as(ctypes.c_void_p), dt, B, H, W, int(u),
                                  ref.ctypes.data_as(ctypes.POINTER(ctypes.c_float)), float(epsilon), out, int(threads))
    elif method == "u":
        rc = _load().cco_track(frames.ctypes.data_as(ctypes.c_void_p), dt, B, H, W, int(u),
                               ref.ctypes.data_as(ctypes.POINTER(ctypes.c_float)), out, int(threads))
    else:
        raise ValueError("method must be 'u' or 'sn'")
    if rc:
        raise RuntimeError("oracle cco_track failed: %d" % rc)
    arr = np.frombuffer(out, dtype=np.dtype([
        ("dy", "f8"), ("dx", "f8"), ("peak", "f8"), ("wy", "i4"), ("wx", "i4"),
        ("m", "i4"), ("n", "i4"), ("cc_top1", "f8"), ("cc_top2", "f8"),
        ("up_top1", "f8"), ("up_top2", "f8")], align=True))[:B]
    return TrackResult(*(arr[k].copy() for k in
                         ("dy", "dx", "peak", "wy", "wx", "m", "n",
                          "cc_top1", "cc_top2", "up_top1", "up_top2")))


def drift_correct(dx, dy, a0: float, max_step: float = 0.0, state=None):
    """PAPER.md:L110-127, Eqs. (10)-(12): returns (dx', dy', state) with state = (Rx, Ry) after the last sample."""
    dx = np.ascontiguousarray(dx, dtype=np.float32)
    dy = np.ascontiguousarray(dy, dtype=np.float32)
    n = dx.size
    st = np.zeros(2) if state is None else np.array(state, dtype=np.float64)
    ox, oy = np.empty(n), np.empty(n)
    fp = ctypes.POINTER(ctypes.c_float)
    rc = _load().cco_drift_correct(dx.ctypes.data_as(fp), dy.ctypes.data_as(fp), n, float(a0), float(max_step),
                                   _d(st), _d(ox), _d(oy))
    if rc:
        raise ValueError("oracle cco_drift_correct failed: %d" % rc)
    return ox, oy, st


_RES_DT = np.dtype([("dy", "f8"), ("dx", "f8"), ("peak", "f8"), ("wy", "i4"), ("wx", "i4"), ("m", "i4"), ("n", "i4"),
                    ("cc_top1", "f8"), ("cc_top2", "f8"), ("up_top1", "f8"), ("up_top2", "f8")], align=True)


def _status(rc, what):
    if rc == -3:
        raise ValueError("oracle %s: CC-SN needs E + epsilon > 0 in every pixel of the current reference" % what)
    if rc:
        raise RuntimeError("oracle %s failed: %d" % (what, rc))


def track_rt(frames, reference, u: int, a0: float, method: str = "u", epsilon: float = 0.0):
    """PAPER.md:L102-108, Eq. (9): sequential tracking with the running reference image.  Returns
    (TrackResult, G) with G the complex spectrum (H, W) of the last reference image.  method "sn": CC-SN (R19)."""
    frames = np.ascontiguousarray(frames)
    if frames.ndim == 2:
        frames = frames[None]
    dt = {np.dtype(np.uint8): 0, np.dtype(np.uint16): 1}[frames.dtype]
    B, H, W = frames.shape
    ref = np.ascontiguousarray(reference, dtype=np.float32)
    out = (_Result * max(B, 1))()
    gr, gi = np.empty((H, W)), np.empty((H, W))
    if method == "sn":
        rc = _load().cco_track_rt_sn(frames.ctypes.data_as(ctypes.c_void_p), dt, B, H, W, int(u),
                                     ref.ctypes.data_as(ctypes.POINTER(ctypes.c_float)), float(epsilon), float(a0), out, _d(gr), _d(gi))
    else:
        rc = _load().cco_track_rt(frames.ctypes.data_as(ctypes.c_void_p), dt, B, H, W, int(u),
                                  ref.ctypes.data_as(ctypes.POINTER(ctypes.c_float)), float(a0), out, _d(gr), _d(gi))
    _status(rc, "cco_track_rt")
    arr = np.frombuffer(out, dtype=_RES_DT)[:B]
    res = TrackResult(*(arr[k].copy() for k in ("dy", "dx", "peak", "wy", "wx", "m", "n", "cc_top1", "cc_top2",
                                                "up_top1", "up_top2")))
    return res, gr + 1j * gi


def iterate_reference(frames, reference, u: int, n_iter: int, method: str = "u", epsilon: float = 0.0):
    """PAPER.md:L94-100, Eq. (8): n_iter passes of the offline analysis.  Returns (TrackResult of the last pass, G).
    method "sn": CC-SN (R19)."""
    frames = np.ascontiguousarray(frames)
    dt = {np.dtype(np.uint8): 0, np.dtype(np.uint16): 1}[frames.dtype]
    B, H, W = frames.shape
    ref = np.ascontiguousarray(reference, dtype=np.float32)
    out = (_Result * B)()
    gr, gi = np.empty((H, W)), np.empty((H, W))
    if method == "sn":
        rc = _load().cco_iterate_reference_sn(frames.ctypes.data_as(ctypes.c_void_p), dt, B, H, W, int(u),
                                              ref.ctypes.data_as(ctypes.POINTER(ctypes.c_float)), float(epsilon), int(n_iter), out,
                                              _d(gr), _d(gi))
    else:
        rc = _load().cco_iterate_reference(frames.ctypes.data_as(ctypes.c_void_p), dt, B, H, W, int(u),
                                           ref.ctypes.data_as(ctypes.POINTER(ctypes.c_float)), int(n_iter), out, _d(gr), _d(gi))
    _status(rc, "cco_iterate_reference")
    arr = np.frombuffer(out, dtype=_RES_DT)[:B]
    res = TrackResult(*(arr[k].copy() for k in ("dy", "dx", "peak", "wy", "wx", "m", "n", "cc_top1", "cc_top2",
                                                "up_top1", "up_top2")))
    return res, gr + 1j * gi


def step_from_spectrum(frame, G, u: int, a0: float, method: str = "u", epsilon: float = 0.0):
    """PAPER.md:L106, Eq. (9), ONE step from a given reference spectrum G (complex (H, W), full spectrum): returns
    (TrackResult of the frame against G, Gn = a0 F[frame aligned] + (1 - a0) G).  a0 = 1: the aligned spectrum (a
    summand of Eq. (8)).  method "sn": the frame is measured by Eq. (7) with the weight 1/(E + epsilon), E = F^-1[G]."""
    frame = np.ascontiguousarray(frame)
    dt = {np.dtype(np.uint8): 0, np.dtype(np.uint16): 1}[frame.dtype]
    H, W = frame.shape
    G = np.asarray(G, dtype=np.complex128)
    gr, gi = _f64(G.real), _f64(G.imag)
    nr, ni = np.empty((H, W)), np.empty((H, W))
    out = (_Result * 1)()
    if method == "sn":
        rc = _load().cco_step_from_spectrum_sn(frame.ctypes.data_as(ctypes.c_void_p), dt, H, W, int(u), _d(gr), _d(gi),
                                               float(epsilon), float(a0), out, _d(nr), _d(ni))
    else:
        rc = _load().cco_step_from_spectrum(frame.ctypes.data_as(ctypes.c_void_p), dt, H, W, int(u), _d(gr), _d(gi), float(a0), out,
                                            _d(nr), _d(ni))
    _status(rc, "cco_step_from_spectrum")
    arr = np.frombuffer(out, dtype=_RES_DT)[:1]
    res = TrackResult(*(arr[k].copy() for k in ("dy", "dx", "peak", "wy", "wx", "m", "n", "cc_top1", "cc_top2",
                                                "up_top1", "up_top2")))
    return res, nr + 1j * ni
