"""Seeded synthetic camera workloads (input generators ONLY).

This module holds none of the tracking method's arithmetic: it only draws the
input frames.  It is the one module that serves both the CPU oracle's tests
and the CUDA path (tests, bench.py, smoke()).

The recipes stand in for the paper's workloads -- its synthetic study
("a Gaussian function integrated over each pixel ... with Poisson shot noise
added", displacements "randomly distributed but exactly known",
PAPER.md:L131) and its 12-bit experimental recording --
neither of which is available here.  Parameters are those of
``BASELINE.json:configs``; the details the configs leave open are fixed in
DESIGN.md ("Input recipe").

Streams: all shifts of a config come from ``default_rng([seed, 0])``; the
noise of frame ``i`` comes from its own stream ``default_rng([seed, 1, i])``,
so any subset of frames can be regenerated without the rest.
"""
from __future__ import annotations

import os
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass

import numpy as np
from scipy.special import erf, j1


@dataclass(frozen=True)
class Config:
    index: int          # 1..5, position in BASELINE.json:configs
    name: str
    H: int
    W: int
    dtype: str          # "uint8" | "uint16"
    n_frames: int
    seed: int
    upsample: int
    mode: str           # "batched" | "streaming"
    oracle_stride: int  # parity subset: frames i % stride == 0 ...
    oracle_count: int   # ... first `oracle_count` of them


CONFIGS = {
    1: Config(1, "cfg1_64x64_u16_u100_batch1000", 64, 64, "uint16", 1000, 0, 100, "batched", 1, 1000),
    2: Config(2, "cfg2_128x128_u8_u20_stream", 128, 128, "uint8", 10000, 1, 20, "streaming", 10, 1000),
    3: Config(3, "cfg3_256x256_u16_u100_batch10000", 256, 256, "uint16", 10000, 2, 100, "batched", 10, 1000),
    4: Config(4, "cfg4_512x512_u16_u50_stream", 512, 512, "uint16", 2000, 3, 50, "streaming", 10, 200),
    5: Config(5, "cfg5_1024x1024_u16_u100_batch1000", 1024, 1024, "uint16", 1000, 4, 100, "batched", 8, 64),
}


def config(index: int) -> Config:
    return CONFIGS[int(index)]


def _gauss_px(t, mu, sigma):
    """Peak-normalised 1-D Gaussian integrated over each pixel [t-1/2, t+1/2]."""
    s = np.sqrt(2.0) * sigma
    return (erf((t - mu + 0.5) / s) - erf((t - mu - 0.5) / s)) / (2.0 * erf(0.5 / s))


def shifts(cfg: Config) -> np.ndarray:
    """(n_frames, 2) float64 true shifts, column 0 = sy (rows), column 1 = sx."""
    rng = np.random.default_rng([cfg.seed, 0])
    n = cfg.n_frames
    if cfg.index == 1:
        return rng.uniform(-5.0, 5.0, size=(n, 2))
    if cfg.index == 2:
        steps = rng.normal(0.0, 0.3, size=(n, 2))
        s = np.zeros((n, 2))
        for i in range(1, n):
            s[i] = np.clip(s[i - 1] + steps[i], -20.0, 20.0)
        return s
    if cfg.index == 3:
        return rng.uniform(-30.0, 30.0, size=(n, 2))
    if cfg.index == 4:
        i = np.arange(n, dtype=np.float64)
        jit = rng.normal(0.0, 0.25, size=(n, 2))
        sy = 40.0 * np.sin(2.0 * np.pi * i / 293.0 + 1.0) + jit[:, 0]
        sx = 40.0 * np.sin(2.0 * np.pi * i / 400.0) + jit[:, 1]
        return np.stack([sy, sx], axis=1)
    if cfg.index == 5:
        return rng.uniform(-100.0, 100.0, size=(n, 2))
    raise ValueError(cfg.index)


def expected_counts(cfg: Config, sy: float, sx: float, template: bool = False) -> np.ndarray:
    """Noise-free expected photon map lambda(y, x) in float64.

    template=True gives the reference template: the spot at the frame centre on
    a FLAT background equal to the mean background level (camera-fixed
    structure -- cfg 3's gradient, cfg 5's fringes -- is in frames only)."""
    H, W = cfg.H, cfg.W
    y = np.arange(H, dtype=np.float64)[:, None]
    x = np.arange(W, dtype=np.float64)[None, :]
    cy, cx = H / 2 + sy, W / 2 + sx
    if cfg.index == 1:
        return 1000.0 * _gauss_px(y, cy, 3.0) * _gauss_px(x, cx, 3.0) + 10.0
    if cfg.index == 2:
        return 200.0 * _gauss_px(y, cy, 4.0) * _gauss_px(x, cx, 4.0) + 5.0
    if cfg.index == 3:
        r = np.hypot(y - cy, x - cx)
        v = 3.8317 * r / 6.0
        with np.errstate(invalid="ignore", divide="ignore"):
            a = np.where(v > 1e-12, 2.0 * j1(v) / np.where(v > 1e-12, v, 1.0), 1.0)
        bg = 50.0 if template else 20.0 + 60.0 * x / 255.0
        return 5000.0 * a * a + bg
    if cfg.index == 4:
        dx_, dy_ = x - cx, y - cy
        c30, s30 = np.cos(np.pi / 6), np.sin(np.pi / 6)
        a = c30 * dx_ + s30 * dy_
        b = -s30 * dx_ + c30 * dy_
        return 2000.0 * np.exp(-a * a / (2 * 5.0 ** 2) - b * b / (2 * 8.0 ** 2)) + 50.0
    if cfg.index == 5:
        spot = 50.0 * _gauss_px(y, cy, 6.0) * _gauss_px(x, cx, 6.0)
        bg = 30.0 if template else 30.0 + 10.0 * np.sin(2 * np.pi * x / 64.0) * np.sin(2 * np.pi * y / 64.0)
        return spot + bg
    raise ValueError(cfg.index)


def _one_frame(cfg: Config, i: int, sy: float, sx: float) -> np.ndarray:
    rng = np.random.default_rng([cfg.seed, 1, int(i)])
    lam = expected_counts(cfg, sy, sx)
    px = rng.poisson(lam).astype(np.float64)
    if cfg.index == 4:
        px = px + rng.normal(0.0, 2.0, size=px.shape)
    px = np.rint(px)
    hi = 255 if cfg.dtype == "uint8" else 65535
    return np.clip(px, 0, hi).astype(cfg.dtype)


def frames(cfg: Config, indices=None, workers: int | None = None) -> np.ndarray:
    """Frames `indices` (default: all) of a config, shape (n, H, W)."""
    if indices is None:
        indices = np.arange(cfg.n_frames)
    indices = np.asarray(indices, dtype=np.int64)
    s = shifts(cfg)
    out = np.empty((len(indices), cfg.H, cfg.W), dtype=cfg.dtype)

    def work(j):
        i = int(indices[j])
        out[j] = _one_frame(cfg, i, s[i, 0], s[i, 1])

    workers = workers or min(32, os.cpu_count() or 1)
    if len(indices) < 4 or workers == 1:
        for j in range(len(indices)):
            work(j)
    else:
        with ThreadPoolExecutor(workers) as ex:
            list(ex.map(work, range(len(indices)), chunksize=max(1, len(indices) // (workers * 8))))
    return out


def reference(cfg: Config) -> np.ndarray:
    """float32 (H, W) reference image of a config."""
    if cfg.index == 2:  # "The reference is the first noisy frame."
        return frames(cfg, [0])[0].astype(np.float32)
    return expected_counts(cfg, 0.0, 0.0, template=True).astype(np.float32)


def oracle_subset(cfg: Config) -> np.ndarray:
    """Indices of the frames the float64 oracle is run on for this config."""
    idx = np.arange(0, cfg.n_frames, cfg.oracle_stride)
    return idx[: cfg.oracle_count]


def checksum(px: np.ndarray) -> dict:
    import hashlib
    return {"sum": int(px.astype(np.uint64).sum()),
            "sha256_frame0": hashlib.sha256(np.ascontiguousarray(px[0]).tobytes()).hexdigest()}
