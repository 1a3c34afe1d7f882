#!/usr/bin/env python
"""bench.py -- frames/s of the fused cross-correlation tracker on B200.

One "step" = one cc_track() pass of the whole hot path (ingest, FFTs, product,
argmax, upsampled DFT, sub-pixel argmax) over one batch of seeded synthetic
frames (BASELINE.json configs[2]: 256x256 uint16, batch 10,000, u = 100 --
the configuration the roofline target is quoted on).  Also reports the
single-frame latency of the streaming configs (configs[1] 128x128 uint8 u = 20, configs[3] 512x512 uint16
u = 50) through cc_track + stream sync and through the real-time session (cc_rt_*).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

Under torchrun (N > 1) every rank runs the same workload on its own frames
(weak scaling, no data-path collective); time = max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2310_08770_b200 import workloads as wl  # noqa: E402

NOMINAL_SM_MHZ = 1965.0
FP32_LANES_PER_SM = 128
# dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel, one 10,000-frame launch, from the committed capture
TRAFFIC_BYTES_PER_10K_LAUNCH = 1.3175e9
TRAFFIC_SOURCE = ("ncu --set full capture of one 10,000-frame launch, raw rows in profiles/r2d_cfg3_raw_metrics.csv "
                  "(dram__bytes_read.sum + dram__bytes_write.sum); algorithmic bytes 1.3108e9")


def flops_per_frame(H, W, u):
    """Algorithmic flop count of SURVEY.md 8(d): FFT pair + product + upsampled DFT stages 1 and 2."""
    Wh, M = W // 2 + 1, (3 * u + 1) // 2
    fft = 5.0 * H * W * np.log2(H * W)
    prod = 6.0 * H * Wh
    s1 = 8.0 * M * H * Wh
    s2 = 4.0 * M * M * Wh
    return fft + prod + s1 + s2


def executed_flops_per_frame(H, W, u):
    """Flops of the formulation the kernel executes: real Dirichlet stage 1 on Q with
    even/odd halves (2 x nd x (H/2+1) x W multiply-adds), stage 2 as E/O pairs (M x nd x W multiply-adds)."""
    M = (3 * u + 1) // 2
    nd = M // 2 + 1
    fft = 5.0 * H * W * np.log2(H * W)
    return fft + 6.0 * H * (W // 2) + 2.0 * (2.0 * nd * (H // 2 + 1) * W) + 2.0 * (M * nd * W)


def tensor_core_flops_per_frame(H, info):
    """Flop the tensor cores are handed per frame when stage 1 runs on them: per CTA, pass over
    the offsets and 8-row step, two accumulators (U, V) x (128 x 256 x 8 + 128 x 128 x 8) multiply-adds: the three TF32
    passes of the hi/lo split, MMA M = 128 whatever the number of offsets in use."""
    if not info.get("tensor_core_stage1"):
        return 0.0
    ksteps = (H // 2 + 1 + 7) // 8
    return 2.0 * info["cluster_size"] * info["super_blocks"] * ksteps * 2 * (128 * 256 * 8 + 128 * 128 * 8)


class ClockSampler:
    def __init__(self, gpu_index: int):
        self.idx = gpu_index
        self.proc = None
        self.lines = []

    def start(self):
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.idx), "--query-gpu=" + q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])), mx.append(float(f[1]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def oracle_rate(cfg, n_frames: int):
    """Frames/s of the float64 CPU oracle, as it stands, on the first n frames of the batch."""
    import oracle
    idx = np.arange(min(n_frames, cfg.n_frames))
    fr = wl.frames(cfg, idx)
    ref = wl.reference(cfg)
    oracle.track(fr[:1], ref, cfg.upsample)  # build + warm
    t0 = time.perf_counter()
    oracle.track(fr, ref, cfg.upsample)
    dt = time.perf_counter() - t0
    return len(idx) / dt, oracle.num_threads(), len(idx), dt


PHASES = ["ingest + row FFT", "column FFT x conj(G) + column inverse", "row C2R + integer argmax", "fp64 integer polish",
          "upsampled stage 1", "upsampled stage 2", "sub-pixel argmax reduction", "fp64 sub-pixel polish"]


def run_phases():
    """--phases: per-phase SM-clock cycles per frame (cc_track_profile, median over frames) of every config,
    batched configs in steady state and the streaming configs at batch 1."""
    import torch
    from paper_2310_08770_b200 import Plan
    for ci, B in ((1, 1000), (2, 1), (3, 2960), (4, 1), (5, 30)):
        cfg = wl.config(ci)
        fr = wl.frames(cfg, np.arange(min(B, 64)))
        if B > len(fr):
            fr = np.concatenate([fr] * ((B + len(fr) - 1) // len(fr)))[:B]
        plan = Plan(cfg.H, cfg.W, fr.dtype, cfg.upsample, wl.reference(cfg))
        d = plan.device_frames(fr)
        for _ in range(3):
            out = plan.track_profile(d, B)
        torch.cuda.synchronize()
        med = np.median(out[3].cpu().numpy().astype(np.float64), axis=0)
        info = plan.info()
        cs = info["lat_cluster_size"] if (B <= info["lat_max_clusters"] and info["lat_cluster_size"]) else info["cluster_size"]
        print("%s  batch %d  cluster size %d" % (cfg.name, B, cs))
        for nm, v in zip(PHASES, med):
            print("   %-40s %9.0f cycles %5.1f %%" % (nm, v, 100 * v / med.sum()))
        print("   %-40s %9.0f cycles = %.1f us at 1965 MHz" % ("total per frame", med.sum(), med.sum() / 1965.0))
        plan.close()


def run_table(args):
    """--table: one JSON line per config for BASELINE.md section 3 -- batched configs: frames/s over the whole batch
    (CUDA events, 3 warm-up + 5 timed calls) and roofline fractions; streaming configs: single-frame latency; every
    config: the oracle's frames/s on a bounded sample."""
    import torch
    from paper_2310_08770_b200 import Plan, RtSession
    import oracle
    peak_tf = 148 * FP32_LANES_PER_SM * 2 * NOMINAL_SM_MHZ * 1e6 / 1e12
    osample = {1: 1000, 2: 1000, 3: 256, 4: 64, 5: 32}
    for ci in (1, 2, 3, 4, 5):
        cfg = wl.config(ci)
        row = {"cfg": ci, "workload": cfg.name}
        ref = wl.reference(cfg)
        if cfg.mode == "batched":
            fr = wl.frames(cfg)
            B = len(fr)
            plan = Plan(cfg.H, cfg.W, fr.dtype, cfg.upsample, ref)
            d = plan.device_frames(fr)
            out = tuple(torch.empty(B, dtype=torch.float32, device="cuda") for _ in range(3))
            for _ in range(3):
                plan.track(d, B, out=out)
            ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(5)]
            for a, b in ev:
                a.record()
                plan.track(d, B, out=out)
                b.record()
            torch.cuda.synchronize()
            ms = float(np.median([a.elapsed_time(b) for a, b in ev]))
            fps = B / (ms * 1e-3)
            row.update({"frames_per_s": fps, "ms_per_batch": ms, "batch": B,
                        "roofline_frac_algorithmic": flops_per_frame(cfg.H, cfg.W, cfg.upsample) * fps / (peak_tf * 1e12),
                        "roofline_frac_executed": executed_flops_per_frame(cfg.H, cfg.W, cfg.upsample) * fps / (peak_tf * 1e12),
                        "input": "%.2f GB per call%s" % (fr.nbytes / 1e9, "" if fr.nbytes > 2e8 else " (fits L2; ALU-bound either way)")})
            plan.close()
            del d, fr
        else:
            n = min(2000, cfg.n_frames)
            fr = wl.frames(cfg, np.arange(n))
            plan = Plan(cfg.H, cfg.W, fr.dtype, cfg.upsample, ref)
            d = plan.device_frames(fr)
            plan.latency_probe(d, 100)
            l0 = plan.latency_probe(d, n)[3]
            torch.cuda.current_stream().synchronize()
            rt = RtSession(plan, 1000)
            try:
                rt.latency_probe(d.data_ptr(), 100)
                l1 = rt.latency_probe(d.data_ptr(), n)[3]
            finally:
                rt.close()
            row.update({"latency_us_cc_track_sync_median_p99": [float(np.median(l0)), float(np.percentile(l0, 99))],
                        "latency_us_rt_session_median_p99": [float(np.median(l1)), float(np.percentile(l1, 99))], "calls": n})
            plan.close()
        idx = wl.oracle_subset(cfg)[: osample[ci]]
        fo = wl.frames(cfg, idx)
        oracle.track(fo[:1], ref, cfg.upsample)
        t0 = time.perf_counter()
        oracle.track(fo, ref, cfg.upsample)
        dt = time.perf_counter() - t0
        row.update({"oracle_frames_per_s": len(idx) / dt, "oracle_cores": oracle.num_threads(), "oracle_sample": len(idx)})
        print(json.dumps(row), flush=True)


def run_table1(args):
    """--table1: the settings of the paper's Table I (CC-SN, one image per call, u = 128 ... 1024)
    on synthetic 12-bit spot frames: images/s of sequential single-frame calls (the paper's mode) and of one batched
    call.  Context for BASELINE.md section 1, not a target."""
    import torch
    from paper_2310_08770_b200 import Plan, RtSession
    rng = np.random.default_rng(7)
    for (H, W) in ((128, 256), (256, 256), (256, 512), (512, 512), (128, 1024)):
        y, x = np.mgrid[0:H, 0:W].astype(np.float64)
        spot = lambda sy, sx: 900.0 * np.exp(-((y - H / 2 - sy) ** 2 + (x - W / 2 - sx) ** 2) / (2 * 4.0 ** 2)) + 15.0
        ref = spot(0.0, 0.0).astype(np.float32)
        nb = 592
        sh = rng.uniform(-9, 9, size=(16, 2))
        fr16 = np.stack([rng.poisson(spot(a, b)) for a, b in sh]).clip(0, 4095).astype(np.uint16)
        fr = np.concatenate([fr16] * (nb // 16))
        for u in (128, 256, 512, 1024):
            plan = Plan(H, W, fr.dtype, u, ref, method="sn", epsilon=200.0)
            d = plan.device_frames(fr)
            out = tuple(torch.empty(nb, dtype=torch.float32, device="cuda") for _ in range(3))
            plan.track(d, nb, out=out)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            plan.track(d, nb, out=out)
            b.record()
            torch.cuda.synchronize()
            batched = nb / (a.elapsed_time(b) * 1e-3)
            plan.latency_probe(d, 20)
            lat = plan.latency_probe(d, 100)[3]
            torch.cuda.current_stream().synchronize()
            rt = RtSession(plan, 1000)           # the resident session kernel: no launch + synchronise per image
            try:
                rt.latency_probe(d.data_ptr(), 20)
                lat_rt = rt.latency_probe(d.data_ptr(), 100)[3]
            finally:
                rt.close()
            # the paper's real-time method like for like ("CC-SN algorithm implementations", with the
            # reference image updated after every image, Eq. (9); R19): cc_track(batch 1) + synchronise per image
            plan.enable_reference_update(0.02)
            plan.latency_probe(d, 20)
            lat_upd = plan.latency_probe(d, 100)[3]
            plan.enable_reference_update(0.0)
            print(json.dumps({"rows_x_cols": "%dx%d" % (H, W), "u": u, "method": "CC-SN",
                              "images_per_s_single_frame_calls_with_reference_update": 1e6 / float(np.median(lat_upd)),
                              "single_frame_latency_us_median_with_reference_update": float(np.median(lat_upd)),
                              "images_per_s_single_frame_calls": 1e6 / float(np.median(lat)),
                              "single_frame_latency_us_median": float(np.median(lat)),
                              "images_per_s_rt_session": 1e6 / float(np.median(lat_rt)),
                              "rt_session_latency_us_median": float(np.median(lat_rt)),
                              "images_per_s_batched": batched, "batch": nb}), flush=True)
            plan.close()
    # the paper's sustained real-time run (256x128, 12-bit, u = 256, 470 Hz, camera-limited): the whole
    # loop of Sec. III -- running reference image of Eq. (9) updated after every frame -- inside the resident session
    for (H, W) in ((128, 256), (256, 128)):
        y, x = np.mgrid[0:H, 0:W].astype(np.float64)
        spot = lambda sy, sx: 900.0 * np.exp(-((y - H / 2 - sy) ** 2 + (x - W / 2 - sx) ** 2) / (2 * 4.0 ** 2)) + 15.0
        sh = np.cumsum(rng.normal(0.0, 0.05, size=(400, 2)), axis=0)           # a slow random walk, a few pixels in total
        fr = np.stack([rng.poisson(spot(a, b)) for a, b in sh]).clip(0, 4095).astype(np.uint16)
        plan = Plan(H, W, fr.dtype, 256, spot(0.0, 0.0).astype(np.float32))
        plan.enable_reference_update(0.02)
        d = plan.device_frames(fr)
        torch.cuda.current_stream().synchronize()
        rt = RtSession(plan, 1000)
        try:
            rt.latency_probe(d.data_ptr(), 100)
            dx, dy, _, lat_rt = rt.latency_probe(d.data_ptr(), len(fr))
        finally:
            rt.close()
        plan.close()
        print(json.dumps({"rows_x_cols": "%dx%d" % (H, W), "u": 256, "method": "CC-U, running reference image (Eq. (9), a0 = 0.02)",
                          "mode": "real-time session, one image per call, reference updated after every image",
                          "images_per_s_rt_session": 1e6 / float(np.median(lat_rt)),
                          "rt_session_latency_us_median": float(np.median(lat_rt)),
                          "rt_session_latency_us_p99": float(np.percentile(lat_rt, 99)),
                          "median_error_px": float(np.median(np.hypot(dx - sh[:, 1], dy - sh[:, 0]))),
                          "paper": "470 Hz sustained, camera/USB3-limited, RTX 3080 Ti (PAPER.md:L210-216)"}), flush=True)


def run_tc_probe():
    """--tc-probe: the measured tensor-core experiment for the upsampled-DFT products (include/cc_bench.h,
    cc_tc_gemm_probe): accuracy of 1 x TF32 / 3 x TF32 against float64 on stage-1 operands of cfg 3
    (even Dirichlet weights x sums of rows of Q of a real frame) and the MMA rate with every SM busy."""
    from paper_2310_08770_b200 import tc_gemm_probe
    cfg = wl.config(3)
    H, W, u = cfg.H, cfg.W, cfg.upsample
    fr = wl.frames(cfg, [5])[0].astype(np.float64)
    ref = wl.reference(cfg).astype(np.float64)
    P = np.fft.fft2(fr - 50.0) * np.conj(np.fft.fft2(ref)) / (H * W)
    P[0, 0] = 0
    y0, _ = np.unravel_index(np.argmax(np.fft.ifft2(P).real), (H, W))
    Q = np.fft.ifft(P, axis=0)[:, 1:65]                                   # the 64 columns of one CTA

    def dirichlet(t):
        x = np.pi * np.asarray(t, dtype=np.float64) / H
        with np.errstate(divide="ignore", invalid="ignore"):
            v = np.sin(np.pi * t) * np.cos(x) / (H * np.sin(x))
        return np.where(np.abs(np.sin(x)) < 1e-15, 1.0, v)
    K = 192
    A, B = np.zeros((128, K)), np.zeros((K, 128))
    for j in range(H // 2 + 1):
        row = Q[(y0 + j) % H] if j in (0, H // 2) else Q[(y0 + j) % H] + Q[(y0 - j) % H]
        B[j, 0::2], B[j, 1::2] = row.real, row.imag
        dd = np.arange(76) / u
        A[:76, j] = dirichlet(dd - j) if j in (0, H // 2) else 0.5 * (dirichlet(dd - j) + dirichlet(dd + j))
    A32, B32 = A.astype(np.float32), B.astype(np.float32)
    Dref = A32.astype(np.float64) @ B32.astype(np.float64)
    scale = np.abs(Dref).max()
    out = {"experiment": "tcgen05.mma kind::tf32, 128x128xK products per SM, accumulator in tensor memory", "K": K,
           "fp32_host_sgemm_err": float(np.abs((A32 @ B32) - Dref).max() / scale)}
    for passes in (1, 3):
        D, sc, mc = tc_gemm_probe(A32, B32, passes=passes, iters=200)
        out["tf32_x%d" % passes] = {"max_err_rel_to_result_scale": float(np.abs(D - Dref).max() / scale),
                                    "staging_cycles_per_product": sc, "mma_cycles_per_product": mc}
    r2 = tc_gemm_probe(A32, B32, passes=3, iters=100, repeat=2)[2]
    r6 = tc_gemm_probe(A32, B32, passes=3, iters=100, repeat=6)[2]
    per_mma = (r6 - r2) / (4 * 3 * (K // 8))
    out["cycles_per_128x128x8_mma_all_sms_busy"] = per_mma
    out["tf32_tflops_chip"] = 2.0 * 128 * 128 * 8 / per_mma * 148 * NOMINAL_SM_MHZ * 1e6 / 1e12
    print(json.dumps(out))


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    n = args.ref_frames
    idx = wl.oracle_subset(cfg)[:n]
    fr = wl.frames(cfg, idx)
    ref = wl.reference(cfg)
    oracle.track(fr[:1], ref, cfg.upsample)
    for _ in range(args.warmup):
        oracle.track(fr, ref, cfg.upsample)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.track(fr, ref, cfg.upsample)
    dt = (time.perf_counter() - t0) / max(1, args.steps)
    val = len(idx) / dt
    sample = "first %d frames of the cfg-3 parity subset per step (bounded sample of the 10,000-frame batch)" % len(idx)
    line = {
        "impl": "reference", "metric": "frames_per_s", "value": val, "unit": "frames/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "H": cfg.H, "W": cfg.W, "pixel": cfg.dtype, "upsample": cfg.upsample,
                   "frames_per_step": len(idx)},
        "cpu_baseline": {"value": val, "unit": "frames/s", "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": "frames/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--batch", type=int, default=0, help="frames per step (default: the config's 10,000)")
    ap.add_argument("--ref-frames", type=int, default=256, help="frames per step of the --impl reference arm")
    ap.add_argument("--cpu-frames", type=int, default=2048, help="sample size of the cpu_baseline leg")
    ap.add_argument("--latency-frames", type=int, default=2000)
    ap.add_argument("--no-latency", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--table", action="store_true", help="per-config numbers for BASELINE.md section 3 and exit")
    ap.add_argument("--table1", action="store_true", help="the paper's Table I settings (context numbers) and exit")
    ap.add_argument("--tc-probe", action="store_true", help="tensor-core experiment for the upsampled-DFT products and exit")
    ap.add_argument("--phases", action="store_true", help="print the per-phase cycle breakdown of every config and exit")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "b200" else args.warmup

    if args.phases:
        run_phases()
        return
    if args.tc_probe:
        run_tc_probe()
        return
    if args.table:
        run_table(args)
        return
    if args.table1:
        run_table1(args)
        return
    cfg = wl.config(3)
    if args.impl == "reference":
        run_reference(args, cfg)
        return

    import torch
    import torch.distributed as dist
    from paper_2310_08770_b200 import Plan, fp32_peak_probe, fp32_tile_probe

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    B = args.batch or cfg.n_frames
    # every rank draws its own frames: same recipe, frame indices offset by rank (weak scaling)
    t_gen = time.perf_counter()
    uniq = min(B, cfg.n_frames)
    idx = (np.arange(uniq) + rank * 7919) % cfg.n_frames
    frames = wl.frames(cfg, idx)
    if uniq < B:
        frames = np.concatenate([frames] * ((B + uniq - 1) // uniq))[:B]
    ref = wl.reference(cfg)
    t_gen = time.perf_counter() - t_gen
    input_checksum = wl.checksum(frames)          # sum of all pixels + SHA-256 of frame 0 of the timed batch
    plan = Plan(cfg.H, cfg.W, frames.dtype, cfg.upsample, ref)
    info = plan.info()
    dfr = plan.device_frames(frames)
    out = (torch.empty(B, dtype=torch.float32, device="cuda"), torch.empty(B, dtype=torch.float32, device="cuda"),
           torch.empty(B, dtype=torch.float32, device="cuda"))

    for _ in range(args.warmup):
        plan.track(dfr, B, out=out)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    t0 = time.perf_counter()
    for a, b in ev:
        a.record()
        plan.track(dfr, B, out=out)
        b.record()
    barrier()
    wall = time.perf_counter() - t0
    clocks = sampler.stop() if rank == 0 else None
    kernel_ms = [a.elapsed_time(b) for a, b in ev]
    step_ms = ev[0][0].elapsed_time(ev[-1][1]) / args.steps
    t = torch.tensor([step_ms, float(np.mean(kernel_ms))], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    step_ms, kern_ms = float(t[0]), float(t[1])
    value = world * B / (step_ms * 1e-3)

    # ---- end to end: pinned host frames -> cc_track_host -> host results
    e2e = None
    if not args.no_e2e:
        hfr = torch.from_numpy(frames.view(np.uint8).reshape(B, -1)).pin_memory()
        hnp = hfr.numpy().view(frames.dtype).reshape(frames.shape)
        hdx = torch.empty(B, dtype=torch.float32).pin_memory()
        hdy = torch.empty(B, dtype=torch.float32).pin_memory()
        hpk = torch.empty(B, dtype=torch.float32).pin_memory()
        plan.track_host(hnp, hdx.numpy(), hdy.numpy(), hpk.numpy())
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            plan.track_host(hnp, hdx.numpy(), hdy.numpy(), hpk.numpy())
        barrier()
        dt = (time.perf_counter() - t0) / args.steps
        tt = torch.tensor([dt], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        e2e = {"value": world * B / float(tt[0]), "unit": "frames/s", "h2d_bytes_per_step": int(frames.nbytes),
               "d2h_bytes_per_step": int(3 * 4 * B), "ms_per_step": float(tt[0]) * 1e3,
               "api": "cc_track_host (pinned host frames in, host dx/dy/peak out)"}
        same = bool(np.array_equal(hdx.numpy(), out[0].cpu().numpy()) and np.array_equal(hdy.numpy(), out[1].cpu().numpy()))
        e2e["matches_device_path"] = same
        if not same:
            raise SystemExit("bench.py: cc_track_host returned displacements that differ from cc_track on the same frames")

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the (single) fused kernel
    flop = flops_per_frame(cfg.H, cfg.W, cfg.upsample)
    peak_tf = 148 * FP32_LANES_PER_SM * 2 * NOMINAL_SM_MHZ * 1e6 / 1e12
    achieved_tf = flop * B / (kern_ms * 1e-3) / 1e12
    probe_tf = fp32_peak_probe()
    tile_tf = fp32_tile_probe()
    hbm_gbs = None
    try:
        hbm_gbs = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
    except Exception:
        hbm_gbs = 6650.0
    t_alu = flop / (peak_tf * 1e12)
    t_hbm = (frames[0].nbytes + 12) / (hbm_gbs * 1e9)
    roofline = {
        "bound": "alu", "achieved": achieved_tf, "peak": peak_tf, "unit": "TFLOP/s", "frac": achieved_tf / peak_tf,
        "achieved_is": "ALGORITHMIC flop of SURVEY.md 8(d) (naive two-product upsampled DFT, 56.7 MFLOP per frame) / kernel time; "
                       "the kernel's even/odd formulation needs 21.3 MFLOP per frame: see frac_executed.  Stage 1 of it (10.0 MFLOP at 256x256, u = 100) "
                       "runs on the tensor cores as three TF32 passes where tensor_core_stage1 is 1, the rest on the FP32 pipes "
                       "the peak is derived from",
        "tensor_core_stage1": int(info.get("tensor_core_stage1", 0)),
        "tensor_core_tflops_issued": tensor_core_flops_per_frame(cfg.H, info) * B / (kern_ms * 1e-3) / 1e12,
        "frac_executed": executed_flops_per_frame(cfg.H, cfg.W, cfg.upsample) * B / (kern_ms * 1e-3) / 1e12 / peak_tf,
        "traffic": TRAFFIC_BYTES_PER_10K_LAUNCH * B / 10000.0, "traffic_source": TRAFFIC_SOURCE,
        "kernel": "cc_fused_kernel<256,256,CS=2>", "kernel_ms": kern_ms,
        "flop_per_frame": flop, "executed_flop_per_frame": executed_flops_per_frame(cfg.H, cfg.W, cfg.upsample),
        "executed_tflops": executed_flops_per_frame(cfg.H, cfg.W, cfg.upsample) * B / (kern_ms * 1e-3) / 1e12,
        "peak_source": "derived: 148 SM x 128 FP32 lanes x 2 flop x 1965 MHz (DESIGN.md); FFMA-loop probe measured %.1f TFLOP/s" % probe_tf,
        "ffma_probe_tflops": probe_tf, "ffma_register_tile_probe_tflops": tile_tf,
        "frac_of_register_tile_rate": achieved_tf / tile_tf,
        "roofline_frames_per_s": 1.0 / max(t_alu, t_hbm), "hbm_leg_frames_per_s": 1.0 / t_hbm,
        "hbm_achieved_gbs": (frames[0].nbytes + 12) * B / (kern_ms * 1e-3) / 1e9, "hbm_peak_gbs": hbm_gbs,
    }

    # ---- single-frame latency, the streaming configs (configs[1]: 128x128 u8 u=20; configs[3]: 512x512 u16 u=50):
    # sequential batch-1 frames, each timed on the host clock from hand-over to result-in-host-memory
    latency = None
    if not args.no_latency:
        from paper_2310_08770_b200 import RtSession
        latency = {"note": "per-frame host-clock latency, sequential frames, native timing loops of the C-ABI "
                           "(cc_track_latency_probe / cc_rt_latency_probe); frame resident in HBM unless stated"}
        stat = lambda l: {"median_us": float(np.median(l)), "p99_us": float(np.percentile(l, 99)), "max_us": float(l.max())}
        for ci in (2, 4):
            c2 = wl.config(ci)
            nlat = min(args.latency_frames, c2.n_frames)
            f2 = wl.frames(c2, np.arange(nlat))
            p2 = Plan(c2.H, c2.W, f2.dtype, c2.upsample, wl.reference(c2))
            d2 = p2.device_frames(f2)
            p2.latency_probe(d2, min(100, nlat))
            leg = {"workload": c2.name, "calls": nlat,
                   "cluster_size": p2.info()["lat_cluster_size"] or p2.info()["cluster_size"]}
            # (a) cc_track(batch = 1) + cudaStreamSynchronize per frame
            leg["cc_track_plus_stream_sync"] = stat(p2.latency_probe(d2, nlat)[3])
            # GPU-only time of the same launches (events around back-to-back calls)
            o2 = tuple(torch.empty(1, dtype=torch.float32, device="cuda") for _ in range(3))
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for i in range(200):
                p2.track(d2[i % nlat], 1, out=o2)
            b.record()
            torch.cuda.current_stream().synchronize()
            leg["gpu_only_us_per_call_back_to_back"] = a.elapsed_time(b) * 1e3 / 200
            # (b) real-time session: resident kernel, mailbox in mapped host memory
            rt = None
            try:
                rt = RtSession(p2, 1000)
                rt.latency_probe(d2.data_ptr(), min(100, nlat))
                rx, ry, _, lat_rt = rt.latency_probe(d2.data_ptr(), nlat)
                leg["rt_session"] = stat(lat_rt)
                if ci == 2:  # the paper's full real-time loop: running reference image, Eq. (9), inside the session
                    rt.close()
                    rt = None
                    p2.enable_reference_update(0.02)
                    rt = RtSession(p2, 1000)
                    rt.latency_probe(d2.data_ptr(), min(100, nlat))
                    leg["rt_session_with_reference_update"] = stat(rt.latency_probe(d2.data_ptr(), nlat)[3])
                    rt.close()
                    rt = None
                    p2.close()
                    p2 = Plan(c2.H, c2.W, f2.dtype, c2.upsample, wl.reference(c2))
                    rt = RtSession(p2, 1000)
                h2 = torch.from_numpy(f2.view(np.uint8).reshape(nlat, -1)).pin_memory()
                rt.latency_probe(h2.data_ptr(), min(100, nlat))
                leg["rt_session_frame_in_pinned_host_memory"] = stat(rt.latency_probe(h2.data_ptr(), nlat)[3])
                bx, by, _ = [t.cpu().numpy() for t in p2.track(d2)]
                leg["rt_matches_cc_track"] = bool(np.array_equal(rx, bx) and np.array_equal(ry, by))
            except Exception as ex:  # e.g. under a profiler that serialises launches the resident kernel cannot be served
                leg["rt_session_error"] = str(ex)[:200]
            finally:
                if rt is not None:
                    rt.close()
            latency["cfg%d" % ci] = leg
            p2.close()

    # ---- CPU oracle beside it
    cpu = None
    if not args.no_cpu:
        v, cores, n, dt = oracle_rate(cfg, args.cpu_frames)
        cpu = {"value": v, "unit": "frames/s", "cores": cores, "kind": "oracle",
               "sample": "first %d frames of the 10,000-frame cfg-3 batch, %.1f s wall" % (n, dt)}

    line = {
        "metric": "frames_per_s", "value": value, "unit": "frames/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": step_ms, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": cfg.name, "H": cfg.H, "W": cfg.W, "pixel": cfg.dtype, "upsample": cfg.upsample,
                   "frames_per_step_per_gpu": B, "unique_frames": int(uniq), "parallelism": "replicas x%d" % world,
                   "l2": "inputs (%.2f GB per step) larger than L2" % (frames.nbytes / 1e9),
                   "cluster_size": info["cluster_size"], "clusters_resident": info["max_clusters"],
                   "threads": info["threads"], "smem_bytes": info["smem_bytes"], "gen_s": round(t_gen, 1),
                   "input_checksum": input_checksum},
        "clocks": clocks, "e2e": e2e, "gpu_launches": args.steps, "roofline": roofline, "cpu_baseline": cpu,
        "latency": latency, "wall_s_timed_region": wall,
    }
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
