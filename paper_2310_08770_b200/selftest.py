"""Self-test of libcc_b200.so without the CPU oracle: every compiled kernel variant is launched on a small batch in
every mode (batched, single-frame cluster variant, Eq. (9) update, Eq. (8) accumulation, real-time session,
cc_track_host) and checked for what must hold by construction -- integer circular shifts of the reference come back
exactly (periodic boundaries) and two runs give identical bits.

    python -m paper_2310_08770_b200.selftest [--only f256] [--upsample 8] [--no-session] [--dump out.npz]
    python -m paper_2310_08770_b200.selftest --compare a.npz b.npz

Race check without compute-sanitizer (closed on the development pool; profiles/sanitizer_r2.md): `--dump` also runs a
batch of NOISY frames per shape (near-ties and rounding-level differences make the results sensitive to any change in
the data the kernel reads) and stores every output; the dump of the plain library must equal, bit for bit, the dumps
of repeated runs of the schedule-fuzzing build (CC_B200_LIB=.../libcc_b200_fuzz.so, build.py --fuzz: random delays
before every synchronisation point).
"""
from __future__ import annotations

import argparse
import sys

import numpy as np


def _shapes():
    from . import build as cuda_build
    seen = []
    for v in cuda_build.variants():
        key = (int(v["H"]), int(v["W"]), np.uint8 if v["PIX"] == "uint8_t" else np.uint16)
        if key not in seen:
            seen.append(key)
    return seen


def run(only: str = "", upsample: int = 8, session: bool = True, verbose: bool = True, dump: dict | None = None) -> int:
    import torch
    from . import Plan, RtSession
    n_checked = 0
    for H, W, dt in _shapes():
        name = "f%dx%d_%s" % (H, W, np.dtype(dt).name)
        if only and only not in name:
            continue
        rng = np.random.default_rng(H * 31 + W)
        hi = 200 if dt == np.uint8 else 3000
        ref = rng.integers(0, hi, size=(H, W)).astype(dt)
        shifts = [(0, 0), (3, W - 5), (H - 2, 1), (H // 2, W // 2)]
        fr = np.stack([np.roll(ref, s, axis=(0, 1)) for s in shifts])
        want_y = np.array([a - H if 2 * a >= H else a for a, _ in shifts], np.float32)
        want_x = np.array([b - W if 2 * b >= W else b for _, b in shifts], np.float32)
        plan = Plan(H, W, dt, upsample, ref.astype(np.float32))
        info = plan.info()
        d = plan.device_frames(fr)
        # batched call on the throughput variant (more frames than the cluster variant takes)
        reps = max(1, (info["lat_max_clusters"] + len(fr)) // len(fr))
        big = plan.device_frames(np.concatenate([fr] * (reps + 1)))
        a = [t.cpu().numpy() for t in plan.track(big)]
        b = [t.cpu().numpy() for t in plan.track(big)]
        assert all(np.array_equal(x, y) for x, y in zip(a, b)), name + ": batched run not deterministic"
        assert np.array_equal(a[0][:4], want_x) and np.array_equal(a[1][:4], want_y), name + ": batched shifts wrong"
        # single-frame calls (the cluster variant where the shape has one)
        for i in range(len(fr)):
            x, y, _ = plan.track(d[i], 1)
            assert (x.item(), y.item()) == (want_x[i], want_y[i]), name + ": single-frame shift wrong"
        # host path, two chunks
        plan.set_host_chunk(2)
        hx, hy, _ = plan.track_host(fr)
        assert np.array_equal(hx, want_x) and np.array_equal(hy, want_y), name + ": host path wrong"
        torch.cuda.synchronize()
        # Eq. (8): accumulate + reference update; Eq. (9): running reference (exact shifts leave it in place)
        ax, ay, _ = plan.track_accumulate(d)
        plan.update_reference_from_accumulator()
        assert np.array_equal(ax.cpu().numpy(), want_x), name + ": accumulate pass wrong"
        plan.enable_reference_update(0.25)
        rx, ry, _ = [t.cpu().numpy() for t in plan.track(d)]
        assert np.array_equal(rx, want_x) and np.array_equal(ry, want_y), name + ": running-reference pass wrong"
        plan.enable_reference_update(0.0)
        if session:
            torch.cuda.current_stream().synchronize()
            rt = RtSession(plan, idle_timeout_ms=20000)
            try:
                for i in range(len(fr)):
                    x, y, _ = rt.track(d.data_ptr() + i * fr[0].nbytes)
                    assert (x, y) == (want_x[i], want_y[i]), name + ": session shift wrong"
            finally:
                rt.close()
        if dump is not None:  # noisy frames, every mode: the outputs go into the dump
            noisy = np.clip(np.stack([np.roll(ref, sft, axis=(0, 1)).astype(np.int64) for sft in shifts * 3])
                            + rng.integers(-hi // 8, hi // 8, size=(12, H, W)), 0, np.iinfo(dt).max).astype(dt)
            dn = plan.device_frames(noisy)
            bign = plan.device_frames(np.concatenate([noisy] * (reps + 1)))
            dump[name + ".batched"] = np.stack([t.cpu().numpy() for t in plan.track(bign)])
            dump[name + ".single"] = np.array([[t.item() for t in plan.track(dn[i], 1)] for i in range(len(noisy))], np.float32)
            dump[name + ".accumulate"] = np.stack([t.cpu().numpy() for t in plan.track_accumulate(dn)])
            plan.update_reference_from_accumulator()
            plan.enable_reference_update(0.1)
            dump[name + ".running"] = np.stack([t.cpu().numpy() for t in plan.track(dn)])
            dump[name + ".spectrum"] = plan.reference_spectrum()
            plan.enable_reference_update(0.0)
        plan.close()
        n_checked += 1
        if verbose:
            print("%-22s ok  (cluster sizes %d / %d, %d B smem)" % (name, info["cluster_size"], info["lat_cluster_size"],
                                                                   info["smem_bytes"]), flush=True)
    # CC-SN ingest path (fp64 pixel transform) on one shape
    if not only or "f64" in only:
        rng = np.random.default_rng(5)
        ref = rng.integers(1, 3000, size=(64, 64)).astype(np.uint16)
        fr = np.stack([np.roll(ref, s, axis=(0, 1)) for s in [(0, 0), (5, 60)]])
        plan = Plan(64, 64, np.uint16, upsample, ref.astype(np.float32), method="sn", epsilon=200.0)
        x, y, _ = [t.cpu().numpy() for t in plan.track(plan.device_frames(fr))]
        assert np.array_equal(x, [0.0, -4.0]) and np.array_equal(y, [0.0, 5.0]), "CC-SN shifts wrong"
        plan.close()
        n_checked += 1
    torch.cuda.synchronize()
    if verbose:
        print("selftest ok: %d shape(s)" % n_checked)
    return n_checked


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--only", default="", help="substring of the shape name, e.g. f256x256_uint16")
    ap.add_argument("--upsample", type=int, default=8)
    ap.add_argument("--no-session", action="store_true", help="skip the resident real-time session kernel")
    ap.add_argument("--dump", default="", help="also run noisy frames in every mode and store all outputs in this .npz")
    ap.add_argument("--compare", nargs=2, default=None, help="compare two dumps bit for bit and exit")
    args = ap.parse_args(argv)
    if args.compare:
        a, b = np.load(args.compare[0]), np.load(args.compare[1])
        assert sorted(a.files) == sorted(b.files), "different sets of outputs"
        bad = [k for k in a.files if not np.array_equal(a[k], b[k], equal_nan=True)]
        print("%d arrays compared, %d differ%s" % (len(a.files), len(bad), (": " + ", ".join(bad)) if bad else ""))
        sys.exit(1 if bad else 0)
    dump = {} if args.dump else None
    run(args.only, args.upsample, not args.no_session, dump=dump)
    if args.dump:
        np.savez(args.dump, **dump)


if __name__ == "__main__":
    main(sys.argv[1:])
