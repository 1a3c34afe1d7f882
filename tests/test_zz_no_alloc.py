"""cc_track_static (include/cc.h): the allocation-free entry point, whose global spectrum scratch is a file-scope
`static __device__` array inside the library, against the existing path cc_track on the same inputs.

Collected last on purpose (the suite runs with `pytest -x`): a failure here hides no other test.  Passes alone in a
fresh process and after the other GPU tests: the static array keeps the previous call's contents and nothing in it has
to start at zero.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL_PX = 2e-3       # the bar of tests/test_parity_gpu.py (north_star): same 1/u grid point
TOL_PEAK = 1e-4     # relative


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2310_08770_b200 import build as cuda_build
    cuda_build.build()
    import paper_2310_08770_b200 as pkg
    pkg.load_library()
    return pkg


def _outs(torch, n):
    return tuple(torch.full((n,), float("nan"), dtype=torch.float32, device="cuda") for _ in range(3))


def _close(a, b, label):
    for name, x, y in zip(("dx", "dy"), a[:2], b[:2]):
        x, y = x.cpu().numpy(), y.cpu().numpy()
        assert np.all(np.isfinite(x)), "%s: %s not written" % (label, name)
        assert np.max(np.abs(x - y)) <= TOL_PX, "%s: %s differs from cc_track: %s vs %s" % (label, name, x, y)
    pa, pb = a[2].cpu().numpy(), b[2].cpu().numpy()
    assert np.all(np.abs(pa - pb) <= TOL_PEAK * np.abs(pb)), "%s: peak differs from cc_track: %s vs %s" % (label, pa, pb)


def test_static_scratch_matches_cc_track_two_calls_in_a_row(gpu):
    """1024 x 1024 (the shape whose spectrum block lives in global scratch): two calls in a row on different frames,
    not synchronised in between (same stream: serialised), each equal to cc_track's result for its frames; then a
    single-frame call.  Device memory in use does not change across the calls."""
    import torch
    from paper_2310_08770_b200 import workloads as wl
    cfg = wl.config(5)
    fr = wl.frames(cfg, np.arange(5))
    plan = gpu.Plan(cfg.H, cfg.W, fr.dtype, cfg.upsample, wl.reference(cfg))
    assert plan.info()["scratch_bytes"] > 0, "this shape is expected to use global spectrum scratch"
    d = plan.device_frames(fr)
    a, b, c = d[0:2], d[2:4], d[4:5]
    want = [plan.track(x, x.shape[0]) for x in (a, b, c)]           # existing path (plan-owned cudaMalloc'ed scratch)
    oa, ob, oc = _outs(torch, 2), _outs(torch, 2), _outs(torch, 1)
    plan.track_static(a, oa)                                        # first call on the device: resolves the array's address
    oa = _outs(torch, 2)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    plan.track_static(a, oa)
    plan.track_static(b, ob)                                        # second call in a row: the array holds a's spectra
    plan.track_static(c, oc)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0, "device memory in use changed across cc_track_static calls"
    _close(oa, want[0], "first call")
    _close(ob, want[1], "second call")
    _close(oc, want[2], "single frame")
    # same kernel, same arithmetic: the results are in fact bit-identical
    for got, ref in zip((oa, ob, oc), want):
        for x, y in zip(got, ref):
            assert torch.equal(x, y)
    plan.close()


def test_static_scratch_rejects_what_does_not_fit(gpu):
    """Three 1024 x 1024 frames in flight need 12 MiB of spectrum scratch; the array holds 8 MiB."""
    import torch
    from paper_2310_08770_b200 import workloads as wl
    from paper_2310_08770_b200.binding import CcError
    cfg = wl.config(5)
    fr = wl.frames(cfg, np.arange(3))
    plan = gpu.Plan(cfg.H, cfg.W, fr.dtype, cfg.upsample, wl.reference(cfg))
    d = plan.device_frames(fr)
    with pytest.raises(CcError) as ei:
        plan.track_static(d, _outs(torch, 3))
    assert ei.value.status == 2 and "largest batch is 2" in str(ei.value), str(ei.value)
    # a plan that rewrites its reference (Eq. (9)) is refused as well
    plan.enable_reference_update(0.05)
    with pytest.raises(CcError) as ei:
        plan.track_static(d[0:1], _outs(torch, 1))
    assert ei.value.status == 2
    plan.close()


def test_static_entry_on_a_shape_without_scratch(gpu):
    """128 x 128 keeps its spectrum in shared memory: no scratch, any batch, same results as cc_track."""
    import torch
    from paper_2310_08770_b200 import workloads as wl
    cfg = wl.config(2)
    fr = wl.frames(cfg, np.arange(300))
    plan = gpu.Plan(cfg.H, cfg.W, fr.dtype, cfg.upsample, fr[0].astype(np.float32))
    d = plan.device_frames(fr)
    for n in (1, 300):
        want = plan.track(d[:n], n)
        got = plan.track_static(d[:n], _outs(torch, n))
        torch.cuda.synchronize()
        _close(got, want, "128x128 batch %d" % n)
    plan.close()
