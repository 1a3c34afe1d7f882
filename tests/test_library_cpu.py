"""CPU-side checks of the C-ABI library: it loads, exports every symbol that
include/cc.h declares, and validates arguments before touching a device."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2310_08770_b200 import build as cuda_build
    from paper_2310_08770_b200 import binding
    cuda_build.build()
    return binding.load_library()


def _declared_functions():
    """Every function declared by include/*.h (cc.h: the tracking interface; cc_bench.h: measurement aids)."""
    names = set()
    inc = os.path.join(ROOT, "include")
    for f in sorted(os.listdir(inc)):
        if f.endswith(".h"):
            txt = re.sub(r"/\*.*?\*/", "", open(os.path.join(inc, f)).read(), flags=re.S)
            names |= set(re.findall(r"\b(cc_[a-z0-9_]+)\s*\(", txt))
    return sorted(names)


def test_header_symbols_exported(lib):
    names = _declared_functions()
    assert {"cc_plan_create", "cc_track", "cc_plan_destroy"} <= set(names)
    for n in names:
        assert hasattr(lib, n), "libcc_b200.so does not export %s" % n


def test_binding_lists_every_header_function():
    from paper_2310_08770_b200 import binding
    assert sorted(binding.EXPORTS) == _declared_functions()


def test_status_strings(lib):
    assert lib.cc_status_string(0) == b"CC_OK"
    assert lib.cc_status_string(2) == b"CC_ERR_UNSUPPORTED"
    assert lib.cc_status_string(5) == b"CC_ERR_ARCH"


def test_argument_validation_needs_no_device(lib):
    h = ctypes.c_void_p()
    ref = np.zeros((64, 64), np.float32)
    rp = ref.ctypes.data_as(ctypes.c_void_p)
    assert lib.cc_plan_create(None, 64, 64, 1, 10, rp) == 1          # NULL out
    assert lib.cc_plan_create(ctypes.byref(h), 64, 64, 1, 10, None) == 1  # NULL reference
    assert lib.cc_plan_create(ctypes.byref(h), 0, 64, 1, 10, rp) == 1
    assert lib.cc_plan_create(ctypes.byref(h), 64, 64, 1, 0, rp) == 1     # upsample < 1
    assert lib.cc_plan_create(ctypes.byref(h), 64, 64, 7, 10, rp) == 1    # bad dtype
    assert lib.cc_plan_create(ctypes.byref(h), 48, 64, 1, 10, rp) == 2    # not a power of two
    assert lib.cc_plan_create(ctypes.byref(h), 2048, 64, 1, 10, rp) == 2  # outside 64..1024
    assert b"power" in lib.cc_last_error()
    assert lib.cc_track(None, None, 4, None, None, None, None) == 1
    assert lib.cc_plan_destroy(None) == 0
    assert lib.cc_plan_info(None, None) == 1
    assert lib.cc_rt_open(None, 0, ctypes.byref(h)) == 1
    assert lib.cc_plan_create_weighted(ctypes.byref(h), 64, 64, 1, 10, rp, 5, ctypes.c_float(1.0)) == 1   # bad method
    assert lib.cc_plan_create_weighted(ctypes.byref(h), 64, 64, 1, 10, rp, 1, ctypes.c_float(-2.0)) == 1  # epsilon < 0
    assert lib.cc_rt_submit(None, None) == 1 and lib.cc_rt_wait(None, None, None, None) == 1
    assert lib.cc_rt_close(None) == 0
    assert lib.cc_plan_enable_reference_update(None, 0.1) == 1
    assert lib.cc_plan_get_reference_spectrum(None, None) == 1
    assert lib.cc_track_accumulate(None, None, 4, None, None, None, None) == 1
    assert lib.cc_plan_update_reference_from_accumulator(None, None) == 1
    assert lib.cc_drift_correct(None, None, -1, 0.1, 0.0, None, None, None, None) == 1
    assert lib.cc_drift_correct(None, None, 4, 0.1, 0.0, None, None, None, None) == 1
    assert lib.cc_track_latency_probe(None, None, 1, None, None, None, None, None) == 1
    assert lib.cc_plan_set_host_chunk(None, 4) == 1


def test_no_device_is_a_loud_error(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    h = ctypes.c_void_p()
    ref = np.zeros((64, 64), np.float32)
    st = lib.cc_plan_create(ctypes.byref(h), 64, 64, 1, 10, ref.ctypes.data_as(ctypes.c_void_p))
    assert st == 5 and not h.value   # CC_ERR_ARCH: there is no CPU fallback
    from paper_2310_08770_b200 import Plan
    with pytest.raises(RuntimeError):
        Plan(64, 64, np.uint16, 10, ref)


def test_variant_list_covers_all_config_shapes():
    from paper_2310_08770_b200 import build as cuda_build
    from paper_2310_08770_b200 import workloads as wl
    have = {(int(v["H"]), int(v["W"]), v["PIX"]) for v in cuda_build.variants()}
    for i in range(1, 6):
        c = wl.config(i)
        assert (c.H, c.W, c.dtype + "_t") in have


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2310_08770_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                s = open(os.path.join(dp, f)).read()
                assert "import oracle" not in s and "cc_oracle" not in s, f


def test_workloads_are_seeded_and_subsettable():
    from paper_2310_08770_b200 import workloads as wl
    c = wl.config(1)
    a = wl.frames(c, [3, 10, 500])
    b = wl.frames(c, [500, 3])
    assert np.array_equal(a[0], b[1]) and np.array_equal(a[2], b[0])
    assert a.dtype == np.uint16 and a.shape == (3, 64, 64)
    assert wl.frames(wl.config(2), [0]).dtype == np.uint8
