"""Build the C-ABI CUDA library (in-tree): one nvcc invocation per kernel
variant of csrc/cc_variant_list.h plus csrc/cc_api.cu, linked into
paper_2310_08770_b200/libcc_b200.so.  sm_100a only.

    python -m paper_2310_08770_b200.build [--force]
"""
from __future__ import annotations

import os
import re
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libcc_b200.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
         "-Xcompiler", "-fPIC", "-Xptxas", "-v"]
_CCV = re.compile(r"^CCV\(([^)]*)\)", re.M)
_KEYS = ["NAME", "H", "W", "CS", "PIX", "NT", "TM1", "TN1", "TM2", "TN2", "SG", "BK1", "G2", "R2", "KS2", "NSTG", "PFD", "KS1", "TC"]


def variants():
    txt = open(os.path.join(CSRC, "cc_variant_list.h")).read()
    out = []
    for m in _CCV.finditer(txt):
        vals = [v.strip() for v in m.group(1).split(",")]
        out.append(dict(zip(_KEYS, vals)))
    return out


def _newest_src():
    """Newest of the sources, the public headers (enums and struct layouts the binding mirrors) and this file (FLAGS)."""
    inc = os.path.join(os.path.dirname(HERE), "include")
    files = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.abspath(__file__)]
    files += [os.path.join(inc, f) for f in os.listdir(inc) if f.endswith(".h")]
    return max(os.path.getmtime(f) for f in files)


def _run(cmd, log):
    r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    with open(log, "w") as fh:
        fh.write(" ".join(cmd) + "\n" + r.stdout)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed: %s\n%s" % (" ".join(cmd), r.stdout[-4000:]))
    return r.stdout


def build(force: bool = False, verbose: bool = False, fuzz: bool = False) -> str:
    """fuzz=True builds libcc_b200_fuzz.so: the same library with -DCC_FUZZ (random delays before every
    synchronisation point; the race check of profiles/sanitizer_r2.md).  Load it with CC_B200_LIB=<path>."""
    global OBJ, LIB
    if fuzz:
        return _build_fuzz(force, verbose)
    return _build(force, verbose, [])


def _build_fuzz(force, verbose):
    global OBJ, LIB
    obj0, lib0 = OBJ, LIB
    OBJ, LIB = os.path.join(HERE, "build_fuzz"), os.path.join(HERE, "libcc_b200_fuzz.so")
    try:
        return _build(force, verbose, ["-DCC_FUZZ"])
    finally:
        OBJ, LIB = obj0, lib0


def _build(force, verbose, extra):
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= _newest_src():
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    jobs = []
    for v in variants():
        obj = os.path.join(OBJ, "v_%s.o" % v["NAME"])
        cmd = [NVCC] + FLAGS + extra + ["-c", os.path.join(CSRC, "cc_variant.cu"), "-o", obj] + \
              ["-DCCV_%s=%s" % (k, v[k]) for k in _KEYS]
        jobs.append((cmd, obj))
    for src in ("cc_api", "cc_refupdate", "cc_tc_probe"):
        o = os.path.join(OBJ, src + ".o")
        jobs.append(([NVCC] + FLAGS + extra + ["-c", os.path.join(CSRC, src + ".cu"), "-o", o], o))
    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as ex:
        outs = list(ex.map(lambda j: _run(j[0], j[1] + ".log"), jobs))
    if verbose:
        for o in outs:
            for line in o.splitlines():
                if "registers" in line or "spill" in line or "warning" in line:
                    print(line)
    tmp = LIB + ".tmp.%d" % os.getpid()
    _run([NVCC, "-shared", "-o", tmp] + [j[1] for j in jobs] + ["-gencode", "arch=compute_100a,code=sm_100a"],
         os.path.join(OBJ, "link.log"))
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True, fuzz="--fuzz" in sys.argv))
