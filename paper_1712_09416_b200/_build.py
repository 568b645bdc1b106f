"""In-tree builds of the package's native parts (no JIT cache: the built .so files travel with the repo).

* ``gen/libtpcgen.so``      -- gcc, the seeded workload generator (host only)
* ``csrc/libtpctrack.so``   -- nvcc for sm_100a, the tracker behind the C ABI of ``include/tpctrack.h``

A target is rebuilt when it is missing or older than one of its sources.
"""
from __future__ import annotations

import os
import shutil
import subprocess
from pathlib import Path

PKG = Path(__file__).resolve().parent
ROOT = PKG.parent

NVCC_ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
# -fmad=false: decision-critical float32 expressions must round like the strict-float oracle mode
# (DESIGN.md "Parity protocol"); division and sqrt stay IEEE (-prec-div/-prec-sqrt default true, no -ftz).
NVCC_FLAGS = ["-O3", "-std=c++17", "-lineinfo", "-fmad=false", "-prec-div=true", "-prec-sqrt=true", "-ftz=false",
              "-Xcompiler", "-fPIC", "-shared"]


def _stale(target: Path, sources) -> bool:
    if not target.exists():
        return True
    t = target.stat().st_mtime
    return any(Path(s).stat().st_mtime > t for s in sources)


def _run(cmd):
    r = subprocess.run([str(c) for c in cmd], capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("build failed: %s\n%s\n%s" % (" ".join(map(str, cmd)), r.stdout, r.stderr))
    return r.stdout + r.stderr


def build_gen(force: bool = False) -> Path:
    src = PKG / "gen" / "tpcgen.c"
    out = PKG / "gen" / "libtpcgen.so"
    if force or _stale(out, [src]):
        _run(["gcc", "-O2", "-std=c11", "-shared", "-fPIC", "-o", out, src, "-lm"])
    return out


def nvcc_path() -> str:
    p = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(p):
        raise RuntimeError("nvcc not found: cannot build libtpctrack.so")
    return p


def tracker_sources():
    c = PKG / "csrc"
    return sorted(c.glob("*.cu")), sorted(c.glob("*.cuh")) + sorted(c.glob("*.h")) + [ROOT / "include" / "tpctrack.h"]


def build_tracker(force: bool = False, verbose: bool = False) -> Path:
    cus, hdrs = tracker_sources()
    out = PKG / "csrc" / "libtpctrack.so"
    if force or _stale(out, list(cus) + list(hdrs)):
        cmd = [nvcc_path(), *NVCC_ARCH, *NVCC_FLAGS, "-I", ROOT / "include", "-I", PKG / "csrc"]
        if verbose:
            cmd += ["-Xptxas", "-v"]
        cmd += ["-o", out, *cus, "-lcudart"]
        log = _run(cmd)
        if verbose:
            print(log)
    return out


def build_all(force: bool = False) -> None:
    build_gen(force)
    build_tracker(force)
