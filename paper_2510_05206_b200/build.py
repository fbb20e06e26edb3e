"""Build libpmforce.so (the C-ABI library of include/pmforce.h) in-tree with nvcc for sm_100a.

    python -m paper_2510_05206_b200.build [--force] [--verbose] [--es-widths 7 --suffix _dev]

One object per translation unit (compiled in parallel), linked against cuFFT.  The objects go to
``paper_2510_05206_b200/build/`` and the library to ``paper_2510_05206_b200/libpmforce.so``; both are
git-ignored but travel to the GPU box with the repo snapshot.  nvcc cross-compiles without a GPU.
"""
from __future__ import annotations

import argparse
import os
import shutil
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
CSRC = os.path.join(PKG, "csrc")
OBJ = os.path.join(PKG, "build")
LIB = os.path.join(PKG, "libpmforce.so")

ES_WIDTHS = (4, 5, 6, 7, 8)  # keep in step with ES_WIDTHS in csrc/nufft_dispatch.cu
SOURCES = ["pm_ctx.cu", "pm_bin.cu", "pm_scatter.cu", "pm_gather.cu", "pm_jvp.cu", "pm_kspace.cu", "pm_xfft.cu",
           "pm_stencil.cu", "pm_step.cu", "pm_power.cu", "pm_resample.cu", "pm_microbench.cu", "pm_noalloc.cu", "pm_api.cu",
           "nufft_dispatch.cu"]
HEADERS = ["pm_internal.cuh", "pm_mesh_kernels.cuh", os.path.join(ROOT, "include", "pmforce.h")]

NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "--expt-relaxed-constexpr"]


def _nvcc() -> str:
    cand = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(cand):
        raise RuntimeError("nvcc not found (needed to build libpmforce.so)")
    return cand


def _cuda_lib_dir(nvcc: str) -> str:
    return os.path.join(os.path.dirname(os.path.dirname(os.path.realpath(nvcc))), "lib64")


def _units(es_widths=ES_WIDTHS, obj=OBJ):
    units = []
    # widest kernels first: they take the longest to compile and should not start last
    for w in sorted(es_widths, reverse=True):
        for part in (2, 1, 0):
            units.append((os.path.join(CSRC, "nufft_mesh.cu"), os.path.join(obj, f"nufft_mesh_w{w}_p{part}.o"),
                          [f"-DES_W={w}", f"-DES_PART={part}"]))
    partial = tuple(es_widths) != ES_WIDTHS
    for s in SOURCES:
        extra = ["-DPMF_ES_WIDTHS(X)=" + " ".join(f"X({w})" for w in es_widths)] if partial and s == "nufft_dispatch.cu" else []
        units.append((os.path.join(CSRC, s), os.path.join(obj, s[:-3] + ".o"), extra))
    return units


def _stale(target: str, deps) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, es_widths=ES_WIDTHS, suffix: str = "") -> str:
    """Compile whatever is out of date and return the path of libpmforce.so.

    ``es_widths`` / ``suffix`` are for development only: a library with fewer ES-kernel widths (they take most of
    the build time) goes to ``libpmforce<suffix>.so`` with its own object directory and is never what the package
    loads; the product is the default build."""
    if tuple(es_widths) != ES_WIDTHS and not suffix:
        raise ValueError("a partial build needs a --suffix: libpmforce.so always holds every width")
    nvcc = _nvcc()
    OBJ = os.path.join(PKG, "build" + suffix)
    LIB = os.path.join(PKG, f"libpmforce{suffix}.so")
    os.makedirs(OBJ, exist_ok=True)
    hdrs = [h if os.path.isabs(h) else os.path.join(CSRC, h) for h in HEADERS]
    jobs = []
    for src, obj, extra in _units(es_widths, OBJ):
        if force or _stale(obj, [src] + hdrs):
            jobs.append([nvcc, *NVCC_FLAGS, *extra, "-Xptxas", "-v", "-c", src, "-o", obj])

    def run(cmd):
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + r.stdout + r.stderr)
        if verbose:
            sys.stderr.write(" ".join(cmd) + "\n" + r.stderr)
        return r.stderr

    logs = []
    if jobs:
        with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 4)) as ex:
            logs = list(ex.map(run, jobs))
        with open(os.path.join(OBJ, "ptxas.log"), "a") as f:
            f.write("\n".join(logs))
    objs = [u[1] for u in _units(es_widths, OBJ)]
    if force or jobs or _stale(LIB, objs):
        libdir = _cuda_lib_dir(nvcc)
        run([nvcc, "-shared", "-o", LIB, *objs, "-gencode", "arch=compute_100a,code=sm_100a",
             "-L" + libdir, "-lcufft", "-Xlinker", "-rpath," + libdir])
    return LIB


def main(argv=None) -> int:
    ap = argparse.ArgumentParser(description=__doc__)
    ap.add_argument("--force", action="store_true")
    ap.add_argument("--verbose", action="store_true")
    ap.add_argument("--es-widths", default="", help="development: comma-separated subset of the ES-kernel widths")
    ap.add_argument("--suffix", default="", help="development: build libpmforce<suffix>.so in build<suffix>/")
    a = ap.parse_args(argv)
    widths = tuple(int(w) for w in a.es_widths.split(",")) if a.es_widths else ES_WIDTHS
    print(build(force=a.force, verbose=a.verbose, es_widths=widths, suffix=a.suffix))
    return 0


if __name__ == "__main__":
    raise SystemExit(main())
