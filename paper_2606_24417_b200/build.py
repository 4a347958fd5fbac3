"""Build the CUDA libraries in-tree (sm_100a):
  csrc/*.cu except sbf_bench*.cu -> paper_2606_24417_b200/libsbf_b200.so        the product (include/sbf.h)
  csrc/sbf_bench*.cu             -> paper_2606_24417_b200/libsbf_bench_b200.so  measurement / test hooks (include/sbf_bench.h)

nvcc cross-compiles without a GPU.  The translation units are compiled in parallel; an object is
rebuilt only when its source or a header is newer.  `python -m paper_2606_24417_b200.build [--force]`.
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
OBJDIR = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libsbf_b200.so")
BENCH_LIB = os.path.join(HERE, "libsbf_bench_b200.so")

SWEEP_S = (24, 26, 28, 30, 31)   # BASELINE.json configs[4]
SWEEP_M = (12, 14, 16, 18, 20)

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-std=c++17", "-O3", "-lineinfo",
    "-Xcompiler", "-fPIC",
    "-I", INCLUDE,
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _headers():
    return glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(CSRC, "*.h")) + \
        glob.glob(os.path.join(INCLUDE, "*.h"))


def _is_bench(src: str) -> bool:
    return os.path.basename(src).startswith("sbf_bench")


def build(force: bool = False, verbose: bool = False, extra_flags=(), lib: str = LIB, objdir: str = OBJDIR) -> str:
    """Both libraries; returns the product library's path.  extra_flags / lib / objdir: build a variant (-D switches) of
    the product library next to it (the bench library is then left alone)."""
    out = _build(False, force, verbose, extra_flags, lib, objdir)
    if lib == LIB:
        _build(True, force, verbose, (), BENCH_LIB, objdir)
    return out


def _build(bench: bool, force: bool, verbose: bool, extra_flags, lib: str, objdir: str) -> str:
    srcs = sorted(s for s in glob.glob(os.path.join(CSRC, "*.cu")) if _is_bench(s) == bench)
    if not srcs:
        raise RuntimeError("no CUDA sources under %s" % CSRC)
    hdr_time = max(os.path.getmtime(h) for h in _headers())
    # a library newer than every source and header is current even when the objects are gone (they do not travel to the
    # GPU box: .gpurunignore): nothing to do
    if not force and os.path.exists(lib) and os.path.getmtime(lib) >= max([hdr_time] + [os.path.getmtime(x) for x in srcs]) \
            and os.path.getmtime(lib) >= os.path.getmtime(os.path.abspath(__file__)):
        return lib
    os.makedirs(objdir, exist_ok=True)
    nvcc = _nvcc()
    jobs = []
    objs = []
    units = []  # (source, object, extra -D flags)
    for src in srcs:
        base = os.path.basename(src)[:-3]
        if base == "sbf_inst_sweep":
            # one object per (s, m) pair of BASELINE config 5, five H instances each (skipped in tuning builds)
            if "-DSBF_ONLY_DEFAULT" not in extra_flags:
                for s_ in SWEEP_S:
                    for m_ in SWEEP_M:
                        units.append((src, os.path.join(objdir, "%s_s%d_m%d.o" % (base, s_, m_)),
                                      ["-DSBF_SWEEP_S=%d" % s_, "-DSBF_SWEEP_M=%d" % m_]))
        else:
            units.append((src, os.path.join(objdir, base + ".o"), []))
    for src, obj, defs in units:
        objs.append(obj)
        stale = force or not os.path.exists(obj) or os.path.getmtime(obj) < max(os.path.getmtime(src), hdr_time)
        if stale:
            cmd = [nvcc] + NVCC_FLAGS + list(extra_flags) + defs + (["-Xptxas", "-v"] if verbose else []) + ["-c", src, "-o", obj]
            jobs.append(cmd)

    def run(cmd):
        r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed: %s\n%s" % (" ".join(cmd), r.stdout))
        return r.stdout

    if jobs:
        with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 4)) as ex:
            for out in ex.map(run, jobs):
                if verbose and out:
                    print(out)
    if jobs or not os.path.exists(lib) or os.path.getmtime(lib) < max(os.path.getmtime(o) for o in objs):
        tmp = lib + ".tmp.%d" % os.getpid()
        run([nvcc, "-shared", "-o", tmp] + objs + ["-gencode", "arch=compute_100a,code=sm_100a"])
        os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
