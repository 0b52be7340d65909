"""Builds libjt.so (the C-ABI library of include/jt.h) and libjtprobe.so (include/jt_probe.h, bench.py's ALU-rate
microbenchmarks) in-tree with nvcc for sm_100a.

    python -m paper_2606_01547_b200.build [--force]

nvcc cross-compiles without a GPU.  Objects go to paper_2606_01547_b200/build/ (git-ignored); the
library lands beside this file so that it travels with the repository snapshot to the GPU box.
"""
import concurrent.futures
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libjt.so")
PROBE_LIB = os.path.join(HERE, "libjtprobe.so")
SOURCES = ["jt_api.cu", "jt_trace.cu", "jt_trace_f32.cu", "jt_trace_f64.cu", "jt_conv.cu", "jt_fft.cu", "jt_batch.cu", "jt_next.cu", "jt_noalloc.cu"]
PROBE_SOURCES = ["jt_probe.cu"]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
         "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden"]


def _deps():
    d = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cuh", ".h", ".cu"))]
    d.append(os.path.join(HERE, "..", "include", "jt.h"))
    d.append(os.path.join(HERE, "..", "include", "jt_probe.h"))
    return d


def _stale(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def _compile(src):
    obj = os.path.join(OBJ, src.replace(".cu", ".o"))
    cmd = [NVCC] + FLAGS + ["-c", os.path.join(CSRC, src), "-o", obj]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed for %s:\n%s\n%s" % (src, r.stdout, r.stderr))
    return obj


def build(force=False, verbose=False):
    deps = _deps()
    if not force and not _stale(LIB, deps) and not _stale(PROBE_LIB, deps):
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    with concurrent.futures.ThreadPoolExecutor(max_workers=8) as ex:
        objs = list(ex.map(_compile, SOURCES + PROBE_SOURCES))
    for lib, members in ((LIB, objs[:len(SOURCES)]), (PROBE_LIB, objs[len(SOURCES):])):
        cmd = [NVCC, "-shared", "-o", lib] + members + ["-cudart", "static"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("link failed:\n%s\n%s" % (r.stdout, r.stderr))
        if verbose:
            print("built", lib)
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
