"""Build steps of the package: libmanta.so (nvcc, sm_100a) and libmanta_workloads.so (gcc).

Deterministic mode: -fmad=false, IEEE division and square root (nvcc defaults
-prec-div=true -prec-sqrt=true, stated explicitly), no fast-math.
"""
import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_HERE)
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libmanta.so")
SOURCES = [os.path.join(CSRC, "manta_api.cu")]
DEPS = SOURCES + [os.path.join(CSRC, "manta_kernels.cuh"), os.path.join(CSRC, "manta_device.cuh"),
                  os.path.join(_ROOT, "include", "manta.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-fmad=false", "-prec-div=true", "-prec-sqrt=true", "-ftz=false",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-pthread", "-shared", "-Xptxas", "-v"]


def nvcc():
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    raise RuntimeError("nvcc not found")


def build_cuda(force=False, verbose=False):
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= max(os.path.getmtime(d) for d in DEPS)):
        return LIB
    cmd = [nvcc()] + NVCC_FLAGS + os.environ.get("MANTA_NVCC_EXTRA", "").split() + ["-o", LIB] + SOURCES + ["-lcudart"]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed")
    with open(os.path.join(_HERE, "libmanta.ptxas.txt"), "w") as f:   # git-ignored build log (registers, spills); a copy per profile round lives under profiles/
        log = "".join(l for l in (res.stdout + res.stderr).splitlines(True) if "Compile time" not in l)
        f.write(" ".join(cmd) + "\n" + log)
    return LIB


LIB_CHECK = os.path.join(_HERE, "libmanta_check.so")


def build_check(force=False):
    """The same sources with -DMANTA_CHECK: device-side bounds checks on every computed index (tests only)."""
    if (not force and os.path.exists(LIB_CHECK)
            and os.path.getmtime(LIB_CHECK) >= max(os.path.getmtime(d) for d in DEPS)):
        return LIB_CHECK
    cmd = [nvcc()] + [f for f in NVCC_FLAGS if f not in ("-Xptxas", "-v")] + ["-DMANTA_CHECK", "-o", LIB_CHECK] + SOURCES + ["-lcudart"]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed (check build)")
    return LIB_CHECK


LIB_FAST = os.path.join(_HERE, "libmanta_fast.so")


def build_fast(force=False):
    """Fast mode: the same sources with FMA contraction allowed (-fmad=true).  Not bit-exact against
    the oracle: held to a per-step tolerance instead (tests/test_gpu_parity.py::test_fast_variant_one_step_and_aggregates, run by test_fast_mode)."""
    if (not force and os.path.exists(LIB_FAST)
            and os.path.getmtime(LIB_FAST) >= max(os.path.getmtime(d) for d in DEPS)):
        return LIB_FAST
    flags = ["-fmad=true" if f == "-fmad=false" else f for f in NVCC_FLAGS if f not in ("-Xptxas", "-v")]
    cmd = [nvcc()] + flags + ["-DMANTA_FAST", "-o", LIB_FAST] + SOURCES + ["-lcudart"]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed (fast build)")
    return LIB_FAST


def build_all(force=False, verbose=False):
    """Everything the package needs; the three nvcc compilations run side by side."""
    from concurrent.futures import ThreadPoolExecutor
    from . import workloads
    workloads.build_routing(force)
    with ThreadPoolExecutor(3) as ex:
        jobs = [ex.submit(build_check, force), ex.submit(build_fast, force), ex.submit(build_cuda, force, verbose)]
        return [j.result() for j in jobs][-1]


if __name__ == "__main__":
    sys.path.insert(0, _ROOT)
    from paper_2007_03614_b200 import workloads as _w
    _w.build_routing("--force" in sys.argv)
    build_check("--force" in sys.argv)
    build_fast("--force" in sys.argv)
    build_cuda("--force" in sys.argv, verbose=True)
    print(LIB)
