"""Builds, in-tree with nvcc (sm_100a only):
  libnfs_b200.so      the product: the C ABI of include/nfs.h and nothing else
  libnfs_b200_dev.so  the same object files plus csrc/nfs_dev.cu and csrc/nfs_probe.cu: additionally exports the
                      measurement / debugging aids of include/nfs_dev.h; loaded by the tests and bench.py
Every source is compiled once; the two libraries differ only in what is linked."""
import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libnfs_b200.so")
DEV_LIB = os.path.join(_HERE, "libnfs_b200_dev.so")
SOURCES = ["nfs_api.cu", "nfs_fft.cu", "nfs_lag.cu", "nfs_bin.cu", "nfs_static.cu"]
DEV_SOURCES = ["nfs_dev.cu", "nfs_probe.cu"]
HEADERS = [os.path.join(CSRC, "nfs_common.cuh"), os.path.join(_HERE, "..", "include", "nfs.h"),
           os.path.join(_HERE, "..", "include", "nfs_dev.h")]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden", "--expt-relaxed-constexpr",
]


def _nvcc() -> str:
    for p in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if p and (os.path.exists(p) or p == "nvcc"):
            return p
    return "nvcc"


def needs_build() -> bool:
    if not os.path.exists(LIB) or not os.path.exists(DEV_LIB):
        return True
    t = min(os.path.getmtime(LIB), os.path.getmtime(DEV_LIB))
    deps = [os.path.join(CSRC, s) for s in SOURCES + DEV_SOURCES] + HEADERS + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compiles the .cu files (in parallel, each once) and links both libraries beside this file; returns the
    product library's path."""
    if not force and not needs_build():
        return LIB
    objs, procs = [], []
    for s in SOURCES + DEV_SOURCES:
        o = os.path.join(CSRC, s.replace(".cu", ".o"))
        cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else [])
        procs.append((s, subprocess.Popen(cmd + ["-c", os.path.join(CSRC, s), "-o", o])))
        objs.append(o)
    failed = [s for s, p in procs if p.wait() != 0]
    if failed:
        raise RuntimeError("nvcc failed on " + ", ".join(failed))
    for lib, n in ((LIB, len(SOURCES)), (DEV_LIB, len(objs))):
        tmp = lib + ".tmp.%d" % os.getpid()
        subprocess.check_call([_nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", tmp] + objs[:n])
        os.replace(tmp, lib)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))
