"""Builds paper_1209_3362_b200/libnfs_b200.so (the C-ABI CUDA library, sm_100a only) in-tree with nvcc."""
import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libnfs_b200.so")
SOURCES = ["nfs_api.cu", "nfs_fft.cu", "nfs_lag.cu", "nfs_bin.cu", "nfs_probe.cu", "nfs_static.cu"]
HEADERS = [os.path.join(CSRC, "nfs_common.cuh"), os.path.join(_HERE, "..", "include", "nfs.h")]
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
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compiles the four .cu files (in parallel) and links libnfs_b200.so beside this file."""
    if not force and not needs_build():
        return LIB
    objs, procs = [], []
    for s in SOURCES:
        o = os.path.join(CSRC, s.replace(".cu", ".o"))
        cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else [])
        procs.append((s, subprocess.Popen(cmd + ["-c", os.path.join(CSRC, s), "-o", o])))
        objs.append(o)
    failed = [s for s, p in procs if p.wait() != 0]
    if failed:
        raise RuntimeError("nvcc failed on " + ", ".join(failed))
    tmp = LIB + ".tmp.%d" % os.getpid()
    subprocess.check_call([_nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", tmp] + objs)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))
