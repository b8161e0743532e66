"""CPU-side checks of the C-ABI boundary (no compute calls, no GPU needed):
the library loads, exports every symbol include/nfs.h declares, validates arguments before it touches
CUDA, and fails loudly (NFS_ERR_CUDA, never a fallback) when no device is present."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1209_3362_b200 import build as nfs_build
    from paper_1209_3362_b200 import binding

    nfs_build.build()
    return binding.load_library()


def _declared_symbols(header="nfs.h"):
    src = open(os.path.join(ROOT, "include", header)).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"NFS_API\s+[\w\s\*]+?\b(nfs_\w+)\s*\(", src)))


def _exported(path):
    """nfs_* functions in the dynamic symbol table of a shared library (binutils nm), or None without nm."""
    import shutil
    import subprocess

    if not shutil.which("nm"):
        return None
    out = subprocess.run(["nm", "-D", "--defined-only", path], capture_output=True, text=True, check=True).stdout
    return sorted(ln.split()[-1] for ln in out.splitlines() if ln.split()[-2:-1] == ["T"] and ln.split()[-1].startswith("nfs_"))


def test_header_declares_the_north_star_calls():
    names = _declared_symbols()
    for required in ("nfs_create", "nfs_push_frames", "nfs_finalize", "nfs_destroy", "nfs_reset", "nfs_strerror",
                     "nfs_get_pair_counts", "nfs_get_D2d", "nfs_get_I2d"):
        assert required in names, names


def test_product_library_exports_exactly_the_public_header(lib):
    """libnfs_b200.so = include/nfs.h, no more (measurement and debug aids do not belong in the product ABI)
    and no less; the binding's product table names the same symbols."""
    from paper_1209_3362_b200 import binding

    raw = C.CDLL(binding.LIB_PATH)
    declared = _declared_symbols()
    assert len(declared) >= 15
    for name in declared:
        assert hasattr(raw, name), "libnfs_b200.so does not export %s" % name
    for name in _declared_symbols("nfs_dev.h"):
        assert not hasattr(raw, name), "libnfs_b200.so exports the dev-only %s" % name
    exported = _exported(binding.LIB_PATH)
    if exported is not None:
        assert exported == declared, sorted(set(exported) ^ set(declared))
    assert {s[0] for s in binding.SYMBOLS} == set(declared)


def test_dev_library_exports_both_headers(lib):
    """libnfs_b200_dev.so (what the tests and bench.py load) = include/nfs.h + include/nfs_dev.h."""
    from paper_1209_3362_b200 import binding

    raw = C.CDLL(binding.DEV_LIB_PATH)
    dev = _declared_symbols("nfs_dev.h")
    both = sorted(set(_declared_symbols()) | set(dev))
    assert len(dev) == 8 and not set(dev) & set(_declared_symbols())
    for name in both:
        assert hasattr(raw, name), "libnfs_b200_dev.so does not export %s" % name
    exported = _exported(binding.DEV_LIB_PATH)
    if exported is not None:
        assert exported == both, sorted(set(exported) ^ set(both))
    assert {s[0] for s in binding.DEV_SYMBOLS} == set(dev)


def test_no_torch_or_python_symbols_in_the_abi():
    """The boundary is plain C: the header includes only stdint.h and uses no C++/torch types."""
    for header, includes in (("nfs.h", ["stdint.h"]), ("nfs_dev.h", ["nfs.h"])):
        src = open(os.path.join(ROOT, "include", header)).read()
        assert re.findall(r"#include\s+[<\"]([^>\"]+)[>\"]", src) == includes
        assert 'extern "C"' in src
        for bad in ("torch", "at::", "std::", "Tensor"):
            assert bad not in src


def test_strerror(lib):
    from paper_1209_3362_b200 import binding as b

    seen = set()
    for st in (b.NFS_OK, b.NFS_ERR_INVALID_ARG, b.NFS_ERR_OOM, b.NFS_ERR_CUDA, b.NFS_ERR_ZERO_MEAN, b.NFS_ERR_STATE,
               b.NFS_ERR_UNSUPPORTED):
        s = lib.nfs_strerror(st).decode()
        assert s and s != "unknown status"
        seen.add(s)
    assert len(seen) == 7
    assert lib.nfs_strerror(-99).decode() == "unknown status"


def _create(lib, W, H, lags, nb, batch=0):
    lg = np.ascontiguousarray(lags, dtype=np.int32)
    h = C.c_void_p()
    ptr = lg.ctypes.data_as(C.POINTER(C.c_int32)) if lg.size else None
    rc = lib.nfs_create_ex(C.byref(h), W, H, ptr, int(lg.size), nb, None, batch)
    return rc, h


@pytest.mark.parametrize("W,H,lags,nb,batch,expect", [
    (48, 48, [1, 2], 8, 0, -1),        # not a power of two
    (16, 16, [1, 2], 8, 0, -1),        # below the paper's range (L33: 32x32 ... 4k x 4k)
    (8192, 8192, [1], 8, 0, -1),       # above it
    (64, 64, [], 8, 0, -1),            # no lags
    (64, 64, [0, 1], 8, 0, -1),        # lag < 1
    (64, 64, [2, 2], 8, 0, -1),        # not strictly increasing
    (64, 64, [3, 1], 8, 0, -1),
    (64, 64, [1, 2], 0, 0, -1),        # no bins
    (64, 64, [1, 2], 8, -3, -1),       # negative batch
    (64, 128, [1, 2], 8, 0, -6),       # W != H: unsupported, not invalid
])
def test_create_validates_before_touching_cuda(lib, W, H, lags, nb, batch, expect):
    rc, h = _create(lib, W, H, lags, nb, batch)
    assert rc == expect
    assert not h.value


def test_null_arguments(lib):
    from paper_1209_3362_b200 import binding as b

    assert lib.nfs_create(None, 64, 64, None, 0, 8, None) == b.NFS_ERR_INVALID_ARG
    assert lib.nfs_push_frames(None, None, 1) == b.NFS_ERR_INVALID_ARG
    assert lib.nfs_finalize(None, None, None, None) == b.NFS_ERR_INVALID_ARG
    assert lib.nfs_get_pair_counts(None, None) == b.NFS_ERR_INVALID_ARG
    assert lib.nfs_get_D2d(None, 0, None) == b.NFS_ERR_INVALID_ARG
    assert lib.nfs_get_I2d(None, None) == b.NFS_ERR_INVALID_ARG
    assert lib.nfs_reset(None) == b.NFS_ERR_INVALID_ARG
    assert lib.nfs_num_frames(None) == 0
    assert lib.nfs_num_launches(None) == 0
    # the calls added for the band schedule, sharding, the Eq. 1 fit and the measurement aids
    assert lib.nfs_push_halo(None, None, 1) == b.NFS_ERR_INVALID_ARG
    assert lib.nfs_partials_count(None) == 0
    assert lib.nfs_export_partials(None, None) == b.NFS_ERR_INVALID_ARG
    assert lib.nfs_import_partials(None, None) == b.NFS_ERR_INVALID_ARG
    assert lib.nfs_fit_eq1(None, None, None, None, None) == b.NFS_ERR_INVALID_ARG
    assert lib.nfs_get_variance(None, None) == b.NFS_ERR_INVALID_ARG
    assert lib.nfs_get_transfer_counts(None, None) == b.NFS_ERR_INVALID_ARG
    assert lib.nfs_check_guards(None, None) == b.NFS_ERR_INVALID_ARG
    assert lib.nfs_probe_lag_traffic(None, 26, 1, None, None) == b.NFS_ERR_INVALID_ARG
    h = C.c_void_p()
    lg = np.array([1, 2, 3], dtype=np.int32)
    ptr = lg.ctypes.data_as(C.POINTER(C.c_int32))
    assert lib.nfs_create_banded(C.byref(h), 64, 64, ptr, 3, 8, None, 0, 0, -1, 0) == b.NFS_ERR_INVALID_ARG   # negative ring cap
    assert lib.nfs_create_banded(C.byref(h), 64, 64, ptr, 3, 8, None, 4, 0, 5, 0) == b.NFS_ERR_INVALID_ARG    # banded without max_frames
    assert lib.nfs_create_banded(C.byref(h), 64, 64, ptr, 3, 8, None, 1, 1, 3, 100) == b.NFS_ERR_UNSUPPORTED  # banded + bin-only
    assert lib.nfs_create_opts(C.byref(h), 64, 64, ptr, 3, 8, None, 0, 8) == b.NFS_ERR_INVALID_ARG            # unknown flag
    assert not h.value
    lib.nfs_destroy(None)  # no-op


def test_fails_loudly_without_a_device(lib):
    """No CPU fallback: on a box without a GPU a valid nfs_create returns NFS_ERR_CUDA and no context."""
    import torch

    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_1209_3362_b200 import binding as b

    rc, h = _create(lib, 64, 64, [1, 2, 3], 16)
    assert rc == b.NFS_ERR_CUDA
    assert not h.value
    with pytest.raises(b.NFSError):
        b.NFS(64, 64, [1, 2, 3], 16)


def test_product_never_imports_the_oracle():
    """oracle/ is test infrastructure: nothing under the package (or the C sources) refers to it."""
    pkg = os.path.join(ROOT, "paper_1209_3362_b200")
    for dp, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dp, fn)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), fn
                assert "nfs_oracle" not in txt and "libnfs_oracle" not in txt, fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", fn)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_1209_3362_b200\b", txt, flags=re.M), fn
            assert "libnfs_b200" not in txt, fn
