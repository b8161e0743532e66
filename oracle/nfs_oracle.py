"""oracle/nfs_oracle.py — ctypes binding of the CPU ORACLE.  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin argument marshalling around oracle/nfs_oracle.c (the plain fp64 definition of
D(q,tau), I(q), counts — SURVEY.md §8(c) steps 1-6).
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from paper_1209_3362_b200.
"""
import ctypes as C

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.nfso_frame_sum.restype = C.c_uint64
        _lib.nfso_num_threads.restype = C.c_int
        _lib.nfso_qbin.restype = C.c_int
    return _lib


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t)) if a is not None else None


def _frames(frames):
    f = np.ascontiguousarray(frames, dtype=np.uint16)
    assert f.ndim == 3, "frames must be [N][H][W] uint16"
    return f


def num_threads() -> int:
    return int(lib().nfso_num_threads())


def frame_sum(frame) -> int:
    f = np.ascontiguousarray(frame, dtype=np.uint16)
    H, W = f.shape
    return int(lib().nfso_frame_sum(_p(f, C.c_uint16), W, H))


def transform_u16(frame, method=0):
    """Unitary full-plane transform of one normalised uint16 frame -> complex128 [H][W]."""
    f = np.ascontiguousarray(frame, dtype=np.uint16)
    H, W = f.shape
    out = np.empty((H, W), dtype=np.complex128)
    rc = lib().nfso_transform_u16(_p(f, C.c_uint16), W, H, int(method), _p(out, C.c_double))
    if rc:
        raise RuntimeError("nfso_transform_u16 rc=%d" % rc)
    return out


def transform_f64(img, method=0):
    """Unitary full-plane transform of a real fp64 image (no normalisation)."""
    a = np.ascontiguousarray(img, dtype=np.float64)
    H, W = a.shape
    out = np.empty((H, W), dtype=np.complex128)
    rc = lib().nfso_transform_f64(_p(a, C.c_double), W, H, int(method), _p(out, C.c_double))
    if rc:
        raise RuntimeError("nfso_transform_f64 rc=%d" % rc)
    return out


def qbin(kx, ky, W, H, n_b) -> int:
    return int(lib().nfso_qbin(int(kx), int(ky), int(W), int(H), int(n_b)))


def azimuthal_mean(map2d, n_b):
    a = np.ascontiguousarray(map2d, dtype=np.float64)
    H, W = a.shape
    out = np.zeros(n_b, dtype=np.float64)
    cnt = np.zeros(n_b, dtype=np.int64)
    lib().nfso_azimuthal_mean(_p(a, C.c_double), W, H, int(n_b), _p(out, C.c_double), _p(cnt, C.c_int64))
    return out, cnt


class Result(dict):
    __getattr__ = dict.__getitem__


def structure_function(frames, lags, n_b, method=0, want_2d=False, windowed=False):
    """The definition, everything in memory (or `windowed`: streamed through Lmax+1 slots).

    Returns Result(D [n_l][n_b], I_q [n_b], counts [n_b] int64, n_pairs [n_l] int64,
                   D2d [n_l][H][W] or None, I2d [H][W] or None)."""
    f = _frames(frames)
    N, H, W = f.shape
    lg = np.ascontiguousarray(lags, dtype=np.int32)
    n_l = lg.size
    D = np.zeros((n_l, n_b), dtype=np.float64)
    I_q = np.zeros(n_b, dtype=np.float64)
    cnt = np.zeros(n_b, dtype=np.int64)
    npairs = np.zeros(n_l, dtype=np.int64)
    D2d = np.zeros((n_l, H, W), dtype=np.float64) if want_2d else None
    I2d = np.zeros((H, W), dtype=np.float64) if want_2d else None
    if windowed:
        rc = lib().nfso_structure_function_windowed(
            _p(f, C.c_uint16), N, W, H, _p(lg, C.c_int32), n_l, int(n_b), _p(D, C.c_double),
            _p(I_q, C.c_double), _p(cnt, C.c_int64), _p(npairs, C.c_int64), _p(D2d, C.c_double),
            _p(I2d, C.c_double))
    else:
        rc = lib().nfso_structure_function(
            _p(f, C.c_uint16), N, W, H, _p(lg, C.c_int32), n_l, int(n_b), int(method), _p(D, C.c_double),
            _p(I_q, C.c_double), _p(cnt, C.c_int64), _p(npairs, C.c_int64), _p(D2d, C.c_double),
            _p(I2d, C.c_double))
    if rc:
        raise RuntimeError("oracle structure_function rc=%d" % rc)
    return Result(D=D, I_q=I_q, counts=cnt, n_pairs=npairs, D2d=D2d, I2d=I2d)


def structure_function_half(frames, lags, n_b, want_2d=False):
    """The definition on the half plane kx <= W/2 (Hermitian weights in the bin means; pin P11: equal to
    structure_function).  Returns Result(D, I_q, counts, n_pairs, D2d [n_l][H][W/2+1] or None, I2d [H][W/2+1] or None)."""
    f = _frames(frames)
    N, H, W = f.shape
    lg = np.ascontiguousarray(lags, dtype=np.int32)
    n_l = lg.size
    D = np.zeros((n_l, n_b), dtype=np.float64)
    I_q = np.zeros(n_b, dtype=np.float64)
    cnt = np.zeros(n_b, dtype=np.int64)
    npairs = np.zeros(n_l, dtype=np.int64)
    D2d = np.zeros((n_l, H, W // 2 + 1), dtype=np.float64) if want_2d else None
    I2d = np.zeros((H, W // 2 + 1), dtype=np.float64) if want_2d else None
    rc = lib().nfso_structure_function_half(
        _p(f, C.c_uint16), N, W, H, _p(lg, C.c_int32), n_l, int(n_b), _p(D, C.c_double), _p(I_q, C.c_double),
        _p(cnt, C.c_int64), _p(npairs, C.c_int64), _p(D2d, C.c_double), _p(I2d, C.c_double))
    if rc:
        raise RuntimeError("oracle structure_function_half rc=%d" % rc)
    return Result(D=D, I_q=I_q, counts=cnt, n_pairs=npairs, D2d=D2d, I2d=I2d)


def last_stage_seconds():
    """(seconds of steps 1-2, seconds of steps 3-4) of the last structure_function call."""
    out = (C.c_double * 2)()
    lib().nfso_last_stage_seconds(out)
    return float(out[0]), float(out[1])


def structure_function_sampled(frames, lags, sample_ky, sample_kx):
    """The definition restricted to sampled Fourier pixels (full transform of every frame).

    Returns Result(D2d [n_l][n_s], I2d [n_s], n_pairs [n_l])."""
    f = _frames(frames)
    N, H, W = f.shape
    lg = np.ascontiguousarray(lags, dtype=np.int32)
    ky = np.ascontiguousarray(sample_ky, dtype=np.int32)
    kx = np.ascontiguousarray(sample_kx, dtype=np.int32)
    n_l, n_s = lg.size, ky.size
    D2d = np.zeros((n_l, n_s), dtype=np.float64)
    I2d = np.zeros(n_s, dtype=np.float64)
    npairs = np.zeros(n_l, dtype=np.int64)
    rc = lib().nfso_structure_function_sampled(
        _p(f, C.c_uint16), N, W, H, _p(lg, C.c_int32), n_l, _p(ky, C.c_int32), _p(kx, C.c_int32), n_s,
        _p(D2d, C.c_double), _p(I2d, C.c_double), _p(npairs, C.c_int64))
    if rc:
        raise RuntimeError("oracle structure_function_sampled rc=%d" % rc)
    return Result(D2d=D2d, I2d=I2d, n_pairs=npairs)


def variance_spectrum(frames, n_b, method=0, want_2d=False):
    """Step 7: V2d(k) = (1/N) sum_t |F_t(k) - <F(k)>_t|^2 and its azimuthal mean.

    Returns Result(V_q [n_b], counts [n_b] int64, V2d [H][W] or None)."""
    f = _frames(frames)
    N, H, W = f.shape
    V_q = np.zeros(n_b, dtype=np.float64)
    cnt = np.zeros(n_b, dtype=np.int64)
    V2d = np.zeros((H, W), dtype=np.float64) if want_2d else None
    rc = lib().nfso_variance_spectrum(_p(f, C.c_uint16), N, W, H, int(n_b), int(method), _p(V_q, C.c_double),
                                      _p(cnt, C.c_int64), _p(V2d, C.c_double))
    if rc:
        raise RuntimeError("oracle variance_spectrum rc=%d" % rc)
    return Result(V_q=V_q, counts=cnt, V2d=V2d)
