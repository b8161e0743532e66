"""Thin Python binding of include/nfs.h (argument marshalling only; every step runs in the CUDA kernels).

Same names as the C ABI: nfs_create / nfs_push_frames / nfs_finalize / getters, plus a small
`NFS` convenience class.  torch is used only for device memory and streams.  There is no CPU
fallback: if the library is missing or does not load, load_library() raises.

Two builds of the same object files exist (paper_1209_3362_b200/build.py): libnfs_b200.so exports include/nfs.h and is
what this module loads by default; libnfs_b200_dev.so additionally exports the measurement / debugging aids of
include/nfs_dev.h (per-kernel timing, launch counts, guard zones, plan introspection, the traffic probe) and is loaded
instead after use_dev_library() — the tests (tests/conftest.py) and bench.py do that before they create a context.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libnfs_b200.so")
DEV_LIB_PATH = os.path.join(_HERE, "libnfs_b200_dev.so")

NFS_OK = 0
NFS_ERR_INVALID_ARG = -1
NFS_ERR_OOM = -2
NFS_ERR_CUDA = -3
NFS_ERR_ZERO_MEAN = -4
NFS_ERR_STATE = -5
NFS_ERR_UNSUPPORTED = -6
NFS_ERR_TOO_LARGE = -7
NFS_STATIC_MAX_QBINS = 1024

# every symbol include/nfs.h declares: (name, restype, argtypes)
_P = C.c_void_p
SYMBOLS = [
    ("nfs_create", C.c_int, [C.POINTER(_P), C.c_int, C.c_int, C.POINTER(C.c_int32), C.c_int, C.c_int, _P]),
    ("nfs_create_ex", C.c_int, [C.POINTER(_P), C.c_int, C.c_int, C.POINTER(C.c_int32), C.c_int, C.c_int, _P, C.c_int]),
    ("nfs_create_opts", C.c_int, [C.POINTER(_P), C.c_int, C.c_int, C.POINTER(C.c_int32), C.c_int, C.c_int, _P, C.c_int, C.c_uint]),
    ("nfs_create_banded", C.c_int, [C.POINTER(_P), C.c_int, C.c_int, C.POINTER(C.c_int32), C.c_int, C.c_int, _P, C.c_int, C.c_uint,
                                    C.c_int, C.c_int64]),
    ("nfs_get_transfer_counts", C.c_int, [_P, C.POINTER(C.c_int64)]),
    ("nfs_push_frames", C.c_int, [_P, _P, C.c_int]),
    ("nfs_push_halo", C.c_int, [_P, _P, C.c_int]),
    ("nfs_partials_count", C.c_int64, [_P]),
    ("nfs_export_partials", C.c_int, [_P, _P]),
    ("nfs_import_partials", C.c_int, [_P, _P]),
    ("nfs_finalize", C.c_int, [_P, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_int64)]),
    ("nfs_get_pair_counts", C.c_int, [_P, C.POINTER(C.c_int64)]),
    ("nfs_get_D2d", C.c_int, [_P, C.c_int, C.POINTER(C.c_double)]),
    ("nfs_get_I2d", C.c_int, [_P, C.POINTER(C.c_double)]),
    ("nfs_get_variance", C.c_int, [_P, C.POINTER(C.c_double)]),
    ("nfs_get_V2d", C.c_int, [_P, C.POINTER(C.c_double)]),
    ("nfs_fit_eq1", C.c_int, [_P, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_double)]),
    ("nfs_num_frames", C.c_int64, [_P]),
    ("nfs_ring_capacity", C.c_int, [_P]),
    ("nfs_device_bytes", C.c_int64, [_P]),
    ("nfs_azimuthal_mean_static", C.c_int, [_P, C.c_int, C.c_int, C.c_int, _P, _P, _P]),
    ("nfs_reset", C.c_int, [_P]),
    ("nfs_destroy", None, [_P]),
    ("nfs_strerror", C.c_char_p, [C.c_int]),
    ("nfs_last_cuda_error", C.c_char_p, [_P]),
]
# include/nfs_dev.h: exported by libnfs_b200_dev.so only
DEV_SYMBOLS = [
    ("nfs_band_plan", C.c_int, [C.c_int64, C.POINTER(C.c_int32), C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int64)]),
    ("nfs_probe_lag_traffic", C.c_int, [_P, C.c_int, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]),
    ("nfs_check_guards", C.c_int, [_P, C.POINTER(C.c_int64)]),
    ("nfs_num_launches", C.c_int64, [_P]),
    ("nfs_set_launch_shape", C.c_int, [_P, C.c_int]),
    ("nfs_plan_lags", C.c_int, [C.POINTER(C.c_int32), C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int32), C.c_int]),
    ("nfs_set_profiling", C.c_int, [_P, C.c_int]),
    ("nfs_get_kernel_times", C.c_int, [_P, C.POINTER(C.c_double), C.POINTER(C.c_int64)]),
]

KERNEL_CLASSES = ["ref_setup", "fft", "unused", "lag_accum", "bin"]
NFS_FLAG_BIN_ONLY = 1
NFS_FLAG_GUARD = 2
NFS_FLAG_DIRECT = 4
SHAPE_AUTO, SHAPE_ONE_TILE, SHAPE_PERSISTENT = 0, 1, 2

_lib = None
_use_dev = False


def use_dev_library():
    """From now on load_library() returns libnfs_b200_dev.so (include/nfs.h + include/nfs_dev.h).  Call it before the
    first context is created: a context belongs to the library that created it."""
    global _lib, _use_dev
    if not _use_dev:
        _use_dev = True
        _lib = None


def load_library(path: str = None):
    """Loads the C-ABI library; raises (never falls back) if it is missing."""
    global _lib
    if _lib is None:
        path = path or (DEV_LIB_PATH if _use_dev else LIB_PATH)
        if not os.path.exists(path):
            raise ImportError(
                "%s not found: build it with `python -m paper_1209_3362_b200.build` "
                "(there is no CPU fallback for the hot path)" % path)
        lib = C.CDLL(path)
        for name, res, args in SYMBOLS + (DEV_SYMBOLS if _use_dev else []):
            fn = getattr(lib, name)  # AttributeError if the symbol is not exported
            fn.restype = res
            fn.argtypes = args
        _lib = lib
    return _lib


def _dev_fn(name):
    """A function of include/nfs_dev.h; a clear error if the product library is the one loaded."""
    lib = load_library()
    if not _use_dev:
        raise RuntimeError("%s is a measurement / debugging aid (include/nfs_dev.h) that libnfs_b200.so does not export: "
                           "call binding.use_dev_library() before creating contexts" % name)
    return getattr(lib, name)


class NFSError(RuntimeError):
    def __init__(self, status, detail=""):
        self.status = status
        msg = load_library().nfs_strerror(status).decode()
        super().__init__("nfs status %d: %s%s" % (status, msg, (" [" + detail + "]") if detail else ""))


def _check(rc, handle=None):
    if rc != NFS_OK:
        detail = ""
        if handle and rc == NFS_ERR_CUDA:
            detail = load_library().nfs_last_cuda_error(handle).decode()
        raise NFSError(rc, detail)


def _dp(a, t):
    return a.ctypes.data_as(C.POINTER(t))


# ---- functions with the C names -----------------------------------------------------------------------
def nfs_create(W, H, lags, n_qbins, cuda_stream=None, batch_frames=0, flags=0, ring_frames_cap=0, max_frames=0):
    lg = np.ascontiguousarray(lags, dtype=np.int32)
    h = _P()
    st = _P(cuda_stream) if cuda_stream else None
    if ring_frames_cap:
        rc = load_library().nfs_create_banded(C.byref(h), int(W), int(H), _dp(lg, C.c_int32), int(lg.size), int(n_qbins), st,
                                              int(batch_frames), int(flags), int(ring_frames_cap), int(max_frames))
    else:
        rc = load_library().nfs_create_opts(C.byref(h), int(W), int(H), _dp(lg, C.c_int32), int(lg.size), int(n_qbins), st,
                                            int(batch_frames), int(flags))
    _check(rc)
    return h


def nfs_band_plan(n_frames, lags, ring_frames_cap, batch_frames=0):
    """Host-only walk of the out-of-core band schedule (include/nfs.h): dict(bands, band_width, batch, old_uploads,
    new_uploads, launches)."""
    lg = np.ascontiguousarray(lags, dtype=np.int32)
    out = np.zeros(6, dtype=np.int64)
    _check(_dev_fn("nfs_band_plan")(int(n_frames), _dp(lg, C.c_int32), int(lg.size), int(ring_frames_cap), int(batch_frames),
                                        _dp(out, C.c_int64)))
    return dict(zip(("bands", "band_width", "batch", "old_uploads", "new_uploads", "launches"), (int(v) for v in out)))


def nfs_push_frames(handle, d_frames_ptr: int, n: int):
    _check(load_library().nfs_push_frames(handle, _P(d_frames_ptr), int(n)), handle)


def nfs_finalize(handle, n_lags, n_qbins):
    D = np.zeros((n_lags, n_qbins), dtype=np.float64)
    I_q = np.zeros(n_qbins, dtype=np.float64)
    cnt = np.zeros(n_qbins, dtype=np.int64)
    _check(load_library().nfs_finalize(handle, _dp(D, C.c_double), _dp(I_q, C.c_double), _dp(cnt, C.c_int64)), handle)
    return D, I_q, cnt


def nfs_plan_lags(lags, n_px=1024 * 513, smem_per_sm=233472, smem_optin=232448, n_sm=148):
    """Host-only lag plan (no CUDA call): dict(stages, smem, tile_px, ctas_per_sm, groups=[...], tasks=[...]); see
    include/nfs.h."""
    lags = np.ascontiguousarray(lags, dtype=np.int32)
    cap = 7 + 27 * (len(lags) + 1)
    out = np.zeros(cap, dtype=np.int32)
    n = _dev_fn("nfs_plan_lags")(_dp(lags, C.c_int32), len(lags), int(n_px), int(smem_per_sm), int(smem_optin), int(n_sm),
                                     _dp(out, C.c_int32), cap)
    if n < 0:
        raise NFSError(n)
    ng, nt, stages, smem, tile_px, per_sm, slots = (int(v) for v in out[:7])
    o = 7
    groups, tasks = [], []
    for _ in range(ng):
        g = out[o:o + 23]
        groups.append(dict(task0=int(g[0]), ntasks=int(g[1]), tau_min=int(g[2]), tau_max=int(g[3]), flags=int(g[4]),
                           warp_task=[int(v) for v in g[5:21]], cta0=int(g[21]), nctas=int(g[22])))
        o += 23
    for _ in range(nt):
        t = out[o:o + 4]
        tasks.append(dict(tau0=int(t[0]), cnt=int(t[1]), l0=int(t[2]), kind=int(t[3])))
        o += 4
    return dict(stages=stages, smem=smem, tile_px=tile_px, ctas_per_sm=per_sm, slots=slots, groups=groups, tasks=tasks)


def nfs_destroy(handle):
    load_library().nfs_destroy(handle)


def nfs_azimuthal_mean_static(d_spec2d_ptr: int, W: int, H: int, n_qbins: int, d_mean_q_ptr: int, d_counts_ptr: int = 0,
                              cuda_stream: int = 0):
    """Azimuthal average of one device-resident [H][W/2+1] float64 spectrum into n_qbins |q| bins without any device
    allocation (include/nfs.h).  It is meant for code that may not call cudaMalloc where it runs: per-frame analysis
    loops, processes whose GPU memory is owned by another pool, plug-ins that only get pointers and a stream.  All
    arguments are raw device addresses / a raw stream handle supplied by the caller; this wrapper allocates nothing
    either.  n_qbins above NFS_STATIC_MAX_QBINS raises NFSError(NFS_ERR_TOO_LARGE).  Asynchronous on `cuda_stream`;
    calls that may overlap on one device race on the library's fixed scratch array, so keep them stream ordered.  The
    first call on a device does a one-time address lookup: make it during set-up."""
    _check(load_library().nfs_azimuthal_mean_static(_P(d_spec2d_ptr), int(W), int(H), int(n_qbins), _P(d_mean_q_ptr),
                                                    _P(d_counts_ptr) if d_counts_ptr else None,
                                                    _P(cuda_stream) if cuda_stream else None))


# ---- convenience wrapper ----------------------------------------------------------------------------------
class NFS:
    """One context on a torch CUDA stream.  `push(frames)` takes a CUDA uint16 torch tensor [n][H][W] (contiguous).

    The context's work is enqueued on `stream` (default: a stream of its own).  push() orders that stream after the
    work already enqueued on torch's current stream (so a tensor written just before the call is complete when the
    kernels read it) and tells the caching allocator that the tensor is in use on the context's stream (so a
    temporary passed to push() is not recycled while the kernels still read it): include/nfs.h puts both duties on
    the caller of nfs_push_frames."""

    def __init__(self, W, H, lags, n_qbins, stream=None, batch_frames=0, bin_only=False, ring_frames_cap=0, max_frames=0,
                 guard=False, direct=False):
        import torch

        self.lib = load_library()
        self.W, self.H, self.n_qbins = int(W), int(H), int(n_qbins)
        self.lags = [int(t) for t in lags]
        self.bin_only = bool(bin_only)
        if stream is None and torch.cuda.is_available():
            stream = torch.cuda.Stream()
        self._stream = stream  # without a device nfs_create itself reports NFS_ERR_CUDA: no fallback
        self.handle = nfs_create(W, H, self.lags, n_qbins, stream.cuda_stream if stream is not None else None, batch_frames,
                                 (NFS_FLAG_BIN_ONLY if bin_only else 0) | (NFS_FLAG_GUARD if guard else 0) |
                                 (NFS_FLAG_DIRECT if direct else 0), ring_frames_cap,
                                 max_frames)

    def transfer_counts(self):
        out = np.zeros(4, dtype=np.int64)
        _check(self.lib.nfs_get_transfer_counts(self.handle, _dp(out, C.c_int64)), self.handle)
        return dict(zip(("bands", "band_width", "h2d_frames", "d2h_frames"), (int(v) for v in out)))

    @property
    def stream(self):
        return self._stream

    def push(self, frames):
        import torch

        assert frames.is_cuda and frames.dtype == torch.uint16 and frames.is_contiguous()
        assert frames.dim() == 3 and frames.shape[1] == self.H and frames.shape[2] == self.W
        cur = torch.cuda.current_stream(frames.device)
        if cur != self._stream:
            self._stream.wait_stream(cur)
            frames.record_stream(self._stream)
        nfs_push_frames(self.handle, frames.data_ptr(), frames.shape[0])

    def push_halo(self, frames):
        """Frames that precede this context's own frames (time-chunk sharding, include/nfs.h)."""
        import torch

        assert frames.is_cuda and frames.dtype == torch.uint16 and frames.is_contiguous()
        cur = torch.cuda.current_stream(frames.device)
        if cur != self._stream:
            self._stream.wait_stream(cur)
            frames.record_stream(self._stream)
        _check(self.lib.nfs_push_halo(self.handle, _P(frames.data_ptr()), int(frames.shape[0])), self.handle)

    def export_partials(self):
        """The context's partial sums as a float64 torch tensor on the context's device (ready for all_reduce).  The
        buffer is allocated on the context's stream, where the library writes it; nfs_export_partials synchronises that
        stream before it returns, and the tensor is then marked as in use on torch's current stream, where the caller
        will read it."""
        import torch

        n = int(self.lib.nfs_partials_count(self.handle))
        with torch.cuda.stream(self._stream):
            buf = torch.empty(n, dtype=torch.float64, device=self._stream.device)
        _check(self.lib.nfs_export_partials(self.handle, _P(buf.data_ptr())), self.handle)
        buf.record_stream(torch.cuda.current_stream(buf.device))
        return buf

    def import_partials(self, buf):
        """`buf`: the sum over all contexts of their exported buffers (the caller's all-reduce, enqueued on torch's
        current stream): the context's stream is ordered after that stream, no host synchronisation of it."""
        import torch

        assert buf.is_cuda and buf.dtype == torch.float64 and buf.is_contiguous()
        assert buf.numel() == int(self.lib.nfs_partials_count(self.handle))
        cur = torch.cuda.current_stream(buf.device)
        if cur != self._stream:
            self._stream.wait_stream(cur)
            buf.record_stream(self._stream)
        _check(self.lib.nfs_import_partials(self.handle, _P(buf.data_ptr())), self.handle)

    def push_ptr(self, ptr, n):
        nfs_push_frames(self.handle, ptr, n)

    def finalize(self):
        return nfs_finalize(self.handle, len(self.lags), self.n_qbins)

    def pair_counts(self):
        out = np.zeros(len(self.lags), dtype=np.int64)
        _check(self.lib.nfs_get_pair_counts(self.handle, _dp(out, C.c_int64)), self.handle)
        return out

    def D2d(self, lag_index):
        out = np.zeros((self.H, self.W // 2 + 1), dtype=np.float64)
        _check(self.lib.nfs_get_D2d(self.handle, int(lag_index), _dp(out, C.c_double)), self.handle)
        return out

    def I2d(self):
        out = np.zeros((self.H, self.W // 2 + 1), dtype=np.float64)
        _check(self.lib.nfs_get_I2d(self.handle, _dp(out, C.c_double)), self.handle)
        return out

    def variance(self):
        out = np.zeros(self.n_qbins, dtype=np.float64)
        _check(self.lib.nfs_get_variance(self.handle, _dp(out, C.c_double)), self.handle)
        return out

    def V2d(self):
        out = np.zeros((self.H, self.W // 2 + 1), dtype=np.float64)
        _check(self.lib.nfs_get_V2d(self.handle, _dp(out, C.c_double)), self.handle)
        return out

    def fit_eq1(self):
        """Per-|q| fit of Eq. 1 to the binned structure function: (A, C, Gamma, chi2), each [n_qbins]."""
        out = [np.zeros(self.n_qbins, dtype=np.float64) for _ in range(4)]
        _check(self.lib.nfs_fit_eq1(self.handle, *[_dp(a, C.c_double) for a in out]), self.handle)
        return tuple(out)

    def probe_lag_traffic(self, batch_frames, reps=20):
        """(ms per launch, algorithmic bytes per launch) of the lag kernel's memory access pattern without its arithmetic."""
        ms, by = C.c_double(0.0), C.c_double(0.0)
        _check(_dev_fn("nfs_probe_lag_traffic")(self.handle, int(batch_frames), int(reps), C.byref(ms), C.byref(by)), self.handle)
        return ms.value, by.value

    def check_guards(self):
        """Overwritten guard bytes around the context's device buffers (0 = intact); needs guard=True at creation."""
        n = C.c_int64(0)
        rc = _dev_fn("nfs_check_guards")(self.handle, C.byref(n))
        if rc not in (NFS_OK, NFS_ERR_STATE) or (rc == NFS_ERR_STATE and n.value == 0):
            _check(rc, self.handle)
        return int(n.value)

    def set_launch_shape(self, shape):
        _check(_dev_fn("nfs_set_launch_shape")(self.handle, int(shape)), self.handle)

    def set_profiling(self, enable):
        _check(_dev_fn("nfs_set_profiling")(self.handle, int(bool(enable))), self.handle)

    def kernel_times(self):
        """-> dict class -> (milliseconds, launches) since the last call (synchronises)."""
        ms = np.zeros(len(KERNEL_CLASSES), dtype=np.float64)
        n = np.zeros(len(KERNEL_CLASSES), dtype=np.int64)
        _check(_dev_fn("nfs_get_kernel_times")(self.handle, _dp(ms, C.c_double), _dp(n, C.c_int64)), self.handle)
        return {k: (float(ms[i]), int(n[i])) for i, k in enumerate(KERNEL_CLASSES)}

    def reset(self):
        _check(self.lib.nfs_reset(self.handle), self.handle)

    @property
    def num_frames(self):
        return int(self.lib.nfs_num_frames(self.handle))

    @property
    def num_launches(self):
        return int(_dev_fn("nfs_num_launches")(self.handle))

    @property
    def ring_capacity(self):
        return int(self.lib.nfs_ring_capacity(self.handle))

    @property
    def device_bytes(self):
        return int(self.lib.nfs_device_bytes(self.handle))

    def close(self):
        if self.handle is not None:
            nfs_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
