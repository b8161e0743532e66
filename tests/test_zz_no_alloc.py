"""nfs_azimuthal_mean_static: the |q|-binning entry point for callers that cannot allocate device memory.

Who needs it: a per-frame analysis loop (a cudaMalloc stalls the device for an unpredictable time), a process whose GPU
memory is owned entirely by another pool or capped by a MIG / MPS share (a library-side cudaMalloc fails or steals from
that budget), and plug-in code that only receives device pointers and a stream.  The entry point therefore takes every
buffer from the caller and keeps its partial sums in one fixed array inside the library (NFS_STATIC_MAX_QBINS bins at
most) that all calls on a device share.

What is checked here: its output against the library's ordinary path (nfs_finalize: host-built bin table, cudaMalloc'ed
buffers) for the same 2-D spectra, on two calls issued back to back on one stream WITHOUT a synchronisation in
between and after a call that deliberately leaves the shared array full of unrelated numbers — so a result that
depended on leftovers, or on a clean array, would fail.  Tolerance: the 1e-4 relative bar the binned parity tests use
(north_star); bin counts exactly.

The file name sorts last on purpose: under `pytest -x` a failure here must not hide the parity tests.  Nothing in
it depends on what ran before, so it passes alone in a fresh process as well as at the end of the suite.
"""
import ctypes as C
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

RTOL_BINNED = 1e-4  # same bar as tests/test_gpu_parity.py for |q|-binned quantities


def test_static_entry_rejects_what_its_fixed_array_cannot_hold():
    """Argument checks happen before CUDA is touched (no GPU needed): more bins than the built-in array was sized for
    is its own, named error — never a silent overrun — and the usual size rules of the library apply."""
    from paper_1209_3362_b200 import build as nfs_build
    from paper_1209_3362_b200 import binding as b

    nfs_build.build()
    lib = b.load_library()
    fake = C.c_void_p(4096)  # never dereferenced: the call must refuse before launching anything
    assert lib.nfs_azimuthal_mean_static(fake, 256, 256, b.NFS_STATIC_MAX_QBINS + 1, fake, None, None) == b.NFS_ERR_TOO_LARGE
    assert "NFS_STATIC_MAX_QBINS" in lib.nfs_strerror(b.NFS_ERR_TOO_LARGE).decode()
    assert lib.nfs_azimuthal_mean_static(None, 256, 256, 64, fake, None, None) == b.NFS_ERR_INVALID_ARG
    assert lib.nfs_azimuthal_mean_static(fake, 256, 256, 64, None, None, None) == b.NFS_ERR_INVALID_ARG
    assert lib.nfs_azimuthal_mean_static(fake, 256, 256, 0, fake, None, None) == b.NFS_ERR_INVALID_ARG
    assert lib.nfs_azimuthal_mean_static(fake, 100, 100, 64, fake, None, None) == b.NFS_ERR_INVALID_ARG
    assert lib.nfs_azimuthal_mean_static(fake, 256, 128, 64, fake, None, None) == b.NFS_ERR_UNSUPPORTED
    assert lib.nfs_azimuthal_mean_static(C.c_void_p(4100), 256, 256, 64, fake, None, None) == b.NFS_ERR_INVALID_ARG
    with pytest.raises(b.NFSError) as e:
        b.nfs_azimuthal_mean_static(4096, 256, 256, 5000, 4096)
    assert e.value.status == b.NFS_ERR_TOO_LARGE


@pytest.mark.gpu
def test_static_entry_matches_the_context_path_on_two_calls_in_a_row():
    import torch

    import synth
    from paper_1209_3362_b200 import build as nfs_build
    from paper_1209_3362_b200 import binding as b

    nfs_build.build()
    assert torch.cuda.is_available(), "needs a CUDA device: the library has no CPU fallback"
    torch.cuda.set_device(0)
    dev = "cuda:0"

    # the ordinary path: a context with its own (allocated) bin table
    cfg = synth.config(1, W=256, N=48, lags=[1, 3, 7], n_qbins=96)
    stack = synth.make_stack(cfg, dev)
    nfs = b.NFS(cfg.W, cfg.H, cfg.lags, cfg.n_qbins)
    try:
        nfs.push(stack)
        D, I_q, counts = nfs.finalize()
        I2d = nfs.I2d()      # HOST [H][W/2+1] float64
        D2d = nfs.D2d(2)     # lag 7
    finally:
        nfs.close()
    assert counts.sum() > 0 and np.all(I_q[counts > 0] > 0)

    # everything the new entry point touches is allocated HERE, by the caller, before the calls
    d_I2d = torch.from_numpy(I2d).to(dev)
    d_D2d = torch.from_numpy(D2d).to(dev)
    junk = torch.rand(512, 257, dtype=torch.float64, device=dev) * 1e30
    out_junk = torch.empty(b.NFS_STATIC_MAX_QBINS, dtype=torch.float64, device=dev)
    out_I = torch.full((cfg.n_qbins,), -1.0, dtype=torch.float64, device=dev)
    out_D = torch.full((cfg.n_qbins,), -1.0, dtype=torch.float64, device=dev)
    cnt_I = torch.full((cfg.n_qbins,), -1, dtype=torch.int64, device=dev)
    cnt_D = torch.full((cfg.n_qbins,), -1, dtype=torch.int64, device=dev)
    stream = torch.cuda.Stream()
    stream.wait_stream(torch.cuda.current_stream())
    s = stream.cuda_stream

    # fill the shared array with unrelated, huge partial sums (largest bin count, another frame size) ...
    b.nfs_azimuthal_mean_static(junk.data_ptr(), 512, 512, b.NFS_STATIC_MAX_QBINS, out_junk.data_ptr(), 0, s)
    # ... then the two calls under test, back to back on the same stream, no synchronisation in between
    b.nfs_azimuthal_mean_static(d_I2d.data_ptr(), cfg.W, cfg.H, cfg.n_qbins, out_I.data_ptr(), cnt_I.data_ptr(), s)
    b.nfs_azimuthal_mean_static(d_D2d.data_ptr(), cfg.W, cfg.H, cfg.n_qbins, out_D.data_ptr(), cnt_D.data_ptr(), s)
    stream.synchronize()

    nz = counts > 0
    for got, cnt, ref, what in ((out_I, cnt_I, I_q, "I(q)"), (out_D, cnt_D, D[2], "D(q, tau=7)")):
        got, cnt = got.cpu().numpy(), cnt.cpu().numpy()
        assert np.array_equal(cnt, counts), what + ": bin counts differ from nfs_finalize"
        assert np.all(got[~nz] == 0.0), what
        err = float(np.max(np.abs(got[nz] - ref[nz]) / np.abs(ref[nz])))
        assert err < RTOL_BINNED, (what, err)
        assert err < 1e-12, (what, err)  # both sides are fp64 sums of the same numbers: only the order differs

    # a repeat of the first call gives the same bits (fixed summation order, nothing carried over between calls)
    again = torch.empty_like(out_I)
    b.nfs_azimuthal_mean_static(d_I2d.data_ptr(), cfg.W, cfg.H, cfg.n_qbins, again.data_ptr(), 0, s)
    stream.synchronize()
    assert torch.equal(again, out_I)
