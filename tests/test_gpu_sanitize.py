"""Small, structurally rich parity cases sized for `compute-sanitizer` (memcheck, racecheck, initcheck, synccheck:
SURVEY.md §5, §7 step 3).  They run as ordinary `-m gpu` parity tests too; the sanitizer summaries under profiles/
come from `compute-sanitizer --tool <tool> python -m pytest tests/test_gpu_sanitize.py -x -q`.

Covered: BASELINE.json configs[0] in every launch shape of the lag kernel, a sparse-lag context whose Fourier ring
wraps around (several lag groups, warm-up, ragged batches, in-launch folds), the one-level FFT at 64 points and the
two-level FFT at 2048 points, bin-only accumulation, and the getters."""
import numpy as np
import pytest
import torch

import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def binding():
    assert torch.cuda.is_available()
    from paper_1209_3362_b200 import binding as b

    b.load_library()
    return b


def _check(g_D, g_I, g_cnt, ref, tol=1e-4):
    assert np.array_equal(g_cnt, ref.counts)
    nz = ref.counts > 0
    rows = ref.n_pairs > 0
    assert np.max(np.abs(g_D[rows][:, nz] - ref.D[rows][:, nz]) / ref.D[rows][:, nz]) < tol
    assert np.max(np.abs(g_I[nz] - ref.I_q[nz]) / ref.I_q[nz]) < tol


@pytest.mark.parametrize("shape", [0, 1, 2])
def test_config0_every_launch_shape(binding, oracle, shape):
    cfg = synth.config(0)
    st = synth.make_stack(cfg, "cuda")
    ref = oracle.structure_function(st.cpu().numpy(), cfg.lags, cfg.n_qbins)
    nfs = binding.NFS(cfg.W, cfg.H, cfg.lags, cfg.n_qbins)
    nfs.set_launch_shape(shape)
    nfs.push(st)
    D, I_q, cnt = nfs.finalize()
    nfs.D2d(0), nfs.I2d(), nfs.V2d(), nfs.variance()
    nfs.close()
    _check(D, I_q, cnt, ref)


@pytest.mark.parametrize("batch", [0, 37])
def test_sparse_lags_ring_wrap(binding, oracle, batch):
    lags = [1, 2, 3, 4, 5, 6, 7, 8, 9, 11, 14, 20, 33, 60, 61, 62, 63, 64, 65, 66, 67, 100, 140]
    cfg = synth.config(3, W=64, N=330, lags=lags, n_qbins=16)
    st = synth.make_stack(cfg, "cuda")
    ref = oracle.structure_function(st.cpu().numpy(), lags, cfg.n_qbins)
    nfs = binding.NFS(cfg.W, cfg.H, lags, cfg.n_qbins, batch_frames=batch)
    if batch:
        assert nfs.ring_capacity < cfg.N, "the ring must wrap"
    for i in range(0, cfg.N, 50):
        nfs.push(st[i:i + 50].contiguous())
    D, I_q, cnt = nfs.finalize()
    nfs.close()
    _check(D, I_q, cnt, ref)


def test_two_level_fft_2048(binding, oracle):
    lags = [1, 2, 3]
    cfg = synth.config(3, W=2048, N=5, lags=lags, n_qbins=64)
    st = synth.make_stack(cfg, "cuda")
    ref = oracle.structure_function(st.cpu().numpy(), lags, cfg.n_qbins)
    nfs = binding.NFS(cfg.W, cfg.H, lags, cfg.n_qbins)
    nfs.push(st)
    D, I_q, cnt = nfs.finalize()
    nfs.close()
    _check(D, I_q, cnt, ref)
