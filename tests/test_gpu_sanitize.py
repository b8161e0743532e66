"""Small, structurally rich parity cases sized for `compute-sanitizer` (memcheck, racecheck, initcheck, synccheck:
SURVEY.md §5, §7 step 3): `compute-sanitizer --tool <tool> python -m pytest tests/test_gpu_sanitize.py -x -q`.
On the pool these tests run on, that tool is closed (profiles/r02_sanitizer.md), so every context here is created
with NFS_FLAG_GUARD: all device buffers lie between canary zones which nfs_check_guards reads back — an out-of-bounds
write of any kernel next to a buffer fails the test — and the results are compared with the CPU oracle as always.

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
    nfs = binding.NFS(cfg.W, cfg.H, cfg.lags, cfg.n_qbins, guard=True)
    nfs.set_launch_shape(shape)
    nfs.push(st)
    D, I_q, cnt = nfs.finalize()
    nfs.D2d(0), nfs.I2d(), nfs.V2d(), nfs.variance(), nfs.fit_eq1()
    assert nfs.check_guards() == 0
    nfs.close()
    _check(D, I_q, cnt, ref)


@pytest.mark.parametrize("batch", [0, 37])
def test_sparse_lags_ring_wrap(binding, oracle, batch):
    lags = [1, 2, 3, 4, 5, 6, 7, 8, 9, 11, 14, 20, 33, 60, 61, 62, 63, 64, 65, 66, 67, 100, 140]
    cfg = synth.config(3, W=64, N=330, lags=lags, n_qbins=16)
    st = synth.make_stack(cfg, "cuda")
    ref = oracle.structure_function(st.cpu().numpy(), lags, cfg.n_qbins)
    nfs = binding.NFS(cfg.W, cfg.H, lags, cfg.n_qbins, batch_frames=batch, guard=True)
    if batch:
        assert nfs.ring_capacity < cfg.N, "the ring must wrap"
    for i in range(0, cfg.N, 50):
        nfs.push(st[i:i + 50].contiguous())
    D, I_q, cnt = nfs.finalize()
    assert nfs.check_guards() == 0
    nfs.close()
    _check(D, I_q, cnt, ref)


def test_two_level_fft_2048(binding, oracle):
    lags = [1, 2, 3]
    cfg = synth.config(3, W=2048, N=5, lags=lags, n_qbins=64)
    st = synth.make_stack(cfg, "cuda")
    ref = oracle.structure_function(st.cpu().numpy(), lags, cfg.n_qbins)
    nfs = binding.NFS(cfg.W, cfg.H, lags, cfg.n_qbins, guard=True)
    nfs.push(st)
    D, I_q, cnt = nfs.finalize()
    assert nfs.check_guards() == 0
    nfs.close()
    _check(D, I_q, cnt, ref)


@pytest.mark.parametrize("mode", ["bin_only", "banded", "sharded"])
def test_guarded_modes(binding, oracle, mode):
    """Bin-only accumulation, the out-of-core band schedule and a halo + partial-sum merge, each between guard zones."""
    lags = list(range(1, 61)) + [75, 90]
    cfg = synth.config(0, N=150, lags=lags, n_qbins=16)
    st = synth.make_stack(cfg, "cuda")
    ref = oracle.structure_function(st.cpu().numpy(), lags, cfg.n_qbins)
    if mode == "bin_only":
        nfs = binding.NFS(cfg.W, cfg.H, lags, cfg.n_qbins, bin_only=True, guard=True, batch_frames=40)
        nfs.push(st)
    elif mode == "banded":
        nfs = binding.NFS(cfg.W, cfg.H, lags, cfg.n_qbins, batch_frames=13, ring_frames_cap=30 + 26, max_frames=cfg.N, guard=True)
        nfs.push(st)
    else:
        from paper_1209_3362_b200 import sharding

        plan = sharding.shard_plan(cfg.N, 2, max(lags))
        other = binding.NFS(cfg.W, cfg.H, lags, cfg.n_qbins, guard=True)
        sharding.push_shard(other, st, plan[0])
        nfs = binding.NFS(cfg.W, cfg.H, lags, cfg.n_qbins, guard=True)
        sharding.push_shard(nfs, st, plan[1])
        total = other.export_partials() + nfs.export_partials()
        nfs.import_partials(total)
        assert other.check_guards() == 0
        other.close()
    D, I_q, cnt = nfs.finalize()
    assert nfs.check_guards() == 0
    nfs.close()
    _check(D, I_q, cnt, ref)
