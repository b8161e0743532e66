"""Time-chunk sharding of one stack over several ranks (the result is a sum over
frame pairs, so it splits by the later frame of each pair).  CPU: the shard plan, and world_size-2 gloo — every rank
sums the pairs of its own chunk (plain numpy on a tiny stack), ONE all-reduce adds them, the total equals the CPU
oracle of the whole stack.  GPU: the ranks are emulated one after the other on one device (separate contexts, their
partial-sum buffers added as the all-reduce would), against the single-context result and the oracle."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import synth
from paper_1209_3362_b200 import sharding


def test_shard_plan_covers_every_pair_once():
    for N, G, L in [(1000, 8, 100), (2000, 2, 100), (97, 4, 30), (10, 3, 9), (5, 8, 2)]:
        plan = sharding.shard_plan(N, G, L)
        assert [s.rank for s in plan] == list(range(G))
        assert plan[0].own_start == 0 and plan[-1].own_end == N
        assert all(a.own_end == b.own_start for a, b in zip(plan, plan[1:])), "own chunks tile the stack"
        assert all(s.n_halo == min(L, s.own_start) for s in plan), "a complete halo wherever frames exist before the chunk"
        assert max(s.n_own for s in plan) - min(s.n_own for s in plan) <= 1
        for tau in range(1, L + 1):
            assert sum(sharding.pairs_on_shard(s, tau) for s in plan) == max(0, N - tau)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _partial_sums(frames, sh, lags):
    """Pair sums of one shard by the plain definition (numpy, unitary FFT): only its halo and own frames are touched."""
    local = frames[sh.halo_start:sh.own_end].astype(np.float64)
    local = local / local.mean(axis=(1, 2), keepdims=True)
    F = np.fft.fft2(local) / np.sqrt(local.shape[1] * local.shape[2])
    out = np.zeros((len(lags),) + F.shape[1:])
    n_pairs = np.zeros(len(lags))
    for li, tau in enumerate(lags):
        for s in range(sh.own_start, sh.own_end):
            if s - tau >= 0:
                out[li] += np.abs(F[s - sh.halo_start] - F[s - tau - sh.halo_start]) ** 2
                n_pairs[li] += 1
    return out, n_pairs


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = synth.config(0, W=16, N=21, lags=[1, 2, 3, 5, 8], n_qbins=4)
        frames = synth.make_stack(cfg, "cpu").numpy()          # same seed on every rank: one stack, sharded
        sh = sharding.shard_plan(cfg.N, world, max(cfg.lags))[rank]
        sums, n_pairs = _partial_sums(frames, sh, cfg.lags)
        buf = torch.from_numpy(np.concatenate([sums.ravel(), n_pairs, [sh.n_own]]))
        sharding.all_reduce_sum(buf, dist)                     # the path's one collective
        q.put((rank, buf.numpy().copy(), (sh.halo_start, sh.own_start, sh.own_end)))
    finally:
        dist.destroy_process_group()


def test_sharded_sums_equal_oracle_world2(oracle):
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    out = sorted((q.get(timeout=180) for _ in range(world)), key=lambda o: o[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    cfg = synth.config(0, W=16, N=21, lags=[1, 2, 3, 5, 8], n_qbins=4)
    frames = synth.make_stack(cfg, "cpu").numpy()
    ref = oracle.structure_function(frames, cfg.lags, cfg.n_qbins, want_2d=True)
    assert out[0][2] == (0, 0, 10) and out[1][2] == (2, 10, 21)     # rank 1: halo of Lmax = 8 frames
    assert np.array_equal(out[0][1], out[1][1]), "after the all-reduce every rank holds the same totals"
    nl, P = len(cfg.lags), cfg.W * cfg.H
    tot = out[0][1][:nl * P].reshape(nl, cfg.H, cfg.W)
    n_pairs = out[0][1][nl * P:nl * P + nl]
    assert n_pairs.tolist() == [cfg.N - t for t in cfg.lags] and out[0][1][-1] == cfg.N
    D2d = tot / n_pairs[:, None, None]
    m = ref.D2d > 1e-9 * ref.D2d.max()
    assert np.max(np.abs(D2d[m] - ref.D2d[m]) / ref.D2d[m]) < 1e-9


@pytest.mark.gpu
@pytest.mark.parametrize("world,bin_only", [(2, False), (3, False), (2, True)])
def test_sharded_contexts_equal_single_context(oracle, world, bin_only):
    from paper_1209_3362_b200 import binding

    assert torch.cuda.is_available()
    lags = list(range(1, 31)) + [40, 55, 70]
    cfg = synth.config(1, W=128, N=300, lags=lags, n_qbins=32)
    st = synth.make_stack(cfg, "cuda")
    ref = oracle.structure_function(st.cpu().numpy(), lags, cfg.n_qbins)
    one = binding.NFS(cfg.W, cfg.H, lags, cfg.n_qbins)
    one.push(st)
    D1, I1, c1 = one.finalize()
    V1 = one.variance()
    one.close()

    plan = sharding.shard_plan(cfg.N, world, max(lags))
    ctxs = [binding.NFS(cfg.W, cfg.H, lags, cfg.n_qbins, bin_only=bin_only) for _ in plan]
    for nfs, sh in zip(ctxs, plan):
        sharding.push_shard(nfs, st, sh, chunk=64)
        assert nfs.pair_counts().tolist() == [sharding.pairs_on_shard(sh, t) for t in lags]
    bufs = [nfs.export_partials() for nfs in ctxs]
    total = torch.stack(bufs).sum(dim=0)                # what all_reduce(SUM) leaves on every rank
    for nfs in ctxs:
        nfs.import_partials(total.clone())
    outs = [nfs.finalize() + (nfs.variance(), nfs.pair_counts()) for nfs in ctxs]
    with pytest.raises(binding.NFSError):
        ctxs[0].push(st[:4])                            # merged sums: no more frames until reset
    ctxs[0].reset()                                     # ... after which the context starts over
    with pytest.raises(binding.NFSError):
        ctxs[0].push_halo(st[:max(lags) + 1])           # a halo is at most Lmax frames
    ctxs[0].push_halo(st[:5])
    ctxs[0].push(st[5:40])
    with pytest.raises(binding.NFSError):
        ctxs[0].push_halo(st[40:44])                    # ... and only precedes the own frames
    assert ctxs[0].pair_counts().tolist() == [max(0, 35 - max(0, t - 5)) for t in lags]
    for nfs in ctxs:
        nfs.close()
    nz = ref.counts > 0
    for D, I_q, cnt, V, npairs in outs:
        assert np.array_equal(cnt, ref.counts) and npairs.tolist() == [cfg.N - t for t in lags]
        assert np.max(np.abs(D[:, nz] - ref.D[:, nz]) / ref.D[:, nz]) < 1e-4
        assert np.max(np.abs(I_q[nz] - ref.I_q[nz]) / ref.I_q[nz]) < 1e-4
        assert np.max(np.abs(D[:, nz] - D1[:, nz]) / D1[:, nz]) < 2e-5      # other reference frames and batch cuts: fp32 rounding
        assert np.max(np.abs(I_q[nz] - I1[nz]) / I1[nz]) < 1e-5
        assert np.max(np.abs(V[nz] - V1[nz]) / V1[nz]) < 1e-4
    for o in outs[1:]:
        assert all(np.array_equal(a, b) for a, b in zip(o, outs[0])), "every rank returns the same result"


@pytest.mark.gpu
def test_more_ranks_than_frames_and_halo_only_contexts(oracle):
    """with fewer frames than ranks some time chunks are empty.  Such a rank must still get through the one
    collective (its export is all zeros, frame count 0) and hold the whole result afterwards; a context that has seen
    only halo frames has no average to give (NFS_ERR_STATE, not NaN)."""
    from paper_1209_3362_b200 import binding

    assert torch.cuda.is_available()
    lags = [1, 2]
    cfg = synth.config(0, W=64, N=3, lags=lags, n_qbins=16)
    st = synth.make_stack(cfg, "cuda")
    ref = oracle.structure_function(st.cpu().numpy(), lags, cfg.n_qbins)
    plan = sharding.shard_plan(cfg.N, 4, max(lags))
    assert [s.n_own for s in plan] == [0, 1, 1, 1]
    ctxs = [binding.NFS(cfg.W, cfg.H, lags, cfg.n_qbins) for _ in plan]
    for nfs, sh in zip(ctxs, plan):
        sharding.push_shard(nfs, st, sh)
    with pytest.raises(binding.NFSError) as e:
        ctxs[0].finalize()                                  # nothing pushed
    assert e.value.status == binding.NFS_ERR_STATE
    bufs = [nfs.export_partials() for nfs in ctxs]
    assert float(bufs[0].abs().max()) == 0.0
    total = torch.stack(bufs).sum(dim=0)
    for nfs in ctxs:
        nfs.import_partials(total.clone())
    with pytest.raises(binding.NFSError) as e:
        ctxs[1].import_partials(total.clone())              # once per context
    assert e.value.status == binding.NFS_ERR_STATE
    nz = ref.counts > 0
    for nfs in ctxs:
        D, I_q, cnt = nfs.finalize()
        assert nfs.pair_counts().tolist() == [2, 1]
        assert np.max(np.abs(D[:, nz] - ref.D[:, nz]) / ref.D[:, nz]) < 1e-4
        assert np.max(np.abs(I_q[nz] - ref.I_q[nz]) / ref.I_q[nz]) < 1e-4
        nfs.close()
    halo_only = binding.NFS(cfg.W, cfg.H, lags, cfg.n_qbins)
    halo_only.push_halo(st[:2])
    for call in (halo_only.finalize, halo_only.I2d, halo_only.variance):
        with pytest.raises(binding.NFSError) as e:
            call()
        assert e.value.status == binding.NFS_ERR_STATE
    assert float(halo_only.export_partials().abs().max()) == 0.0
    halo_only.close()
