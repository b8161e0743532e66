"""The N>1 path is "replicas only": every rank analyses its own stack, the only
cross-rank step is the max-over-ranks of the device time.  Covered here with world_size-2 gloo on CPU."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import synth
from paper_1209_3362_b200 import replicas


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # each rank "measures" a different time; everyone must agree on the max
        ms = 10.0 + 5.0 * rank
        mx = replicas.max_over_ranks(ms, dist)
        cfg = replicas.rank_config(synth.config(0), rank)
        st = synth.make_stack(cfg, "cpu", n=2)
        q.put((rank, mx, cfg.seed, int(st.to(torch.int64).sum())))
    finally:
        dist.destroy_process_group()


def test_max_over_ranks_and_rate_world2():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [o[1] for o in out] == [15.0, 15.0]           # max over ranks, identical everywhere
    assert out[0][2] != out[1][2] and out[0][3] != out[1][3]  # independent stacks per rank
    # whole-job rate: all ranks' units / slowest rank's time
    assert replicas.whole_job_rate(2000, 15.0, world) == pytest.approx(2 * 2000 / 0.015)


def test_single_process_is_identity():
    assert replicas.max_over_ranks(3.5, None) == 3.5
    assert replicas.whole_job_rate(100, 50.0, 1) == pytest.approx(2000.0)
    cfg = synth.config(0)
    assert replicas.rank_config(cfg, 0) is cfg
    assert replicas.rank_config(cfg, 3).seed == cfg.seed + 300
