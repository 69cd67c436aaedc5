"""N > 1 host logic ("replicas only") under gloo, world_size 2, on CPU."""
import os
import socket

import pytest


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    import torch.distributed as dist
    from paper_2607_04230_b200 import replicas, synth
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # each replica builds the same seeded scene (no broadcast): segment counts must agree
        sc = synth.config(4, scale=0.002, res_scale=0.05)
        n_full = sum(int(g["strands_per_tri"].sum()) * (g["pos"].shape[0] - 1) * g["style"]["spi"] for g in sc["grooms"])
        same = replicas.same_on_all_ranks(n_full, dist)
        differs = replicas.same_on_all_ranks(n_full + rank, dist)
        ms = replicas.max_over_ranks(1.0 + 0.5 * rank, dist)  # rank 1 is the slow one
        dist.barrier()
        q.put((rank, same, differs, ms, replicas.job_rate(1000, world, ms)))
    finally:
        dist.destroy_process_group()


def test_replicas_timing_rule_gloo_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, same, differs, ms, rate in out:
        assert same and not differs
        assert ms == pytest.approx(1.5)                      # the MAX over ranks, on every rank
        assert rate == pytest.approx(2 * 1000 / 1.5e-3)      # both replicas' units over the slowest rank's time


def test_single_process_is_identity():
    from paper_2607_04230_b200 import replicas
    assert replicas.max_over_ranks(2.5) == 2.5
    assert replicas.same_on_all_ranks(7)
    assert replicas.job_rate(10, 1, 2.0) == pytest.approx(5000.0)
