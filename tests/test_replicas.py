"""Multi-GPU host logic (replicas over independent states) on CPU: world size 2, gloo backend."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2509_26309_b200 import replicas as R


def test_shards_cover_all_states_once():
    for total in (0, 1, 7, 32, 64):
        for world in (1, 2, 3, 8):
            seen = []
            for r in range(world):
                sh = R.strong_shard(total, r, world)
                seen += list(range(sh.first_state, sh.first_state + sh.n_state))
            assert seen == list(range(total))
    for world in (1, 2, 8):
        firsts = [R.weak_shard(4, r, world).first_state for r in range(world)]
        assert firsts == [4 * r for r in range(world)]


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        sh = R.strong_shard(5, rank, world)                       # ragged: 3 + 2 states
        n_step = 4
        corr = torch.zeros((sh.n_state, n_step), dtype=torch.complex128)
        for b in range(sh.n_state):
            for n in range(n_step):
                corr[b, n] = complex(sh.first_state + b, n)
        R.barrier()
        t = R.max_over_ranks([1.0 + rank, 5.0 - rank])
        rate = R.whole_job_rate(10.0 * (rank + 1), 2.0 + rank)    # (10 + 20) / max(2, 3)
        g = R.gather_corr(corr, sh)
        if rank == 0:
            out.put((t, rate, g.clone()))
        else:
            assert g is None
        R.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(120)
def test_two_ranks_gloo():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    t, rate, g = out.get(timeout=90)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    assert t == [2.0, 5.0]
    assert rate == pytest.approx(10.0)
    assert g.shape == (5, 4)
    for b in range(5):
        for n in range(4):
            assert g[b, n] == complex(b, n)
