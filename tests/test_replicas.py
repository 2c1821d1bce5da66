"""The N > 1 path of bench.py is N independent replicas: the only
cross-rank traffic is the barrier and the max of the timed duration.  World-size-2 gloo on CPU."""
import os
import socket

import numpy as np
import torch.multiprocessing as mp

from paper_2510_19047_b200 import replicas, synth


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    info = replicas.RankInfo.from_env()
    replicas.init(info, "gloo")
    replicas.barrier(info)
    w = synth.scaled(synth.WORKLOADS["cfg2"], Nt=64, Nf=64, n_templates=100)
    bank = synth.make_templates(w, seed=replicas.bank_seed(w.seed, info.rank))
    my_time = 1.0 + 0.5 * rank                       # stand-in for the device-timed region
    t = replicas.max_over_ranks(my_time, info)
    replicas.barrier(info)
    out.put((rank, t, replicas.aggregate_rate(len(bank), t, info), float(bank[:, 0].sum())))
    replicas.finish(info)


def test_two_replicas_gloo():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[0] for r in res] == [0, 1]
    assert all(r[1] == 1.5 for r in res)                       # max over ranks, on every rank
    assert all(abs(r[2] - 2 * 100 / 1.5) < 1e-12 for r in res)  # whole-job rate
    assert res[0][3] != res[1][3]                               # each replica has its own bank


def test_single_rank_is_a_noop():
    info = replicas.RankInfo.from_env({})
    assert (info.rank, info.world, info.local_rank) == (0, 1, 0)
    assert replicas.init(info, "gloo") is None
    replicas.barrier(info)
    assert replicas.max_over_ranks(3.25, info) == 3.25
    assert replicas.bank_seed(5, 0) == 5
