"""N > 1 path on CPU: world_size-2 gloo group, the replica bookkeeping bench.py uses (DESIGN.md section 8:
replicas only, no data-path collective; barrier + max-over-ranks timing; value = units of all ranks / max time)."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1908_00587_b200 import replicas, synth


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = replicas.rank_config(synth.scaled_config(0, N_r=12, M=4, K=4), rank)
        r = 1.0 + np.linspace(0.0, 1.0, cfg["N_r"])
        st = synth.make_state(cfg, r)
        dist.barrier()
        ms = replicas.max_over_ranks(10.0 + 5.0 * rank, dist, "cpu")     # rank 1 is the slow one
        value = replicas.aggregate_rate(world, 4, ms / 1e3)
        # fingerprint of this rank's synthetic state, gathered on every rank
        fp = torch.tensor([float(np.abs(st[0]).sum())], dtype=torch.float64)
        got = [torch.zeros(1, dtype=torch.float64) for _ in range(world)]
        dist.all_gather(got, fp)
        out.put((rank, ms, value, [float(g) for g in got]))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_replicas_over_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, value, fps in res:
        assert ms == 15.0                                  # max over ranks, on every rank
        assert value == world * 4 / 15.0e-3                # whole-job aggregate
        assert fps[0] != fps[1]                            # replicas carry different seeded states
    assert res[0][3] == res[1][3]


def test_single_process_is_identity():
    assert replicas.max_over_ranks(3.5) == 3.5
    assert replicas.aggregate_rate(1, 10, 0.5) == 20.0
