"""NEXT-2 bookkeeping: the slab plan and the two exchanges between the
mode-slab layout of the linear stage and the radial-slab layout of the nonlinear stage, over a world_size-2 and a
world_size-4 gloo group on CPU, against plain numpy slicing of the global array."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1908_00587_b200.slabs import SlabPlan, to_mode_slab, to_radial_slab


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _global_field(N_r, n_modes):
    j = np.arange(N_r)[:, None]
    e = np.arange(n_modes)[None, :]
    return (j * 1000 + e) + 1j * (e * 7 - j)                 # every entry identifies its (level, mode)


def test_plan_partitions_levels_and_modes():
    plan = SlabPlan(N_r=32, n_modes=9 * 17, world=4)
    lev = [plan.levels(r) for r in range(4)]
    assert lev == [(0, 8), (8, 16), (16, 24), (24, 32)]
    assert [plan.levels_with_halo(r) for r in range(4)] == [(0, 12), (4, 20), (12, 28), (20, 32)]
    # slabs of four levels: the one-sided stencils next to a wall reach nine levels (s0 = clamp(j - 4, 0, N_r - 9))
    assert [SlabPlan(N_r=16, n_modes=153, world=4).levels_with_halo(r) for r in range(4)] == [(0, 9), (0, 12), (4, 16), (7, 16)]
    assert [SlabPlan(N_r=32, n_modes=153, world=8).levels_with_halo(r) for r in (0, 1, 6, 7)] == [(0, 9), (0, 12), (20, 32), (23, 32)]
    assert SlabPlan(N_r=16, n_modes=153, world=16).levels_with_halo(15) == (7, 16)
    assert SlabPlan(N_r=16, n_modes=153, world=16).levels_with_halo(8) == (4, 13)
    mo = [plan.modes(r) for r in range(4)]
    assert mo[0][0] == 0 and mo[-1][1] == 153 and all(a[1] == b[0] for a, b in zip(mo, mo[1:]))
    assert sorted(e1 - e0 for e0, e1 in mo) == [38, 38, 38, 39]
    with pytest.raises(ValueError):
        SlabPlan(N_r=30, n_modes=100, world=4)               # the number of ranks must divide N_r
    # one rank: everything local, nothing sent
    one = SlabPlan(N_r=16, n_modes=40, world=1)
    assert one.levels_with_halo(0) == (0, 16) and one.modes(0) == (0, 40)
    assert one.bytes_per_exchange(0, 3, True) == 0
    # bytes: rank 1 of 4 sends its 38 columns of the 16 + 16 + 12 halo-extended rows of the others
    assert plan.bytes_per_exchange(1, 3, True) == 16 * 3 * 38 * (12 + 16 + 12)
    assert plan.bytes_per_exchange(1, 3, False) == 16 * 3 * 8 * (153 - 38)


def test_single_process_exchanges_are_slicing():
    plan = SlabPlan(N_r=12, n_modes=30, world=1)
    g = torch.from_numpy(_global_field(12, 30))
    assert torch.equal(to_radial_slab(plan, g, 0), g)
    assert torch.equal(to_mode_slab(plan, g, 0), g)


def _worker(rank, world, port, N_r, n_modes, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        plan = SlabPlan(N_r=N_r, n_modes=n_modes, world=world)
        G = _global_field(N_r, n_modes)
        e0, e1 = plan.modes(rank)
        j0, j1 = plan.levels(rank)
        h0, h1 = plan.levels_with_halo(rank)
        mine = torch.from_numpy(np.ascontiguousarray(G[:, e0:e1]))
        rad = to_radial_slab(plan, mine, rank, dist)                     # linear -> nonlinear layout, with halo
        ok_fwd = bool(np.array_equal(rad.numpy(), G[h0:h1]))
        own = rad[j0 - h0:j1 - h0]                                       # the nonlinear stage returns its own levels
        back = to_mode_slab(plan, own * 2.0, rank, dist)                 # nonlinear -> linear layout
        ok_bwd = bool(np.array_equal(back.numpy(), 2.0 * G[:, e0:e1]))
        out.put((rank, ok_fwd, ok_bwd, tuple(rad.shape), tuple(back.shape)))
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,N_r,n_modes", [(2, 12, 9 * 17), (4, 16, 33 * 65 // 5)])
def test_exchanges_over_gloo(world, N_r, n_modes):
    port = _free_port()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, N_r, n_modes, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=180) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    plan = SlabPlan(N_r=N_r, n_modes=n_modes, world=world)
    for rank, ok_fwd, ok_bwd, s_rad, s_back in res:
        h0, h1 = plan.levels_with_halo(rank)
        e0, e1 = plan.modes(rank)
        assert ok_fwd and ok_bwd
        assert s_rad == (h1 - h0, n_modes) and s_back == (N_r, e1 - e0)
