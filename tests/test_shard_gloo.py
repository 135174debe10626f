"""N > 1 host logic on CPU (gloo, world_size 2): channel sharding needs no collective on the data path
(channels are independent; the paper's multi-GPU plan is one channel range per GPU,
PAPER.md:285).  Each rank correlates only its own channel range (here with the CPU oracle standing in
for the device), the gathered cube must equal the single-process result, and the timing reduction
bench.py uses (max over ranks) must behave."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import paper_1107_4264_b200 as xcb
import xc_workloads as wl
from oracle import xo


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, N, F, T, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        x = wl.gaussian(N, F, T, seed=77, sigma=10.0)              # every rank can regenerate the seeded input
        lo, hi = xcb.shard_channels(F, world, rank)
        mine = xo.correlate_i8(np.ascontiguousarray(x[:, lo:hi]))  # [hi-lo][NB][2][2][2]: a disjoint output slice
        # no collective was needed to compute `mine`; gather only to check the result
        parts = [None] * world
        dist.all_gather_object(parts, (lo, hi, mine))
        cube = np.concatenate([p[2] for p in sorted(parts, key=lambda p: p[0])], axis=0)
        # timing reduction as in bench.py: max over ranks
        t = torch.tensor([1.0 + rank], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        if rank == 0:
            np.save(os.path.join(out_dir, "cube.npy"), cube)
            np.save(os.path.join(out_dir, "tmax.npy"), t.numpy())
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_channel_sharding_world_size_2(tmp_path):
    N, F, T = 12, 5, 40                                            # F odd: uneven shards
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), N, F, T, str(tmp_path)), nprocs=world, join=True)
    cube = np.load(tmp_path / "cube.npy")
    ref = xo.correlate_i8(wl.gaussian(N, F, T, seed=77, sigma=10.0))
    assert np.array_equal(cube, ref)
    assert np.load(tmp_path / "tmax.npy")[0] == float(world)


def _fx_worker(rank, world, port, N, F, T, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import fo
        volt = wl.voltages(N, F, T, seed=78)                       # every rank receives the station time series
        scale = wl.fengine_scale(F)
        lo, hi = xcb.shard_channels(F, world, rank)
        # what xc_fx_channels does on a rank, with the two oracles standing in for the device: full F-point transforms, only
        # the rank's channels of the corner turn are kept (the pruned cube), then the X-engine on them
        cube, _ = fo.fengine(volt, F, scale)
        pruned = np.ascontiguousarray(cube[:, lo:hi])
        mine = xo.correlate_i8(pruned)
        plan = xcb.Plan(N, F, T)                                   # host logic only: sizes of the rank's pruned cube
        pruned_bytes = plan.scratch_pitch * (hi - lo) * T
        parts = [None] * world
        dist.all_gather_object(parts, (lo, hi, mine, pruned_bytes))
        if rank == 0:
            parts.sort(key=lambda p: p[0])
            assert parts[0][0] == 0 and parts[-1][1] == F and all(a[1] == b[0] for a, b in zip(parts[:-1], parts[1:]))
            assert sum(p[3] for p in parts) == int(xcb.lib().xc_cube_bytes(plan._h))      # the shards' cubes add up to the full one
            np.save(os.path.join(out_dir, "fx_cube.npy"), np.concatenate([p[2] for p in parts], axis=0))
        plan.close()
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_fx_channel_sharding_world_size_2(tmp_path):
    """The FX chain under channel sharding (xc_fx_channels): every rank transforms all stations, keeps its
    own channels, correlates them; no collective on the data path; the gathered visibilities equal the unsharded chain and the
    ranks' pruned cubes add up to the full cube's size."""
    from oracle import fo
    N, F, T = 5, 8, 12
    world = 2
    mp.spawn(_fx_worker, args=(world, _free_port(), N, F, T, str(tmp_path)), nprocs=world, join=True)
    cube, _ = fo.fengine(wl.voltages(N, F, T, seed=78), F, wl.fengine_scale(F))
    assert np.array_equal(np.load(tmp_path / "fx_cube.npy"), xo.correlate_i8(cube))
