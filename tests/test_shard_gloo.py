"""The N>1 path on CPU (gloo, world_size 2): the x3-slab decomposition of SURVEY.md section 8(e) has no
exchange step, so rank-local results concatenated in rank order must equal the single-process result
on the global lattice, in both layouts, and the job throughput is sum(units) / max(time)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
import su3gen
from paper_1710_09409_b200 import shard  # host logic only; importing the package also loads libsu3stream.so


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, gL, nl, W, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        lL, s0, vol = shard.local_extents(gL, rank, world)
        m0, m1 = shard.matrix_range(gL, nl, rank, world)
        n = m1 - m0
        assert n == vol * nl and m0 == s0 * nl
        x = su3gen.su3_field(5, su3gen.FIELD_X, n, m0=m0).view(np.float64).reshape(-1)
        y = su3gen.su3_field(5, su3gen.FIELD_Y, n, m0=m0).view(np.float64).reshape(-1)
        gs = oracle.Geom(lL, nl=nl)
        gv = oracle.Geom(lL, nl=nl, layout=oracle.su3_oracle.VECTOR, W=W)  # virtual nodes INSIDE the rank
        zs = oracle.mul(gs, x, y)
        zv = oracle.mul(gv, oracle.convert(gv, gs, x), oracle.convert(gv, gs, y))
        assert np.array_equal(oracle.convert(gs, gv, zv), zs)
        np.save(os.path.join(out_dir, "z%d.npy" % rank), zs)
        # throughput aggregation: rank r pretends to have taken (r+1) ms for n units
        rate, worst, total = shard.job_throughput(n, float(rank + 1), dist)
        assert worst == float(world) and total == float(n * world) and abs(rate - total / (world * 1e-3)) < 1e-6
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("gL,nl,W", [((4, 4, 2, 8), 1, 4), ((2, 4, 4, 4), 4, 2)])
def test_two_ranks_equal_one_process(tmp_path, gL, nl, W):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), gL, nl, W, str(tmp_path)), nprocs=world, join=True)
    g = oracle.Geom(gL, nl=nl)
    n = g.nmat
    x = su3gen.su3_field(5, su3gen.FIELD_X, n).view(np.float64).reshape(-1)
    y = su3gen.su3_field(5, su3gen.FIELD_Y, n).view(np.float64).reshape(-1)
    zg = oracle.mul(g, x, y)
    zr = np.concatenate([np.load(tmp_path / ("z%d.npy" % r)) for r in range(world)])
    assert np.array_equal(zr, zg)


def test_slabs_partition_the_lattice():
    gL = (6, 4, 2, 12)
    for world in (1, 2, 3, 4, 6):
        ranges = [shard.matrix_range(gL, 4, r, world) for r in range(world)]
        assert ranges[0][0] == 0 and ranges[-1][1] == 6 * 4 * 2 * 12 * 4
        assert all(ranges[r][1] == ranges[r + 1][0] for r in range(world - 1))
        assert shard.weak_global_extents(shard.local_extents(gL, 0, world)[0], world) == gL
    with pytest.raises(ValueError):
        shard.local_extents(gL, 0, 5)
    with pytest.raises(ValueError):
        shard.local_extents(gL, 2, 2)
    assert shard.job_throughput(10, 2.0) == (5000.0, 2.0, 10.0)
