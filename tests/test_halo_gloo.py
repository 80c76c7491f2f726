"""The one exchange step of the multi-GPU path (su3_cshift is periodic on the LOCAL
slab): a shift along x3 on x3 slabs.  On CPU: (1) shard.cshift_plan against brute force on plane labels, (2) the
sequencing of paper_1710_09409_b200/halo.py (SlabShift + DistComm) under gloo with world_size 2 and 3, its kernels
replaced by the ORACLE's (an `ops` object defined here, in the tests), compared with the oracle's Cshift and shifted
product on the GLOBAL lattice.  The CUDA kernels of the same sequence are tested in test_gpu_halo.py."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
import su3gen
from paper_1710_09409_b200 import halo, shard

VEC = oracle.su3_oracle.VECTOR


def test_plan_matches_brute_force_on_plane_labels():
    rng = np.random.default_rng(3)
    cases = [(l3, w, d) for l3 in (1, 2, 3, 4, 6) for w in (1, 2, 3, 4, 5) for d in range(-2 * l3 * w - 1, 2 * l3 * w + 2)]
    for l3, world, disp in cases:
        G3 = l3 * world
        glob = rng.integers(0, 1 << 30, G3)                       # a label per global plane
        want = np.roll(glob, -disp)                               # z[p] = x[p + disp]
        slabs = [glob[r * l3:(r + 1) * l3] for r in range(world)]
        for rank in range(world):
            pl = shard.cshift_plan(l3, rank, world, disp)
            assert abs(pl["shift"]) < l3 and pl["nface"] == abs(pl["shift"])
            z = np.roll(slabs[pl["bulk_from"]], -pl["shift"])     # the local periodic shift of the bulk source
            n = pl["nface"]
            if n:
                owner = shard.cshift_plan(l3, pl["face_from"], world, disp)
                assert owner["face_to"] == rank                    # the sender's plan names me
                face = slabs[pl["face_from"]][owner["send_plane0"]:owner["send_plane0"] + n]
                z[pl["dst_plane0"]:pl["dst_plane0"] + n] = face
            assert shard.cshift_plan(l3, pl["bulk_from"], world, disp)["bulk_to"] == rank
            assert np.array_equal(z, want[rank * l3:(rank + 1) * l3]), (l3, world, disp, rank, pl)
    with pytest.raises(ValueError):
        shard.cshift_plan(4, 2, 2, 1)


class _F:
    """a rank's field for OracleOps: geometry + flat fp64 reals in that layout"""
    kind = "matrix"

    def __init__(self, g, a):
        self.g, self.a = g, a


class OracleOps:
    """halo.SlabShift's kernels, restated with the oracle and numpy (test infrastructure)."""

    def _gs(self, g):
        return oracle.Geom(tuple(g.L), nl=g.nl)

    def l3(self, f):
        return f.g.L[3]

    def key(self, f):
        return (tuple(f.g.L), f.g.nl, f.g.layout, f.g.W)

    def _plane_reals(self, f):
        return f.g.L[0] * f.g.L[1] * f.g.L[2] * f.g.nl * 18

    def face_buffer(self, f, n):
        return torch.zeros(n * self._plane_reals(f), dtype=torch.float64)

    def slab_like(self, f):
        return _F(f.g, np.zeros_like(f.a))

    def payload(self, f):
        return torch.from_numpy(f.a)

    def face_pack(self, buf, x, plane0, n):
        s = oracle.convert(self._gs(x.g), x.g, x.a).reshape(x.g.L[3], -1)
        buf.copy_(torch.from_numpy(s[plane0:plane0 + n].reshape(-1).copy()))

    def face_unpack(self, z, buf, plane0, n):
        s = oracle.convert(self._gs(z.g), z.g, z.a).reshape(z.g.L[3], -1)
        s[plane0:plane0 + n] = buf.numpy().reshape(n, -1)
        z.a[:] = oracle.convert(z.g, self._gs(z.g), s.reshape(-1))

    def cshift(self, z, y, dim, disp):
        z.a[:] = oracle.cshift(y.g, y.a, dim, disp)

    def mul_shift(self, z, x, y, dim, disp):
        z.a[:] = oracle.mul_shift(x.g, x.a, y.a, dim, disp)

    def copy(self, z, y):
        z.a[:] = y.a

    def mul(self, z, x, y):
        z.a[:] = oracle.mul(x.g, x.a, y.a)

    def face_mul(self, zb, xb, hb, like, n):
        g = oracle.Geom((like.g.L[0], like.g.L[1], like.g.L[2], n), nl=like.g.nl)
        zb.copy_(torch.from_numpy(oracle.mul(g, xb.numpy(), hb.numpy())))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _fields(gL, nl):
    g = oracle.Geom(gL, nl=nl)
    x = su3gen.su3_field(11, su3gen.FIELD_X, g.nmat).view(np.float64).reshape(-1)
    y = su3gen.su3_field(11, su3gen.FIELD_Y, g.nmat).view(np.float64).reshape(-1)
    return g, x, y


def _worker(rank, world, port, gL, nl, W, disps, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        lL, _, _ = shard.local_extents(gL, rank, world)
        m0, m1 = shard.matrix_range(gL, nl, rank, world)
        _, gx, gy = _fields(gL, nl)
        gs = oracle.Geom(lL, nl=nl)
        g = oracle.Geom(lL, nl=nl, layout=VEC, W=W) if W > 1 else gs
        x = _F(g, oracle.convert(g, gs, gx[m0 * 18:m1 * 18].copy()))
        y = _F(g, oracle.convert(g, gs, gy[m0 * 18:m1 * 18].copy()))
        sh = halo.SlabShift(halo.DistComm(dist), ops=OracleOps())
        for k, (dim, disp) in enumerate(disps):
            zc, zm = _F(g, np.zeros_like(x.a)), _F(g, np.zeros_like(x.a))
            sh.cshift(zc, y, dim, disp)
            sh.mul_shift(zm, x, y, dim, disp)
            xi = _F(g, x.a.copy())
            sh.mul_shift(xi, xi, y, dim, disp)                     # in place: z is x (allowed for the product)
            np.save(os.path.join(out_dir, "i%d_%d.npy" % (k, rank)), oracle.convert(gs, g, xi.a))
            np.save(os.path.join(out_dir, "c%d_%d.npy" % (k, rank)), oracle.convert(gs, g, zc.a))
            np.save(os.path.join(out_dir, "m%d_%d.npy" % (k, rank)), oracle.convert(gs, g, zm.a))
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,gL,nl,W", [(2, (4, 2, 2, 8), 1, 4), (3, (2, 2, 4, 6), 4, 1), (2, (2, 4, 2, 4), 1, 2)])
def test_sharded_shift_equals_global_shift(tmp_path, world, gL, nl, W):
    l3 = gL[3] // world
    disps = [(3, 1), (3, -1), (3, l3), (3, l3 + 1), (3, -(l3 + 1)), (3, gL[3] // 2), (3, 0), (3, gL[3]), (1, 1), (0, -1)]
    if l3 > 2:
        disps.append((3, 2))
    mp.spawn(_worker, args=(world, _free_port(), gL, nl, W, disps, str(tmp_path)), nprocs=world, join=True)
    g, gx, gy = _fields(gL, nl)
    for k, (dim, disp) in enumerate(disps):
        # dim < 3: the shift stays inside every x3 plane, so the slab-local shift IS the global one
        want_c = oracle.cshift(g, gy, dim, disp)
        want_m = oracle.mul_shift(g, gx, gy, dim, disp)
        got_c = np.concatenate([np.load(tmp_path / ("c%d_%d.npy" % (k, r))) for r in range(world)])
        got_m = np.concatenate([np.load(tmp_path / ("m%d_%d.npy" % (k, r))) for r in range(world)])
        assert np.array_equal(got_c, want_c), (dim, disp)
        assert np.array_equal(got_m, want_m), (dim, disp)
        got_i = np.concatenate([np.load(tmp_path / ("i%d_%d.npy" % (k, r))) for r in range(world)])
        assert np.array_equal(got_i, want_m), ("z is x", dim, disp)


def test_second_start_before_finish_is_refused():
    """the face buffers are cached per field shape: two shifts of same-shaped fields in flight would share them, so the
    second start() raises instead of corrupting the first; after the matching finish a new shift may start"""
    gL, world = (2, 2, 2, 8), 2
    g, gx, gy = _fields(gL, 1)
    hub = halo.LoopbackComm(world)
    sh = [halo.SlabShift(hub.for_rank(r), ops=OracleOps()) for r in range(world)]
    ys, zs = [], []
    for r in range(world):
        m0, m1 = shard.matrix_range(gL, 1, r, world)
        gl = oracle.Geom(shard.local_extents(gL, r, world)[0], nl=1)
        ys.append(_F(gl, gy[m0 * 18:m1 * 18].copy()))
        zs.append(_F(gl, np.zeros(ys[-1].a.shape)))
    for _ in range(2):                                             # the guard is released by finish_*: a second round works
        st = [sh[r].start(ys[r], 3, 1) for r in range(world)]
        with pytest.raises(RuntimeError, match="finish"):
            sh[0].start(ys[0], 3, -1)
        local = sh[0].start(ys[0], 1, 1)                           # no exchange: never restricted
        sh[0].finish_cshift(_F(ys[0].g, np.zeros(ys[0].a.shape)), local)
        for r in range(world):
            sh[r].finish_cshift(zs[r], st[r])
        assert np.array_equal(np.concatenate([z.a for z in zs]), oracle.cshift(g, gy, 3, 1))
