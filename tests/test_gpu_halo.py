"""-m gpu: the kernels of the multi-GPU shift (su3_face_pack / unpack / copy) against the oracle, bit for bit, and
halo.SlabShift with its CUDA kernels on several slabs held by ONE process (LoopbackComm: a send is a device copy;
no kernel waits on another), compared with the oracle's Cshift / shifted product on the GLOBAL lattice."""
import numpy as np
import pytest
import torch

import oracle
import paper_1710_09409_b200 as su3
import su3gen
from gpu_util import NPDT, download, geom_of, scalar_desc, upload
from helpers import TOL, flat, rel_err
from paper_1710_09409_b200 import halo, shard

pytestmark = pytest.mark.gpu
VEC = su3.SU3_VECTOR


def _slab_desc(gL, world, nl, prec, W):
    lL = (gL[0], gL[1], gL[2], gL[3] // world)
    return su3.make_desc(lL, n_lorentz=nl, prec=prec, layout=VEC if W > 1 else su3.SU3_SCALAR, W=W)


def _global(gL, nl, prec, fid):
    g = oracle.Geom(gL, nl=nl)
    return g, flat(su3gen.su3_field(23, fid, g.nmat), NPDT[prec])


def _slabs(gL, world, nl, prec, W, gflat):
    d = _slab_desc(gL, world, nl, prec, W)
    out = []
    for r in range(world):
        m0, m1 = shard.matrix_range(gL, nl, r, world)
        loc = gflat[m0 * 18:m1 * 18].copy()
        out.append(upload(d, oracle.convert(geom_of(d), geom_of(scalar_desc(d)), loc)))
    return d, out


def _gather(d, fields):
    return np.concatenate([oracle.convert(geom_of(scalar_desc(d)), geom_of(d), download(f)) for f in fields])


@pytest.mark.parametrize("prec", [su3.SU3_F64, su3.SU3_F32])
@pytest.mark.parametrize("L,nl,W,simd", [((6, 4, 2, 8), 1, 1, None), ((4, 4, 4, 8), 4, 4, None), ((4, 2, 4, 4), 1, 8, None),
                                          ((8, 2, 2, 6), 1, 2, (2, 1, 1, 1)), ((2, 4, 4, 4), 1, 32, None)])
def test_face_pack_unpack_copy_bit_exact(prec, L, nl, W, simd):
    d = su3.make_desc(L, n_lorentz=nl, prec=prec, layout=VEC if W > 1 else su3.SU3_SCALAR, W=W, simd=simd)
    g, gs = geom_of(d), geom_of(scalar_desc(d))
    xs = flat(su3gen.gaussian_field(5, 0, gs.nmat), NPDT[prec])
    x = upload(d, oracle.convert(g, gs, xs))
    A = xs.reshape(L[3], L[2], L[1], L[0], nl * 18)                # scalar site order, x0 fastest
    rng = np.random.default_rng(1)
    for dim in range(4):
        for _ in range(3):
            n = int(rng.integers(1, L[dim] + 1))
            p0 = int(rng.integers(0, L[dim] - n + 1))
            q0 = int(rng.integers(0, L[dim] - n + 1))
            sl = [slice(None)] * 4
            sl[3 - dim] = slice(p0, p0 + n)
            want = np.ascontiguousarray(A[tuple(sl)]).reshape(-1)   # the packed face = a scalar field of n planes
            nb = su3.su3_face_bytes(x, dim, n)
            assert nb == want.nbytes
            buf = torch.empty(nb + 64, dtype=torch.uint8, device="cuda")
            buf[nb:] = 0xAB
            su3.su3_face_pack(buf, x, dim, p0, n)
            torch.cuda.synchronize()
            assert np.array_equal(buf[:nb].cpu().numpy().view(NPDT[prec]), want), (dim, p0, n)
            assert bool((buf[nb:] == 0xAB).all())                  # nothing written past the face
            # unpack into other planes of a field full of canaries; the rest must stay untouched
            z = su3.alloc_field(d)
            z.tensor.fill_(0x5C)
            before = download(z)
            su3.su3_face_unpack(z, buf, dim, q0, n)
            B = oracle.convert(gs, g, before).reshape(L[3], L[2], L[1], L[0], nl * 18).copy()
            sq = [slice(None)] * 4
            sq[3 - dim] = slice(q0, q0 + n)
            B[tuple(sq)] = A[tuple(sl)]
            assert np.array_equal(download(z).view(np.uint8), oracle.convert(g, gs, B.reshape(-1)).view(np.uint8)), (dim, q0, n)
            # field -> field copy of the same planes = pack + unpack in one launch
            z2 = su3.alloc_field(d)
            z2.tensor.fill_(0x5C)
            su3.su3_face_copy(z2, q0, x, p0, dim, n)
            torch.cuda.synchronize()
            assert torch.equal(z2.tensor, z.tensor), (dim, p0, q0, n)


def test_face_of_a_colour_vector_field():
    d = su3.make_desc((4, 4, 2, 6), prec=su3.SU3_F64, layout=VEC, W=4)
    g, gs = geom_of(d), geom_of(scalar_desc(d))
    V = 4 * 4 * 2 * 6
    ps = np.random.default_rng(2).standard_normal(V * 6)
    psi = su3.alloc_vec(d)
    psi.tensor.copy_(torch.from_numpy(oracle.convert_vec(g, gs, ps).view(np.uint8)))
    nb = su3.su3_face_bytes(psi, 3, 2)
    assert nb == 4 * 4 * 2 * 2 * 48
    buf = torch.empty(nb, dtype=torch.uint8, device="cuda")
    su3.su3_face_pack(buf, psi, 3, 3, 2)
    torch.cuda.synchronize()
    assert np.array_equal(buf.cpu().numpy().view(np.float64), ps.reshape(6, -1)[3:5].reshape(-1))


@pytest.mark.parametrize("prec", [su3.SU3_F64, su3.SU3_F32])
@pytest.mark.parametrize("world,gL,nl,W", [(2, (8, 4, 4, 12), 1, 1), (2, (8, 4, 4, 12), 1, 4), (3, (4, 4, 4, 12), 4, 4),
                                           (4, (6, 2, 4, 16), 1, 8), (2, (16, 8, 8, 16), 1, 4)])
def test_sharded_shifts_equal_the_oracle_on_the_global_lattice(prec, world, gL, nl, W):
    g, gx = _global(gL, nl, prec, su3gen.FIELD_X)
    _, gy = _global(gL, nl, prec, su3gen.FIELD_Y)
    d, xs = _slabs(gL, world, nl, prec, W, gx)
    _, ys = _slabs(gL, world, nl, prec, W, gy)
    l3 = gL[3] // world
    hub = halo.LoopbackComm(world)
    sh = [halo.SlabShift(hub.for_rank(r)) for r in range(world)]
    for dim, disp in [(3, 1), (3, -1), (3, 2), (3, l3 - 1), (3, l3), (3, l3 + 1), (3, -(l3 + 1)), (3, gL[3] // 2), (3, 5 * gL[3] - 1),
                      (0, 1), (2, -1)]:
        zc = [su3.alloc_field(d) for _ in range(world)]
        zm = [su3.alloc_field(d) for _ in range(world)]
        n0 = su3.su3_launch_count()
        st = [sh[r].start(ys[r], dim, disp) for r in range(world)]          # every rank posts its sends first
        for r in range(world):
            sh[r].finish_cshift(zc[r], st[r])
        st = [sh[r].start(ys[r], dim, disp) for r in range(world)]
        for r in range(world):
            sh[r].finish_mul_shift(zm[r], xs[r], st[r])
        assert su3.su3_launch_count() > n0                                   # the library's own kernels ran
        assert np.array_equal(_gather(d, zc), oracle.cshift(g, gy, dim, disp)), (dim, disp)
        ref = oracle.mul_shift(g, gx, gy, dim, disp)
        e, _ = rel_err(_gather(d, zm), ref, 1)
        assert e <= TOL[prec], (dim, disp, e)
        # and bit-identical to the sharded Cshift followed by the site-local product
        for r in range(world):
            t = su3.alloc_field(d)
            su3.su3_mul(t, xs[r], zc[r])
            torch.cuda.synchronize()
            assert torch.equal(t.tensor, zm[r].tensor), (dim, disp, r)
        # in place (z is x, which su3stream.h allows for the product): x's face is packed before the bulk kernel
        xi = [su3.alloc_field(d) for _ in range(world)]
        for r in range(world):
            xi[r].tensor.copy_(xs[r].tensor)
        st = [sh[r].start(ys[r], dim, disp) for r in range(world)]
        for r in range(world):
            sh[r].finish_mul_shift(xi[r], xi[r], st[r])
        torch.cuda.synchronize()
        for r in range(world):
            assert torch.equal(xi[r].tensor, zm[r].tensor), ("z is x", dim, disp, r)


@pytest.mark.parametrize("prec", [su3.SU3_F64, su3.SU3_F32])
@pytest.mark.parametrize("world,gL,nl,W,simd", [(2, (8, 4, 4, 12), 1, 1, None), (3, (4, 4, 4, 12), 4, 1, None), (2, (8, 4, 4, 12), 1, 4, None),
                                                (2, (8, 4, 4, 8), 1, 4, (2, 2, 1, 1)), (4, (4, 2, 4, 16), 1, 8, (2, 2, 2, 1)),
                                                (2, (16, 8, 8, 16), 1, 1, None), (2, (6, 2, 2, 6), 1, 1, None), (2, (3, 3, 3, 4), 1, 1, None)])
def test_peer_mapped_slabs_one_kernel_exchange(prec, world, gL, nl, W, simd):
    """su3_cshift_slab / halo.PeerShift: the neighbour's slab is read by the shift kernel itself (here: another field on the
    same device stands for peer memory).  Fused (scalar layout, simd[3] = 1) and two-launch (x3 split) variants."""
    g, gx = _global(gL, nl, prec, su3gen.FIELD_X)
    _, gy = _global(gL, nl, prec, su3gen.FIELD_Y)
    lL = (gL[0], gL[1], gL[2], gL[3] // world)
    d = su3.make_desc(lL, n_lorentz=nl, prec=prec, layout=VEC if W > 1 else su3.SU3_SCALAR, W=W, simd=simd)

    def slabs(gflat):
        out = []
        for r in range(world):
            m0, m1 = shard.matrix_range(gL, nl, r, world)
            out.append(upload(d, oracle.convert(geom_of(d), geom_of(scalar_desc(d)), gflat[m0 * 18:m1 * 18].copy())))
        return out
    xs, ys = slabs(gx), slabs(gy)
    ps = halo.PeerShift()
    l3 = lL[3]
    for disp in sorted({v for v in (1, -1, 2, -(l3 - 1), l3 - 1, 0) if abs(v) < l3}):
        zc = [su3.alloc_field(d) for _ in range(world)]
        zm = [su3.alloc_field(d) for _ in range(world)]
        for r in range(world):
            nxt, prv = ys[(r + 1) % world], ys[(r - 1) % world]
            n0 = su3.su3_launch_count()
            ps.cshift(zc[r], ys[r], nxt, prv, disp)
            fused = W == 1 or su3.su3_desc_normalize(d).simd[3] == 1
            if prec == su3.SU3_F32 and W == 1 and (lL[0] * lL[1] * lL[2] * nl) % 2:
                fused = False          # 72-byte records with odd run boundaries: bulk copies cannot be 16-byte aligned
            if disp != 0:
                assert su3.su3_launch_count() - n0 == (1 if fused else 2)
            ps.mul_shift(zm[r], xs[r], ys[r], nxt, prv, disp)
            xi = su3.alloc_field(d)
            xi.tensor.copy_(xs[r].tensor)
            ps.mul_shift(xi, xi, ys[r], nxt, prv, disp)            # in place: z is x
            torch.cuda.synchronize()
            assert torch.equal(xi.tensor, zm[r].tensor), ("z is x", disp, r)
        with pytest.raises(ValueError):
            ps.mul_shift(zm[0], xs[0], ys[0], ys[1 % world], ys[-1 % world], l3)   # refused before any launch
        assert np.array_equal(_gather(d, zc), oracle.cshift(g, gy, 3, disp)), disp
        e, _ = rel_err(_gather(d, zm), oracle.mul_shift(g, gx, gy, 3, disp), 1)
        assert e <= TOL[prec], (disp, e)
    with pytest.raises(su3.Su3Error):
        su3.su3_cshift_slab(zc[0], ys[0], ys[1], l3)
    with pytest.raises(su3.Su3Error):
        su3.su3_cshift_slab(ys[0], ys[0], ys[1], 1)


def test_slab_shift_fuzz():
    """random slab counts, extents, virtual-node splits, precisions and displacements (up to two turns around the global
    lattice): both executors -- packed faces through a communicator, and neighbour slabs read directly -- against the
    oracle's Cshift / shifted product on the global lattice"""
    rng = np.random.default_rng(2026)
    for it in range(40):
        world = int(rng.integers(2, 5))
        W = int(2 ** rng.integers(0, 5))
        simd, w = [1, 1, 1, 1], W
        while w > 1:
            simd[int(rng.integers(0, 4))] *= 2
            w //= 2
        lL = [int(s * rng.integers(1, 5)) for s in simd]
        gL = (lL[0], lL[1], lL[2], lL[3] * world)
        nl, prec = int(rng.choice([1, 4])), int(rng.choice([su3.SU3_F64, su3.SU3_F32]))
        d = su3.make_desc(tuple(lL), n_lorentz=nl, prec=prec, layout=VEC if W > 1 else su3.SU3_SCALAR, W=W,
                          simd=simd if W > 1 else None)
        g, gx = _global(gL, nl, prec, su3gen.FIELD_X)
        _, gy = _global(gL, nl, prec, su3gen.FIELD_Y)

        def slabs(gf):
            out = []
            for r in range(world):
                m0, m1 = shard.matrix_range(gL, nl, r, world)
                out.append(upload(d, oracle.convert(geom_of(d), geom_of(scalar_desc(d)), gf[m0 * 18:m1 * 18].copy())))
            return out
        xs, ys = slabs(gx), slabs(gy)
        hub = halo.LoopbackComm(world)
        sh = [halo.SlabShift(hub.for_rank(r)) for r in range(world)]
        ps = halo.PeerShift()
        zc = [su3.alloc_field(d) for _ in range(world)]
        zm = [su3.alloc_field(d) for _ in range(world)]
        disp = int(rng.integers(-2 * gL[3], 2 * gL[3] + 1))
        st = [sh[r].start(ys[r], 3, disp) for r in range(world)]
        for r in range(world):
            sh[r].finish_cshift(zc[r], st[r])
        st = [sh[r].start(ys[r], 3, disp) for r in range(world)]
        for r in range(world):
            sh[r].finish_mul_shift(zm[r], xs[r], st[r])
        assert np.array_equal(_gather(d, zc), oracle.cshift(g, gy, 3, disp)), (it, gL, world, W, simd, disp)
        e, _ = rel_err(_gather(d, zm), oracle.mul_shift(g, gx, gy, 3, disp), 1)
        assert e <= TOL[prec], (it, gL, world, W, simd, disp, e)
        if lL[3] > 1:
            dp = int(rng.integers(-(lL[3] - 1), lL[3]))
            for r in range(world):
                ps.cshift(zc[r], ys[r], ys[(r + 1) % world], ys[(r - 1) % world], dp)
                ps.mul_shift(zm[r], xs[r], ys[r], ys[(r + 1) % world], ys[(r - 1) % world], dp)
            assert np.array_equal(_gather(d, zc), oracle.cshift(g, gy, 3, dp)), (it, gL, world, W, simd, dp)
            e, _ = rel_err(_gather(d, zm), oracle.mul_shift(g, gx, gy, 3, dp), 1)
            assert e <= TOL[prec], (it, gL, world, W, simd, dp, e)
