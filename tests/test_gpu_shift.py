"""-m gpu: Cshift and the shifted product against the oracle.
su3_cshift is a permutation: bit-exact.  su3_mul_shift: north_star tolerances, and bit-identical to
su3_cshift followed by su3_mul."""
import numpy as np
import pytest
import torch

import oracle
import paper_1710_09409_b200 as su3
from gpu_util import download, geom_of, host_field, upload
from helpers import TOL, rel_err

pytestmark = pytest.mark.gpu
F64, F32, SC, VE = su3.SU3_F64, su3.SU3_F32, su3.SU3_SCALAR, su3.SU3_VECTOR

CASES = [((4, 6, 4, 8), 1, SC, 1), ((3, 3, 3, 3), 1, SC, 1), ((5, 3, 1, 7), 4, SC, 1), ((6, 2, 10, 2), 4, VE, 8),
         ((8, 8, 8, 8), 1, VE, 4), ((2, 2, 2, 2), 4, VE, 16), ((4, 4, 4, 8), 1, VE, 32), ((10, 6, 6, 2), 1, VE, 2),
         ((12, 12, 12, 12), 1, VE, 8)]


@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("L,nl,layout,W", CASES)
def test_cshift_bit_exact_and_mul_shift(prec, L, nl, layout, W):
    desc = su3.make_desc(L, n_lorentz=nl, prec=prec, layout=layout, W=W)
    g = geom_of(desc)
    x, y = host_field(desc, 51, 0), host_field(desc, 51, 1)
    fx, fy, fz, fs = upload(desc, x), upload(desc, y), su3.alloc_field(desc), su3.alloc_field(desc)
    Wn = su3.su3_desc_normalize(desc).W
    for dim in range(4):
        for disp in (1, -1, 3, L[dim], -2 * L[dim] - 1):
            fz.tensor.fill_(0xFF)
            su3.su3_cshift(fz, fy, dim, disp)
            assert np.array_equal(download(fz), oracle.cshift(g, y, dim, disp)), (dim, disp)
        for disp in (1, -1):
            fz.tensor.fill_(0xFF)
            su3.su3_mul_shift(fz, fx, fy, dim, disp)
            z = download(fz)
            err, _ = rel_err(z, oracle.mul_shift(g, x, y, dim, disp), Wn)
            assert np.isfinite(z).all() and err <= TOL[prec], (dim, disp, err)
            # fused == two passes, bit for bit (same FMA chain)
            su3.su3_cshift(fs, fy, dim, disp)
            su3.su3_tune_set(path=1)
            su3.su3_mul(fs, fx, fs)
            su3.su3_tune_set()
            assert torch.equal(fs.tensor, fz.tensor)


def test_custom_split_and_aliasing_rules():
    desc = su3.make_desc((8, 4, 4, 4), layout=VE, W=8, simd=(4, 2, 1, 1), prec=F32)
    g = geom_of(desc)
    x, y = host_field(desc, 53, 0), host_field(desc, 53, 1)
    fx, fy, fz = upload(desc, x), upload(desc, y), su3.alloc_field(desc)
    for dim in range(4):
        su3.su3_cshift(fz, fx, dim, 1)
        assert np.array_equal(download(fz), oracle.cshift(g, x, dim, 1))
    ref = oracle.mul_shift(g, x, y, 0, 1)
    su3.su3_mul_shift(fx, fx, fy, 0, 1)           # z may be x
    assert rel_err(download(fx), ref, 8)[0] <= TOL[F32]
    n0 = su3.su3_launch_count()
    for call in (lambda: su3.su3_cshift(fy, fy, 0, 1), lambda: su3.su3_mul_shift(fy, fx, fy, 0, 1)):
        with pytest.raises(su3.Su3Error) as e:
            call()
        assert e.value.status == su3.SU3_ERR_MISMATCH
    with pytest.raises(su3.Su3Error) as e:
        su3.su3_cshift(fz, fy, 4, 1)
    assert e.value.status == su3.SU3_ERR_INVALID
    assert su3.su3_launch_count() == n0


def test_cshift_full_size_32x4_lorentz_properties():
    """any-size properties at config 3's size: shift by +1 then -1 is the identity; L shifts of 1 are the identity"""
    desc = su3.make_desc(32, n_lorentz=4, layout=VE, W=4)
    a, b, c = (su3.alloc_field(desc) for _ in range(3))
    a.tensor.view(torch.float64).normal_()
    for dim in range(4):
        su3.su3_cshift(b, a, dim, 1)
        su3.su3_cshift(c, b, dim, -1)
        assert torch.equal(c.tensor, a.tensor)
        assert not torch.equal(b.tensor, a.tensor)
        su3.su3_cshift(c, a, dim, 32)
        assert torch.equal(c.tensor, a.tensor)


def test_random_geometries_and_splits_fuzz():
    """random extents, vector lengths, custom virtual-node splits, Lorentz index and precision: layout permutation
    and Cshift bit-exact against the oracle, products within tolerance"""
    from gpu_util import scalar_desc
    rng = np.random.default_rng(77)
    for it in range(80):
        W = int(2 ** rng.integers(0, 6))
        simd, w = [1, 1, 1, 1], W
        while w > 1:
            simd[int(rng.integers(0, 4))] *= 2
            w //= 2
        L = tuple(int(s * rng.integers(1, 4 if it < 40 else 9)) for s in simd)
        nl = int(rng.choice([1, 4]))
        prec = int(rng.choice([F64, F32]))
        desc = su3.make_desc(L, n_lorentz=nl, prec=prec, layout=VE, W=W, simd=simd)
        g, ds = geom_of(desc), scalar_desc(desc)
        xs = host_field(ds, 90 + it, 0)
        x, y = host_field(desc, 90 + it, 0), host_field(desc, 90 + it, 1)
        fs, fx, fy, fz = upload(ds, xs), su3.alloc_field(desc), upload(desc, y), su3.alloc_field(desc)
        su3.su3_convert(fx, fs)
        assert np.array_equal(download(fx), x), (L, W, simd)
        back = su3.alloc_field(ds)
        su3.su3_convert(back, fx)
        assert np.array_equal(download(back), xs), (L, W, simd)
        dim, disp = int(rng.integers(0, 4)), int(rng.integers(-5, 6))
        su3.su3_tune_set(path=int(rng.choice([0, 0, 1, 2, 3])))          # any of the shift kernels
        su3.su3_cshift(fz, fx, dim, disp)
        assert np.array_equal(download(fz), oracle.cshift(g, x, dim, disp)), (L, W, simd, dim, disp)
        su3.su3_tune_set(path=int(rng.choice([0, 0, 1, 2])))
        su3.su3_mul_shift(fz, fx, fy, dim, disp)
        su3.su3_tune_set()
        err, _ = rel_err(download(fz), oracle.mul_shift(g, x, y, dim, disp), W)
        assert err <= TOL[prec], (L, W, simd, dim, disp, err)
        su3.su3_mul(fz, fx, fy)
        err, _ = rel_err(download(fz), oracle.mul(g, x, y), W)
        assert err <= TOL[prec], (L, W, simd, err)


@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("L,nl,layout,W", [((2, 8, 8, 12), 1, SC, 1), ((4, 2, 6, 16), 1, SC, 1), ((6, 6, 6, 6), 4, SC, 1),
                                           ((3, 5, 2, 16), 1, SC, 1), ((8, 8, 4, 8), 1, VE, 4), ((4, 4, 8, 8), 1, VE, 8),
                                           ((16, 4, 4, 4), 1, VE, 2), ((2, 32, 32, 64), 1, SC, 1), ((4, 16, 16, 64), 1, VE, 2)])
def test_every_shift_kernel_agrees_bitwise(prec, L, nl, layout, W):
    """the kernels behind the `path` knob -- pure TMA copy / pipeline with a shifted slot (runs issued by all lanes, incl.
    tiles with MORE than 32 runs: cycles of 2-4 records along dim 0, and the 8-byte run ends of 72-byte records),
    register kernel, cp.async gather -- give the same bits as the default, which is checked against the oracle"""
    desc = su3.make_desc(L, n_lorentz=nl, prec=prec, layout=layout, W=W)
    g = geom_of(desc)
    x, y = host_field(desc, 53, 0), host_field(desc, 53, 1)
    fx, fy, fz, fr = upload(desc, x), upload(desc, y), su3.alloc_field(desc), su3.alloc_field(desc)
    Wn = su3.su3_desc_normalize(desc).W
    for dim in range(4):
        for disp in (1, -1, 2):
            su3.su3_tune_set()
            su3.su3_cshift(fr, fy, dim, disp)
            assert np.array_equal(download(fr), oracle.cshift(g, y, dim, disp)), (dim, disp)
            for path in (1, 2, 3):
                su3.su3_tune_set(path=path)
                fz.tensor.fill_(0xEE)
                su3.su3_cshift(fz, fy, dim, disp)
                torch.cuda.synchronize()
                assert torch.equal(fz.tensor, fr.tensor), ("cshift", path, dim, disp)
            su3.su3_tune_set()
            su3.su3_mul_shift(fr, fx, fy, dim, disp)
            err, _ = rel_err(download(fr), oracle.mul_shift(g, x, y, dim, disp), Wn)
            assert err <= TOL[prec], (dim, disp, err)
            for path in (1, 2):
                su3.su3_tune_set(path=path)
                fz.tensor.fill_(0xEE)
                su3.su3_mul_shift(fz, fx, fy, dim, disp)
                torch.cuda.synchronize()
                assert torch.equal(fz.tensor, fr.tensor), ("mul_shift", path, dim, disp)
    su3.su3_tune_set()


@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("L,layout,W,simd", [((1, 1, 1, 1), SC, 1, None), ((1, 1, 1, 5), SC, 1, None), ((2, 1, 1, 1), VE, 2, (2, 1, 1, 1)),
                                             ((1, 2, 1, 2), VE, 4, (1, 2, 1, 2)), ((1, 1, 3, 1), SC, 1, None)])
def test_degenerate_lattices(prec, L, layout, W, simd):
    """a single site, a single record, extents of 1: every shift is (partly) the identity, every tile is ragged; shifts,
    the shifted product, the interpreter and the face calls (incl. zero planes) against the oracle"""
    desc = su3.make_desc(L, prec=prec, layout=layout, W=W, simd=simd)
    g = geom_of(desc)
    x, y = host_field(desc, 59, 0), host_field(desc, 59, 1)
    fx, fy, fz = upload(desc, x), upload(desc, y), su3.alloc_field(desc)
    Wn = su3.su3_desc_normalize(desc).W
    for path in (0, 1, 2, 3):
        su3.su3_tune_set(path=path)
        for dim in range(4):
            for disp in (0, 1, -1, 7):
                fz.tensor.fill_(0xEE)
                su3.su3_cshift(fz, fy, dim, disp)
                assert np.array_equal(download(fz), oracle.cshift(g, y, dim, disp)), (path, dim, disp)
                if path < 3:
                    su3.su3_mul_shift(fz, fx, fy, dim, disp)
                    err, _ = rel_err(download(fz), oracle.mul_shift(g, x, y, dim, disp), Wn)
                    assert err <= TOL[prec], (path, dim, disp, err)
    su3.su3_tune_set(path=3)
    for prog in ("01*", "01*01*+", "010**"):
        su3.su3_expr(fz, prog, [fx, fy])
        err, _ = rel_err(download(fz), oracle.expr(g, prog, x, y), Wn)
        assert err <= 4 * TOL[prec], (prog, err)
    su3.su3_tune_set()
    for dim in range(4):
        nb = su3.su3_face_bytes(fx, dim, L[dim])
        assert nb == fx.nbytes and su3.su3_face_bytes(fx, dim, 0) == 0
        buf = torch.empty(max(nb, 16), dtype=torch.uint8, device="cuda")
        n0 = su3.su3_launch_count()
        su3.su3_face_pack(buf, fx, dim, 0, 0)                      # zero planes: nothing is launched
        assert su3.su3_launch_count() == n0
        su3.su3_face_pack(buf, fx, dim, 0, L[dim])                 # all planes: the packed face is the scalar-layout field
        gs = oracle.Geom(L)
        assert np.array_equal(buf[:nb].cpu().numpy().view(x.dtype), oracle.convert(gs, g, x))
