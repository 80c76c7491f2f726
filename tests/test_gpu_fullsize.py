"""-m gpu: parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (library
defaults), on sampled outputs the oracle computes one matrix at a time, plus properties that hold at
any size (scalar result == vector result bit-for-bit after the permutation, convert round trip = identity,
copy bit-exact, closure of SU(3)).  Element positions inside full-size fields come from the ORACLE's
index function (oracle.index), never from the library's."""
import numpy as np
import pytest
import torch

import oracle
import paper_1710_09409_b200 as su3
import su3gen
from gpu_util import NPDT, geom_of
from helpers import TOL, rel_err

pytestmark = pytest.mark.gpu
F64, F32, SC, VE = su3.SU3_F64, su3.SU3_F32, su3.SU3_SCALAR, su3.SU3_VECTOR
NS = 1500  # sampled sites per check


@pytest.fixture(autouse=True)
def _defaults():
    su3.su3_tune_set()
    yield
    su3.su3_tune_set()
    torch.cuda.empty_cache()


def sample_sites(V, seed):
    """random sites + the places a tiling bug would hit: both ends and tile boundaries"""
    rng = np.random.default_rng(seed)
    edge = [0, 1, 31, 32, 33, 63, 64, 65, 127, 128, 129, 255, 256, V // 2 - 1, V // 2, V - 130, V - 129, V - 128,
            V - 65, V - 64, V - 33, V - 32, V - 2, V - 1]
    s = np.unique(np.concatenate([rng.integers(0, V, NS), np.array([e for e in edge if 0 <= e < V])]))
    return s.astype(np.int64)


def offsets(g, sites):
    """real offsets [len(sites), nl, 18] of the sampled matrices in layout g, from the oracle's index map"""
    out = np.empty((len(sites), g.nl, 18), dtype=np.int64)
    for a, s in enumerate(sites):
        for mu in range(g.nl):
            base = oracle.index(g, int(s), mu, 0, 0, 0)
            if g.layout == oracle.su3_oracle.SCALAR:
                out[a, mu] = base + np.arange(18)
            else:  # element e of lane l: stride 2*W reals between elements (S3); check two of them below
                out[a, mu] = base + (np.arange(18) // 2) * 2 * g.W + np.arange(18) % 2
        if a < 4:  # the closed form above against the oracle, element by element
            for mu in range(g.nl):
                for e in range(9):
                    for ri in range(2):
                        assert out[a, mu, 2 * e + ri] == oracle.index(g, int(s), mu, e // 3, e % 3, ri)
    return out


def gather(field, off):
    t = field.tensor.view(torch.float64 if field.desc.prec == F64 else torch.float32)
    idx = torch.from_numpy(off.reshape(-1)).to(t.device)
    return t[idx].cpu().numpy().reshape(-1)


def host_logical(desc, seed, fid, gauss=False):
    """logical-order (scalar layout) host field in desc's precision, as flat reals"""
    nmat = int(np.prod(list(desc.L))) * desc.n_lorentz
    a = (su3gen.gaussian_field if gauss else su3gen.su3_field)(seed, fid, nmat)
    return a.view(np.float64).reshape(-1).astype(NPDT[desc.prec], copy=False)


def up(desc, h):
    f = su3.alloc_field(desc)
    f.tensor.copy_(torch.from_numpy(h.view(np.uint8)))
    return f


def run_config(L, nl, prec, W, seed, ops):
    ds = su3.make_desc(L, n_lorentz=nl, prec=prec)
    dv = su3.make_desc(L, n_lorentz=nl, prec=prec, layout=VE, W=W)
    gs, gv = geom_of(ds), geom_of(dv)
    V = gs.volume
    sites = sample_sites(V, seed)
    off_s, off_v = offsets(gs, sites), offsets(gv, sites)
    small = oracle.Geom((len(sites), 1, 1, 1), nl=nl)  # the sampled matrices as a tiny scalar-layout field
    hx, hy, hw = (host_logical(ds, seed, f) for f in (su3gen.FIELD_X, su3gen.FIELD_Y, su3gen.FIELD_W))
    hv = host_logical(ds, seed, su3gen.FIELD_V, gauss=True)
    sx, sy, sw, sv = (h[off_s.reshape(-1)] for h in (hx, hy, hw, hv))
    xs, ys, ws, vs = up(ds, hx), up(ds, hy), up(ds, hw), up(ds, hv)
    del hy, hw, hv
    xv, yv, wv, vv = (su3.alloc_field(dv) for _ in range(4))
    for d_, s_ in ((xv, xs), (yv, ys), (wv, ws), (vv, vs)):
        su3.su3_convert(d_, s_)
    # A5 at full size: sampled elements sit where the oracle's map says; round trip is the identity
    assert np.array_equal(gather(xv, off_v), sx)
    back = su3.alloc_field(ds)
    su3.su3_convert(back, xv)
    assert torch.equal(back.tensor, xs.tensor)
    # A6: copy bit-exact
    su3.su3_copy(back, ys)
    assert torch.equal(back.tensor, ys.tensor)
    ref = {"mul": oracle.mul(small, sx, sy), "mul3": oracle.mul3(small, sx, sy, sw),
           "mul_add": oracle.mul_add(small, sx, sy, sv)}
    zs, zv = su3.alloc_field(ds), su3.alloc_field(dv)
    for op in ops:
        third = {"mul": (), "mul3": (ws,), "mul_add": (vs,)}[op]
        third_v = {"mul": (), "mul3": (wv,), "mul_add": (vv,)}[op]
        fn = {"mul": su3.su3_mul, "mul3": su3.su3_mul3, "mul_add": su3.su3_mul_add}[op]
        zs.tensor.fill_(0xFF)
        zv.tensor.fill_(0xFF)
        fn(zs, xs, ys, *third)
        fn(zv, xv, yv, *third_v)
        gz = gather(zs, off_s)
        err, _ = rel_err(gz, ref[op], 1)
        assert np.isfinite(gz).all() and err <= TOL[prec], (op, "scalar", err)
        err, _ = rel_err(gather(zv, off_v), ref[op], 1)
        assert err <= TOL[prec], (op, "vector", err)
        # any-size property: the vector-layout result is the scalar-layout result, bit for bit
        su3.su3_convert(back, zv)
        assert torch.equal(back.tensor, zs.tensor), op
        if op == "mul" and prec == F64:  # closure of SU(3) on the sampled products
            zz = gz.view(np.complex128).reshape(-1, 3, 3)
            assert np.abs(zz @ zz.conj().transpose(0, 2, 1) - np.eye(3)).max() <= 1e-13
            assert np.abs(np.linalg.det(zz) - 1).max() <= 1e-13
    # every byte of the output was written (no 0xFF.. pattern left: NaN payload in both precisions)
    assert not torch.isnan(zs.tensor.view(torch.float64 if prec == F64 else torch.float32)).any()


def test_config5_top_64x4_fp64_bench_configuration():
    run_config(64, 1, F64, 4, su3gen.config_seed(5), ["mul", "mul3", "mul_add"])


def test_config5_64x4_fp32_W8():
    run_config(64, 1, F32, 8, su3gen.config_seed(5), ["mul"])


def test_config3_32x4_lorentz4_fp64():
    run_config(32, 4, F64, 4, su3gen.config_seed(3), ["mul"])


def test_config4_48x4_fp32_W8_fused():
    run_config(48, 1, F32, 8, su3gen.config_seed(4), ["mul3", "mul_add"])


def test_maximum_size_64x4_lorentz4_fp64():
    """the largest field of the configs' shapes: 64^4 x 4 Lorentz matrices, fp64 = 9.66 GB per field (byte
    offsets beyond 2^32, 67M matrices): sampled parity for mul in both layouts, convert, Cshift"""
    L, nl, seed = 64, 4, su3gen.config_seed(3)
    ds = su3.make_desc(L, n_lorentz=nl)
    dv = su3.make_desc(L, n_lorentz=nl, layout=VE, W=4)
    gs, gv = geom_of(ds), geom_of(dv)
    sites = sample_sites(gs.volume, seed)[::3]
    off_s, off_v = offsets(gs, sites), offsets(gv, sites)
    small = oracle.Geom((len(sites), 1, 1, 1), nl=nl)
    hx = host_logical(ds, seed, su3gen.FIELD_X)
    sx = hx[off_s.reshape(-1)]
    xs = up(ds, hx)
    # neighbours of the sampled sites in x3 (the slowest dimension: source 64^3*4 matrices = 151 MB away)
    nb_sites = np.array([oracle.neighbour(gs, int(s), 3, 1) for s in sites], dtype=np.int64)
    sx_nb = hx[offsets(gs, nb_sites).reshape(-1)]
    del hx
    hy = host_logical(ds, seed, su3gen.FIELD_Y)
    sy = hy[off_s.reshape(-1)]
    ys = up(ds, hy)
    del hy
    zs = su3.alloc_field(ds)
    zs.tensor.fill_(0xFF)
    su3.su3_mul(zs, xs, ys)
    ref = oracle.mul(small, sx, sy)
    err, _ = rel_err(gather(zs, off_s), ref, 1)
    assert err <= TOL[F64], err
    assert not torch.isnan(zs.tensor.view(torch.float64)[-18 * 4096:]).any()      # the far end was written
    # Cshift along x3, then the scalar -> vector permutation, at full size
    su3.su3_cshift(zs, xs, 3, 1)
    assert np.array_equal(gather(zs, off_s), sx_nb)
    xv = su3.alloc_field(dv)
    su3.su3_convert(xv, xs)
    assert np.array_equal(gather(xv, off_v), sx)
    del zs
    yv, zv = su3.alloc_field(dv), su3.alloc_field(dv)
    su3.su3_convert(yv, ys)
    su3.su3_mul(zv, xv, yv)
    err, _ = rel_err(gather(zv, off_v), ref, 1)
    assert err <= TOL[F64], err
    su3.su3_mul_shift(zv, xv, yv, 3, 1)
    err, _ = rel_err(gather(zv, off_v), oracle.mul(small, sx, hy_nb(gs, ys, sites)), 1)
    assert err <= TOL[F64], err


def hy_nb(gs, ys, sites):
    """y at the x3-neighbours of the sampled sites, gathered from the device copy of the scalar-layout field"""
    nb_sites = np.array([oracle.neighbour(gs, int(s), 3, 1) for s in sites], dtype=np.int64)
    return gather(ys, offsets(gs, nb_sites))
