"""-m gpu: the shared-memory rings in their STEADY STATE.  The small parity tests give every persistent CTA
1-4 tiles, so a ring stage is hardly ever reused and an mbarrier phase never comes back to 0.  Here the launch
is pinned (su3_tune_set) to 32-matrix tiles, ring depth 2 or 3 and ONE CTA per SM on lattices of 1e5-4e5
matrices, so that every CTA (pipeline, matvec) or warp (expression interpreter, Cshift) runs >= 20 tiles --
>= 6 phase flips per stage -- and EVERY element is compared with the oracle (the kernels
are those of DESIGN.md sections 6.1, 11)."""
import functools

import numpy as np
import pytest
import torch

import oracle
import paper_1710_09409_b200 as su3
import su3gen
from gpu_util import download, geom_of, host_field, upload
from helpers import TOL, rel_err

pytestmark = pytest.mark.gpu
F64, F32, SC, VE = su3.SU3_F64, su3.SU3_F32, su3.SU3_SCALAR, su3.SU3_VECTOR
L_CTA = (16, 16, 20, 20)    # 102400 matrices = 3200 tiles of 32: 21.6 tiles per CTA on 148 CTAs
L_WARP = (16, 16, 32, 48)   # 393216 matrices = 12288 tiles of 32: 20.8 tiles per warp on 148 x 4 warps
LAYOUTS = [(SC, 1), (VE, 4), (VE, 8), (VE, 32)]


@pytest.fixture(autouse=True)
def _defaults():
    su3.su3_tune_set()
    yield
    su3.su3_tune_set()


def tiles_per_worker(nmat, workers):
    sms = su3.su3_device_info()["sm_count"]
    return (nmat // 32) / (sms * workers)


@functools.lru_cache(maxsize=16)
def fields(L, prec, layout, W, seed, kinds):
    desc = su3.make_desc(L, prec=prec, layout=layout, W=W)
    return desc, [host_field(desc, seed, f, kind=k) for f, k in enumerate(kinds)]


@pytest.mark.parametrize("stages", [2, 3])
@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("layout,W", LAYOUTS)
def test_pipe_kernel_steady_state_all_ops(prec, layout, W, stages):
    desc, (x, y, w, v) = fields(L_CTA, prec, layout, W, 61, ("su3", "su3", "su3", "gauss"))
    g = geom_of(desc)
    assert tiles_per_worker(g.nmat, 1) >= 20
    fx, fy, fw, fv, z = upload(desc, x), upload(desc, y), upload(desc, w), upload(desc, v), su3.alloc_field(desc)
    su3.su3_tune_set(tile_mats=32, stages=stages, ctas_per_sm=1, path=1)
    for op, call, ref in (("mul", lambda: su3.su3_mul(z, fx, fy), lambda: oracle.mul(g, x, y)),
                          ("mul3", lambda: su3.su3_mul3(z, fx, fy, fw), lambda: oracle.mul3(g, x, y, w)),
                          ("mul_add", lambda: su3.su3_mul_add(z, fx, fy, fv), lambda: oracle.mul_add(g, x, y, v))):
        z.tensor.fill_(0xFF)
        call()
        zg = download(z)
        err, _ = rel_err(zg, ref(), W)
        assert np.isfinite(zg).all() and err <= TOL[prec], (op, err)
    z.tensor.fill_(0xFF)
    su3.su3_add(z, fx, fy)                       # OP_ADD of the same pipeline; one rounding per element: exact
    assert np.array_equal(download(z), x + y)
    # and the launch knobs never change results: the default launch gives the same bits
    su3.su3_mul(z, fx, fy)
    a = download(z)
    su3.su3_tune_set(path=1)
    su3.su3_mul(z, fx, fy)
    assert np.array_equal(download(z), a)


@pytest.mark.parametrize("stages", [2, 3])
@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("layout,W", LAYOUTS)
def test_matvec_kernel_steady_state(prec, layout, W, stages):
    desc, (U, ) = fields(L_CTA, prec, layout, W, 67, ("su3",))
    g = geom_of(desc)
    NPDT = {F64: np.float64, F32: np.float32}
    psi_l = np.ascontiguousarray(su3gen.gaussian_field(67, su3gen.FIELD_V, g.nmat)[:, 0, :]).view(np.float64).reshape(-1)
    gs = oracle.Geom(L_CTA)
    psi = oracle.convert_vec(g, gs, psi_l.astype(NPDT[prec]))
    fU, fpsi, fy = upload(desc, U), su3.alloc_vec(desc), su3.alloc_vec(desc)
    fpsi.tensor.copy_(torch.from_numpy(psi.view(np.uint8)))
    fy.tensor.fill_(0xFF)
    su3.su3_tune_set(tile_mats=32, stages=stages, ctas_per_sm=1)
    su3.su3_matvec(fy, fU, fpsi)
    torch.cuda.synchronize()
    yg = fy.tensor.cpu().numpy().view(NPDT[prec]).astype(np.float64).reshape(-1, 3, W, 2)
    yref = oracle.matvec(g, U, psi).reshape(-1, 3, W, 2)
    err = float((np.abs(yg - yref).max(axis=(1, 3)) / np.abs(yref).max(axis=(1, 3))).max())
    assert np.isfinite(yg).all() and err <= TOL[prec], err


@pytest.mark.parametrize("stages", [2, 3])
@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("layout,W", LAYOUTS)
def test_expr_kernel_steady_state(prec, layout, W, stages):
    desc, hosts = fields(L_WARP, prec, layout, W, 71, ("su3", "gauss", "su3", "gauss"))
    g = geom_of(desc)
    assert tiles_per_worker(g.nmat, 4) >= 20
    fs, z = [upload(desc, h) for h in hosts], su3.alloc_field(desc)
    su3.su3_tune_set(stages=stages, ctas_per_sm=1)
    for prog, n in (("01+01*+", 2), ("01*23*+", 4), ("01*21*-", 3)):
        z.tensor.fill_(0xFF)
        su3.su3_expr(z, prog, fs[:n])
        zg = download(z)
        err, _ = rel_err(zg, oracle.expr(g, prog, *hosts[:n]), W)
        assert np.isfinite(zg).all() and err <= 4 * TOL[prec], (prog, err)   # 4 x: as in test_gpu_expr (several roundings)


@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("layout,W", LAYOUTS)
def test_cshift_ring_steady_state(prec, layout, W):
    desc, (x, y) = fields(L_WARP, prec, layout, W, 73, ("su3", "su3"))
    g = geom_of(desc)
    fx, fy, z = upload(desc, x), upload(desc, y), su3.alloc_field(desc)
    su3.su3_tune_set(ctas_per_sm=1)
    for dim, disp in ((0, 1), (1, -1), (3, 1), (2, 5)):
        z.tensor.fill_(0xFF)
        su3.su3_cshift(z, fy, dim, disp)
        assert np.array_equal(download(z), oracle.cshift(g, y, dim, disp)), (dim, disp)
    for dim, disp in ((0, 1), (3, -1)):
        z.tensor.fill_(0xFF)
        su3.su3_mul_shift(z, fx, fy, dim, disp)
        zg = download(z)
        err, _ = rel_err(zg, oracle.mul_shift(g, x, y, dim, disp), W)
        assert np.isfinite(zg).all() and err <= TOL[prec], (dim, disp, err)
