"""-m gpu: colour-vector fields and y = U.psi against the oracle."""
import numpy as np
import pytest
import torch

import oracle
import paper_1710_09409_b200 as su3
import su3gen
from gpu_util import NPDT, const_field, download, geom_of, host_field, scalar_desc, upload
from helpers import TOL, load_integer_case

pytestmark = pytest.mark.gpu
IC = load_integer_case()
F64, F32, SC, VE = su3.SU3_F64, su3.SU3_F32, su3.SU3_SCALAR, su3.SU3_VECTOR


def host_vec(desc, seed, ints=False):
    """seeded colour-vector field in desc's layout and precision"""
    d = su3.su3_desc_normalize(desc)
    nmat = d.L[0] * d.L[1] * d.L[2] * d.L[3] * d.n_lorentz
    if ints:
        a = (np.arange(nmat * 3).reshape(nmat, 3) % 5 - 2) + 1j * (np.arange(nmat * 3).reshape(nmat, 3) % 3 - 1)
    else:
        a = su3gen.gaussian_field(seed, su3gen.FIELD_V, nmat)[:, 0, :]
    f = np.ascontiguousarray(a, dtype=np.complex128).view(np.float64).reshape(-1).astype(NPDT[d.prec])
    if d.layout == VE:
        f = oracle.convert_vec(geom_of(d), geom_of(scalar_desc(d)), f)
    return f


def upload_vec(desc, h):
    f = su3.alloc_vec(desc)
    assert h.nbytes == f.nbytes
    f.tensor.copy_(torch.from_numpy(h.view(np.uint8)))
    return f


def vec_err(y, yref, W):
    a = y.astype(np.float64).reshape(-1, 3, W, 2)
    b = yref.reshape(-1, 3, W, 2)
    num = np.abs(a - b).max(axis=(1, 3))
    den = np.abs(b).max(axis=(1, 3))
    with np.errstate(divide="ignore", invalid="ignore"):
        return float(np.where(num == 0, 0.0, num / den).max())


CASES = [((4, 6, 4, 8), 1, SC, 1), ((3, 3, 3, 3), 1, SC, 1), ((1, 1, 1, 1), 1, SC, 1), ((5, 3, 1, 7), 4, SC, 1),
         ((6, 2, 10, 2), 4, VE, 8), ((8, 8, 8, 8), 1, VE, 4), ((2, 2, 2, 2), 4, VE, 16), ((4, 4, 4, 8), 1, VE, 32),
         ((12, 12, 12, 12), 1, VE, 8), ((16, 16, 8, 9), 1, SC, 1)]


@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("L,nl,layout,W", CASES)
def test_matvec_against_oracle(prec, L, nl, layout, W):
    desc = su3.make_desc(L, n_lorentz=nl, prec=prec, layout=layout, W=W)
    g = geom_of(desc)
    Wn = su3.su3_desc_normalize(desc).W
    U, psi = host_field(desc, 61, su3gen.FIELD_X), host_vec(desc, 61)
    fU, fpsi, fy = upload(desc, U), upload_vec(desc, psi), su3.alloc_vec(desc)
    ref = oracle.matvec(g, U, psi)
    for tile, stages in ((0, 0), (32, 2), (128, 4)):
        su3.su3_tune_set(tile_mats=tile, stages=stages)
        fy.tensor.fill_(0xFF)
        su3.su3_matvec(fy, fU, fpsi)
        y = download(fy)
        assert np.isfinite(y).all() and vec_err(y, ref, Wn) <= TOL[prec], (tile, stages)
    su3.su3_tune_set()
    # exact integer inputs: bit-equal to the oracle
    Ui, pi = const_field(desc, IC["A"] * np.arange(1, 4).reshape(-1, 1, 1)), host_vec(desc, 0, ints=True)
    su3.su3_matvec(fy, upload(desc, Ui), upload_vec(desc, pi))
    assert np.array_equal(download(fy).astype(np.float64), oracle.matvec(g, Ui, pi))
    # y may be psi's field
    su3.su3_matvec(fpsi, fU, fpsi)
    assert vec_err(download(fpsi), ref, Wn) <= TOL[prec]
    # vector-kind fields convert and copy bit-exactly
    if layout == VE:
        ds = scalar_desc(desc)
        ps = host_vec(ds, 61)
        fs, fv, fs2 = upload_vec(ds, ps), su3.alloc_vec(desc), su3.alloc_vec(ds)
        su3.su3_convert(fv, fs)
        su3.su3_convert(fs2, fv)
        assert np.array_equal(download(fv), psi) and np.array_equal(download(fs2), ps)
    fc = su3.alloc_vec(desc)
    su3.su3_copy(fc, upload_vec(desc, psi))
    assert np.array_equal(download(fc), psi)


def test_field_kinds_are_checked():
    desc = su3.make_desc(4)
    m, v = su3.alloc_field(desc), su3.alloc_vec(desc)
    n0 = su3.su3_launch_count()
    for call in (lambda: su3.su3_mul(m, m, v), lambda: su3.su3_matvec(v, v, v), lambda: su3.su3_matvec(m, m, v),
                 lambda: su3.su3_copy(m, v), lambda: su3.su3_cshift(v, v, 0, 1), lambda: su3.su3_expr(m, "01*", [m, v])):
        with pytest.raises(su3.Su3Error) as e:
            call()
        assert e.value.status == su3.SU3_ERR_MISMATCH
    assert su3.su3_launch_count() == n0
