"""-m gpu: real scalar fields and the paper's own example of the expression engine (Listing 2:
v1 = 1.0; v2 = 2.0; v3 = v1+v2; v3 = v1+v2+v1*v2) through su3_fill and su3_expr, against the golden fixture and
the oracle's orc_expr_real."""
import numpy as np
import pytest
import torch

import oracle
import paper_1710_09409_b200 as su3
from test_oracle_pins import load_listing2

pytestmark = pytest.mark.gpu
F64, F32 = su3.SU3_F64, su3.SU3_F32
NP = {F64: np.float64, F32: np.float32}


def down(f):
    torch.cuda.synchronize()
    return f.tensor.cpu().numpy().view(NP[f.desc.prec]).copy()


@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("L", [(8, 8, 8, 8), (3, 3, 3, 3), (1, 1, 1, 1), (5, 3, 1, 7)])
def test_listing2_of_the_paper(prec, L):
    desc = su3.make_desc(L, prec=prec)
    v1, v2, v3 = (su3.alloc_real(desc) for _ in range(3))
    for prog, a, b, want in load_listing2():
        su3.su3_fill(v1, a)
        su3.su3_fill(v2, b)
        v3.tensor.fill_(0xFF)
        su3.su3_expr(v3, prog, [v1, v2])
        got = down(v3)
        assert got.size == int(np.prod(L)) and np.array_equal(got, np.full(got.size, want, dtype=NP[prec])), (prog, L)


@pytest.mark.parametrize("prec", [F64, F32])
def test_real_expressions_against_the_oracle(prec):
    desc = su3.make_desc((6, 5, 7, 3), n_lorentz=4, prec=prec)      # 2520 reals: ragged tail for both vector widths
    n = 6 * 5 * 7 * 3 * 4
    rng = np.random.default_rng(5)
    hosts = [rng.standard_normal(n).astype(NP[prec]) for _ in range(4)]
    fs = []
    for h in hosts:
        f = su3.alloc_real(desc)
        f.tensor.copy_(torch.from_numpy(h.view(np.uint8)))
        fs.append(f)
    z = su3.alloc_real(desc)
    for prog in ["01+", "01*", "01-", "0", "01+01*+", "01*2-0+", "012-*", "01*23*+01-*", "0123+++", "00*0*0*"]:
        k = max(int(c) for c in prog if c.isdigit()) + 1
        z.tensor.fill_(0xFF)
        su3.su3_expr(z, prog, fs[:k])
        ref = oracle.expr_real(prog, *hosts[:k])
        got = down(z).astype(np.float64)
        tol = 1e-14 if prec == F64 else 1e-5
        assert np.isfinite(got).all() and np.abs(got - ref).max() <= tol * max(1.0, np.abs(ref).max()), prog
    # the fixed-menu program `a+b` under every path knob
    for path in (0, 1, 2, 3):
        su3.su3_tune_set(path=path)
        su3.su3_expr(z, "01+", fs[:2])
        assert np.array_equal(down(z), hosts[0] + hosts[1]), path
    su3.su3_tune_set()
    # z may be an operand
    su3.su3_expr(fs[0], "01+", fs[:2])
    assert np.array_equal(down(fs[0]), hosts[0] + hosts[1])


def test_real_kind_is_checked():
    desc = su3.make_desc(4)
    r, m = su3.alloc_real(desc), su3.alloc_field(desc)
    assert su3.su3_real_bytes(desc) == 256 * 8
    n0 = su3.su3_launch_count()
    for call in (lambda: su3.su3_fill(m, 1.0), lambda: su3.su3_expr(r, "01*", [r, m]), lambda: su3.su3_mul(m, m, r),
                 lambda: su3.su3_copy(r, r), lambda: su3.su3_cshift(r, r, 0, 1)):
        with pytest.raises(su3.Su3Error) as e:
            call()
        assert e.value.status == su3.SU3_ERR_MISMATCH
    assert su3.su3_launch_count() == n0


@pytest.mark.parametrize("prec", [F64, F32])
def test_real_menu_programs_equal_the_interpreter(prec):
    """Listing 2's programs on real fields run on ahead-of-time rows of the pipeline kernel: same bits as the interpreter"""
    desc = su3.make_desc((16, 12, 10, 9), n_lorentz=4, prec=prec)     # 69120 reals = 3840 records of 18
    n = 16 * 12 * 10 * 9 * 4
    rng = np.random.default_rng(9)
    hosts = [rng.standard_normal(n).astype(NP[prec]) for _ in range(4)]
    fs = []
    for h in hosts:
        f = su3.alloc_real(desc)
        f.tensor.copy_(torch.from_numpy(h.view(np.uint8)))
        fs.append(f)
    z = su3.alloc_real(desc)
    for prog in ["01+", "01*", "10*", "01-", "01+01*+", "01+2+", "01+2+3+"]:
        k = max(int(c) for c in prog if c.isdigit()) + 1
        assert su3.su3_expr_plan(prog, k, real_fields=True)[0] == "menu", prog
        su3.su3_tune_set()
        z.tensor.fill_(0xFF)
        su3.su3_expr(z, prog, fs[:k])
        got = down(z)
        ref = oracle.expr_real(prog, *hosts[:k])
        tol = 1e-14 if prec == F64 else 1e-5
        assert np.abs(got.astype(np.float64) - ref).max() <= tol * max(1.0, np.abs(ref).max()), prog
        su3.su3_tune_set(path=3)
        z.tensor.fill_(0xFF)
        su3.su3_expr(z, prog, fs[:k])
        assert np.array_equal(down(z), got), prog
    su3.su3_tune_set()
