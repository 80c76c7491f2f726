"""-m gpu: the one-pass expression evaluator su3_expr (PAPER.md P:76-109,
Listings 1-2) against the oracle's orc_expr, element by element; exact on integer inputs; bit-identical to
the fixed calls on their three programs."""
import numpy as np
import pytest
import torch

import oracle
import paper_1710_09409_b200 as su3
import su3gen
from gpu_util import const_field, download, geom_of, host_field, upload
from helpers import TOL, load_integer_case, rel_err

pytestmark = pytest.mark.gpu
IC = load_integer_case()
F64, F32, SC, VE = su3.SU3_F64, su3.SU3_F32, su3.SU3_SCALAR, su3.SU3_VECTOR
PROGS = ["01*", "10*", "01*2*", "012**", "01*2+", "01+01*+", "01-2*0+", "0", "00*0*1-", "01*21*-", "0123+*-",
         "01*23*+", "01*23*45*++", "01234567*******", "01+2+3+", "01*23*-01+23+*-"]


@pytest.fixture(autouse=True)
def _defaults():
    su3.su3_tune_set()
    yield
    su3.su3_tune_set()


def nops(prog):
    return max(int(c) for c in prog if c.isdigit()) + 1


def run_expr(desc, prog, hosts):
    fs = [upload(desc, h) for h in hosts]
    z = su3.alloc_field(desc)
    z.tensor.fill_(0xFF)
    su3.su3_expr(z, prog, fs)
    return download(z)


@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("layout,W", [(SC, 1), (VE, 4), (VE, 8), (VE, 32)])
def test_expr_integer_inputs_bit_exact(prec, layout, W):
    desc = su3.make_desc((4, 4, 4, 8), prec=prec, layout=layout, W=W)
    k = np.arange(1, 4).reshape(-1, 1, 1)
    mats = [IC["A"] * k, IC["B"], IC["C"], IC["A"] - IC["C"], IC["B"] + IC["C"], IC["C"], IC["A"], IC["B"]]
    hosts = [const_field(desc, m) for m in mats]
    for prog in PROGS:
        if prog in ("01234567*******", "00*0*1-"):   # entries beyond 2^24 would not be exact in fp32
            continue
        n = nops(prog)
        z = run_expr(desc, prog, hosts[:n])
        assert np.array_equal(z.astype(np.float64), oracle.expr(geom_of(desc), prog, *hosts[:n])), prog


@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("L,nl,layout,W", [((4, 6, 4, 8), 1, SC, 1), ((3, 3, 3, 3), 1, SC, 1), ((6, 2, 10, 2), 4, VE, 8),
                                           ((8, 8, 8, 8), 1, VE, 4), ((2, 2, 2, 2), 4, VE, 16)])
def test_expr_random_su3_against_oracle(prec, L, nl, layout, W):
    desc = su3.make_desc(L, n_lorentz=nl, prec=prec, layout=layout, W=W)
    hosts = [host_field(desc, 41, f, kind="su3" if f % 2 == 0 else "gauss") for f in range(8)]
    Wn = su3.su3_desc_normalize(desc).W
    for prog in PROGS:
        n = nops(prog)
        z = run_expr(desc, prog, hosts[:n])
        err, _ = rel_err(z, oracle.expr(geom_of(desc), prog, *hosts[:n]), Wn)
        # products of up to 8 unit-variance Gaussian matrices: a few more roundings than one product
        assert np.isfinite(z).all() and err <= 4 * TOL[prec], (prog, err)


def test_expr_is_bit_identical_to_the_fixed_calls_and_tuning_invariant():
    for desc in (su3.make_desc((8, 8, 8, 6)), su3.make_desc((8, 8, 8, 6), prec=F32, layout=VE, W=8)):
        x, y, w = (host_field(desc, 43, f) for f in (0, 1, 2))
        v = host_field(desc, 43, 3, kind="gauss")
        fx, fy, fw, fv, z = upload(desc, x), upload(desc, y), upload(desc, w), upload(desc, v), su3.alloc_field(desc)
        su3.su3_tune_set(path=1)
        su3.su3_mul(z, fx, fy)
        assert np.array_equal(download(z), run_expr(desc, "01*", [x, y]))
        su3.su3_mul3(z, fx, fy, fw)
        ref3 = download(z)
        assert np.array_equal(ref3, run_expr(desc, "01*2*", [x, y, w]))
        su3.su3_mul_add(z, fx, fy, fv)
        assert np.array_equal(download(z), run_expr(desc, "01*2+", [x, y, v]))
        for tile, stages, ctas in [(32, 2, 1), (64, 4, 1), (32, 3, 3)]:
            su3.su3_tune_set(tile_mats=tile, stages=stages, ctas_per_sm=ctas)
            assert np.array_equal(ref3, run_expr(desc, "01*2*", [x, y, w]))
        su3.su3_tune_set()
        # z may alias an operand
        su3.su3_expr(fx, "01*2*", [fx, fy, fw])
        assert np.array_equal(download(fx), ref3)


def test_expr_errors_launch_nothing():
    desc = su3.make_desc(4)
    a, b = su3.alloc_field(desc), su3.alloc_field(su3.make_desc(4, prec=F32))
    n0 = su3.su3_launch_count()
    with pytest.raises(su3.Su3Error) as e:
        su3.su3_expr(a, "01*", [a, b])
    assert e.value.status == su3.SU3_ERR_MISMATCH
    with pytest.raises(su3.Su3Error) as e:
        su3.su3_expr(a, "0+", [a])
    assert e.value.status == su3.SU3_ERR_INVALID
    assert su3.su3_launch_count() == n0


def _random_program(rng, n_ops, n_operators):
    """a random valid postfix program that uses every operand 0..n_ops-1 (and more pushes as needed)"""
    pushes = n_operators + 1
    leaves = list(range(n_ops)) + [int(rng.integers(0, n_ops)) for _ in range(pushes - n_ops)]
    rng.shuffle(leaves)
    prog, depth, li, ops_left = [], 0, 0, n_operators
    while li < len(leaves) or ops_left:
        can_push = li < len(leaves) and depth < 8
        can_op = depth >= 2 and ops_left
        if can_push and (not can_op or rng.random() < 0.55):
            prog.append(str(leaves[li])); li += 1; depth += 1
        else:
            prog.append("+-*"[int(rng.integers(0, 3))]); depth -= 1; ops_left -= 1
    return "".join(prog)


@pytest.mark.parametrize("prec,layout,W", [(F64, SC, 1), (F32, VE, 8), (F64, VE, 4)])
def test_expr_random_programs_fuzz(prec, layout, W):
    """random trees (deep stacks, several live temporaries, repeated operands) against the oracle's stack machine"""
    rng = np.random.default_rng(20251104 + W)
    desc = su3.make_desc((4, 4, 6, 4), prec=prec, layout=layout, W=W)
    g = geom_of(desc)
    hosts = [host_field(desc, 71, f) for f in range(6)]          # SU(3): products keep unit scale
    fs = [upload(desc, h) for h in hosts]
    z = su3.alloc_field(desc)
    Wn = su3.su3_desc_normalize(desc).W
    abs_hosts = []                                               # (|a|, 0) for every complex number a, in fp64
    for h in hosts:
        a = np.zeros(h.size, dtype=np.float64).reshape(-1, 2)
        a[:, 0] = np.hypot(*h.astype(np.float64).reshape(-1, 2).T)
        abs_hosts.append(a.reshape(-1))
    seen_temps = 0
    for _ in range(60):
        n_ops = int(rng.integers(1, 7))
        n_operators = int(rng.integers(max(1, n_ops - 1), 13))
        prog = _random_program(rng, n_ops, n_operators)
        st, fl = su3.su3_expr_cost(prog, n_ops)
        assert st == n_ops + 1 and fl == 198 * prog.count("*") + 18 * (prog.count("+") + prog.count("-"))
        z.tensor.fill_(0xFF)
        su3.su3_expr(z, prog, fs[:n_ops])
        got, ref = download(z), oracle.expr(g, prog, *hosts[:n_ops])
        # x - x style cancellations make per-matrix relative norms meaningless, so the bar is the componentwise forward
        # error bound of the expression (Higham, Accuracy and Stability, ch. 3): |fl(E) - E| <= gamma_k * E_abs, where E_abs
        # is the SAME program evaluated on the moduli |a_ij| with '-' replaced by '+' (no cancellation left) and
        # k counts the roundings on the longest path: <= 8 per complex product-and-sum of three terms (gamma_3 for the sum,
        # gamma_2 * sqrt(2) for each complex product, FMA or not: about 4.8 u per '*') and 1 per '+'/'-'; K = 8 per operator.
        u = 2.0 ** -53 if prec == F64 else 2.0 ** -24
        K = 8 * (prog.count("*") + prog.count("+") + prog.count("-")) + 4     # + 4: the oracle's own fp64 roundings in fp32 runs
        e_abs = oracle.expr(g, prog.replace("-", "+"), *abs_hosts[:n_ops]).reshape(-1, 2)[:, 0]
        diff = np.hypot(*(got.astype(np.float64) - ref).reshape(-1, 2).T)
        assert np.isfinite(got).all() and (diff <= K * u * e_abs).all(), (prog, float((diff / (u * e_abs)).max()), K)
        seen_temps += prog.count("*") > 2
    assert seen_temps > 10


def test_lattice_front_end_assign():
    from paper_1710_09409_b200.lattice import Lattice
    desc = su3.make_desc((4, 4, 4, 6), prec=F32, layout=VE, W=8)
    hosts = [host_field(desc, 97, f) for f in range(3)]
    x, y, w = (Lattice(upload(desc, h)) for h in hosts)
    z = Lattice(su3.alloc_field(desc))
    z.assign(x * y)
    ref = su3.alloc_field(desc)
    su3.su3_mul(ref, x.field, y.field)
    assert np.array_equal(download(z.field), download(ref))
    z.assign(x + y + x * y - w * x)
    err, _ = rel_err(download(z.field), oracle.expr(geom_of(desc), "01+01*+20*-", *hosts), 8)
    assert err <= 4 * TOL[F32]
    # real scalar fields: the paper's Listing 2, written the paper's way
    v1, v2, v3 = (Lattice(su3.alloc_real(desc)) for _ in range(3))
    su3.su3_fill(v1.field, 1.0)
    su3.su3_fill(v2.field, 2.0)
    v3.assign(v1 + v2 + v1 * v2)
    torch.cuda.synchronize()
    assert bool((v3.field.tensor.view(torch.float32) == 5.0).all())


MENU = [("01+01*+", 2), ("10+01*+", 2), ("01*23*+", 4), ("32*10*+", 4), ("01*23*-", 4), ("01*2-", 3), ("01+2+", 3),
        ("01+2+3+", 4), ("01-", 2), ("10-", 2), ("201*+", 3), ("01*2*3*", 4), ("012**", 3), ("210**", 3), ("01*23**", 4),
        ("32*10**", 4)]


@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("L,nl,layout,W", [((4, 6, 4, 8), 1, SC, 1), ((3, 3, 3, 3), 1, SC, 1), ((6, 2, 10, 2), 4, VE, 8),
                                           ((8, 8, 8, 8), 1, VE, 4), ((2, 2, 2, 2), 4, VE, 16), ((4, 4, 4, 8), 1, VE, 32),
                                           ((16, 16, 8, 10), 1, VE, 2)])
def test_menu_programs_against_oracle_and_interpreter(prec, L, nl, layout, W):
    """the ahead-of-time rows of the pipeline kernel: within tolerance of the oracle, and bit-identical to what the
    interpreter gives for the same program (same order of operations, same FMA chains)"""
    desc = su3.make_desc(L, n_lorentz=nl, prec=prec, layout=layout, W=W)
    g = geom_of(desc)
    hosts = [host_field(desc, 47, f, kind="su3" if f % 2 == 0 else "gauss") for f in range(4)]
    fs, z = [upload(desc, h) for h in hosts], su3.alloc_field(desc)
    Wn = su3.su3_desc_normalize(desc).W
    for prog, n in MENU:
        assert su3.su3_expr_plan(prog, n)[0] == "menu", prog
        su3.su3_tune_set()
        z.tensor.fill_(0xFF)
        su3.su3_expr(z, prog, fs[:n])
        got = download(z)
        ref = oracle.expr(g, prog, *hosts[:n])
        scale = max(np.abs(ref).max(), 1.0)
        assert np.isfinite(got).all() and np.abs(got - ref).max() / scale <= 4 * TOL[prec], prog
        if "-" not in prog:                      # no cancellation: the per-matrix norm of S15 applies as well
            assert rel_err(got, ref, Wn)[0] <= 4 * TOL[prec], prog
        su3.su3_tune_set(path=3)                 # the interpreter
        z.tensor.fill_(0xFF)
        su3.su3_expr(z, prog, fs[:n])
        assert np.array_equal(download(z), got), prog
        for tile, stages, ctas in [(32, 2, 1), (128, 2, 1)]:
            su3.su3_tune_set(tile_mats=tile, stages=stages, ctas_per_sm=ctas)
            su3.su3_expr(z, prog, fs[:n])
            assert np.array_equal(download(z), got), (prog, tile)
    # z may alias any operand of a menu program
    su3.su3_tune_set()
    su3.su3_expr(z, "01*23*+", fs)
    want = download(z)
    su3.su3_expr(fs[3], "01*23*+", fs)
    assert np.array_equal(download(fs[3]), want)


def test_menu_programs_integer_inputs_bit_exact_against_oracle():
    for prec, layout, W in ((F64, SC, 1), (F32, VE, 8), (F64, VE, 4)):
        desc = su3.make_desc((4, 4, 4, 8), prec=prec, layout=layout, W=W)
        k = np.arange(1, 4).reshape(-1, 1, 1)
        hosts = [const_field(desc, m) for m in (IC["A"] * k, IC["B"], IC["C"], IC["A"] - IC["C"])]
        for prog, n in MENU:
            z = run_expr(desc, prog, hosts[:n])
            assert np.array_equal(z.astype(np.float64), oracle.expr(geom_of(desc), prog, *hosts[:n])), prog
