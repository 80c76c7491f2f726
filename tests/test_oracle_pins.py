"""Pins for the CPU oracle (oracle/su3_oracle.c) against things OTHER than itself:
hand-computed integer products (tests/golden), identity / zero, closed-form SU(3)
elements, group invariants, numpy.matmul, pure-Python brute force, hand-computed index
spot values.  PAPER.md prints no worked numeric example (section 4), so every
pin is a closed form, an invariant, an exact integer case or an independent routine.
CPU only (-m "not gpu")."""
import itertools

import numpy as np
import pytest

import oracle
import su3gen
from helpers import flat, load_integer_case, load_vector_map_spots, logical, rel_err

IC = load_integer_case()


def fill(g, mat, dtype=np.float64):
    """every matrix of the (scalar-layout) field = mat"""
    return flat(np.broadcast_to(mat, (g.nmat, 3, 3)).copy(), dtype)


# ---------------------------------------------------------------- arithmetic pins
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_integer_case_exact(dtype):
    g = oracle.Geom(2)
    A, B, C = fill(g, IC["A"], dtype), fill(g, IC["B"], dtype), fill(g, IC["C"], dtype)
    assert np.array_equal(logical(oracle.mul(g, A, B)), np.broadcast_to(IC["AB"], (16, 3, 3)))
    assert np.array_equal(logical(oracle.mul(g, B, A)), np.broadcast_to(IC["BA"], (16, 3, 3)))
    assert np.array_equal(logical(oracle.mul3(g, A, B, C)), np.broadcast_to(IC["ABC"], (16, 3, 3)))
    assert np.array_equal(logical(oracle.mul_add(g, A, B, C)), np.broadcast_to(IC["AB+C"], (16, 3, 3)))
    # operand order matters (catches swapped/transposed operands); traces agree
    assert not np.array_equal(IC["AB"], IC["BA"])
    assert np.trace(IC["AB"]) == np.trace(IC["BA"]) == 6 + 4j


def test_integer_case_fixture_is_self_consistent():
    """exact Gaussian-integer brute force (pure Python ints) on the stored fixture"""
    def ints(m):
        return [[(int(m[i, j].real), int(m[i, j].imag)) for j in range(3)] for i in range(3)]

    def cm(a, b):
        return (a[0] * b[0] - a[1] * b[1], a[0] * b[1] + a[1] * b[0])

    def mm(a, b):
        return [[tuple(map(sum, zip(*[cm(a[i][k], b[k][j]) for k in range(3)]))) for j in range(3)]
                for i in range(3)]

    def det(a):
        def sub(p, q):
            return (p[0] - q[0], p[1] - q[1])
        t0 = cm(a[0][0], sub(cm(a[1][1], a[2][2]), cm(a[1][2], a[2][1])))
        t1 = cm(a[0][1], sub(cm(a[1][0], a[2][2]), cm(a[1][2], a[2][0])))
        t2 = cm(a[0][2], sub(cm(a[1][0], a[2][1]), cm(a[1][1], a[2][0])))
        return (t0[0] - t1[0] + t2[0], t0[1] - t1[1] + t2[1])

    A, B, C = ints(IC["A"]), ints(IC["B"]), ints(IC["C"])
    assert mm(A, B) == ints(IC["AB"]) and mm(B, A) == ints(IC["BA"])
    assert mm(mm(A, B), C) == ints(IC["ABC"]) == mm(A, mm(B, C))
    assert det(A) == (-4, 8) == (IC["detA"].real, IC["detA"].imag)
    assert det(B) == (-2, 6) and det(mm(A, B)) == (-40, -40) == cm(det(A), det(B))


def test_site_dependent_integer_field_both_layouts():
    """A scaled by (1 + site mod 7): tests indexing as well as arithmetic, exactly."""
    for layout, W in [(0, 1), (1, 4), (1, 8)]:
        g = oracle.Geom(4, nl=4, layout=layout, W=W)
        gs = oracle.Geom(4, nl=4)
        scale = (1 + (np.arange(gs.nmat) // 4) % 7).astype(np.float64)
        mu = (np.arange(gs.nmat) % 4 + 1).astype(np.float64)
        xa = IC["A"][None] * scale[:, None, None]
        yb = IC["B"][None] * mu[:, None, None]
        x, y = oracle.convert(g, gs, flat(xa)), oracle.convert(g, gs, flat(yb))
        z = logical(oracle.convert(gs, g, oracle.mul(g, x, y)))
        assert np.array_equal(z, IC["AB"][None] * (scale * mu)[:, None, None])


def test_identity_and_zero():
    g = oracle.Geom(4)
    x = flat(su3gen.su3_field(11, 0, g.nmat))
    v = flat(su3gen.gaussian_field(11, 3, g.nmat))
    one, zero = fill(g, np.eye(3)), fill(g, np.zeros((3, 3)))
    assert np.array_equal(oracle.mul(g, x, one), x)   # x.1 = x (value-equal)
    assert np.array_equal(oracle.mul(g, one, x), x)   # 1.y = y
    assert np.all(oracle.mul(g, x, zero) == 0)
    assert np.all(oracle.mul(g, zero, x) == 0)
    assert np.array_equal(oracle.mul_add(g, zero, x, v), v)
    assert np.array_equal(oracle.mul3(g, x, one, one), x)


def test_closed_form_su3_elements():
    g = oracle.Geom(2)
    P = np.array([[0, 1, 0], [0, 0, 1], [1, 0, 0]], dtype=complex)
    PP = logical(oracle.mul(g, fill(g, P), fill(g, P)))[0]
    assert np.array_equal(PP, np.array([[0, 0, 1], [1, 0, 0], [0, 1, 0]]))
    assert np.array_equal(logical(oracle.mul3(g, fill(g, P), fill(g, P), fill(g, P)))[3], np.eye(3))

    def D(a, b):
        return np.diag([np.exp(1j * a), np.exp(1j * b), np.exp(-1j * (a + b))])
    got = logical(oracle.mul(g, fill(g, D(0.3, -1.1)), fill(g, D(0.9, 0.25))))[5]
    assert np.abs(got - D(1.2, -0.85)).max() < 4e-16

    R = np.array([[.6, .8, 0], [-.8, .6, 0], [0, 0, 1]], dtype=complex)
    RR = np.array([[-.28, .96, 0], [-.96, -.28, 0], [0, 0, 1]])
    assert np.abs(logical(oracle.mul(g, fill(g, R), fill(g, R)))[0] - RR).max() < 3e-16
    U = np.array([[.6, .8j, 0], [.8j, .6, 0], [0, 0, 1]])
    UR = np.array([[.36 - .64j, .48 + .48j, 0], [-.48 + .48j, .36 + .64j, 0], [0, 0, 1]])
    assert np.abs(logical(oracle.mul(g, fill(g, U), fill(g, R)))[7] - UR).max() < 3e-16


def test_group_invariants_random_su3():
    g = oracle.Geom(8)
    seed = su3gen.config_seed(1)
    x, y = su3gen.su3_field(seed, 0, g.nmat), su3gen.su3_field(seed, 1, g.nmat)
    z = logical(oracle.mul(g, flat(x), flat(y)))
    eye = np.eye(3)
    assert np.abs(z @ z.conj().transpose(0, 2, 1) - eye).max() <= 1e-13       # closure: unitarity
    assert np.abs(np.linalg.det(z) - 1).max() <= 1e-13                        # det = 1
    assert np.abs(np.linalg.norm(z, axis=(1, 2)) - np.sqrt(3)).max() < 1e-14  # Frobenius norm
    zyx = logical(oracle.mul(g, flat(y), flat(x)))
    assert np.abs(np.trace(z, axis1=1, axis2=2) - np.trace(zyx, axis1=1, axis2=2)).max() < 1e-14
    # (x y)^dagger = y^dagger x^dagger
    xd, yd = x.conj().transpose(0, 2, 1), y.conj().transpose(0, 2, 1)
    zd = logical(oracle.mul(g, flat(np.ascontiguousarray(yd)), flat(np.ascontiguousarray(xd))))
    assert np.abs(zd - z.conj().transpose(0, 2, 1)).max() < 1e-15


def test_associativity_of_mul3():
    g = oracle.Geom(4)
    x, y, w = (flat(su3gen.su3_field(7, f, g.nmat)) for f in (0, 1, 2))
    left = oracle.mul3(g, x, y, w)                 # (x y) w
    right = oracle.mul(g, x, oracle.mul(g, y, w))  # x (y w)
    assert rel_err(left, right, 1)[0] < 5e-15
    assert np.array_equal(left, oracle.mul(g, oracle.mul(g, x, y), w))  # left-assoc. by definition


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_numpy_matmul_crosscheck(dtype):
    """the product reduces to a batched complex matmul: an independent library routine"""
    g = oracle.Geom(8, nl=4)
    seed = su3gen.config_seed(3)
    xs, ys, ws = (flat(su3gen.su3_field(seed, f, g.nmat), dtype) for f in (0, 1, 2))
    vs = flat(su3gen.gaussian_field(seed, 3, g.nmat), dtype)
    x, y, w, v = (logical(a.astype(np.float64)) for a in (xs, ys, ws, vs))  # the rounded inputs (S16)
    assert rel_err(oracle.mul(g, xs, ys), flat(x @ y), 1)[0] <= 1e-15
    assert rel_err(oracle.mul3(g, xs, ys, ws), flat((x @ y) @ w), 1)[0] <= 2e-15
    assert rel_err(oracle.mul_add(g, xs, ys, vs), flat(x @ y + v), 1)[0] <= 1e-15


def test_brute_force_tiny():
    """pure-Python triple loop with Python complex numbers on a 2^4 lattice, vector layout"""
    g = oracle.Geom(2, layout=1, W=2)
    gs = oracle.Geom(2)
    x, y = su3gen.su3_field(3, 0, 16), su3gen.gaussian_field(3, 1, 16)
    z = oracle.mul(g, oracle.convert(g, gs, flat(x)), oracle.convert(g, gs, flat(y)))
    for site in range(16):
        for i in range(3):
            for j in range(3):
                ref = sum(complex(x[site, i, k]) * complex(y[site, k, j]) for k in range(3))
                got = complex(z[oracle.index(g, site, 0, i, j, 0)], z[oracle.index(g, site, 0, i, j, 1)])
                assert abs(got - ref) < 1e-15 * max(1.0, abs(ref))


def test_det_multiplicative_integer_case():
    assert IC["detA"] * IC["detB"] == IC["detAB"]
    assert np.linalg.det(IC["AB"]) == pytest.approx(IC["detAB"], abs=1e-12)


# ---------------------------------------------------------------- layout pins
def test_vector_map_spot_values():
    spots, splits = load_vector_map_spots()
    for W, s in splits.items():
        assert oracle.default_simd(W) == s
    for sp in spots:
        L = sp["L"]
        g = oracle.Geom(L, layout=1, W=sp["W"])
        x = sp["x"]
        site = x[0] + L * (x[1] + L * (x[2] + L * x[3]))
        assert site == sp["site"]
        assert oracle.site_to_outer(g, site) == (sp["outer"], sp["lane"])
        assert oracle.index(g, site, 0, 1, 2, 1) == ((sp["outer"] * 9 + 5) * sp["W"] + sp["lane"]) * 2 + 1


def test_scalar_index_formula():
    g = oracle.Geom((2, 3, 4, 5), nl=4)
    # site 37 = x0 + 2*(x1 + 3*(x2 + 4*x3)): element (i=2,j=1) of mu=3, imaginary part
    assert oracle.index(g, 37, 3, 2, 1, 1) == ((37 * 4 + 3) * 9 + 7) * 2 + 1
    assert oracle.index(g, 0, 0, 0, 0, 0) == 0
    assert oracle.index(g, g.volume - 1, 3, 2, 2, 1) == g.nreals - 1


@pytest.mark.parametrize("L,W,nl,simd", [
    (4, 1, 1, None), (4, 2, 1, None), (8, 4, 1, None), (8, 8, 4, None), (4, 16, 1, None),
    (4, 32, 1, None), (12, 8, 1, None), ((4, 6, 2, 8), 4, 4, None), (4, 4, 1, (4, 1, 1, 1)),
    ((8, 4, 4, 2), 8, 1, (2, 2, 2, 1))])
def test_vector_index_is_a_bijection(L, W, nl, simd):
    g = oracle.Geom(L, nl=nl, layout=1, W=W, simd=simd)
    seen = np.zeros(g.nreals, dtype=np.int32)
    Lx = g.L
    for site in range(g.volume):
        o, l = oracle.site_to_outer(g, site)
        assert 0 <= o < g.volume // W and 0 <= l < W
        # the sites of one outer site are one per sub-lattice (far apart), reading S3
        x = [site % Lx[0], site // Lx[0] % Lx[1], site // (Lx[0] * Lx[1]) % Lx[2], site // (Lx[0] * Lx[1] * Lx[2])]
        r = [Lx[d] // g.simd[d] for d in range(4)]
        assert l == sum((x[d] // r[d]) * int(np.prod(g.simd[:d])) for d in range(4))
        for mu in range(nl):
            seen[oracle.index(g, site, mu, 0, 0, 0)] += 1
            seen[oracle.index(g, site, mu, 2, 2, 1)] += 1
    assert seen.max() == 1 and seen.sum() == 2 * g.nmat
    # full bijection through convert: a ramp maps to a permutation of itself
    gs = oracle.Geom(L, nl=nl)
    ramp = np.arange(g.nreals, dtype=np.float64)
    v = oracle.convert(g, gs, ramp)
    assert np.array_equal(np.sort(v), ramp)


def test_inadmissible_geometries():
    for kw in [dict(L=8, nl=3), dict(L=8, layout=0, W=4), dict(L=8, layout=1, W=3), dict(L=8, layout=1, W=64),
               dict(L=(8, 8, 8, 3), layout=1, W=2), dict(L=8, layout=1, W=4, simd=(2, 1, 1, 1)),
               dict(L=(8, 8, 0, 8)), dict(L=8, layout=2)]:
        with pytest.raises(ValueError):
            oracle.Geom(**kw)


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_layout_agreement_bit_exact(dtype):
    """oracle on the vector layout, converted back, equals oracle on the scalar layout bit for bit"""
    seed = su3gen.config_seed(2)
    for L, W, nl in [(8, 4, 1), (8, 8, 4), (4, 16, 1), (4, 2, 4)]:
        gs, gv = oracle.Geom(L, nl=nl), oracle.Geom(L, nl=nl, layout=1, W=W)
        xs, ys, ws = (flat(su3gen.su3_field(seed, f, gs.nmat), dtype) for f in (0, 1, 2))
        vs = flat(su3gen.gaussian_field(seed, 3, gs.nmat), dtype)
        xv, yv, wv, vv = (oracle.convert(gv, gs, a) for a in (xs, ys, ws, vs))
        assert np.array_equal(oracle.convert(gs, gv, oracle.mul(gv, xv, yv)), oracle.mul(gs, xs, ys))
        assert np.array_equal(oracle.convert(gs, gv, oracle.mul3(gv, xv, yv, wv)), oracle.mul3(gs, xs, ys, ws))
        assert np.array_equal(oracle.convert(gs, gv, oracle.mul_add(gv, xv, yv, vv)),
                              oracle.mul_add(gs, xs, ys, vs))


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_convert_round_trip_and_w1(dtype):
    rng = np.random.default_rng(5)
    for L, W, nl in [(8, 4, 1), (4, 8, 4), (4, 32, 1)]:
        gs, gv = oracle.Geom(L, nl=nl), oracle.Geom(L, nl=nl, layout=1, W=W)
        a = rng.standard_normal(gs.nreals).astype(dtype)
        v = oracle.convert(gv, gs, a)
        assert not np.array_equal(v, a)
        assert np.array_equal(oracle.convert(gs, gv, v), a)               # s -> v -> s
        assert np.array_equal(oracle.convert(gv, gs, oracle.convert(gs, gv, a)), a)  # v -> s -> v
        # explicit definition: vec[o][mu][e][l] = sca[site(o,l)][mu][e]
        vv = v.reshape(-1, nl, 9, W, 2)
        aa = a.reshape(-1, nl, 9, 2)
        for site in rng.integers(0, gs.volume, 50):
            o, l = oracle.site_to_outer(gv, int(site))
            assert np.array_equal(vv[o, :, :, l, :], aa[site])
    g1, gs = oracle.Geom(4, nl=4, layout=1, W=1), oracle.Geom(4, nl=4)
    a = rng.standard_normal(gs.nreals).astype(dtype)
    assert np.array_equal(oracle.convert(g1, gs, a), a)  # W=1 vector layout == scalar layout, byte for byte
    with pytest.raises(ValueError):
        oracle.convert(oracle.Geom((2, 8, 4, 4), nl=4), gs, a)  # same size, different extents


def test_fp32_inputs_are_promoted_not_rounded():
    """S16: fp32 storage is read, promoted exactly, result kept in double"""
    g = oracle.Geom(2)
    x = flat(su3gen.su3_field(9, 0, g.nmat), np.float32)
    y = flat(su3gen.su3_field(9, 1, g.nmat), np.float32)
    z32 = oracle.mul(g, x, y)
    assert z32.dtype == np.float64
    assert np.array_equal(z32, oracle.mul(g, x.astype(np.float64), y.astype(np.float64)))
    assert np.abs(z32 - z32.astype(np.float32)).max() > 0  # not rounded to fp32


# ---------------------------------------------------------------- the postfix expression evaluator (f2)
def _py_postfix(prog, mats):
    """pure-Python reference: exact Gaussian-integer 3x3 arithmetic on lists of Python complex/int"""
    st = []
    for t in prog:
        if t.isdigit():
            st.append(mats[int(t)])
        else:
            b, a = st.pop(), st.pop()
            if t == "*":
                st.append([[sum(a[i][k] * b[k][j] for k in range(3)) for j in range(3)] for i in range(3)])
            else:
                sg = 1 if t == "+" else -1
                st.append([[a[i][j] + sg * b[i][j] for j in range(3)] for i in range(3)])
    assert len(st) == 1
    return np.array(st[0], dtype=np.complex128)


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("prog", ["01*", "10*", "01*2*", "012**", "01*2+", "01+01*+", "01-2*0+", "0", "00*0*1-",
                                  "01*21*-", "0123+*-"])
def test_expr_integer_cases_exact(prog, dtype):
    """Listing 2's pattern (P:104-106 `v3=v1+v2+v1*v2`) and friends on the exact integer matrices of the
    golden fixture: brute force in Python integers, independent of the oracle"""
    g = oracle.Geom(2, layout=oracle.su3_oracle.VECTOR, W=4) if dtype == np.float32 else oracle.Geom(2)
    names = ["A", "B", "C", "AB"]
    gs = oracle.Geom(2)
    fields = [fill(gs, IC[n], dtype) for n in names]
    if g.layout:
        fields = [oracle.convert(g, gs, f) for f in fields]
    z = oracle.expr(g, prog, *fields)
    if g.layout:
        z = oracle.convert(gs, g, z)
    want = _py_postfix(prog, [[[complex(v) for v in row] for row in IC[n]] for n in names])
    assert np.array_equal(logical(z), np.broadcast_to(want, (16, 3, 3)))


def test_expr_matches_fixed_calls_and_numpy():
    g = oracle.Geom((4, 2, 2, 3), nl=4)
    x, y, w = (flat(su3gen.su3_field(3, f, g.nmat)) for f in (0, 1, 2))
    v = flat(su3gen.gaussian_field(3, 3, g.nmat))
    assert np.array_equal(oracle.expr(g, "01*", x, y), oracle.mul(g, x, y))
    assert np.array_equal(oracle.expr(g, "01*2*", x, y, w), oracle.mul3(g, x, y, w))
    assert np.array_equal(oracle.expr(g, "01*2+", x, y, v), oracle.mul_add(g, x, y, v))
    X, Y, W_, V = logical(x), logical(y), logical(w), logical(v)
    z = logical(oracle.expr(g, "01+01*+23*-", x, y, w, v))
    want = X + Y + X @ Y - W_ @ V
    assert np.abs(z - want).max() <= 1e-14
    # algebra: x - x = 0 exactly; (x+y)*w = x*w + y*w to rounding
    assert not oracle.expr(g, "00-", x).any()
    d = oracle.expr(g, "01+2*", x, y, w) - oracle.expr(g, "02*12*+", x, y, w)
    assert np.abs(d).max() <= 1e-14


def test_expr_rejects_malformed_programs():
    g = oracle.Geom(2)
    x = fill(g, IC["A"])
    for bad in ["", "0+", "00", "01*", "0a*", "00*+", "000000000********"]:
        with pytest.raises(ValueError):
            oracle.expr(g, bad, x)


# ---------------------------------------------------------------- Cshift and the shifted product (f3)
def test_neighbour_spot_values_by_hand():
    g = oracle.Geom((4, 2, 3, 2))  # strides 1, 4, 8, 24
    assert oracle.neighbour(g, 0, 0, 1) == 1 and oracle.neighbour(g, 3, 0, 1) == 0      # wrap in x0
    assert oracle.neighbour(g, 0, 0, -1) == 3 and oracle.neighbour(g, 5, 1, 1) == 1      # x=(1,1,..) -> (1,0,..)
    assert oracle.neighbour(g, 5, 2, 1) == 13 and oracle.neighbour(g, 21, 2, 1) == 5     # x2: 2 -> 0 wraps
    assert oracle.neighbour(g, 47, 3, 1) == 23 and oracle.neighbour(g, 47, 3, 2) == 47
    assert oracle.neighbour(g, 7, 0, 9) == oracle.neighbour(g, 7, 0, 1)


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("L,nl,W", [((4, 2, 6, 2), 1, 1), ((4, 4, 4, 4), 4, 4), ((2, 4, 6, 4), 1, 8), ((4, 4, 4, 8), 1, 32)])
def test_cshift_equals_numpy_roll_in_every_layout(L, nl, W, dtype):
    gs = oracle.Geom(L, nl=nl)
    g = gs if W == 1 else oracle.Geom(L, nl=nl, layout=oracle.su3_oracle.VECTOR, W=W)
    a = su3gen.gaussian_field(9, 0, gs.nmat)
    x = flat(a, dtype)
    xl = x if W == 1 else oracle.convert(g, gs, x)
    grid = x.reshape(L[3], L[2], L[1], L[0], nl, 18)
    for dim in range(4):
        for disp in (1, -1, 2, L[dim], -L[dim] - 1):
            z = oracle.cshift(g, xl, dim, disp)
            zs = z if W == 1 else oracle.convert(gs, g, z)
            want = np.roll(grid, -disp, axis=3 - dim).reshape(-1)   # z[x] = x[x + disp]
            assert np.array_equal(zs, want), (dim, disp)


def test_cshift_group_structure_and_mul_shift():
    g = oracle.Geom((4, 4, 2, 6), nl=1, layout=oracle.su3_oracle.VECTOR, W=4)
    gs = oracle.Geom((4, 4, 2, 6))
    x, y = (oracle.convert(g, gs, flat(su3gen.su3_field(9, f, gs.nmat))) for f in (0, 1))
    assert np.array_equal(oracle.cshift(g, oracle.cshift(g, x, 2, 1), 2, -1), x)
    assert np.array_equal(oracle.cshift(g, oracle.cshift(g, x, 3, 2), 3, 3), oracle.cshift(g, x, 3, 5))
    assert np.array_equal(oracle.cshift(g, oracle.cshift(g, x, 0, 1), 3, 1), oracle.cshift(g, oracle.cshift(g, x, 3, 1), 0, 1))
    assert np.array_equal(oracle.cshift(g, x, 1, 4), x)
    for dim, disp in [(0, 1), (3, -1), (2, 1)]:
        assert np.array_equal(oracle.mul_shift(g, x, y, dim, disp), oracle.mul(g, x, oracle.cshift(g, y, dim, disp)))
    # the shifted product of SU(3) fields is SU(3); with y = x^dagger-free check: unitarity only
    z = logical(oracle.convert(gs, g, oracle.mul_shift(g, x, y, 1, 1)))
    assert np.abs(z @ z.conj().transpose(0, 2, 1) - np.eye(3)).max() <= 1e-13
    with pytest.raises(ValueError):
        oracle.cshift(g, x, 4, 1)


# ---------------------------------------------------------------- colour vectors and y = U.psi (f4)
def test_matvec_integer_case_by_hand_and_numpy():
    """A.(1, i, 2-i)^T by hand: row0 = (1+2i) + (-i)(i) + 3(2-i) = 8-i; row1 = (2-i) + (1+i)i = 1;
    row2 = i - 2i + (1-i)(2-i) = 1-4i"""
    g = oracle.Geom(2)
    psi1 = np.array([1, 1j, 2 - 1j])
    U = fill(g, IC["A"])
    psi = np.ascontiguousarray(np.broadcast_to(psi1, (g.nmat, 3))).view(np.float64).reshape(-1)
    y = oracle.matvec(g, U, psi).view(np.complex128).reshape(-1, 3)
    assert np.array_equal(y, np.broadcast_to(np.array([8 - 1j, 1, 1 - 4j]), (16, 3)))
    assert np.array_equal(IC["A"] @ psi1, np.array([8 - 1j, 1, 1 - 4j]))


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_matvec_invariants_layouts_and_einsum(dtype):
    L, nl = (4, 2, 4, 2), 4
    gs = oracle.Geom(L, nl=nl)
    U = flat(su3gen.su3_field(21, 0, gs.nmat), dtype)
    V = flat(su3gen.su3_field(21, 1, gs.nmat), dtype)
    psi = su3gen.gaussian_field(21, 3, gs.nmat)[:, 0, :].copy().view(np.float64).reshape(-1).astype(dtype)
    y = oracle.matvec(gs, U, psi)
    Ul, pl = logical(U), psi.astype(np.float64).view(np.complex128).reshape(-1, 3)
    want = np.einsum("mij,mj->mi", Ul, pl)
    assert np.abs(y.view(np.complex128).reshape(-1, 3) - want).max() <= 1e-14
    # SU(3) preserves the norm (fp32 storage perturbs unitarity of U at the 1e-7 level)
    ny, npsi = np.linalg.norm(want, axis=1), np.linalg.norm(pl, axis=1)
    assert np.abs(ny / npsi - 1).max() <= (1e-13 if dtype == np.float64 else 1e-6)
    # identity and zero, exact
    one = flat(np.broadcast_to(np.eye(3), (gs.nmat, 3, 3)).copy(), dtype)
    assert np.array_equal(oracle.matvec(gs, one, psi), psi.astype(np.float64))
    assert not oracle.matvec(gs, np.zeros_like(U), psi).any()
    # (U.V).psi = U.(V.psi) to rounding (fp64 operands only: the intermediate is fp64)
    if dtype == np.float64:
        lhs = oracle.matvec(gs, oracle.mul(gs, U, V), psi)
        rhs = oracle.matvec(gs, U, oracle.matvec(gs, V, psi))
        assert np.abs(lhs - rhs).max() <= 1e-14
    # every vector layout gives the same numbers, bit for bit, after the permutation
    for W in (2, 4, 8, 16):
        gv = oracle.Geom(L, nl=nl, layout=oracle.su3_oracle.VECTOR, W=W)
        yv = oracle.matvec(gv, oracle.convert(gv, gs, U), oracle.convert_vec(gv, gs, psi))
        assert np.array_equal(oracle.convert_vec(gs, gv, yv), y)
        back = oracle.convert_vec(gs, gv, oracle.convert_vec(gv, gs, psi))
        assert np.array_equal(back, psi)


def test_index_vec_is_a_bijection_and_matches_the_matrix_map():
    g = oracle.Geom((4, 2, 2, 4), nl=4, layout=oracle.su3_oracle.VECTOR, W=8)
    seen = set()
    for site in range(g.volume):
        for mu in range(4):
            for i in range(3):
                for c in range(2):
                    seen.add(oracle.index_vec(g, site, mu, i, c))
        # same (outer site, lane) as the matrix map: component i of the vector sits where column-0 element i would
        # sit in a 3-component record
        o, l = oracle.site_to_outer(g, site)
        assert oracle.index_vec(g, site, 2, 1, 1) == (((o * 4 + 2) * 3 + 1) * 8 + l) * 2 + 1
    assert seen == set(range(g.nmat * 6))
    gs = oracle.Geom((4, 2, 2, 4), nl=4)
    assert oracle.index_vec(gs, 5, 3, 2, 1) == ((5 * 4 + 3) * 3 + 2) * 2 + 1


# ---------------------------------------------------------------- real scalar fields: the paper's Listing 2
def load_listing2():
    import os
    from helpers import GOLDEN
    rows = []
    with open(os.path.join(GOLDEN, "listing2_example.txt")) as f:
        for line in f:
            t = line.split("#")[0].split()
            if t:
                rows.append((t[0], float(t[1]), float(t[2]), float(t[3])))
    return rows


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_expr_real_reproduces_the_papers_listing2(dtype):
    n = 8 ** 4
    for prog, a, b, want in load_listing2():
        v1, v2 = np.full(n, a, dtype=dtype), np.full(n, b, dtype=dtype)
        assert np.array_equal(oracle.expr_real(prog, v1, v2), np.full(n, want))


def test_expr_real_against_numpy_and_rejects_malformed():
    rng = np.random.default_rng(3)
    a, b, c = (rng.standard_normal(1001) for _ in range(3))
    assert np.array_equal(oracle.expr_real("01+01*+", a, b), (a + b) + a * b)
    assert np.array_equal(oracle.expr_real("01*2-0+", a, b, c), (a * b - c) + a)
    assert np.array_equal(oracle.expr_real("012-*", a, b, c), a * (b - c))
    a32 = a.astype(np.float32)
    assert np.array_equal(oracle.expr_real("00*", a32), a32.astype(np.float64) ** 2)   # promoted exactly, kept in fp64
    for bad in ["", "0+", "00", "01*", "0a*"]:
        with pytest.raises(ValueError):
            oracle.expr_real(bad, a)
