"""The C-ABI boundary without a GPU: the library loads, exports every symbol that
include/su3stream.h declares, validates descriptors as the header states, and its host-side
index map reproduces the hand-computed spot values of tests/golden (reading S3/S4).
No compute call is made here (-m "not gpu")."""
import ctypes
import os
import re

import pytest

import paper_1710_09409_b200 as su3
from helpers import load_vector_map_spots

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_exports_match_header():
    text = open(os.path.join(ROOT, "include", "su3stream.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    declared = set(re.findall(r"\b(su3_[a-z0-9_]+)\s*\(", text))
    assert declared == set(su3.EXPORTS)
    for name in declared:
        assert hasattr(su3.lib, name), name
    assert su3.su3_version().startswith("su3stream")


def test_field_bytes_for_the_configs():
    assert su3.su3_field_bytes(su3.make_desc(8)) == 4096 * 144
    assert su3.su3_field_bytes(su3.make_desc(16, layout=su3.SU3_VECTOR, W=4)) == 65536 * 144
    assert su3.su3_field_bytes(su3.make_desc(32, n_lorentz=4)) == 4 * 32 ** 4 * 144
    assert su3.su3_field_bytes(su3.make_desc(48, prec=su3.SU3_F32, layout=su3.SU3_VECTOR, W=8)) == 48 ** 4 * 72
    assert su3.su3_field_bytes(su3.make_desc(64)) == 64 ** 4 * 144  # > 2^31: 64-bit sizes


@pytest.mark.parametrize("kw", [
    dict(L=(8, 8, 0, 8)), dict(L=8, n_lorentz=2), dict(L=8, prec=2), dict(L=8, layout=3),
    dict(L=8, layout=1, W=3), dict(L=8, layout=1, W=64), dict(L=8, layout=0, W=4),
    dict(L=8, layout=1, W=4, simd=(1, 1, 1, 2)), dict(L=(8, 8, 8, 9), layout=1, W=2),
    dict(L=8, layout=1, W=4, simd=(1, 1, -2, -2)),
])
def test_invalid_descriptors(kw):
    with pytest.raises(su3.Su3Error) as ei:
        su3.su3_field_bytes(su3.make_desc(**kw))
    assert ei.value.status == su3.SU3_ERR_INVALID
    assert su3.su3_last_error()


def test_default_split_and_normalize():
    _, splits = load_vector_map_spots()
    for W, simd in splits.items():
        d = su3.su3_desc_normalize(su3.make_desc(8, layout=su3.SU3_VECTOR if W > 1 else su3.SU3_SCALAR, W=W))
        assert tuple(d.simd) == simd
    d = su3.su3_desc_normalize(su3.make_desc(8, layout=su3.SU3_VECTOR, W=4, simd=(2, 2, 1, 1)))
    assert tuple(d.simd) == (2, 2, 1, 1)


def test_index_spot_values():
    spots, _ = load_vector_map_spots()
    for s in spots:
        d = su3.make_desc(s["L"], layout=su3.SU3_VECTOR, W=s["W"])
        for (i, j, c) in [(0, 0, 0), (1, 2, 1), (2, 2, 1)]:
            want = (((s["outer"]) * 9 + 3 * i + j) * s["W"] + s["lane"]) * 2 + c
            assert su3.su3_index(d, s["site"], 0, i, j, c) == want
    d = su3.make_desc(4, n_lorentz=4)
    assert su3.su3_index(d, 7, 3, 2, 1, 1) == ((7 * 4 + 3) * 9 + 7) * 2 + 1
    with pytest.raises(su3.Su3Error):
        su3.su3_index(d, 256, 0, 0, 0, 0)
    with pytest.raises(su3.Su3Error):
        su3.su3_index(d, 0, 4, 0, 0, 0)


def test_index_is_a_bijection_small():
    for kw in [dict(L=4, layout=1, W=8), dict(L=(4, 2, 6, 4), n_lorentz=4, layout=1, W=4), dict(L=2, n_lorentz=4)]:
        d = su3.su3_desc_normalize(su3.make_desc(**kw))
        V = d.L[0] * d.L[1] * d.L[2] * d.L[3]
        seen = set()
        for site in range(V):
            for mu in range(d.n_lorentz):
                for e in (0, 4, 8):
                    seen.add(su3.su3_index(d, site, mu, e // 3, e % 3, 0))
        assert len(seen) == V * d.n_lorentz * 3
        assert max(seen) < V * d.n_lorentz * 18


def test_wrap_errors_without_touching_memory():
    d = su3.make_desc(2)
    h = ctypes.c_void_p()
    need = su3.su3_field_bytes(d)
    assert su3.lib.su3_field_wrap(ctypes.byref(d), ctypes.c_void_p(0), need, ctypes.byref(h)) == su3.SU3_ERR_NULL
    assert su3.lib.su3_field_wrap(ctypes.byref(d), ctypes.c_void_p(0x1008), need, ctypes.byref(h)) == su3.SU3_ERR_ALIGN
    assert su3.lib.su3_field_wrap(ctypes.byref(d), ctypes.c_void_p(0x1000), need - 1, ctypes.byref(h)) == su3.SU3_ERR_SIZE
    assert su3.lib.su3_field_wrap(ctypes.byref(d), ctypes.c_void_p(0x1000), need, None) == su3.SU3_ERR_NULL
    assert su3.lib.su3_field_wrap(ctypes.byref(d), ctypes.c_void_p(0x1000), need, ctypes.byref(h)) == su3.SU3_OK
    out = su3.su3_desc()
    assert su3.lib.su3_field_desc(h, ctypes.byref(out)) == su3.SU3_OK and tuple(out.simd) == (1, 1, 1, 1)
    # mismatching operands are rejected before anything is launched (fake pointers are never touched)
    d2 = su3.make_desc(2, prec=su3.SU3_F32)
    h2 = ctypes.c_void_p()
    assert su3.lib.su3_field_wrap(ctypes.byref(d2), ctypes.c_void_p(0x2000), need, ctypes.byref(h2)) == su3.SU3_OK
    assert su3.lib.su3_mul(h, h, h2, None) == su3.SU3_ERR_MISMATCH
    assert su3.lib.su3_mul(h, None, h, None) == su3.SU3_ERR_NULL
    assert su3.lib.su3_convert(h, h, None) == su3.SU3_ERR_MISMATCH
    assert su3.lib.su3_copy(h, h2, None) == su3.SU3_ERR_MISMATCH
    assert su3.lib.su3_field_free(h) == su3.SU3_OK and su3.lib.su3_field_free(h2) == su3.SU3_OK
    assert su3.lib.su3_field_free(None) == su3.SU3_ERR_NULL


def test_tune_validation_roundtrip():
    su3.su3_tune_set(tile_mats=64, stages=3, ctas_per_sm=2, l2_hint=1, path=1)
    assert su3.su3_tune_get() == dict(tile_mats=64, stages=3, ctas_per_sm=2, l2_hint=1, path=1, l2_pin_mb=0)
    with pytest.raises(su3.Su3Error):
        su3.su3_tune_set(tile_mats=100)
    with pytest.raises(su3.Su3Error):
        su3.su3_tune_set(stages=1)
    su3.su3_tune_set()
    assert su3.su3_tune_get()["tile_mats"] == 0


def test_no_cpu_fallback_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    d = su3.make_desc(2)
    h = ctypes.c_void_p()
    su3.lib.su3_field_wrap(ctypes.byref(d), ctypes.c_void_p(0x1000), su3.su3_field_bytes(d), ctypes.byref(h))
    assert su3.lib.su3_mul(h, h, h, None) == su3.SU3_ERR_CUDA  # fails loudly, computes nothing
    assert "CUDA" in su3.su3_last_error()
    su3.lib.su3_field_free(h)


def test_expr_program_validation_and_cost():
    """host-only: su3_expr_cost runs the same compiler as su3_expr (no launch)"""
    assert su3.su3_expr_cost("01*", 2) == (3, 198)
    assert su3.su3_expr_cost("01*2*", 3) == (4, 396)
    assert su3.su3_expr_cost("01*2+", 3) == (4, 216)
    assert su3.su3_expr_cost("01+01*+", 2) == (3, 198 + 36)
    assert su3.su3_expr_cost("0", 1) == (2, 0)
    for bad, n in [("", 1), ("0+", 1), ("00", 1), ("01*", 1), ("0a*", 1), ("00*+", 1), ("01*", 3), ("0" * 9 + "*" * 8, 1),
                   ("00*" + "0*" * 16, 1), ("0", 0), ("0", 9)]:
        with pytest.raises(su3.Su3Error) as e:
            su3.su3_expr_cost(bad, n)
        assert e.value.status == su3.SU3_ERR_INVALID, bad


def test_colour_vector_boundary_host_side():
    d = su3.make_desc((4, 2, 2, 4), n_lorentz=4, layout=su3.SU3_VECTOR, W=8, prec=su3.SU3_F32)
    assert su3.su3_vec_bytes(d) == 64 * 4 * 6 * 4
    assert su3.su3_vec_bytes(su3.make_desc(8)) == 4096 * 48
    import oracle
    g = oracle.Geom((4, 2, 2, 4), nl=4, layout=1, W=8)
    for site in (0, 5, 17, 63):
        for mu in (0, 3):
            for i in range(3):
                assert su3.su3_vec_index(d, site, mu, i, 1) == oracle.index_vec(g, site, mu, i, 1)
    with pytest.raises(su3.Su3Error) as e:
        su3.su3_vec_index(d, 0, 0, 3, 0)
    assert e.value.status == su3.SU3_ERR_INVALID


def _run_listing(listing, mats):
    """execute the compiled register machine on one site with numpy (what the interpreter kernel does per thread)"""
    import numpy as np
    acc, temps = None, {}

    def get(s):
        return acc if s == "acc" else (temps[s] if s[0] == "t" else mats[int(s[1:])])
    for op, a, b, spill in listing:
        if spill is not None:
            temps[spill] = acc
        A = get(a)
        B = get(b) if op != "copy" else None
        acc = {"mul": lambda: A @ B, "add": lambda: A + B, "sub": lambda: A - B, "copy": lambda: A}[op]()
    return np.array(acc)


def _postfix(prog, mats):
    st = []
    for t in prog:
        if t.isdigit():
            st.append(mats[int(t)])
        else:
            b, a = st.pop(), st.pop()
            st.append(a @ b if t == "*" else (a + b if t == "+" else a - b))
    return st[0]


def test_expr_compiler_listing_evaluates_like_the_postfix_program():
    """host-only pin of the postfix -> register-machine compiler: known listings, and 300 random programs whose
    listing, executed with numpy on random integer matrices, equals direct postfix evaluation exactly"""
    import numpy as np
    assert su3.su3_expr_disasm("01*2*", 3) == [("mul", "o0", "o1", None), ("mul", "acc", "o2", None)]
    assert su3.su3_expr_disasm("01+01*+", 2) == [("add", "o0", "o1", None), ("mul", "o0", "o1", "t0"), ("add", "t0", "acc", None)]
    assert su3.su3_expr_disasm("0", 1) == [("copy", "o0", "-", None)]
    assert su3.su3_expr_disasm("012**", 3) == [("mul", "o1", "o2", None), ("mul", "o0", "acc", None)]
    rng = np.random.default_rng(7)
    mats = [rng.integers(-3, 4, (3, 3)).astype(np.int64).astype(object) for _ in range(8)]   # exact Python integers
    deepest = 0
    for _ in range(300):
        n_ops = int(rng.integers(1, 9))
        n_operators = int(rng.integers(max(1, n_ops - 1), 16))
        leaves = list(range(n_ops)) + [int(rng.integers(0, n_ops)) for _ in range(n_operators + 1 - n_ops)]
        rng.shuffle(leaves)
        prog, depth, li, left = [], 0, 0, n_operators
        while li < len(leaves) or left:
            if li < len(leaves) and depth < 8 and (depth < 2 or not left or rng.random() < 0.6):
                prog.append(str(leaves[li])); li += 1; depth += 1
            else:
                prog.append("+-*"[int(rng.integers(0, 3))]); depth -= 1; left -= 1
        prog = "".join(prog)
        listing = su3.su3_expr_disasm(prog, n_ops)
        assert len(listing) == n_operators
        deepest = max(deepest, len({sp for *_, sp in listing if sp}))
        assert (_run_listing(listing, mats) == _postfix(prog, mats)).all(), prog
    assert deepest >= 3  # programs with several live temporaries were among them


def test_library_and_oracle_index_maps_agree_on_random_geometries():
    """two independent implementations of readings S1-S6 (su3_index / su3_vec_index in the library, orc_index /
    orc_index_vec in the oracle) must give the same offsets for random admissible geometries and custom splits"""
    import numpy as np
    import oracle
    rng = np.random.default_rng(11)
    checked = 0
    while checked < 60:
        W = int(2 ** rng.integers(0, 6))
        simd, w = [1, 1, 1, 1], W
        while w > 1:                       # random split of W over the dimensions
            simd[int(rng.integers(0, 4))] *= 2
            w //= 2
        L = [int(s * rng.integers(1, 4)) for s in simd]
        nl = int(rng.choice([1, 4]))
        layout = su3.SU3_VECTOR if (W > 1 or rng.random() < 0.5) else su3.SU3_SCALAR
        if layout == su3.SU3_SCALAR:
            W, simd = 1, [1, 1, 1, 1]
        d = su3.make_desc(L, n_lorentz=nl, layout=layout, W=W, simd=simd)
        g = oracle.Geom(L, nl=nl, layout=layout, W=W, simd=simd)
        V = int(np.prod(L))
        seen = set()
        for site in rng.integers(0, V, 12):
            mu, i, j, c = int(rng.integers(0, nl)), int(rng.integers(0, 3)), int(rng.integers(0, 3)), int(rng.integers(0, 2))
            off = su3.su3_index(d, int(site), mu, i, j, c)
            assert off == oracle.index(g, int(site), mu, i, j, c)
            assert su3.su3_vec_index(d, int(site), mu, i, c) == oracle.index_vec(g, int(site), mu, i, c)
            assert 0 <= off < V * nl * 18
            seen.add(off)
        checked += 1
    # default split (simd all zero) agrees too
    for W in (2, 4, 8, 16, 32):
        assert tuple(su3.su3_desc_normalize(su3.make_desc(32, layout=su3.SU3_VECTOR, W=W)).simd) == oracle.default_simd(W)


def test_expression_front_end_builds_postfix_programs():
    """the Lattice front end (Listing 3 style `z = x*y`) only builds the tree: check the programs it emits"""
    from paper_1710_09409_b200.lattice import Lattice, postfix
    x, y, w, v = (Lattice(None) for _ in range(4))
    assert postfix(x * y) == ("01*", [x, y])
    assert postfix(x * y * w) == ("01*2*", [x, y, w])                 # left-associative, as C++ parses it
    assert postfix(x * y + v) == ("01*2+", [x, y, v])
    assert postfix(x + y + x * y) == ("01+01*+", [x, y])             # Listing 2: v1+v2+v1*v2, fields deduplicated
    assert postfix(x * (y - w) - v * x)[0] == "012-*30*-"
    assert postfix(x) == ("0", [x])
    with pytest.raises(TypeError):
        x + 1.0


def test_tune_is_per_thread_and_argument_checks_do_not_race():
    """no global state except thread-local data.  Two threads set different launch knobs and hammer the
    argument checks of the launching calls; each must always read back ITS knobs and ITS error string."""
    import threading
    d = su3.make_desc(2)
    need = su3.su3_field_bytes(d)
    d32 = su3.make_desc(2, prec=su3.SU3_F32)
    errors = []

    def worker(k):
        try:
            su3.su3_tune_set(tile_mats=(32, 64, 128)[k % 3], stages=2 + k, ctas_per_sm=1 + k, path=1 + k % 3)
            mine = su3.su3_tune_get()
            h, h2 = ctypes.c_void_p(), ctypes.c_void_p()
            assert su3.lib.su3_field_wrap(ctypes.byref(d), ctypes.c_void_p(0x1000 * (k + 1)), need, ctypes.byref(h)) == su3.SU3_OK
            assert su3.lib.su3_field_wrap(ctypes.byref(d32), ctypes.c_void_p(0x100000), need, ctypes.byref(h2)) == su3.SU3_OK
            for it in range(400):
                if k % 2:
                    assert su3.lib.su3_mul(h, h, h2, None) == su3.SU3_ERR_MISMATCH
                    assert "descriptors differ" in su3.su3_last_error()
                else:
                    assert su3.lib.su3_cshift(h, h2, 9, 1, None) in (su3.SU3_ERR_MISMATCH, su3.SU3_ERR_INVALID)
                    assert su3.lib.su3_mul(h, None, h, None) == su3.SU3_ERR_NULL
                    assert "NULL" in su3.su3_last_error()
                assert su3.su3_tune_get() == mine
            su3.lib.su3_field_free(h)
            su3.lib.su3_field_free(h2)
        except BaseException as e:   # noqa: BLE001 - reported below
            errors.append((k, repr(e)))

    su3.su3_tune_set()
    ts = [threading.Thread(target=worker, args=(k,)) for k in range(6)]
    for t in ts:
        t.start()
    for t in ts:
        t.join()
    assert not errors, errors
    assert su3.su3_tune_get()["tile_mats"] == 0    # the main thread's knobs were never touched


def test_eval_host_rejects_absurd_chunk_counts_before_any_cuda_work():
    d = su3.make_desc(2)
    h = ctypes.c_void_p()
    su3.lib.su3_field_wrap(ctypes.byref(d), ctypes.c_void_p(0x1000), su3.su3_field_bytes(d), ctypes.byref(h))
    import torch
    if torch.cuda.is_available():
        assert su3.lib.su3_eval_host(0, None, None, None, None, h, h, h, None, 1 << 20, None) == su3.SU3_ERR_INVALID
    else:
        assert su3.lib.su3_eval_host(0, None, None, None, None, h, h, h, None, 1 << 20, None) in (su3.SU3_ERR_INVALID, su3.SU3_ERR_CUDA)
    assert su3.lib.su3_host_release() == su3.SU3_OK
    su3.lib.su3_field_free(h)


def test_ahead_of_time_menu_rows_and_matching():
    """host-only: every row of the ahead-of-time menu is reached by its own postfix program, by any renaming of the
    operands and by either order of the sources of '+'; everything else goes to the interpreter"""
    rows = {}
    for prog, n in [("01*", 2), ("01*2*", 3), ("01*2+", 3), ("01+", 2), ("01+01*+", 2), ("01*23*+", 4), ("01*23*-", 4),
                    ("01*2-", 3), ("01+2+", 3), ("01+2+3+", 4), ("01-", 2), ("01*2*3*", 4), ("012**", 3), ("01*23**", 4)]:
        plan = su3.su3_expr_plan(prog, n)
        assert plan[0] == "menu" and plan[2] == prog and plan[3] == list(range(n)), (prog, plan)
        rows[prog] = plan[1]
    assert sorted(rows.values()) == list(range(11)) + [13, 14, 15]   # fourteen distinct rows for matrix fields (11, 12: real fields)
    # renamed operands: slot k of the row holds the operand that plays its part
    assert su3.su3_expr_plan("10*", 2) == ("menu", rows["01*"], "01*", [1, 0])
    assert su3.su3_expr_plan("20*1+", 3) == ("menu", rows["01*2+"], "01*2+", [2, 0, 1])
    assert su3.su3_expr_plan("201*+", 3) == ("menu", rows["01*2+"], "01*2+", [0, 1, 2])       # v + x*y = x*y + v
    assert su3.su3_expr_plan("10+01*+", 2)[:2] == ("menu", rows["01+01*+"])
    assert su3.su3_expr_plan("32*10*+", 4) == ("menu", rows["01*23*+"], "01*23*+", [3, 2, 1, 0])
    # not on the menu: repeated fields, other shapes, non-commutative swaps
    assert su3.su3_expr_plan("210**", 3) == ("menu", rows["012**"], "012**", [2, 1, 0])
    for prog, n in [("00*", 1), ("01*2*3*4*", 5), ("0123***", 4), ("201*-", 3), ("01*21*-", 3), ("01*23*45*++", 6), ("0", 1), ("01-2-", 3)]:
        assert su3.su3_expr_plan(prog, n) == "interpreter", prog
    # real scalar fields: '*' is element-wise; Listing 2's two programs are on the menu
    assert su3.su3_expr_plan("01+", 2, real_fields=True)[:2] == ("menu", rows["01+"])
    p1, p2 = su3.su3_expr_plan("01*", 2, real_fields=True), su3.su3_expr_plan("01+01*+", 2, real_fields=True)
    assert p1[0] == "menu" and p2[0] == "menu" and p1[1] not in rows.values() and p2[1] not in rows.values()
    assert su3.su3_expr_plan("01*2*", 3, real_fields=True) == "interpreter"


def test_face_calls_validate_before_any_cuda_work():
    """su3_face_*: sizes by the header's formula; bad dim / plane range / buffer are rejected host-side"""
    d = su3.make_desc((6, 4, 2, 8), n_lorentz=4, prec=su3.SU3_F32, layout=su3.SU3_VECTOR, W=4)
    h, hv, hr = ctypes.c_void_p(), ctypes.c_void_p(), ctypes.c_void_p()
    assert su3.lib.su3_field_wrap(ctypes.byref(d), ctypes.c_void_p(0x1000), su3.su3_field_bytes(d), ctypes.byref(h)) == su3.SU3_OK
    assert su3.lib.su3_vec_wrap(ctypes.byref(d), ctypes.c_void_p(0x1000), su3.su3_vec_bytes(d), ctypes.byref(hv)) == su3.SU3_OK
    assert su3.lib.su3_real_wrap(ctypes.byref(d), ctypes.c_void_p(0x1000), su3.su3_real_bytes(d), ctypes.byref(hr)) == su3.SU3_OK
    n = ctypes.c_size_t()
    for dim, L in enumerate((6, 4, 2, 8)):
        assert su3.lib.su3_face_bytes(h, dim, 1, ctypes.byref(n)) == su3.SU3_OK
        assert n.value == (6 * 4 * 2 * 8 // L) * 4 * 72           # one plane of 72-byte matrices, 4 Lorentz indices
        assert su3.lib.su3_face_bytes(hv, dim, L, ctypes.byref(n)) == su3.SU3_OK
        assert n.value == su3.su3_vec_bytes(d)                     # all planes = the whole field
        assert su3.lib.su3_face_bytes(h, dim, L + 1, ctypes.byref(n)) == su3.SU3_ERR_INVALID
    assert su3.lib.su3_face_bytes(h, 4, 1, ctypes.byref(n)) == su3.SU3_ERR_INVALID
    assert su3.lib.su3_face_bytes(hr, 3, 1, ctypes.byref(n)) == su3.SU3_ERR_MISMATCH
    assert su3.lib.su3_face_bytes(None, 3, 1, ctypes.byref(n)) == su3.SU3_ERR_NULL
    buf, big = ctypes.c_void_p(0x4000), 1 << 30
    assert su3.lib.su3_face_pack(buf, big, h, 3, 7, 2, None) == su3.SU3_ERR_INVALID          # planes 7..8 of 0..7
    assert su3.lib.su3_face_pack(buf, big, h, 3, -1, 1, None) == su3.SU3_ERR_INVALID
    assert su3.lib.su3_face_pack(None, big, h, 3, 0, 1, None) == su3.SU3_ERR_NULL
    assert su3.lib.su3_face_pack(ctypes.c_void_p(0x4008), big, h, 3, 0, 1, None) == su3.SU3_ERR_ALIGN
    assert su3.lib.su3_face_pack(buf, 100, h, 3, 0, 1, None) == su3.SU3_ERR_SIZE
    assert su3.lib.su3_face_unpack(h, buf, 100, 3, 0, 1, None) == su3.SU3_ERR_SIZE
    assert su3.lib.su3_face_copy(h, 0, h, 1, 3, 1, None) == su3.SU3_ERR_MISMATCH              # same field
    assert su3.lib.su3_face_copy(h, 0, hv, 1, 3, 1, None) == su3.SU3_ERR_MISMATCH             # kinds differ
    for x in (h, hv, hr):
        su3.lib.su3_field_free(x)
