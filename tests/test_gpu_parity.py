"""-m gpu: the CUDA path (through the C ABI) against the CPU oracle, element by element on
the same seeded inputs.  Tolerances are north_star's: per-matrix max-norm relative error
(reading S15) <= 1e-12 in fp64 and <= 2e-5 in fp32; integer cases, convert and copy are
bit-exact."""
import numpy as np
import pytest
import torch

import oracle
import paper_1710_09409_b200 as su3
import su3gen
from gpu_util import const_field, download, geom_of, host_field, scalar_desc, upload
from helpers import TOL, load_integer_case, rel_err

pytestmark = pytest.mark.gpu
IC = load_integer_case()
F64, F32, SC, VE = su3.SU3_F64, su3.SU3_F32, su3.SU3_SCALAR, su3.SU3_VECTOR


@pytest.fixture(autouse=True)
def _default_tuning():
    su3.su3_tune_set()
    yield
    su3.su3_tune_set()


def run_op(op, desc, hosts):
    fs = [upload(desc, h) for h in hosts]
    z = su3.alloc_field(desc)
    z.tensor.fill_(0xFF)
    {"mul": su3.su3_mul, "mul3": su3.su3_mul3, "mul_add": su3.su3_mul_add, "add": su3.su3_add}[op](z, *fs)
    return download(z)


def oracle_op(op, desc, hosts):
    g = geom_of(desc)
    return {"mul": oracle.mul, "mul3": oracle.mul3, "mul_add": oracle.mul_add}[op](g, *hosts)


def check(op, desc, hosts, tol=None):
    z = run_op(op, desc, hosts)
    zref = oracle_op(op, desc, hosts)
    W = su3.su3_desc_normalize(desc).W
    err, _ = rel_err(z, zref, W)
    assert np.isfinite(z).all()
    assert err <= (TOL[desc.prec] if tol is None else tol), (op, err)
    return z, zref


ALL_W = [(SC, 1), (VE, 1), (VE, 2), (VE, 4), (VE, 8), (VE, 16), (VE, 32)]


# ------------------------------------------------------------------ exact integer case (bit-equal)
@pytest.mark.parametrize("path", [0, 1, 2, 3])
@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("layout,W", ALL_W)
def test_integer_case_bit_exact(prec, layout, W, path):
    su3.su3_tune_set(path=path)
    desc = su3.make_desc((4, 4, 4, 8), prec=prec, layout=layout, W=W)
    k = np.arange(1, 8).reshape(-1, 1, 1)  # site-dependent integer multiples: tests indexing too
    A, B, C = const_field(desc, IC["A"] * k), const_field(desc, IC["B"]), const_field(desc, IC["C"])
    for op, hosts in [("mul", [A, B]), ("mul", [B, A]), ("mul3", [A, B, C]), ("mul_add", [A, B, C])]:
        z = run_op(op, desc, hosts)
        assert np.array_equal(z.astype(np.float64), oracle_op(op, desc, hosts)), (op, prec, W)
    # and against the stored hand-computed product directly (site 0 holds 1*A)
    z = run_op("mul", scalar_desc(desc), [const_field(scalar_desc(desc), IC["A"]), const_field(scalar_desc(desc), IC["B"])])
    assert np.array_equal(z[:18].astype(np.float64).view(np.complex128).reshape(3, 3), IC["AB"])


def test_identity_and_zero():
    desc = su3.make_desc(4)
    x = host_field(desc, 7, su3gen.FIELD_X)
    one, zero = const_field(desc, np.eye(3)), const_field(desc, np.zeros((3, 3)))
    v = host_field(desc, 7, su3gen.FIELD_V, kind="gauss")
    assert np.array_equal(run_op("mul", desc, [x, one]), x)
    assert np.array_equal(run_op("mul", desc, [one, x]), x)
    assert not run_op("mul", desc, [x, zero]).any()
    assert np.array_equal(run_op("mul_add", desc, [zero, x, v]), v)
    assert np.array_equal(run_op("mul3", desc, [one, x, one]), x)


# ------------------------------------------------------------------ BASELINE.json configs 1 and 2
def test_config1_8x4_fp64_scalar():
    desc = su3.make_desc(8)
    seed = su3gen.config_seed(1)
    x, y = host_field(desc, seed, su3gen.FIELD_X), host_field(desc, seed, su3gen.FIELD_Y)
    z, _ = check("mul", desc, [x, y])
    # closure of SU(3): the GPU product is unitary with det 1
    zz = z.view(np.complex128).reshape(-1, 3, 3)
    assert np.abs(zz @ zz.conj().transpose(0, 2, 1) - np.eye(3)).max() <= 1e-13
    assert np.abs(np.linalg.det(zz) - 1).max() <= 1e-13


def test_config2_16x4_both_layouts_and_roundtrip():
    ds, dv = su3.make_desc(16), su3.make_desc(16, layout=VE, W=4)
    seed = su3gen.config_seed(2)
    xs, ys = host_field(ds, seed, su3gen.FIELD_X), host_field(ds, seed, su3gen.FIELD_Y)
    xv, yv = host_field(dv, seed, su3gen.FIELD_X), host_field(dv, seed, su3gen.FIELD_Y)
    zs, _ = check("mul", ds, [xs, ys])
    zv, _ = check("mul", dv, [xv, yv])
    # scalar and vector kernels share the FMA chain: bit-equal after the layout permutation
    assert np.array_equal(oracle.convert(geom_of(dv), geom_of(ds), zs), zv)
    # GPU convert == oracle permutation, both ways, and the round trip is the identity (bit-exact)
    fs, fv, fs2 = upload(ds, xs), su3.alloc_field(dv), su3.alloc_field(ds)
    su3.su3_convert(fv, fs)
    su3.su3_convert(fs2, fv)
    assert np.array_equal(download(fv), xv)
    assert np.array_equal(download(fs2), xs)


# ------------------------------------------------------------------ every W, ragged sizes, Lorentz index
@pytest.mark.parametrize("path", [0, 1, 2, 3])
@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("layout,W", ALL_W)
def test_all_ops_every_W(prec, layout, W, path):
    su3.su3_tune_set(path=path)
    desc = su3.make_desc((4, 6, 4, 8), prec=prec, layout=layout, W=W)  # 768 sites: 6 tiles of 128
    x, y, w = (host_field(desc, 11, f) for f in (su3gen.FIELD_X, su3gen.FIELD_Y, su3gen.FIELD_W))
    v = host_field(desc, 11, su3gen.FIELD_V, kind="gauss")
    check("mul", desc, [x, y])
    check("mul3", desc, [x, y, w])
    check("mul_add", desc, [x, y, v])


@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("L,nl,layout,W", [
    ((3, 3, 3, 3), 1, SC, 1),    # 81 matrices: odd count -> fp32 field ends on an 8-byte tail
    ((1, 1, 1, 1), 1, SC, 1),    # a single matrix
    ((5, 3, 1, 7), 1, SC, 1),    # 105: one ragged tile
    ((3, 5, 2, 6), 4, VE, 4),    # simd {1,1,2,2}; 720 matrices
    ((6, 2, 10, 2), 4, VE, 8),   # r = {6,1,5,1}
    ((10, 6, 6, 2), 1, VE, 2),
    ((2, 2, 2, 2), 4, VE, 16),
    ((12, 12, 12, 12), 1, VE, 8),  # L = 12 of the volume sweep, r = {12,6,6,6}
])
def test_ragged_and_lorentz(prec, L, nl, layout, W):
    desc = su3.make_desc(L, n_lorentz=nl, prec=prec, layout=layout, W=W)
    x, y, w = (host_field(desc, 13, f) for f in (su3gen.FIELD_X, su3gen.FIELD_Y, su3gen.FIELD_W))
    for tile in (0, 32, 128):
        su3.su3_tune_set(tile_mats=tile)
        check("mul", desc, [x, y])
    su3.su3_tune_set()
    check("mul3", desc, [x, y, w])
    # convert against the oracle permutation, both directions
    ds = scalar_desc(desc)
    if layout == VE:
        xs = host_field(ds, 13, su3gen.FIELD_X)
        fs, fv, fs2 = upload(ds, xs), su3.alloc_field(desc), su3.alloc_field(ds)
        su3.su3_convert(fv, fs)
        su3.su3_convert(fs2, fv)
        assert np.array_equal(download(fv), x)
        assert np.array_equal(download(fs2), xs)
    # copy is bit-exact, add matches numpy exactly (one rounding per element)
    fx, fc = upload(desc, x), su3.alloc_field(desc)
    fc.tensor.fill_(0)
    su3.su3_copy(fc, fx)
    assert np.array_equal(download(fc), x)
    assert np.array_equal(run_op("add", desc, [x, y]), x + y)


def test_custom_simd_split():
    desc = su3.make_desc((8, 4, 4, 4), layout=VE, W=8, simd=(4, 2, 1, 1), prec=F32)
    x, y = host_field(desc, 17, su3gen.FIELD_X), host_field(desc, 17, su3gen.FIELD_Y)
    check("mul", desc, [x, y])
    ds = scalar_desc(desc)
    fs, fv = upload(ds, host_field(ds, 17, su3gen.FIELD_X)), su3.alloc_field(desc)
    su3.su3_convert(fv, fs)
    assert np.array_equal(download(fv), x)


# ------------------------------------------------------------------ launch configurations, aliasing
@pytest.mark.parametrize("tile,stages,ctas,hint", [(32, 2, 1, 1), (64, 3, 2, 2), (128, 2, 4, 1), (128, 6, 1, 2),
                                                   (128, 3, 3, 1), (32, 2, 4, 2), (64, 16, 1, 1)])
def test_launch_configurations_are_equivalent(tile, stages, ctas, hint):
    desc = su3.make_desc((16, 16, 8, 9), prec=F32)  # 18432 matrices; many tiles per CTA at ctas=1
    x, y = host_field(desc, 19, su3gen.FIELD_X), host_field(desc, 19, su3gen.FIELD_Y)
    ref = run_op("mul", desc, [x, y])
    su3.su3_tune_set(tile_mats=tile, stages=stages, ctas_per_sm=ctas, l2_hint=hint)
    assert np.array_equal(run_op("mul", desc, [x, y]), ref)
    check("mul", desc, [x, y])


def test_output_may_alias_an_input():
    for desc in (su3.make_desc((8, 8, 8, 6)), su3.make_desc((8, 8, 8, 6), prec=F32, layout=VE, W=8)):
        x, y = host_field(desc, 23, su3gen.FIELD_X), host_field(desc, 23, su3gen.FIELD_Y)
        ref = run_op("mul", desc, [x, y])
        fx, fy = upload(desc, x), upload(desc, y)
        su3.su3_mul(fx, fx, fy)
        assert np.array_equal(download(fx), ref)
        fx, fy = upload(desc, x), upload(desc, y)
        su3.su3_mul(fy, fx, fy)
        assert np.array_equal(download(fy), ref)


def test_side_stream_and_launch_count():
    desc = su3.make_desc(8)
    x, y = host_field(desc, 29, su3gen.FIELD_X), host_field(desc, 29, su3gen.FIELD_Y)
    fx, fy, fz = upload(desc, x), upload(desc, y), su3.alloc_field(desc)
    torch.cuda.synchronize()
    n0 = su3.su3_launch_count()
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        su3.su3_mul(fz, fx, fy)
    s.synchronize()
    assert su3.su3_launch_count() == n0 + 1
    err, _ = rel_err(download(fz), oracle.mul(geom_of(desc), x, y), 1)
    assert err <= 1e-12


def test_mul_host_end_to_end():
    for desc in (su3.make_desc((8, 8, 8, 10)), su3.make_desc((3, 3, 3, 3), prec=F32),
                 su3.make_desc((8, 8, 8, 8), prec=F32, layout=VE, W=8)):
        x, y = host_field(desc, 31, su3gen.FIELD_X), host_field(desc, 31, su3gen.FIELD_Y)
        hx, hy = torch.from_numpy(x).pin_memory(), torch.from_numpy(y).pin_memory()
        hz = torch.empty_like(hx).pin_memory()
        zd, xd, yd = (su3.alloc_field(desc) for _ in range(3))
        for chunks in (0, 1, 5):
            hz.zero_()
            su3.su3_mul_host(hz, hx, hy, zd, xd, yd, chunks=chunks)
            torch.cuda.synchronize()
            err, _ = rel_err(hz.numpy(), oracle.mul(geom_of(desc), x, y), su3.su3_desc_normalize(desc).W)
            assert err <= TOL[desc.prec]


def test_eval_host_resident_operands_and_fused_ops():
    desc = su3.make_desc((8, 8, 8, 10), prec=F32, layout=VE, W=8)
    Wn = 8
    x, y, w = (host_field(desc, 37, f) for f in (su3gen.FIELD_X, su3gen.FIELD_Y, su3gen.FIELD_W))
    v = host_field(desc, 37, su3gen.FIELD_V, kind="gauss")
    hx, hy, hw, hv = (torch.from_numpy(a).pin_memory() for a in (x, y, w, v))
    hz = torch.empty_like(hx).pin_memory()
    zd, xd, yd, ud = (su3.alloc_field(desc) for _ in range(4))
    g = geom_of(desc)
    # everything from the host
    su3.su3_eval_host(su3.SU3_OP_MUL3, hz, hx, hy, hw, zd, xd, yd, ud, chunks=3)
    torch.cuda.synchronize()
    assert rel_err(hz.numpy(), oracle.mul3(g, x, y, w), Wn)[0] <= TOL[F32]
    # x, y already resident (left there by the call above); only v travels; result also stays on the device
    hz.zero_()
    su3.su3_eval_host(su3.SU3_OP_MUL_ADD, hz, None, None, hv, zd, xd, yd, ud, chunks=0)
    torch.cuda.synchronize()
    ref = oracle.mul_add(g, x, y, v)
    assert rel_err(hz.numpy(), ref, Wn)[0] <= TOL[F32]
    assert np.array_equal(download(zd), hz.numpy())
    su3.su3_eval_host(su3.SU3_OP_MUL, None, None, None, None, zd, xd, yd, None, chunks=2)
    assert rel_err(download(zd), oracle.mul(g, x, y), Wn)[0] <= TOL[F32]
    for bad in (lambda: su3.su3_eval_host(7, hz, hx, hy, None, zd, xd, yd, None),
                lambda: su3.su3_eval_host(su3.SU3_OP_MUL, hz, hx, hy, hw, zd, xd, yd, ud)):
        with pytest.raises(su3.Su3Error) as e:
            bad()
        assert e.value.status in (su3.SU3_ERR_INVALID, su3.SU3_ERR_MISMATCH)


@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("L,nl,layout,W", [((3, 3, 3, 3), 1, SC, 1), ((5, 3, 1, 7), 1, SC, 1), ((6, 2, 10, 2), 4, VE, 8),
                                           ((2, 2, 2, 2), 4, VE, 16), ((4, 6, 4, 8), 1, VE, 4)])
def test_no_write_outside_the_output_field(prec, L, nl, layout, W):
    """compute-sanitizer is not available on the GPU pool: every kernel family writes its result into a field that
    sits between two canary bands, for ragged sizes and every path, and the bands must come back untouched"""
    desc = su3.make_desc(L, n_lorentz=nl, prec=prec, layout=layout, W=W)
    ds = scalar_desc(desc)
    nb, nvb, G = su3.su3_field_bytes(desc), su3.su3_vec_bytes(desc), 4096
    buf = torch.empty(nb + 2 * G, dtype=torch.uint8, device="cuda")

    def guarded(kind="matrix", d=desc):
        buf.fill_(0xA5)
        n = nb if kind == "matrix" else nvb
        wrap = su3.su3_field_wrap if kind == "matrix" else su3.su3_vec_wrap
        return wrap(d, buf[G:G + n]), n

    def intact(n, what):
        torch.cuda.synchronize()
        assert bool((buf[:G] == 0xA5).all()) and bool((buf[G + n:] == 0xA5).all()), what

    x, y, w = (upload(desc, host_field(desc, 83, f)) for f in (0, 1, 2))
    xs = upload(ds, host_field(ds, 83, 0))
    psi = su3.alloc_vec(desc)
    psi.tensor.zero_()
    for path in (0, 1, 2, 3):
        su3.su3_tune_set(path=path)
        for name, call in [("mul", lambda z: su3.su3_mul(z, x, y)), ("mul3", lambda z: su3.su3_mul3(z, x, y, w)),
                           ("mul_add", lambda z: su3.su3_mul_add(z, x, y, w)), ("add", lambda z: su3.su3_add(z, x, y)),
                           ("copy", lambda z: su3.su3_copy(z, x)), ("expr", lambda z: su3.su3_expr(z, "01+01*+2-", [x, y, w])),
                           ("cshift", lambda z: su3.su3_cshift(z, x, 3, 1)), ("cshift0", lambda z: su3.su3_cshift(z, x, 0, -1)),
                           ("mul_shift", lambda z: su3.su3_mul_shift(z, x, y, 2, 1))]:
            z, n = guarded()
            call(z)
            intact(n, (name, path))
        if layout == VE:
            z, n = guarded()
            su3.su3_convert(z, xs)
            intact(n, ("convert s->v", path))
            z, n = guarded(d=ds)
            su3.su3_convert(z, x)
            intact(n, ("convert v->s", path))
        z, n = guarded("vector")
        su3.su3_matvec(z, x, psi)
        intact(n, ("matvec", path))
    su3.su3_tune_set()


def test_eval_host_from_two_threads_on_two_streams():
    """su3_eval_host keeps its copy streams and events per (device, caller stream): two host threads, each on its own
    stream, run chunked end-to-end products concurrently and both match the oracle; thread-local tune knobs differ."""
    import threading
    descs = [su3.make_desc((8, 8, 8, 12)), su3.make_desc((8, 8, 8, 12), prec=F32, layout=VE, W=8)]
    data, results, errors = [], [None, None], []
    for k, desc in enumerate(descs):
        x, y = host_field(desc, 91 + k, su3gen.FIELD_X), host_field(desc, 91 + k, su3gen.FIELD_Y)
        hx, hy = torch.from_numpy(x).pin_memory(), torch.from_numpy(y).pin_memory()
        data.append((desc, x, y, hx, hy, torch.empty_like(hx).pin_memory(), [su3.alloc_field(desc) for _ in range(3)]))
    torch.cuda.synchronize()

    def worker(k):
        try:
            torch.cuda.set_device(0)
            desc, x, y, hx, hy, hz, (zd, xd, yd) = data[k]
            su3.su3_tune_set(path=1, tile_mats=32 if k else 64, stages=2 + k)
            s = torch.cuda.Stream()
            for it in range(25):
                su3.su3_eval_host(su3.SU3_OP_MUL, hz, hx, hy, None, zd, xd, yd, None, chunks=3 + it % 5, stream=s.cuda_stream)
            s.synchronize()
            results[k] = hz.numpy().copy()
        except BaseException as e:   # noqa: BLE001
            errors.append((k, repr(e)))

    ts = [threading.Thread(target=worker, args=(k,)) for k in range(2)]
    for t in ts:
        t.start()
    for t in ts:
        t.join()
    assert not errors, errors
    for k, (desc, x, y, *_rest) in enumerate(data):
        err, _ = rel_err(results[k], oracle.mul(geom_of(desc), x, y), su3.su3_desc_normalize(desc).W)
        assert err <= TOL[desc.prec], (k, err)
    assert su3.su3_tune_get()["path"] == 0          # the workers' knobs were thread-local
    su3.su3_host_release()
    with pytest.raises(su3.Su3Error) as e:
        su3.su3_eval_host(su3.SU3_OP_MUL, None, None, None, None, data[0][6][0], data[0][6][1], data[0][6][2], None, chunks=65)
    assert e.value.status == su3.SU3_ERR_INVALID
