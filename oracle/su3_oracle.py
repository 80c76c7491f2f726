"""ctypes wrapper around su3_oracle.c (argument marshalling only; see the C file
for what each routine follows in PAPER.md).  TEST INFRASTRUCTURE ONLY."""
import ctypes

import numpy as np

from .build import build as _build


class _CGeom(ctypes.Structure):
    _fields_ = [("L", ctypes.c_int32 * 4), ("nl", ctypes.c_int32), ("layout", ctypes.c_int32),
                ("W", ctypes.c_int32), ("simd", ctypes.c_int32 * 4)]


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(_build())
        P, I, I64, V = ctypes.POINTER(_CGeom), ctypes.c_int, ctypes.c_int64, ctypes.c_void_p
        I32P = ctypes.POINTER(ctypes.c_int32)
        lib.orc_default_simd.argtypes = [I, I32P]
        lib.orc_default_simd.restype = None
        lib.orc_geom_init.argtypes = [P, I32P, I, I, I, I32P]
        lib.orc_geom_init.restype = I
        lib.orc_volume.argtypes = [P]
        lib.orc_volume.restype = I64
        lib.orc_site_to_outer.argtypes = [P, I64, ctypes.POINTER(I64), I32P]
        lib.orc_site_to_outer.restype = None
        lib.orc_index.argtypes = [P, I64, I, I, I, I]
        lib.orc_index.restype = I64
        lib.orc_mul.argtypes = [P, I, V, V, V]
        lib.orc_mul.restype = None
        lib.orc_mul3.argtypes = [P, I, V, V, V, V]
        lib.orc_mul3.restype = None
        lib.orc_mul_add.argtypes = [P, I, V, V, V, V]
        lib.orc_mul_add.restype = None
        lib.orc_expr.argtypes = [P, I, I, ctypes.POINTER(V), ctypes.c_char_p, V]
        lib.orc_expr.restype = I
        lib.orc_cshift.argtypes = [P, I, V, V, I, I]
        lib.orc_cshift.restype = I
        lib.orc_mul_shift.argtypes = [P, I, V, V, I, I, V]
        lib.orc_mul_shift.restype = I
        lib.orc_neighbour.argtypes = [P, I64, I, I]
        lib.orc_neighbour.restype = I64
        lib.orc_index_vec.argtypes = [P, I64, I, I, I]
        lib.orc_index_vec.restype = I64
        lib.orc_matvec.argtypes = [P, I, V, V, V]
        lib.orc_matvec.restype = None
        lib.orc_convert_vec.argtypes = [P, P, I, V, V]
        lib.orc_convert_vec.restype = I
        lib.orc_expr_real.argtypes = [I64, I, I, ctypes.POINTER(V), ctypes.c_char_p, V]
        lib.orc_expr_real.restype = I
        lib.orc_convert.argtypes = [P, P, I, V, V]
        lib.orc_convert.restype = I
        lib.orc_num_threads.restype = I
        lib.orc_set_num_threads.argtypes = [I]
        lib.orc_set_num_threads.restype = None
        _lib = lib
    return _lib


SCALAR, VECTOR = 0, 1


class Geom:
    """Lattice geometry + layout (L[4], n_lorentz, layout, W, simd[4])."""

    def __init__(self, L, nl=1, layout=SCALAR, W=1, simd=None):
        if np.isscalar(L):
            L = (int(L),) * 4
        self.c = _CGeom()
        Larr = (ctypes.c_int32 * 4)(*[int(v) for v in L])
        sarr = (ctypes.c_int32 * 4)(*([int(v) for v in simd] if simd is not None else [0, 0, 0, 0]))
        rc = _load().orc_geom_init(ctypes.byref(self.c), Larr, int(nl), int(layout), int(W), sarr)
        if rc:
            raise ValueError("inadmissible geometry (orc_geom_init -> %d)" % rc)

    L = property(lambda s: tuple(s.c.L))
    nl = property(lambda s: int(s.c.nl))
    layout = property(lambda s: int(s.c.layout))
    W = property(lambda s: int(s.c.W))
    simd = property(lambda s: tuple(s.c.simd))
    volume = property(lambda s: int(_load().orc_volume(ctypes.byref(s.c))))
    nmat = property(lambda s: s.volume * s.nl)
    nreals = property(lambda s: s.nmat * 18)


def default_simd(W):
    out = (ctypes.c_int32 * 4)()
    _load().orc_default_simd(int(W), out)
    return tuple(out)


def site_to_outer(g, site):
    o, l = ctypes.c_int64(), ctypes.c_int32()
    _load().orc_site_to_outer(ctypes.byref(g.c), int(site), ctypes.byref(o), ctypes.byref(l))
    return int(o.value), int(l.value)


def index(g, site, mu, i, j, reim):
    return int(_load().orc_index(ctypes.byref(g.c), int(site), int(mu), int(i), int(j), int(reim)))


def _prec(a, g):
    assert a.flags.c_contiguous and a.size == g.nreals, (a.shape, g.nreals)
    if a.dtype == np.float64:
        return 8
    if a.dtype == np.float32:
        return 4
    raise TypeError(a.dtype)


def _out(g, out=None):
    """result buffer: a fresh fp64 array, or the caller's (bench.py times the oracle with first-touched outputs)"""
    if out is None:
        return np.empty(g.nreals, dtype=np.float64)
    assert out.dtype == np.float64 and out.flags.c_contiguous and out.size == g.nreals
    return out


def mul(g, x, y, out=None):
    """z = x*y; x, y flat real arrays (fp32 or fp64) in layout g; returns fp64, layout g."""
    p = _prec(x, g)
    assert _prec(y, g) == p
    z = _out(g, out)
    _load().orc_mul(ctypes.byref(g.c), p, x.ctypes.data, y.ctypes.data, z.ctypes.data)
    return z


def mul3(g, x, y, w, out=None):
    p = _prec(x, g)
    assert _prec(y, g) == p and _prec(w, g) == p
    z = _out(g, out)
    _load().orc_mul3(ctypes.byref(g.c), p, x.ctypes.data, y.ctypes.data, w.ctypes.data, z.ctypes.data)
    return z


def mul_add(g, x, y, v, out=None):
    p = _prec(x, g)
    assert _prec(y, g) == p and _prec(v, g) == p
    z = _out(g, out)
    _load().orc_mul_add(ctypes.byref(g.c), p, x.ctypes.data, y.ctypes.data, v.ctypes.data, z.ctypes.data)
    return z


def expr(g, prog, *ops):
    """z = postfix expression `prog` ('0'..'7' push ops[k]; '+', '-', '*') over fields ops, all in layout g."""
    p = _prec(ops[0], g)
    assert all(_prec(o, g) == p for o in ops)
    z = _out(g)
    arr = (ctypes.c_void_p * len(ops))(*[o.ctypes.data for o in ops])
    rc = _load().orc_expr(ctypes.byref(g.c), p, len(ops), arr, prog.encode(), z.ctypes.data)
    if rc:
        raise ValueError("malformed expression %r (orc_expr -> %d)" % (prog, rc))
    return z


def neighbour(g, site, dim, disp):
    return int(_load().orc_neighbour(ctypes.byref(g.c), int(site), int(dim), int(disp)))


def cshift(g, x, dim, disp):
    """z[s] = x[s + disp*dim_hat] (Grid's Cshift), bit copy in x's precision, layout g."""
    p = _prec(x, g)
    z = np.empty_like(x)
    if _load().orc_cshift(ctypes.byref(g.c), p, z.ctypes.data, x.ctypes.data, int(dim), int(disp)):
        raise ValueError("dim %r outside 0..3" % (dim,))
    return z


def mul_shift(g, x, y, dim, disp):
    """z[s] = x[s] * y[s + disp*dim_hat]; fp64 result."""
    p = _prec(x, g)
    assert _prec(y, g) == p
    z = _out(g)
    if _load().orc_mul_shift(ctypes.byref(g.c), p, x.ctypes.data, y.ctypes.data, int(dim), int(disp), z.ctypes.data):
        raise ValueError("dim %r outside 0..3" % (dim,))
    return z


def index_vec(g, site, mu, i, reim):
    return int(_load().orc_index_vec(ctypes.byref(g.c), int(site), int(mu), int(i), int(reim)))


def matvec(g, U, psi):
    """y = U.psi per (site, mu): U a matrix field, psi a colour-vector field (nmat*6 reals), layout g; fp64 result."""
    p = _prec(U, g)
    assert psi.flags.c_contiguous and psi.size == g.nmat * 6 and psi.dtype == U.dtype
    y = np.empty(g.nmat * 6, dtype=np.float64)
    _load().orc_matvec(ctypes.byref(g.c), p, U.ctypes.data, psi.ctypes.data, y.ctypes.data)
    return y


def convert_vec(g_dst, g_src, src):
    assert src.flags.c_contiguous and src.size == g_src.nmat * 6
    dst = np.empty_like(src)
    if _load().orc_convert_vec(ctypes.byref(g_dst.c), ctypes.byref(g_src.c), src.dtype.itemsize, dst.ctypes.data, src.ctypes.data):
        raise ValueError("geometry mismatch")
    return dst


def expr_real(prog, *ops):
    """element-wise postfix expression over real scalar fields (flat fp32/fp64 arrays of equal length); fp64 result"""
    n = ops[0].size
    assert all(o.flags.c_contiguous and o.size == n and o.dtype == ops[0].dtype for o in ops)
    z = np.empty(n, dtype=np.float64)
    arr = (ctypes.c_void_p * len(ops))(*[o.ctypes.data for o in ops])
    rc = _load().orc_expr_real(n, ops[0].dtype.itemsize, len(ops), arr, prog.encode(), z.ctypes.data)
    if rc:
        raise ValueError("malformed expression %r (orc_expr_real -> %d)" % (prog, rc))
    return z


def convert(g_dst, g_src, src, out=None):
    """Bit-exact permutation of the reals of `src` (layout g_src) into layout g_dst."""
    p = _prec(src, g_src)
    dst = np.empty_like(src) if out is None else out
    assert dst.dtype == src.dtype and dst.size == src.size and dst.flags.c_contiguous
    rc = _load().orc_convert(ctypes.byref(g_dst.c), ctypes.byref(g_src.c), p, dst.ctypes.data, src.ctypes.data)
    if rc:
        raise ValueError("geometry mismatch (orc_convert -> %d)" % rc)
    return dst


def stream_triad(n, reps=3):
    """host STREAM triad a = b + s*c over n doubles, best of `reps`, in GB/s (24 B per element; arrays first-touched
    by the same OpenMP schedule).  A measurement aid for bench.py's cpu_baseline leg (the paper draws the STREAM
    triad next to its curves); not part of the method."""
    lib = _load()
    lib.orc_stream_triad.argtypes = [ctypes.c_int64, ctypes.c_int]
    lib.orc_stream_triad.restype = ctypes.c_double
    return float(lib.orc_stream_triad(int(n), int(reps)))


def num_threads():
    return int(_load().orc_num_threads())


def set_num_threads(n):
    _load().orc_set_num_threads(int(n))
