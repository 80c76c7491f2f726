"""Thin Python binding of libsu3stream (include/su3stream.h): argument marshalling only.

Every step of the hot path (z = x*y, the fused expressions, the layout permutation, the
copy ceiling; arXiv:1710.09409 section 4/5) runs
in the library's CUDA kernels.  PyTorch supplies device memory and streams, nothing else.
There is no CPU fallback: if the shared library cannot be built or loaded, importing this
package raises.
"""
import ctypes

from ._build import build as _build_lib

SU3_OK, SU3_ERR_NULL, SU3_ERR_INVALID, SU3_ERR_MISMATCH, SU3_ERR_ALIGN, SU3_ERR_SIZE, SU3_ERR_CUDA = range(7)
SU3_F32, SU3_F64 = 4, 8
SU3_SCALAR, SU3_VECTOR = 0, 1

EXPORTS = ["su3_last_error", "su3_version", "su3_field_bytes", "su3_desc_normalize", "su3_field_wrap",
           "su3_field_free", "su3_field_desc", "su3_field_ptr", "su3_index", "su3_mul", "su3_mul3",
           "su3_mul_add", "su3_add", "su3_expr", "su3_expr_cost", "su3_expr_disasm", "su3_expr_plan", "su3_cshift", "su3_mul_shift", "su3_real_bytes", "su3_real_wrap", "su3_fill", "su3_vec_bytes", "su3_vec_wrap", "su3_vec_index", "su3_matvec", "su3_convert", "su3_copy", "su3_mul_host", "su3_eval_host", "su3_tune_set",
           "su3_tune_get", "su3_launch_count", "su3_device_info", "su3_device_name", "su3_host_release",
           "su3_face_bytes", "su3_face_pack", "su3_face_unpack", "su3_face_copy", "su3_cshift_slab",
           "su3_face_move_static", "su3_launch_plan"]


class su3_desc(ctypes.Structure):
    _fields_ = [("L", ctypes.c_int32 * 4), ("n_lorentz", ctypes.c_int32), ("prec", ctypes.c_int32),
                ("layout", ctypes.c_int32), ("W", ctypes.c_int32), ("simd", ctypes.c_int32 * 4)]


class su3_tune(ctypes.Structure):
    _fields_ = [("tile_mats", ctypes.c_int32), ("stages", ctypes.c_int32), ("ctas_per_sm", ctypes.c_int32),
                ("l2_hint", ctypes.c_int32), ("path", ctypes.c_int32), ("l2_pin_mb", ctypes.c_int32),
                ("reserved", ctypes.c_int32 * 2)]


class Su3Error(RuntimeError):
    def __init__(self, status, message):
        super().__init__("su3_status %d: %s" % (status, message))
        self.status = status


def _load():
    lib = ctypes.CDLL(_build_lib())
    vp, i32, i64, sz = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_size_t
    D, T = ctypes.POINTER(su3_desc), ctypes.POINTER(su3_tune)
    sig = {
        "su3_last_error": (ctypes.c_char_p, []),
        "su3_version": (ctypes.c_char_p, []),
        "su3_field_bytes": (i32, [D, ctypes.POINTER(sz)]),
        "su3_desc_normalize": (i32, [D, D]),
        "su3_field_wrap": (i32, [D, vp, sz, ctypes.POINTER(vp)]),
        "su3_field_free": (i32, [vp]),
        "su3_field_desc": (i32, [vp, D]),
        "su3_field_ptr": (i32, [vp, ctypes.POINTER(vp), ctypes.POINTER(sz)]),
        "su3_index": (i32, [D, i64, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.POINTER(i64)]),
        "su3_mul": (i32, [vp, vp, vp, vp]),
        "su3_mul3": (i32, [vp, vp, vp, vp, vp]),
        "su3_mul_add": (i32, [vp, vp, vp, vp, vp]),
        "su3_add": (i32, [vp, vp, vp, vp]),
        "su3_real_bytes": (i32, [D, ctypes.POINTER(sz)]),
        "su3_real_wrap": (i32, [D, vp, sz, ctypes.POINTER(vp)]),
        "su3_fill": (i32, [vp, ctypes.c_double, vp]),
        "su3_vec_bytes": (i32, [D, ctypes.POINTER(sz)]),
        "su3_vec_wrap": (i32, [D, vp, sz, ctypes.POINTER(vp)]),
        "su3_vec_index": (i32, [D, i64, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.POINTER(i64)]),
        "su3_matvec": (i32, [vp, vp, vp, vp]),
        "su3_cshift": (i32, [vp, vp, ctypes.c_int, ctypes.c_int, vp]),
        "su3_mul_shift": (i32, [vp, vp, vp, ctypes.c_int, ctypes.c_int, vp]),
        "su3_expr": (i32, [vp, ctypes.c_char_p, ctypes.POINTER(vp), ctypes.c_int, vp]),
        "su3_expr_disasm": (i32, [ctypes.c_char_p, ctypes.c_int, ctypes.c_char_p, sz]),
        "su3_expr_plan": (i32, [ctypes.c_char_p, ctypes.c_int, ctypes.c_int, ctypes.c_char_p, sz]),
        "su3_expr_cost": (i32, [ctypes.c_char_p, ctypes.c_int, ctypes.POINTER(i32), ctypes.POINTER(i32)]),
        "su3_convert": (i32, [vp, vp, vp]),
        "su3_copy": (i32, [vp, vp, vp]),
        "su3_mul_host": (i32, [vp, vp, vp, vp, vp, vp, ctypes.c_int, vp]),
        "su3_eval_host": (i32, [ctypes.c_int, vp, vp, vp, vp, vp, vp, vp, vp, ctypes.c_int, vp]),
        "su3_tune_set": (i32, [T]),
        "su3_tune_get": (i32, [T]),
        "su3_launch_count": (i64, []),
        "su3_device_info": (i32, [ctypes.POINTER(i32), ctypes.POINTER(i64), ctypes.POINTER(i32), ctypes.POINTER(i32)]),
        "su3_device_name": (i32, [ctypes.c_char_p, sz, ctypes.POINTER(i32)]),
        "su3_host_release": (i32, []),
        "su3_face_bytes": (i32, [vp, ctypes.c_int, ctypes.c_int, ctypes.POINTER(sz)]),
        "su3_face_pack": (i32, [vp, sz, vp, ctypes.c_int, ctypes.c_int, ctypes.c_int, vp]),
        "su3_face_unpack": (i32, [vp, vp, sz, ctypes.c_int, ctypes.c_int, ctypes.c_int, vp]),
        "su3_face_copy": (i32, [vp, ctypes.c_int, vp, ctypes.c_int, ctypes.c_int, ctypes.c_int, vp]),
        "su3_cshift_slab": (i32, [vp, vp, vp, ctypes.c_int, vp]),
        "su3_launch_plan": (i32, [D, ctypes.c_int, ctypes.c_char_p, sz]),
        "su3_face_move_static": (i32, [vp, ctypes.c_int, vp, ctypes.c_int, ctypes.c_int, ctypes.c_int, vp]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    return lib


lib = _load()  # fails loudly if the CUDA library is missing


def _ck(status):
    if status != SU3_OK:
        raise Su3Error(status, lib.su3_last_error().decode())


def su3_last_error():
    return lib.su3_last_error().decode()


def su3_version():
    return lib.su3_version().decode()


def make_desc(L, n_lorentz=1, prec=SU3_F64, layout=SU3_SCALAR, W=1, simd=None):
    d = su3_desc()
    L = (int(L),) * 4 if isinstance(L, int) else tuple(int(v) for v in L)
    d.L[:] = L
    d.n_lorentz, d.prec, d.layout, d.W = int(n_lorentz), int(prec), int(layout), int(W)
    d.simd[:] = tuple(int(v) for v in simd) if simd is not None else (0, 0, 0, 0)
    return d


def su3_field_bytes(desc):
    n = ctypes.c_size_t()
    _ck(lib.su3_field_bytes(ctypes.byref(desc), ctypes.byref(n)))
    return n.value


def su3_desc_normalize(desc):
    out = su3_desc()
    _ck(lib.su3_desc_normalize(ctypes.byref(desc), ctypes.byref(out)))
    return out


def su3_index(desc, site, mu, i, j, reim):
    off = ctypes.c_int64()
    _ck(lib.su3_index(ctypes.byref(desc), int(site), int(mu), int(i), int(j), int(reim), ctypes.byref(off)))
    return off.value


class Field:
    """A su3_field handle plus the torch tensor that owns its device memory (kind: "matrix" or "vector")."""

    def __init__(self, desc, tensor, kind="matrix"):
        self.tensor = tensor  # keeps the memory alive as long as the handle
        self.kind = kind
        h = ctypes.c_void_p()
        wrap = {"matrix": lib.su3_field_wrap, "vector": lib.su3_vec_wrap, "real": lib.su3_real_wrap}[kind]
        _ck(wrap(ctypes.byref(desc), ctypes.c_void_p(tensor.data_ptr()),
                 tensor.numel() * tensor.element_size(), ctypes.byref(h)))
        self.handle = h
        self.desc = su3_field_desc(self)
        self.nbytes = {"matrix": su3_field_bytes, "vector": su3_vec_bytes, "real": su3_real_bytes}[kind](self.desc)

    def __del__(self):
        h, self.handle = getattr(self, "handle", None), None
        if h and lib is not None:  # lib is None while the interpreter shuts down
            lib.su3_field_free(h)


def su3_field_wrap(desc, tensor):
    return Field(desc, tensor)


def su3_field_desc(field):
    out = su3_desc()
    _ck(lib.su3_field_desc(field.handle, ctypes.byref(out)))
    return out


def su3_field_ptr(field):
    p, n = ctypes.c_void_p(), ctypes.c_size_t()
    _ck(lib.su3_field_ptr(field.handle, ctypes.byref(p), ctypes.byref(n)))
    return p.value, n.value


def alloc_field(desc, device="cuda"):
    """north_star "allocate a field": su3_field_bytes -> torch.empty -> su3_field_wrap."""
    import torch
    return Field(desc, torch.empty(su3_field_bytes(desc), dtype=torch.uint8, device=device))


def _stream(stream):
    if stream is None:
        import torch
        return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    return ctypes.c_void_p(int(stream))


def su3_mul(z, x, y, stream=None):
    _ck(lib.su3_mul(z.handle, x.handle, y.handle, _stream(stream)))


def su3_mul3(z, x, y, w, stream=None):
    _ck(lib.su3_mul3(z.handle, x.handle, y.handle, w.handle, _stream(stream)))


def su3_mul_add(z, x, y, v, stream=None):
    _ck(lib.su3_mul_add(z.handle, x.handle, y.handle, v.handle, _stream(stream)))


def su3_add(z, x, y, stream=None):
    _ck(lib.su3_add(z.handle, x.handle, y.handle, _stream(stream)))


def su3_expr(z, program, operands, stream=None):
    """z = postfix `program` over `operands` (digits push operands[k]; '+', '-', '*'), one pass."""
    arr = (ctypes.c_void_p * len(operands))(*[o.handle.value for o in operands])
    _ck(lib.su3_expr(z.handle, program.encode(), arr, len(operands), _stream(stream)))


def su3_expr_disasm(program, n_operands):
    """the compiled register-machine listing, one (op, a, b, spill-or-None) tuple per instruction"""
    buf = ctypes.create_string_buffer(2048)
    _ck(lib.su3_expr_disasm(program.encode(), int(n_operands), buf, len(buf)))
    out = []
    for line in buf.value.decode().splitlines():
        t = line.split()
        out.append((t[0], t[1], t[2], t[4] if len(t) > 3 else None))
    return out


def su3_expr_plan(program, n_operands, real_fields=False):
    """"interpreter", or ("menu", row, row's postfix, [operand held by each slot]) for the ahead-of-time kernels"""
    buf = ctypes.create_string_buffer(256)
    _ck(lib.su3_expr_plan(program.encode(), int(n_operands), int(bool(real_fields)), buf, len(buf)))
    t = buf.value.decode().split()
    return "interpreter" if t[0] == "interpreter" else ("menu", int(t[1]), t[2], [int(v) for v in t[3:]])


def su3_expr_cost(program, n_operands):
    """(field streams, flops per matrix) of a program by reading S9"""
    st, fl = ctypes.c_int32(), ctypes.c_int32()
    _ck(lib.su3_expr_cost(program.encode(), int(n_operands), ctypes.byref(st), ctypes.byref(fl)))
    return st.value, fl.value


def su3_cshift(z, x, dim, disp, stream=None):
    _ck(lib.su3_cshift(z.handle, x.handle, int(dim), int(disp), _stream(stream)))


def su3_mul_shift(z, x, y, dim, disp, stream=None):
    _ck(lib.su3_mul_shift(z.handle, x.handle, y.handle, int(dim), int(disp), _stream(stream)))


def su3_real_bytes(desc):
    n = ctypes.c_size_t()
    _ck(lib.su3_real_bytes(ctypes.byref(desc), ctypes.byref(n)))
    return n.value


def su3_real_wrap(desc, tensor):
    return Field(desc, tensor, kind="real")


def alloc_real(desc, device="cuda"):
    import torch
    return Field(desc, torch.empty(su3_real_bytes(desc), dtype=torch.uint8, device=device), kind="real")


def su3_fill(z, value, stream=None):
    _ck(lib.su3_fill(z.handle, float(value), _stream(stream)))


def su3_vec_bytes(desc):
    n = ctypes.c_size_t()
    _ck(lib.su3_vec_bytes(ctypes.byref(desc), ctypes.byref(n)))
    return n.value


def su3_vec_wrap(desc, tensor):
    return Field(desc, tensor, kind="vector")


def alloc_vec(desc, device="cuda"):
    import torch
    return Field(desc, torch.empty(su3_vec_bytes(desc), dtype=torch.uint8, device=device), kind="vector")


def su3_vec_index(desc, site, mu, i, reim):
    off = ctypes.c_int64()
    _ck(lib.su3_vec_index(ctypes.byref(desc), int(site), int(mu), int(i), int(reim), ctypes.byref(off)))
    return off.value


def su3_matvec(y, U, psi, stream=None):
    _ck(lib.su3_matvec(y.handle, U.handle, psi.handle, _stream(stream)))


def su3_convert(dst, src, stream=None):
    _ck(lib.su3_convert(dst.handle, src.handle, _stream(stream)))


def su3_copy(dst, src, stream=None):
    _ck(lib.su3_copy(dst.handle, src.handle, _stream(stream)))


def su3_mul_host(z_host, x_host, y_host, zd, xd, yd, chunks=0, stream=None):
    """z_host, x_host, y_host: host tensors/arrays exposing .data_ptr() or .ctypes.data."""
    def hp(a):
        return ctypes.c_void_p(a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data)
    _ck(lib.su3_mul_host(hp(z_host), hp(x_host), hp(y_host), zd.handle, xd.handle, yd.handle, int(chunks),
                         _stream(stream)))


SU3_OP_MUL, SU3_OP_MUL3, SU3_OP_MUL_ADD = 0, 1, 2


def su3_eval_host(op, z_host, x_host, y_host, u_host, zd, xd, yd, ud, chunks=0, stream=None):
    """chunked H2D -> op -> D2H; a host argument of None means the operand is already resident (or, for z_host,
    that the result stays on the device)"""
    def hp(a):
        if a is None:
            return None
        return ctypes.c_void_p(a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data)
    _ck(lib.su3_eval_host(int(op), hp(z_host), hp(x_host), hp(y_host), hp(u_host), zd.handle, xd.handle, yd.handle,
                          ud.handle if ud is not None else None, int(chunks), _stream(stream)))


def su3_tune_set(tile_mats=0, stages=0, ctas_per_sm=0, l2_hint=0, path=0, l2_pin_mb=0):
    t = su3_tune(int(tile_mats), int(stages), int(ctas_per_sm), int(l2_hint), int(path), int(l2_pin_mb))
    _ck(lib.su3_tune_set(ctypes.byref(t)))


def su3_tune_get():
    t = su3_tune()
    _ck(lib.su3_tune_get(ctypes.byref(t)))
    return dict(tile_mats=t.tile_mats, stages=t.stages, ctas_per_sm=t.ctas_per_sm, l2_hint=t.l2_hint, path=t.path,
                l2_pin_mb=t.l2_pin_mb)


def su3_launch_count():
    return int(lib.su3_launch_count())


def su3_device_info():
    sm, l2, mk, bw = ctypes.c_int32(), ctypes.c_int64(), ctypes.c_int32(), ctypes.c_int32()
    _ck(lib.su3_device_info(ctypes.byref(sm), ctypes.byref(l2), ctypes.byref(mk), ctypes.byref(bw)))
    return dict(sm_count=sm.value, l2_bytes=l2.value, mem_clock_khz=mk.value, bus_width_bits=bw.value)


def su3_device_name():
    """(name, ordinal) of the current CUDA device"""
    buf, o = ctypes.create_string_buffer(128), ctypes.c_int32()
    _ck(lib.su3_device_name(buf, len(buf), ctypes.byref(o)))
    return buf.value.decode(), o.value


def su3_host_release():
    _ck(lib.su3_host_release())


def su3_face_bytes(field, dim, nplanes):
    n = ctypes.c_size_t()
    _ck(lib.su3_face_bytes(field.handle, int(dim), int(nplanes), ctypes.byref(n)))
    return n.value


def su3_face_pack(buf, x, dim, plane0, nplanes, stream=None):
    """buf (a uint8 device tensor) <- planes [plane0, plane0+nplanes) of x along dim, in plane order"""
    _ck(lib.su3_face_pack(ctypes.c_void_p(buf.data_ptr()), buf.numel() * buf.element_size(), x.handle, int(dim),
                          int(plane0), int(nplanes), _stream(stream)))


def su3_face_unpack(z, buf, dim, plane0, nplanes, stream=None):
    _ck(lib.su3_face_unpack(z.handle, ctypes.c_void_p(buf.data_ptr()), buf.numel() * buf.element_size(), int(dim),
                            int(plane0), int(nplanes), _stream(stream)))


def su3_face_copy(z, z_plane0, x, x_plane0, dim, nplanes, stream=None):
    _ck(lib.su3_face_copy(z.handle, int(z_plane0), x.handle, int(x_plane0), int(dim), int(nplanes), _stream(stream)))


def su3_launch_plan(desc, op=0):
    """the launch su3_mul (op 0) / su3_mul3 (1) / su3_mul_add (2) would make for this descriptor, as a dict:
    family ("direct" | "warp" | "pipe"), tile, depth, ctas, grid, block, smem, l2 ("none" | "evict_first" | "pin"), pin_bytes"""
    buf = ctypes.create_string_buffer(256)
    _ck(lib.su3_launch_plan(ctypes.byref(desc), int(op), buf, len(buf)))
    words = buf.value.decode().split()
    out = {"family": words[0]}
    for w in words[1:]:
        k, v = w.split("=")
        out[k] = v if k == "l2" else int(v)
    return out


SU3_STATIC_SCRATCH_BYTES = 16 << 20


def su3_face_move_static(z, z_plane0, x, x_plane0, dim, nplanes, stream=None):
    """planes [z_plane0, +nplanes) of z <- planes [x_plane0, +nplanes) of x along dim, staged through the 16 MiB area
    that lives inside the library's device image -- for callers that cannot allocate device memory where they need a
    face moved (all of HBM already belongs to a framework's pool, a communication thread that must not stall the device
    in cudaMalloc/cudaFree, an embedding that owns no allocator).  Nothing is allocated here either: no tensor is
    created, the arguments are passed through.  Same result as su3_face_pack + su3_face_unpack; z and x may differ in
    layout and may be the same field.  Faces above SU3_STATIC_SCRATCH_BYTES raise Su3Error(SU3_ERR_SIZE).  Make the
    first call per device during start-up, before any stream capture; calls that overlap on the GPU race on the shared
    area (include/su3stream.h has the full contract)."""
    _ck(lib.su3_face_move_static(z.handle, int(z_plane0), x.handle, int(x_plane0), int(dim), int(nplanes),
                                 _stream(stream)))


def su3_cshift_slab(z, x, x_nbr, disp, stream=None):
    """Cshift along x3 of slab x continued by the neighbouring slab x_nbr (next rank's for disp > 0, previous for disp < 0)"""
    _ck(lib.su3_cshift_slab(z.handle, x.handle, x_nbr.handle, int(disp), _stream(stream)))
