"""Seeded synthetic lattice fields for the SU(3)xSU(3) streaming test.

Input generation only: no matrix product and no layout map live here (those are
the method, implemented twice and independently in ``oracle/`` and in the CUDA
library).  Recipe = SURVEY.md section 8(c) readings S10-S14 (the paper is
silent on how x, y are initialised), restated in DESIGN.md.

Fields come back in the LOGICAL order ``a[m, i, j]`` (complex128), with
``m = site * n_lorentz + mu`` and ``site = x0 + L0*(x1 + L1*(x2 + L2*x3))``.
"""
import ctypes

import numpy as np

from .build import build as _build

FIELD_X, FIELD_Y, FIELD_W, FIELD_V = 0, 1, 2, 3
BASE_SEED = 171009409  # + config number (S13)

_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(_build())
        u64, i64, dbl = ctypes.c_uint64, ctypes.c_int64, ctypes.c_double
        lib.su3gen_raw.argtypes = [u64, u64, u64, i64, ctypes.c_void_p]
        lib.su3gen_uniform.argtypes = [u64, u64, u64, i64, ctypes.c_void_p]
        lib.su3gen_gaussian.argtypes = [u64, u64, i64, i64, dbl, ctypes.c_void_p]
        lib.su3gen_su3.argtypes = [u64, u64, i64, i64, ctypes.c_void_p]
        for f in (lib.su3gen_raw, lib.su3gen_uniform, lib.su3gen_gaussian, lib.su3gen_su3):
            f.restype = None
        _lib = lib
    return _lib


def config_seed(config_number: int) -> int:
    return BASE_SEED + int(config_number)


def raw_draws(seed: int, field_id: int, ctr0: int, n: int) -> np.ndarray:
    out = np.empty(n, dtype=np.uint64)
    _load().su3gen_raw(seed, field_id, ctr0, n, out.ctypes.data)
    return out


def uniforms(seed: int, field_id: int, ctr0: int, n: int) -> np.ndarray:
    out = np.empty(n, dtype=np.float64)
    _load().su3gen_uniform(seed, field_id, ctr0, n, out.ctypes.data)
    return out


def gaussian_field(seed: int, field_id: int, count: int, m0: int = 0, variance: float = 1.0,
                   out: np.ndarray = None) -> np.ndarray:
    """Complex Gaussian 3x3 matrices m0..m0+count-1, E|a_ij|^2 = variance (S14)."""
    if out is None:
        out = np.empty((count, 3, 3), dtype=np.complex128)
    assert out.dtype == np.complex128 and out.flags.c_contiguous and out.size == 9 * count
    _load().su3gen_gaussian(seed, field_id, m0, count, variance, out.ctypes.data)
    return out


def su3_field(seed: int, field_id: int, count: int, m0: int = 0, out: np.ndarray = None) -> np.ndarray:
    """Random SU(3) matrices m0..m0+count-1 (S10-S13)."""
    if out is None:
        out = np.empty((count, 3, 3), dtype=np.complex128)
    assert out.dtype == np.complex128 and out.flags.c_contiguous and out.size == 9 * count
    _load().su3gen_su3(seed, field_id, m0, count, out.ctypes.data)
    return out
