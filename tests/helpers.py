"""Shared test helpers: golden fixtures, logical<->flat packing, the S15 error norm.
Holds no product code; numpy only."""
import os

import numpy as np

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")

TOL = {8: 1e-12, 4: 2e-5}  # north_star: max relative error, fp64 / fp32 (per-matrix max-norm, S15)


def load_integer_case():
    """{name: (3,3) complex128} for matrices, {name: complex} for determinants."""
    out = {}
    with open(os.path.join(GOLDEN, "su3_integer_case.txt")) as f:
        for line in f:
            line = line.split("#")[0].split()
            if not line:
                continue
            vals = [float(v) for v in line[1:]]
            if len(vals) == 18:
                out[line[0]] = (np.array(vals[0::2]) + 1j * np.array(vals[1::2])).reshape(3, 3)
            else:
                out[line[0]] = complex(vals[0], vals[1])
    return out


def load_vector_map_spots():
    spots, splits = [], {}
    with open(os.path.join(GOLDEN, "vector_map_spots.txt")) as f:
        for line in f:
            line = line.split("#")[0].split()
            if not line:
                continue
            if line[0] == "split":
                splits[int(line[1])] = tuple(int(v) for v in line[2:6])
            else:
                v = [int(t) for t in line]
                spots.append(dict(L=v[0], W=v[1], x=tuple(v[2:6]), site=v[6], outer=v[7], lane=v[8]))
    return spots, splits


def flat(a, dtype=np.float64):
    """logical (M,3,3) complex128 -> flat reals in the SCALAR layout (S1, S2, S6)."""
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return a.view(np.float64).reshape(-1).astype(dtype)


def logical(f):
    """flat reals in the SCALAR layout -> (M,3,3) complex128"""
    f = np.ascontiguousarray(f, dtype=np.float64)
    return f.view(np.complex128).reshape(-1, 3, 3)


def per_matrix_view(f, W):
    """flat reals of a field whose records hold W matrices lane-interleaved
    -> (nrec, 9, W, 2) view; W=1 is the scalar layout."""
    return f.reshape(-1, 9, W, 2)


def rel_err(z, zref, W):
    """S15: max over matrices of max_ij|z - zref| / max_ij|zref| (0 where the numerator is 0).
    Returns (per_matrix_max, worst elementwise abs diff)."""
    d = np.abs(per_matrix_view(z.astype(np.float64), W) - per_matrix_view(zref, W))
    num = d.max(axis=(1, 3))
    den = np.abs(per_matrix_view(zref, W)).max(axis=(1, 3))
    with np.errstate(divide="ignore", invalid="ignore"):
        r = np.where(num == 0, 0.0, num / den)
    return float(r.max()) if r.size else 0.0, float(d.max()) if d.size else 0.0


def rel_err_chunked(z, zref, W, chunk_records=1 << 20):
    """rel_err over a whole large field, evaluated in slices of `chunk_records` records so that the temporaries
    stay small next to the field (64^4 fp64 = 2.4 GB per array)."""
    step = chunk_records * 18 * W
    worst, worst_abs = 0.0, 0.0
    assert z.size == zref.size and z.size % (18 * W) == 0
    for a in range(0, z.size, step):
        e, d = rel_err(z[a:a + step], zref[a:a + step], W)
        worst, worst_abs = max(worst, e), max(worst_abs, d)
    return worst, worst_abs
