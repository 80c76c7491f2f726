"""-m gpu: z = x*y at EVERY point of the volume sweep (BASELINE.json configs[4]: L = 8..64, fp64 and fp32, scalar and
vector W=4/8) in the launch configuration bench.py times: library defaults, su3_tune_set untouched, the same fields
called several times back to back (Listing 3: the Nloop loop on the same x, y, z).

The library picks kernel family, ring depth and L2 policy from the footprint (su3_launch_plan reports the choice):
direct / warp-staged kernels while everything is L2-resident, the TMA pipeline with a depth-4 ring and PINNED operand
prefixes (evict_last) between 0.6 and 2 x L2, depth 4 up to 3 x L2, depth 3 beyond.  The other parity tests force those
paths by knob on small lattices; here the automatic choice itself runs, on the sizes where it switches, and the THIRD
call is the one compared with the oracle (whole field, S15) -- it sees the L2 lines the first two calls pinned.  The
48^4 and 64^4 points are in test_gpu_wholefield.py / test_gpu_fullsize.py (defaults as well)."""
import numpy as np
import pytest
import torch

import oracle
import paper_1710_09409_b200 as su3
from gpu_util import download, geom_of, host_field, scalar_desc, upload
from helpers import TOL, rel_err_chunked

pytestmark = pytest.mark.gpu
F64, F32, VEC = su3.SU3_F64, su3.SU3_F32, su3.SU3_VECTOR


@pytest.fixture(autouse=True)
def _defaults():
    su3.su3_tune_set()
    yield
    su3.su3_tune_set()
    torch.cuda.empty_cache()


def _b200_l2():
    return 120e6 < su3.su3_device_info()["l2_bytes"] < 140e6


# what the automatic choice is on a B200 (L2 = 126 MiB), per (L, precision, vector layout?):  family, ring depth, l2
EXPECT = {
    (8, F64, False): ("warp", 0, "none"), (8, F64, True): ("direct", 0, "none"),
    (12, F64, False): ("warp", 0, "none"), (12, F64, True): ("direct", 0, "none"),
    (16, F64, False): ("warp", 0, "none"), (16, F64, True): ("direct", 0, "none"),
    (24, F64, False): ("pipe", 4, "pin"), (24, F64, True): ("pipe", 4, "pin"),          # 143 MB: the knee
    (32, F64, False): ("pipe", 3, "none"), (32, F64, True): ("pipe", 3, "none"),        # 453 MB > 3 x L2
    (8, F32, False): ("warp", 0, "none"), (8, F32, True): ("direct", 0, "none"),
    (12, F32, False): ("warp", 0, "none"), (12, F32, True): ("direct", 0, "none"),
    (16, F32, False): ("warp", 0, "none"), (16, F32, True): ("direct", 0, "none"),
    (24, F32, False): ("pipe", 4, "none"), (24, F32, True): ("direct", 0, "none"),      # 72 MB: between L2/2 and 0.6 x L2
    (32, F32, False): ("pipe", 4, "pin"), (32, F32, True): ("pipe", 4, "pin"),          # 226 MB
}


def _run_point(L, prec, vector, calls=3):
    W = (4 if prec == F64 else 8) if vector else 1
    d = su3.make_desc(L, prec=prec, layout=VEC if vector else su3.SU3_SCALAR, W=W)
    hx, hy = host_field(d, 171009409 + 5, 0), host_field(d, 171009409 + 5, 1)
    x, y, z = upload(d, hx), upload(d, hy), su3.alloc_field(d)
    z.tensor.fill_(0xFF)
    for _ in range(calls):
        su3.su3_mul(z, x, y)
    zg = download(z)
    err, _ = rel_err_chunked(zg, oracle.mul(geom_of(d), hx, hy), W)
    assert np.isfinite(zg).all() and err <= TOL[prec], (L, prec, vector, err)
    return d, zg


@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("L", [8, 12, 16, 24, 32])
def test_mul_at_library_defaults_on_every_sweep_point(L, prec):
    assert su3.su3_tune_get() == dict(tile_mats=0, stages=0, ctas_per_sm=0, l2_hint=0, path=0, l2_pin_mb=0)
    out = {}
    for vector in (False, True):
        d, zg = _run_point(L, prec, vector)
        plan = su3.su3_launch_plan(d, 0)
        if _b200_l2():
            fam, depth, l2 = EXPECT[(L, prec, vector)]
            assert (plan["family"], plan["depth"], plan["l2"]) == (fam, depth, l2), (L, prec, vector, plan)
            assert (plan["pin_bytes"] > 0) == (l2 == "pin")
        out[vector] = (d, zg)
    # the scalar-layout and the vector-layout results agree bit for bit after the (oracle's) layout permutation,
    # whichever kernel family each of them ran on
    (ds, zs), (dv, zv) = out[False], out[True]
    assert np.array_equal(oracle.convert(geom_of(scalar_desc(dv)), geom_of(dv), zv).view(np.uint8), zs.view(np.uint8))


@pytest.mark.parametrize("vector", [False, True])
@pytest.mark.parametrize("knobs", [dict(l2_hint=3, l2_pin_mb=1), dict(l2_hint=3, l2_pin_mb=8), dict(l2_hint=3, l2_pin_mb=40),
                                   dict(l2_hint=3, l2_pin_mb=40, stages=4), dict(l2_hint=1, stages=4), dict(l2_hint=2, stages=3),
                                   dict(path=1, l2_hint=3, l2_pin_mb=1000)])
def test_knee_with_explicit_pinning_knobs(knobs, vector):
    """24^4 fp64 (143 MB, between 0.6 and 2 x L2): the pinned-prefix policy with small, medium and larger-than-the-field
    prefixes, and the ring depths around the default, five calls in a row"""
    su3.su3_tune_set(**knobs)
    d, _ = _run_point(24, F64, vector, calls=5)
    plan = su3.su3_launch_plan(d, 0)
    assert plan["family"] == "pipe" and plan["l2"] == {1: "none", 2: "evict_first", 3: "pin"}[knobs["l2_hint"]]
    if "stages" in knobs:
        assert plan["depth"] == knobs["stages"]
    if knobs["l2_hint"] == 3:
        assert plan["pin_bytes"] == knobs["l2_pin_mb"] * 1000000


def test_fused_expressions_at_the_knee_defaults():
    """mul3 / mul_add at 32^4 fp32 W=8 (4 fields = 302 MB... above 2 x L2: depth 4, no pin) and 24^4 fp64 (191 MB: pinned)"""
    for L, prec, W in ((24, F64, 4), (24, F64, 1), (32, F32, 8)):
        d = su3.make_desc(L, prec=prec, layout=VEC if W > 1 else su3.SU3_SCALAR, W=W)
        hx, hy, hw = (host_field(d, 171009409 + 4, i) for i in range(3))
        hv = host_field(d, 171009409 + 4, 3, kind="gauss")
        x, y, w, v, z = upload(d, hx), upload(d, hy), upload(d, hw), upload(d, hv), su3.alloc_field(d)
        g = geom_of(d)
        for _ in range(3):
            su3.su3_mul3(z, x, y, w)
        e3, _ = rel_err_chunked(download(z), oracle.mul3(g, hx, hy, hw), W)
        for _ in range(3):
            su3.su3_mul_add(z, x, y, v)
        ea, _ = rel_err_chunked(download(z), oracle.mul_add(g, hx, hy, hv), W)
        assert e3 <= TOL[prec] and ea <= TOL[prec], (L, prec, W, e3, ea)
        if _b200_l2():
            assert su3.su3_launch_plan(d, 1)["l2"] == ("pin" if L == 24 else "none")
