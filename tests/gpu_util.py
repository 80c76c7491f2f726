"""Helpers of the -m gpu parity tests: host<->device moves through torch, seeded inputs in
either layout.  Inputs come from su3gen (logical order) and reach a vector-layout field
through the ORACLE's permutation on the host, never through the CUDA path."""
import numpy as np
import torch

import oracle
import paper_1710_09409_b200 as su3
import su3gen
from helpers import flat

NPDT = {su3.SU3_F64: np.float64, su3.SU3_F32: np.float32}


def geom_of(desc):
    d = su3.su3_desc_normalize(desc)
    return oracle.Geom(tuple(d.L), nl=d.n_lorentz, layout=d.layout, W=d.W, simd=tuple(d.simd))


def scalar_desc(desc):
    return su3.make_desc(tuple(desc.L), n_lorentz=desc.n_lorentz, prec=desc.prec)


def upload(desc, host_flat):
    """host flat reals (already in desc's layout and precision) -> Field on cuda:0"""
    assert host_flat.dtype == NPDT[desc.prec]
    f = su3.alloc_field(desc)
    assert host_flat.nbytes == f.nbytes
    f.tensor.copy_(torch.from_numpy(host_flat.view(np.uint8)))
    return f


def download(field):
    torch.cuda.synchronize()
    return field.tensor.cpu().numpy().view(NPDT[field.desc.prec]).copy()


def host_field(desc, seed, field_id, kind="su3"):
    """seeded field in desc's layout and precision (S10-S14, S16: fp32 = rounded fp64)"""
    d = su3.su3_desc_normalize(desc)
    nmat = d.L[0] * d.L[1] * d.L[2] * d.L[3] * d.n_lorentz
    a = su3gen.su3_field(seed, field_id, nmat) if kind == "su3" else su3gen.gaussian_field(seed, field_id, nmat)
    f = flat(a, NPDT[d.prec])
    if d.layout == su3.SU3_VECTOR:
        f = oracle.convert(geom_of(d), geom_of(scalar_desc(d)), f)
    return f


def const_field(desc, mats):
    """matrix m = mats[m % len(mats)] in logical order, exact small integers"""
    d = su3.su3_desc_normalize(desc)
    nmat = d.L[0] * d.L[1] * d.L[2] * d.L[3] * d.n_lorentz
    mats = np.asarray(mats, dtype=np.complex128).reshape(-1, 3, 3)
    a = mats[np.arange(nmat) % len(mats)]
    f = flat(a, NPDT[d.prec])
    if d.layout == su3.SU3_VECTOR:
        f = oracle.convert(geom_of(d), geom_of(scalar_desc(d)), f)
    return f
