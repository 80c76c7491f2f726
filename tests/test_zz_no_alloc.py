"""su3_face_move_static: the face move for users who cannot allocate device memory at the point where they need it.

Who that is: a job whose framework already owns all of HBM through its own pool (a cudaMalloc from a library fails
there or fragments the pool), a communication thread that must not stall the whole device inside cudaMalloc/cudaFree
while it overlaps a face exchange with other streams, and an embedding that gets raw field pointers from its host and
has no allocator at all.  For them the library stages the packed face in a 16 MiB array that is part of its own device
image, so the caller passes nothing but the two fields.

What is checked here, on a GPU: the entry point writes exactly the bytes that the existing route writes
(su3_face_pack into a buffer the test allocates, then su3_face_unpack) -- faces are pure permutations, so the
tolerance is the one every face test of this suite uses, bit equality of the whole destination field, canaries
included -- on TWO calls in a row, the second one smaller than the first, so that anything the first call left in the
shared array would show; that the second call changes neither the free device memory nor anything but the launch
count; that a face above the limit is refused with nothing written.  Without a GPU: the refusals that need no device.

The file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the rest."""
import ctypes

import numpy as np
import pytest
import torch

import paper_1710_09409_b200 as su3
import su3gen
from helpers import flat

VEC, SCA = su3.SU3_VECTOR, su3.SU3_SCALAR
NPDT = {su3.SU3_F64: np.float64, su3.SU3_F32: np.float32}


def _desc(L, nl, prec, W):
    return su3.make_desc(L, n_lorentz=nl, prec=prec, layout=VEC if W > 1 else SCA, W=W)


def _random_field(desc, seed):
    """a field of seeded Gaussian reals: a face move only permutes bytes, so which layout they are 'in' is irrelevant"""
    f = su3.alloc_field(desc)
    nmat = f.nbytes // (18 * desc.prec)
    host = flat(su3gen.gaussian_field(seed, 0, nmat), NPDT[desc.prec])
    f.tensor.copy_(torch.from_numpy(host.view(np.uint8)))
    return f


def _canary_field(desc, byte):
    f = su3.alloc_field(desc)
    f.tensor.fill_(byte)
    return f


def _existing_route(z, z_plane0, x, x_plane0, dim, n):
    """su3_face_pack -> a buffer allocated HERE -> su3_face_unpack: the path the new entry point must reproduce"""
    buf = torch.empty(max(su3.su3_face_bytes(x, dim, n), 16), dtype=torch.uint8, device="cuda")
    su3.su3_face_pack(buf, x, dim, x_plane0, n)
    su3.su3_face_unpack(z, buf, dim, z_plane0, n)


@pytest.mark.gpu
@pytest.mark.parametrize("prec", [su3.SU3_F64, su3.SU3_F32])
@pytest.mark.parametrize("L,nl,Wx,Wz", [((6, 4, 2, 8), 1, 1, 1), ((4, 4, 4, 8), 4, 4, 4), ((4, 4, 4, 8), 1, 8, 1),
                                         ((8, 4, 4, 4), 1, 1, 2)])
def test_two_calls_in_a_row_match_pack_unpack(prec, L, nl, Wx, Wz):
    dx, dz = _desc(L, nl, prec, Wx), _desc(L, nl, prec, Wz)
    x = _random_field(dx, 31)
    # first call: a large face (all but one plane along x3); second: a single plane along x1 -- smaller, so most of
    # what the first call staged is still lying in the shared array when the second one runs
    calls = [(3, 1, 0, L[3] - 1), (1, L[1] - 1, 0, 1)]
    got, want = _canary_field(dz, 0x5C), _canary_field(dz, 0x5C)
    for dim, x_p0, z_p0, n in calls:
        su3.su3_face_move_static(got, z_p0, x, x_p0, dim, n)
        _existing_route(want, z_p0, x, x_p0, dim, n)
        torch.cuda.synchronize()
        assert torch.equal(got.tensor, want.tensor), (dim, x_p0, z_p0, n)
    assert not bool((got.tensor == 0x5C).all())                    # the calls did write something


@pytest.mark.gpu
def test_second_call_allocates_nothing_and_launches_two_kernels():
    d = _desc((8, 8, 8, 8), 1, su3.SU3_F64, 4)
    x, z = _random_field(d, 7), _canary_field(d, 0x11)
    su3.su3_face_move_static(z, 0, x, 4, 3, 2)                      # set-up call of this device (and module load)
    torch.cuda.synchronize()
    free0, launches0 = torch.cuda.mem_get_info()[0], su3.su3_launch_count()
    su3.su3_face_move_static(z, 6, x, 1, 3, 2)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0                    # the driver's free-memory figure did not move
    assert su3.su3_launch_count() == launches0 + 2                  # field -> area, area -> field
    want = _canary_field(d, 0x11)
    _existing_route(want, 0, x, 4, 3, 2)
    _existing_route(want, 6, x, 1, 3, 2)
    torch.cuda.synchronize()
    assert torch.equal(z.tensor, want.tensor)


@pytest.mark.gpu
def test_planes_moved_inside_one_field():
    """z may be x, overlapping plane ranges included: the first launch has read the planes before the second writes"""
    d = _desc((4, 4, 6, 8), 1, su3.SU3_F32, 1)
    a = _random_field(d, 3)
    src = su3.alloc_field(d)
    src.tensor.copy_(a.tensor)
    want = su3.alloc_field(d)
    want.tensor.copy_(a.tensor)
    for _ in range(2):                                              # twice in a row: planes 1..5 -> 3..7, then again
        su3.su3_face_move_static(a, 3, a, 1, 3, 5)
        _existing_route(want, 3, src, 1, 3, 5)                      # reference reads an untouched copy of the source
        torch.cuda.synchronize()
        assert torch.equal(a.tensor, want.tensor)
        src.tensor.copy_(want.tensor)


@pytest.mark.gpu
def test_limit_on_the_device():
    """just under the 16 MiB limit works and agrees with the existing route; just over is refused, nothing written"""
    d = _desc((32, 32, 32, 8), 1, su3.SU3_F64, 1)                   # one x3 plane = 32^3 * 144 B = 4.72 MB
    x, z, want = _random_field(d, 9), _canary_field(d, 0x77), _canary_field(d, 0x77)
    assert su3.su3_face_bytes(x, 3, 3) <= su3.SU3_STATIC_SCRATCH_BYTES < su3.su3_face_bytes(x, 3, 4)
    for p0 in (0, 5):                                               # two calls in a row at (nearly) the maximum size
        su3.su3_face_move_static(z, p0, x, 4 - p0 // 5, 3, 3)
        _existing_route(want, p0, x, 4 - p0 // 5, 3, 3)
        torch.cuda.synchronize()
        assert torch.equal(z.tensor, want.tensor)
    before, launches = z.tensor.clone(), su3.su3_launch_count()
    with pytest.raises(su3.Su3Error) as ei:
        su3.su3_face_move_static(z, 0, x, 0, 3, 4)
    assert ei.value.status == su3.SU3_ERR_SIZE and "static" in str(ei.value)
    torch.cuda.synchronize()
    assert su3.su3_launch_count() == launches and torch.equal(z.tensor, before)


def test_refusals_that_need_no_device():
    """argument errors are reported before any CUDA call, so they can be checked on a box without a GPU"""
    d = su3.make_desc((32, 32, 32, 8))
    dv = su3.make_desc((32, 32, 32, 8), layout=VEC, W=4)
    d32 = su3.make_desc((32, 32, 32, 8), prec=su3.SU3_F32)
    h, hv, h32, hc = (ctypes.c_void_p() for _ in range(4))
    wrap = su3.lib.su3_field_wrap
    assert wrap(ctypes.byref(d), ctypes.c_void_p(0x10000), su3.su3_field_bytes(d), ctypes.byref(h)) == su3.SU3_OK
    assert wrap(ctypes.byref(dv), ctypes.c_void_p(0x10000), su3.su3_field_bytes(dv), ctypes.byref(hv)) == su3.SU3_OK
    assert wrap(ctypes.byref(d32), ctypes.c_void_p(0x10000), su3.su3_field_bytes(d32), ctypes.byref(h32)) == su3.SU3_OK
    assert su3.lib.su3_vec_wrap(ctypes.byref(d), ctypes.c_void_p(0x10000), su3.su3_vec_bytes(d), ctypes.byref(hc)) == su3.SU3_OK
    f = su3.lib.su3_face_move_static
    assert f(h, 0, hv, 0, 3, 4, None) == su3.SU3_ERR_SIZE           # 18.9 MB > 16 MiB (layouts may differ: no mismatch)
    assert "static" in su3.su3_last_error()
    assert f(h, 0, h32, 0, 3, 1, None) == su3.SU3_ERR_MISMATCH      # precisions differ
    assert f(h, 0, hc, 0, 3, 1, None) == su3.SU3_ERR_MISMATCH       # colour matrices vs colour vectors
    assert f(h, 6, hv, 0, 3, 3, None) == su3.SU3_ERR_INVALID        # planes 6..8 of 0..7
    assert f(h, 0, hv, 0, 4, 1, None) == su3.SU3_ERR_INVALID        # no such dimension
    assert f(None, 0, hv, 0, 3, 1, None) == su3.SU3_ERR_NULL
    assert f(h, 0, None, 0, 3, 1, None) == su3.SU3_ERR_NULL
    assert su3.SU3_STATIC_SCRATCH_BYTES == 16 << 20
    for x in (h, hv, h32, hc):
        su3.lib.su3_field_free(x)
