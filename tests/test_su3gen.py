"""The seeded input generator (su3gen/): SU(3)-ness, moments, counter-based determinism."""
import numpy as np

import su3gen


def test_su3_unitarity_and_det():
    x = su3gen.su3_field(su3gen.config_seed(5), su3gen.FIELD_X, 1 << 18)
    assert np.abs(x @ x.conj().transpose(0, 2, 1) - np.eye(3)).max() <= 1e-13
    assert np.abs(np.linalg.det(x) - 1).max() <= 1e-13


def test_counter_based_any_order_any_chunk():
    a = su3gen.su3_field(42, 1, 1000)
    b = np.concatenate([su3gen.su3_field(42, 1, 300, m0=0), su3gen.su3_field(42, 1, 700, m0=300)])
    assert np.array_equal(a, b)
    assert not np.array_equal(a, su3gen.su3_field(43, 1, 1000))
    assert not np.array_equal(a, su3gen.su3_field(42, 2, 1000))
    assert np.array_equal(su3gen.gaussian_field(42, 3, 50, m0=950), su3gen.gaussian_field(42, 3, 1000)[950:])


def test_uniforms_open_interval_and_moments():
    u = su3gen.uniforms(1, 0, 0, 1 << 20)
    assert u.min() > 0 and u.max() < 1
    assert abs(u.mean() - 0.5) < 2e-3 and abs(u.var() - 1 / 12) < 1e-3
    r = su3gen.raw_draws(1, 0, 0, 1 << 16)
    bits = np.unpackbits(r.view(np.uint8))
    assert abs(bits.mean() - 0.5) < 2e-3
    assert len(np.unique(r)) == len(r)


def test_gaussian_unit_variance():
    v = su3gen.gaussian_field(7, su3gen.FIELD_V, 1 << 17)
    assert abs((np.abs(v) ** 2).mean() - 1.0) < 5e-3          # E|v_ij|^2 = 1 (S14)
    assert abs(v.real.var() - 0.5) < 5e-3 and abs(v.imag.var() - 0.5) < 5e-3
    assert abs(v.mean()) < 5e-3
    assert abs(np.mean(v.real * v.imag)) < 5e-3
    k = np.mean(v.real ** 4) / v.real.var() ** 2             # Gaussian kurtosis = 3
    assert abs(k - 3) < 0.05


def test_haar_like_first_moments():
    x = su3gen.su3_field(3, 0, 1 << 16)
    tr = np.trace(x, axis1=1, axis2=2)
    assert abs(tr.mean()) < 2e-2                  # <tr U> = 0 under Haar
    assert abs((np.abs(tr) ** 2).mean() - 1.0) < 3e-2  # <|tr U|^2> = 1 under Haar
