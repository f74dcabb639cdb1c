"""Pins for the oracle's real spherical harmonics and segment-integrated basis matrix (Eq. 3).
CPU only.  Each test is a closed form, an invariant or a library cross-check — none re-types the oracle."""
import math

import numpy as np
import pytest
from numpy.polynomial import legendre as leg


def _rand_units(n, seed):
    rng = np.random.default_rng(seed)
    v = rng.standard_normal((n, 3))
    return v / np.linalg.norm(v, axis=1, keepdims=True)


def test_index_order_and_count(ora):
    for lmax, K in ((0, 1), (2, 6), (4, 15), (6, 28), (8, 45)):
        idx = ora.sh_index(lmax)
        assert len(idx) == K == (lmax + 1) * (lmax + 2) // 2
        assert idx[0] == (0, 0)
        assert all(l % 2 == 0 for l, _ in idx)
    assert ora.sh_index(2)[1:] == [(2, -2), (2, -1), (2, 0), (2, 1), (2, 2)]


def test_closed_forms_l0_l2(ora):
    """Y_00 = 1 and the Cartesian l = 2 forms of 4pi-normalised real harmonics (SURVEY.md §8c pin)."""
    n = _rand_units(200, 1)
    x, y, z = n.T
    assert np.allclose(ora.real_sh(0, 0, n), 1.0, atol=1e-15)
    s15, s5 = math.sqrt(15.0), math.sqrt(5.0)
    want = {-2: s15 * x * y, -1: s15 * y * z, 0: 0.5 * s5 * (3 * z * z - 1), 1: s15 * x * z,
            2: 0.5 * s15 * (x * x - y * y)}
    for m, w in want.items():
        assert np.allclose(ora.real_sh(2, m, n), w, atol=1e-13), m


def test_closed_form_l4_m0_and_sectoral(ora):
    n = _rand_units(100, 2)
    x, y, z = n.T
    assert np.allclose(ora.real_sh(4, 0, n), 3.0 / 8.0 * (35 * z ** 4 - 30 * z ** 2 + 3), atol=1e-13)
    # sectoral l = m = 4: sqrt(2) sqrt(9/8!) 105 Re (x+iy)^4
    c = math.sqrt(2.0) * math.sqrt(9.0 / math.factorial(8)) * 105.0
    assert np.allclose(ora.real_sh(4, 4, n), c * np.real((x + 1j * y) ** 4), atol=1e-12)
    assert np.allclose(ora.real_sh(4, -4, n), c * np.imag((x + 1j * y) ** 4), atol=1e-12)


def test_sphere_mean_orthonormal(ora):
    """(1/4pi) int Y_i Y_j = delta_ij for all even l <= 8: Gauss-Legendre in cos(theta) x uniform phi."""
    xs, ws = leg.leggauss(24)
    nphi = 40
    ph = 2 * math.pi * np.arange(nphi) / nphi
    ct, pp = np.meshgrid(xs, ph, indexing="ij")
    st = np.sqrt(1 - ct ** 2)
    n = np.stack([st * np.cos(pp), st * np.sin(pp), ct], axis=-1)
    wq = (ws[:, None] / 2.0) * np.full((1, nphi), 1.0 / nphi)
    idx = ora.sh_index(8)
    Y = np.stack([ora.real_sh(l, m, n) for l, m in idx], axis=0)
    G = np.einsum("iab,jab,ab->ij", Y, Y, wq)
    assert np.allclose(G, np.eye(len(idx)), atol=1e-12)


def test_addition_theorem(ora):
    """sum_m Y_lm(n) Y_lm(q) = (2l+1) P_l(n.q): fixes normalisation and rotation invariance for every l."""
    n, q = _rand_units(50, 3), _rand_units(50, 4)
    for l in range(0, 9, 2):
        s = sum(ora.real_sh(l, m, n) * ora.real_sh(l, m, q) for m in range(-l, l + 1))
        want = (2 * l + 1) * leg.Legendre.basis(l)(np.sum(n * q, axis=1))
        assert np.allclose(s, want, atol=1e-11), l


def test_against_scipy(ora):
    """library cross-check: real harmonics assembled from scipy's complex Y_l^m (Condon-Shortley, orthonormal)."""
    sp = pytest.importorskip("scipy.special")
    n = _rand_units(64, 5)
    theta, phi = np.arccos(n[:, 2]), np.arctan2(n[:, 1], n[:, 0])
    f = getattr(sp, "sph_harm_y", None)
    for l, m in ora.sh_index(8):
        am = abs(m)
        Y = f(l, am, theta, phi) if f is not None else sp.sph_harm(am, l, phi, theta)
        Y = Y * math.sqrt(4 * math.pi) * (-1) ** am
        want = Y.real if m == 0 else math.sqrt(2) * (Y.real if m > 0 else Y.imag)
        assert np.allclose(ora.real_sh(l, m, n), want, atol=1e-12), (l, m)


def test_poles_finite(ora):
    n = np.array([[0.0, 0.0, 1.0], [0.0, 0.0, -1.0]])
    for l, m in ora.sh_index(8):
        v = ora.real_sh(l, m, n)
        assert np.all(np.isfinite(v))
        assert np.allclose(v, math.sqrt(2 * l + 1) if m == 0 else 0.0, atol=1e-12)


# ----------------------------------------------------------------------------- basis matrix (Eq. 3)
def _geom(ora, rot, tilt):
    return ora.Geometry((4, 4, 4), (4, 4), rot, tilt)


def _segs(D):
    c = np.arange(D)
    return c * math.pi / D, (c + 1) * math.pi / D


def test_B_isotropic_channel_is_one(ora):
    g = _geom(ora, [0.0, 0.7, 2.0], [0.0, 0.3, 0.78])
    B = ora.basis_matrix(g, 4, *_segs(8))
    assert B.shape == (3, 15, 8)
    assert np.allclose(B[:, 0, :], 1.0, atol=1e-14)


def test_B_identity_rotation_analytic(ora):
    """R_s = I: q(phi) = (cos phi, sin phi, 0) so Y_lm = N P_l^m(0) sqrt2 {cos|sin}(m phi) and the segment
    mean is the elementary integral of cos(m phi) / sin(m phi)."""
    g = _geom(ora, [0.0], [0.0])
    a, b = _segs(8)
    B = ora.basis_matrix(g, 8, a, b)
    for i, (l, m) in enumerate(ora.sh_index(8)):
        am = abs(m)
        amp = ora.real_sh(l, am, np.array([[1.0, 0.0, 0.0]]))[0]          # value at phi = 0 on the equator
        if m == 0:
            want = np.full(8, amp)
        elif m > 0:
            want = amp * (np.sin(m * b) - np.sin(m * a)) / (m * (b - a))
        else:
            # sin harmonics: amplitude = that of the cos harmonic of the same |m|
            want = amp * (np.cos(am * a) - np.cos(am * b)) / (am * (b - a))
        assert np.allclose(B[0, i], want, atol=1e-13), (l, m)


def test_B_quadrature_converged_and_variants(ora):
    g = _geom(ora, [0.4, 1.9], [0.2, 0.6])
    a, b = _segs(8)
    B32 = ora.basis_matrix(g, 8, a, b, n_quad=32)
    B64 = ora.basis_matrix(g, 8, a, b, n_quad=64)
    Bs = ora.basis_matrix(g, 8, a, b, n_quad=400, rule="simpson")
    Bc = ora.basis_matrix(g, 8, a, b, rule="central")
    assert np.abs(B32 - B64).max() < 1e-13
    assert np.abs(B32 - Bs).max() < 1e-9
    assert 1e-3 < np.abs(B32 - Bc).max() < 1.5            # the central-angle variant is only an approximation


def test_B_rotation_covariance(ora):
    """Rotating the sample by R about the beam-normal plane mixes harmonics of equal l orthogonally:
    sum_m B[s][lm][c]^2-type invariants are not available per segment, but the l-block of B reproduces a
    rotated zonal function exactly: sum_i B[s][i][c] Y_i(n) = mean over the segment of (2l+1) P_l(n . R^T q)."""
    g = _geom(ora, [0.9], [0.5])
    a, b = _segs(8)
    B = ora.basis_matrix(g, 8, a, b)
    n = _rand_units(1, 7)[0]
    xs, ws = leg.leggauss(48)
    Rt = g.rotation_matrix(0).T
    idx = ora.sh_index(8)
    for l in range(0, 9, 2):
        sel = [i for i, (ll, _) in enumerate(idx) if ll == l]
        lhs = sum(B[0, i, :] * ora.real_sh(idx[i][0], idx[i][1], n[None])[0] for i in sel)
        for c in range(8):
            phi = 0.5 * (a[c] + b[c]) + 0.5 * (b[c] - a[c]) * xs
            q = (np.cos(phi)[:, None] * g.vecs["q0"] + np.sin(phi)[:, None] * g.vecs["q90"]) @ Rt.T
            rhs = np.dot(ws / 2, (2 * l + 1) * leg.Legendre.basis(l)(q @ n))
            assert abs(lhs[c] - rhs) < 1e-11, (l, c)


def test_full_two_theta_scattering_vector(ora):
    """NEXT-4: first line of Eq. 1.  q stays a unit vector; 2theta = 0 is the small-angle line; with
    R_s = 1 and p = z the z-component is -sin(theta) for every phi, so the segment average of
    Y_20 = (sqrt5/2)(3 z^2 - 1) is (sqrt5/2)(3 sin^2 theta - 1) in every segment, and Y_00 stays 1."""
    import math
    g = ora.Geometry((4, 4, 4), (4, 4), [0.0, 0.9], [0.0, 0.4])
    phi = np.linspace(0, 2 * math.pi, 13)
    for tt in (0.0, 0.3, 1.1):
        q = ora.q_hat(g, phi, tt)
        assert np.allclose(np.linalg.norm(q, axis=-1), 1.0, atol=1e-15)
        assert np.allclose(q @ g.vecs["p"], -math.sin(tt / 2), atol=1e-15)
    c = np.arange(8)
    s0, s1 = c * 2 * math.pi / 8, (c + 1) * 2 * math.pi / 8            # WAXS: segments over the full circle
    B0 = ora.basis_matrix(g, 4, s0, s1)
    assert np.array_equal(B0, ora.basis_matrix(g, 4, s0, s1, two_theta=0.0))
    tt = 0.8
    B = ora.basis_matrix(g, 4, s0, s1, two_theta=tt)
    idx = ora.sh_index(4)
    i20 = idx.index((2, 0))
    assert np.allclose(B[0, i20], math.sqrt(5) / 2 * (3 * math.sin(tt / 2) ** 2 - 1), atol=1e-12)
    assert np.allclose(B[:, 0, :], 1.0, atol=1e-13)
    assert np.abs(B[1] - B0[1]).max() > 1e-2                          # and it does change the tilted projection
