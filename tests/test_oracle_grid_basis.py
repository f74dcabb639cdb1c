"""Pins of the oracle's grid-of-orientations basis matrices (NEXT-2, reading S20)."""
import math

import numpy as np
import pytest


def segs(D):
    c = np.arange(D)
    return c * math.pi / D, (c + 1) * math.pi / D


def fib_dirs(n):
    i = np.arange(n) + 0.5
    z = i / n                                             # upper half sphere: lines, not vectors
    ph = i * math.pi * (3.0 - math.sqrt(5.0))
    rr = np.sqrt(1 - z * z)
    return np.stack([rr * np.cos(ph), rr * np.sin(ph), z], axis=1)


def test_nn_partition_of_unity_and_single_direction(ora):
    g = ora.Geometry((4, 4, 4), (4, 4), [0.3, 1.7, 4.0], [0.0, 0.4, -0.6])
    B = ora.basis_matrix_grid(g, fib_dirs(18), "nn", *segs(8), n_quad=12)
    assert np.allclose(B.sum(axis=1), 1.0, atol=1e-15) and B.min() >= 0
    assert set(np.unique(np.round(B * 12))) <= set(range(13))          # multiples of 1/n_quad
    one = ora.basis_matrix_grid(g, np.array([[0.0, 0.6, 0.8]]), "nn", *segs(8))
    assert np.all(one == 1.0)


def test_nn_axis_grid_closed_form(ora):
    """alpha = beta = 0: q(phi) = (cos phi, sin phi, 0).  Grid {x, y, z}: x is nearest for phi in [0, pi/4) and
    (3pi/4, pi), y for (pi/4, 3pi/4), z never.  With 4 segments every segment has one owner."""
    g = ora.Geometry((4, 4, 4), (4, 4), [0.0], [0.0])
    B = ora.basis_matrix_grid(g, np.eye(3), "nn", *segs(4), n_quad=8)
    assert np.array_equal(B[0], np.array([[1, 0, 0, 1], [0, 1, 1, 0], [0, 0, 0, 0]], dtype=float))


def test_gk_closed_forms(ora):
    g = ora.Geometry((4, 4, 4), (4, 4), [0.0], [0.0])
    s0, s1 = np.array([-0.1]), np.array([0.1])                         # one segment centred on phi = 0: q = x
    sig = 0.4
    dirs = np.array([[1.0, 0, 0], [0, 1.0, 0], [0, 0, 1.0], [-1.0, 0, 0], [math.cos(0.3), math.sin(0.3), 0]])
    B = ora.basis_matrix_grid(g, dirs, "gk", s0, s1, sigma=sig, n_quad=1)[0, :, 0]
    want = np.exp(-np.array([0.0, math.pi / 2, math.pi / 2, 0.0, 0.3]) ** 2 / (2 * sig * sig))
    assert np.abs(B - want).max() < 1e-12                              # includes the antipodal direction -x
    wide = ora.basis_matrix_grid(g, dirs, "gk", *segs(8), sigma=1e6)
    assert np.abs(wide - 1.0).max() < 1e-10
    # quadrature converges to the integral of exp(-phi^2/2 sigma^2) over the segment (direction x, q in the plane)
    fine = ora.basis_matrix_grid(g, dirs[:1], "gk", s0, s1, sigma=sig, n_quad=2000)[0, 0, 0]
    exact = sig * math.sqrt(2 * math.pi) * math.erf(0.1 / (sig * math.sqrt(2))) / 0.2
    assert abs(fine - exact) < 1e-8


def test_gk_rotates_with_the_sample(ora):
    """tilt 0, rotation alpha about y: R_s^T q(phi) for phi = 0 is x rotated by -alpha about y; a grid direction
    placed there has theta = 0 for that projection."""
    al = 0.7
    g = ora.Geometry((4, 4, 4), (4, 4), [al], [0.0])
    d = np.array([[math.cos(al), 0.0, math.sin(al)], [math.cos(al), 0.0, -math.sin(al)]])
    B = ora.basis_matrix_grid(g, d, "gk", np.array([0.0]), np.array([0.0]), sigma=0.2, n_quad=1)[0, :, 0]
    assert max(B) == pytest.approx(1.0, abs=1e-12) and min(B) == pytest.approx(math.exp(-(2 * al) ** 2 / 0.08), rel=1e-9)
