"""Pins of the oracle's bilinear back-projector (NEXT-1: the adjoint as PAPER.md:314 words it, "bilinear interpolation
... of the projection for the adjoint"; reading S9).  None of these re-types the routine's loop:
  * hat-function closed form, dense, on tiny problems (no floor(), no tap loop);
  * bilinear interpolation reproduces affine functions: an affine projection a*j + b*k + c back-projects to
    sum_s w_s (a*j0 + b*k0 + c) with (j0,k0) from Eq. 4 written out here independently;
  * a constant projection on a detector that covers the sample back-projects to sum_s w_s (partition of unity);
  * for axis-aligned projections with integer offsets it coincides with the exact transpose of the Joseph forward;
  * for oblique projections it does NOT satisfy <Ax,y> = <x,A^T y> (that is why the exact transpose is primary);
  * channels are independent, pixels outside the detector count as zero."""
import math

import numpy as np
import pytest


def rodrigues(n, t):
    n = np.asarray(n, float)
    Kx = np.array([[0, -n[2], n[1]], [n[2], 0, -n[0]], [-n[1], n[0], 0]])
    return np.eye(3) * math.cos(t) + math.sin(t) * Kx + (1 - math.cos(t)) * np.outer(n, n)


def detector_positions(shape, det, rot, tilt, joff=0.0, koff=0.0, a=1.0, b=1.0):
    """(j0, k0, w) of every voxel, standard geometry (Table I), straight from Eq. 4."""
    R = rodrigues((1, 0, 0), tilt) @ rodrigues((0, 1, 0), rot)            # R_s = R_beta R_alpha
    d, js, ks = R.T @ np.array([0, 0, 1.0]), R.T @ np.array([0, 1.0, 0]), R.T @ np.array([1.0, 0, 0])
    gx = np.stack(np.meshgrid(*[np.arange(n) - (n - 1) / 2 for n in shape], indexing="ij"), -1)
    j0 = (det[0] - 1) / 2 + joff + (a / b) * gx @ js
    k0 = (det[1] - 1) / 2 + koff + (a / b) * gx @ ks
    return j0, k0, a / np.abs(d).max()


def hat(t):
    return np.maximum(0.0, 1.0 - np.abs(t))


@pytest.mark.parametrize("rot,tilt,joff,koff", [(0.3, 0.0, 0.0, 0.0), (1.1, 0.4, 0.37, -0.61), (2.5, -0.7, -1.2, 0.9)])
def test_hat_function_closed_form(ora, rot, tilt, joff, koff):
    shape, det = (5, 4, 6), (7, 6)
    g = ora.Geometry(shape, det, [rot], [tilt], j_offsets=[joff], k_offsets=[koff])
    r = np.random.default_rng(3)
    y = r.standard_normal((1,) + det + (2,))
    got = ora.john_backproject_bilinear(g, y)
    j0, k0, w = detector_positions(shape, det, rot, tilt, joff, koff)
    want = np.zeros(shape + (2,))
    for j in range(det[0]):
        for k in range(det[1]):
            want += (w * hat(j0 - j) * hat(k0 - k))[..., None] * y[0, j, k]
    assert np.abs(got - want).max() < 1e-12


def test_affine_projection_is_reproduced(ora):
    shape, det = (6, 7, 5), (40, 40)                     # detector covers the sample for every angle
    rot, tilt = np.array([0.2, 1.0, 2.2, 4.0]), np.array([0.0, 0.3, -0.5, 0.7])
    joff, koff = np.array([0.0, 0.4, -0.8, 1.3]), np.array([0.2, -0.6, 0.0, 0.9])
    g = ora.Geometry(shape, det, rot, tilt, j_offsets=joff, k_offsets=koff)
    jj, kk = np.meshgrid(np.arange(det[0]), np.arange(det[1]), indexing="ij")
    y = np.stack([(0.3 * jj - 0.7 * kk + 2.0)] * 4)[..., None] * (1.0 + np.arange(4))[:, None, None, None]
    got = ora.john_backproject_bilinear(g, y)[..., 0]
    want = np.zeros(shape)
    ones = np.zeros(shape)
    for s in range(4):
        j0, k0, w = detector_positions(shape, det, rot[s], tilt[s], joff[s], koff[s])
        want += w * (0.3 * j0 - 0.7 * k0 + 2.0) * (1.0 + s)
        ones += w
    assert np.abs(got - want).max() < 1e-11
    const = ora.john_backproject_bilinear(g, np.ones((4,) + det + (1,)))[..., 0]
    assert np.abs(const - ones).max() < 1e-12            # partition of unity: sum_s w_s


def test_equals_exact_transpose_when_axis_aligned(ora):
    shape, det = (6, 5, 7), (5, 6)
    r = np.random.default_rng(5)
    for rot, joff, koff in [(0.0, 0.0, 0.0), (math.pi / 2, 1.0, -1.0), (math.pi, 0.0, 2.0)]:
        g = ora.Geometry(shape, det, [rot], [0.0], j_offsets=[joff], k_offsets=[koff])
        y = r.standard_normal((1,) + det + (3,))
        exact = ora.john_adjoint(g, y, form="scatter")
        assert np.abs(ora.john_backproject_bilinear(g, y) - exact).max() < 1e-12


def test_is_not_the_transpose_for_oblique_rays(ora):
    shape, det = (12, 12, 12), (14, 14)
    g = ora.Geometry(shape, det, [0.6, 2.0], [0.3, 0.5])
    r = np.random.default_rng(6)
    x = r.standard_normal(shape + (1,)).astype(np.float32)
    y = r.standard_normal((2,) + det + (1,))
    lhs = float((ora.john_forward(g, x, 1) * y).sum())
    matched = float((x * ora.john_adjoint(g, y, form="scatter")).sum())
    unmatched = float((x * ora.john_backproject_bilinear(g, y)).sum())
    assert abs(lhs - matched) < 1e-10 * abs(lhs)
    assert abs(lhs - unmatched) > 1e-3 * abs(lhs)        # reading S9: the paper's adjoint is unmatched


def test_channels_independent_and_outside_is_zero(ora):
    shape, det = (5, 5, 5), (4, 4)
    g = ora.Geometry(shape, det, [0.4, 1.9], [0.2, -0.3], j_offsets=[30.0, 0.5], k_offsets=[0.0, -40.0])
    y = np.random.default_rng(8).standard_normal((2,) + det + (3,))
    assert np.all(ora.john_backproject_bilinear(g, y) == 0.0)            # every voxel projects off the detector
    g2 = ora.Geometry(shape, det, [0.4, 1.9], [0.2, -0.3])
    full = ora.john_backproject_bilinear(g2, y)
    for i in range(3):
        assert np.array_equal(full[..., i], ora.john_backproject_bilinear(g2, y[..., i:i + 1])[..., 0])


def test_sampled_voxels_equal_full(ora):
    shape, det = (6, 5, 7), (8, 9)
    g = ora.Geometry(shape, det, [0.4, 1.9, 3.0], [0.2, -0.3, 0.6])
    y = np.random.default_rng(9).standard_normal((3,) + det + (2,))
    full = ora.john_backproject_bilinear(g, y)
    xyz = np.array([[0, 0, 0], [5, 4, 6], [2, 3, 1], [3, 0, 6]])
    assert np.array_equal(ora.john_backproject_bilinear_voxels(g, y, xyz), full[xyz[:, 0], xyz[:, 1], xyz[:, 2]])
