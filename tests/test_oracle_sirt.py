"""Pins of the oracle's SIRT/MITRA step (reading S19 for the weights).
  * one axis-aligned projection of a scalar volume: closed form (row sum = Z, column sum = 1), so one step from
    zero smears each pixel's value evenly along its ray and reproduces the data exactly;
  * a consistent problem (data = A c*) has c* as a fixed point, with either back-projector;
  * with the matched adjoint, ||W^1/2 A C^1/2|| <= 1 (row/column sums of |A|), so the weighted loss never rises;
  * rays that miss the sample and voxels no ray sees get weight / preconditioner 0, not infinity."""
import numpy as np


def test_single_axis_aligned_projection_closed_form(ora):
    shape, det = (5, 4, 6), (4, 5)                       # J = Y, Kd = X: pixel (j,k) sums voxel column (x=k, y=j)
    g = ora.Geometry(shape, det, [0.0], [0.0])
    B = np.ones((1, 1, 1))
    W, C = ora.sirt_preconditioners(g, B, matched=True)
    assert np.allclose(W, 1.0 / shape[2]) and np.allclose(C, 1.0)
    data = np.random.default_rng(1).uniform(1, 2, (1,) + det + (1,))
    c1, L0 = ora.sirt_step(g, B, np.zeros(shape + (1,), np.float32), data, W, C, matched=True)
    want = np.transpose(data[0, :, :, 0], (1, 0))[:, :, None] / shape[2] * np.ones(shape)   # [x][y][z] = I[y][x] / Z
    assert np.abs(c1[..., 0] - want).max() < 1e-12
    assert abs(L0 - 0.5 * np.sum(data ** 2 / shape[2])) < 1e-10
    c2, L1 = ora.sirt_step(g, B, c1.astype(np.float32), data, W, C, matched=True)
    assert L1 < 1e-10 and np.abs(c2 - c1).max() < 1e-6   # already consistent


def test_fixed_point_and_monotone_loss(ora):
    r = np.random.default_rng(2)
    shape, det, P, K, D = (7, 6, 8), (11, 10), 5, 3, 4
    g = ora.Geometry(shape, det, r.uniform(0, 6.28, P), r.uniform(-0.6, 0.6, P))
    B = r.standard_normal((P, K, D))
    cstar = r.standard_normal(shape + (K,)).astype(np.float32)
    data = ora.forward(g, B, cstar)
    for matched in (True, False):
        W, C = ora.sirt_preconditioners(g, B, matched=matched)
        assert np.all(np.isfinite(W)) and np.all(np.isfinite(C)) and W.min() >= 0 and C.min() >= 0
        c1, L = ora.sirt_step(g, B, cstar, data, W, C, matched=matched)
        assert L < 1e-20 and np.abs(c1 - cstar).max() < 1e-9
    W, C = ora.sirt_preconditioners(g, B, matched=True)
    c, losses = np.zeros(shape + (K,)), []
    for _ in range(6):
        c, L = ora.sirt_step(g, B, c.astype(np.float32), data, W, C, matched=True)
        losses.append(L)
    assert all(b <= a * (1 + 1e-6) for a, b in zip(losses, losses[1:])) and losses[-1] < 0.7 * losses[0]


def test_unseen_rays_and_voxels_get_zero(ora):
    g = ora.Geometry((4, 4, 4), (12, 2), [0.0], [0.0], k_offsets=[2.0])   # taller than the sample, and shifted off part of it
    W, C = ora.sirt_preconditioners(g, np.ones((1, 1, 1)), matched=False)
    assert (W == 0).any() and (W > 0).any() and (C == 0).any() and (C > 0).any()
