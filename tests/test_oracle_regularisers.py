"""Pins of the oracle's regulariser gradients and momentum step (NEXT-3, readings S21, S22)."""
import math

import numpy as np


def test_laplacian_dirichlet_eigenfunctions(ora):
    """sin(pi a (x+1)/(X+1)) sin(pi b (y+1)/(Y+1)) sin(pi c (z+1)/(Z+1)) vanishes on the padding planes and is an exact
    eigenvector of the zero-padded 7-point Laplacian with eigenvalue sum(2 cos(pi k/(N+1)) - 2)."""
    X, Y, Z = 7, 5, 6
    for a, b, c in [(1, 1, 1), (2, 3, 1), (4, 2, 5)]:
        fx = np.sin(math.pi * a * (np.arange(X) + 1) / (X + 1))
        fy = np.sin(math.pi * b * (np.arange(Y) + 1) / (Y + 1))
        fz = np.sin(math.pi * c * (np.arange(Z) + 1) / (Z + 1))
        f = (fx[:, None, None] * fy[None, :, None] * fz[None, None, :])[..., None]
        lam = sum(2 * math.cos(math.pi * k / (n + 1)) - 2 for k, n in ((a, X), (b, Y), (c, Z)))
        assert np.abs(ora.laplacian(f) - lam * f).max() < 1e-12


def test_laplacian_polynomials_and_symmetry(ora):
    X, Y, Z = 6, 7, 5
    x, y, z = np.meshgrid(np.arange(X), np.arange(Y), np.arange(Z), indexing="ij")
    f = np.stack([x * x + 2.0 * y * y - z * z, 3.0 * x - y + 0.5 * z, np.ones_like(x, dtype=float)], axis=-1).astype(float)
    l = ora.laplacian(f)
    inner = (slice(1, -1),) * 3
    assert np.allclose(l[inner + (0,)], 2 + 4 - 2) and np.allclose(l[inner + (1,)], 0) and np.allclose(l[inner + (2,)], 0)
    assert l[0, 3, 2, 2] == -1.0 and l[0, 0, 0, 2] == -3.0            # faces / corners see the zero padding
    r = np.random.default_rng(0)
    a_, b_ = r.standard_normal((X, Y, Z, 2)), r.standard_normal((X, Y, Z, 2))
    assert abs(np.sum(ora.laplacian(a_) * b_) - np.sum(a_ * ora.laplacian(b_))) < 1e-10


def test_regulariser_gradients_by_finite_differences(ora):
    r = np.random.default_rng(1)
    c = r.standard_normal((5, 4, 6, 3))
    d = r.standard_normal(c.shape)
    for reg in (ora.laplacian_regulariser, ora.l2_regulariser):
        R0, g = reg(c)
        h = 1e-5
        fd = (reg(c + h * d)[0] - reg(c - h * d)[0]) / (2 * h)
        assert abs(fd - np.sum(g * d)) < 1e-6 * max(1.0, abs(fd))
        assert R0 >= 0


def test_nesterov_reduces_to_plain_descent_and_accelerates(ora):
    c, v = np.array([1.0, -2.0]), np.zeros(2)
    c1, v1 = ora.nesterov_step(c, v, np.array([0.5, 0.5]), eta=0.1, momentum=0.0)
    assert np.allclose(c1, c - 0.05) and np.allclose(v1, -0.05)
    # quadratic bowl f = 1/2 x' A x, ill-conditioned: momentum 0.9 beats plain descent after 60 steps
    A = np.diag([1.0, 100.0])
    def run(m):
        x, vel = np.array([1.0, 1.0]), np.zeros(2)
        for _ in range(60):
            x, vel = ora.nesterov_step(x, vel, A @ (x + m * vel), eta=0.009, momentum=m)
        return 0.5 * x @ A @ x
    assert run(0.9) < 1e-2 * run(0.0)


def test_l1_huber_norm_total_variation(ora):
    """PAPER.md:336-338, reading S24.  Closed forms: a linear ramp c = a x + b y has |grad c| = sqrt(a^2+b^2) at every
    voxel that has both forward neighbours; HuberNorm tends to L1 - delta/2 per element for delta -> 0 and to
    L2/(delta) for large delta; gradients by finite differences (the Huberised terms are C^1)."""
    r = np.random.default_rng(4)
    c = r.standard_normal((6, 5, 7, 2))
    R1, g1 = ora.l1_regulariser(c)
    assert abs(R1 - np.abs(c).sum()) < 1e-12 and np.array_equal(g1, np.sign(c))
    Rh, gh = ora.huber_norm_regulariser(c, 1e-9)
    assert abs(Rh - (R1 - 0.5e-9 * c.size)) < 1e-9 and np.array_equal(gh, np.sign(c))
    Rh, gh = ora.huber_norm_regulariser(c, 1e3)
    assert abs(Rh - 0.5 * np.sum(c * c) / 1e3) < 1e-12 and np.allclose(gh, c / 1e3)
    X, Y, Z = 6, 5, 4
    x, y, z = np.meshgrid(np.arange(X), np.arange(Y), np.arange(Z), indexing="ij")
    ramp = (3.0 * x + 4.0 * y)[..., None].astype(float)
    Rt, gt = ora.total_variation_regulariser(ramp, 0.1)
    full = (X - 1) * (Y - 1) * Z * (5.0 - 0.05)                       # both differences present: |grad| = 5
    edge_x = (Y - 1) * Z * (4.0 - 0.05)                               # last x plane: only d_y = 4
    edge_y = (X - 1) * Z * (3.0 - 0.05)                               # last y row: only d_x = 3
    assert abs(Rt - (full + edge_x + edge_y)) < 1e-10                 # the corner column has no difference at all
    assert abs(gt[2, 2, 1, 0]) < 1e-12                                # interior of a linear ramp: zero TV gradient
    for reg in (lambda v: ora.huber_norm_regulariser(v, 0.3), lambda v: ora.total_variation_regulariser(v, 0.3)):
        d = r.standard_normal(c.shape)
        h = 1e-6
        fd = (reg(c + h * d)[0] - reg(c - h * d)[0]) / (2 * h)
        assert abs(fd - np.sum(reg(c)[1] * d)) < 1e-5 * max(1.0, abs(fd))
