"""Pins for the oracle's forward model (Eq. 6-8), loss and gradient (Eq. 9, 13) — CPU only.
Kronecker structure on tiny volumes, separability, scalar-CT reduction of the l=0 channel, finite
differences of the loss, zero-residual and zero-weight special cases, per-voxel gradient sampler."""
import math

import numpy as np


def _rng(seed):
    return np.random.default_rng(seed)


def _segs(D):
    c = np.arange(D)
    return c * math.pi / D, (c + 1) * math.pi / D


def _setup(ora, shape=(5, 6, 4), det=(7, 6), ell=2, D=4, seed=0):
    r = _rng(seed)
    rot = np.array([0.0, 0.9, math.pi / 4, 2.6])
    tilt = np.array([0.0, 0.3, 0.0, math.pi / 4])
    g = ora.Geometry(shape, det, rot, tilt, j_offsets=r.uniform(-1, 1, 4), k_offsets=r.uniform(-1, 1, 4))
    B = ora.basis_matrix(g, ell, *_segs(D))
    K = B.shape[1]
    vol = r.standard_normal(shape + (K,)).astype(np.float32)
    return g, B, vol, r


def test_kronecker_structure(ora):
    """Eq. 8: A_s = P_s (x) B_s.  Dense P_s from the oracle's closed-form builder (itself pinned against
    numpy in test_oracle_john), B_s^T applied per pixel."""
    g, B, vol, _ = _setup(ora)
    I = ora.forward(g, B, vol)
    K = B.shape[1]
    for s in range(g.P):
        Ps = ora.dense_john_matrix(g, s)                                   # [J*Kd][N]
        As = np.kron(Ps, B[s].T)                                           # [(J*Kd)*D][N*K]
        want = As @ vol.astype(np.float64).reshape(-1)
        assert np.abs(I[s].reshape(-1) - want).max() < 1e-11


def test_separability(ora):
    """c_i(x) = rho(x) gamma_i  =>  I[s,j,k,c] = Proj[rho][s,j,k] * sum_i B[s][i][c] gamma_i."""
    g, B, _, r = _setup(ora, ell=4, D=8)
    K = B.shape[1]
    rho = r.uniform(0, 1, g.shape).astype(np.float32)
    gamma = r.standard_normal(K).astype(np.float32)
    vol = (rho[..., None] * gamma).astype(np.float32)
    I = ora.forward(g, B, vol)
    # the products rho*gamma were rounded to fp32 per voxel; rebuild the expectation from those roundings
    pr = ora.john_forward(g, vol, K)                                        # [P][J][Kd][K]
    scal = ora.john_forward(g, np.ascontiguousarray(rho[..., None]), 1)[..., 0]
    want = scal[..., None] * np.einsum("sic,i->sc", B, gamma.astype(np.float64))[:, None, None, :]
    assert np.abs(I - want).max() < 2e-6 * np.abs(want).max()               # fp32 rounding of rho*gamma only
    assert np.abs(I - ora.basis_forward(B, pr)).max() < 1e-13


def test_l0_channel_is_scalar_ct(ora):
    """Only the isotropic coefficient non-zero: every segment sees the scalar John transform (B[s][0][c] = 1)."""
    g, B, vol, _ = _setup(ora, ell=4, D=8)
    vol[..., 1:] = 0
    I = ora.forward(g, B, vol)
    scal = ora.john_forward(g, np.ascontiguousarray(vol[..., :1]), 1)[..., 0]
    assert np.abs(I - scal[..., None]).max() < 1e-12


def test_forward_adjoint_dot_product(ora):
    g, B, vol, r = _setup(ora, ell=4, D=8)
    y = r.standard_normal((g.P,) + g.det + (8,))
    lhs = float(np.sum(ora.forward(g, B, vol) * y))
    rhs = float(np.sum(vol.astype(np.float64) * ora.adjoint(g, B, y)))
    assert abs(lhs - rhs) < 1e-11 * abs(lhs)
    assert np.abs(ora.adjoint(g, B, y, form="scatter") - ora.adjoint(g, B, y, form="gather")).max() < 1e-11


def test_loss_value_definition(ora):
    g, B, vol, r = _setup(ora)
    data = r.uniform(0, 2, (g.P,) + g.det + (4,)).astype(np.float32)
    w = r.uniform(0.5, 1.5, data.shape).astype(np.float32)
    L, grad, wr = ora.loss_gradient(g, B, vol, data, w)
    I = ora.forward(g, B, vol)
    want = 0.0
    for idx in np.ndindex(*data.shape):                                    # plain loop: 1/2 sum w (Ac - I)^2
        want += 0.5 * float(w[idx]) * (I[idx] - float(data[idx])) ** 2
    assert abs(L - want) < 1e-10 * want
    assert np.abs(wr - w.astype(np.float64) * (I - data)).max() < 1e-13


def test_gradient_finite_difference(ora):
    """central differences of L along random directions (fp32 inputs exactly representable: h = 2^-7)."""
    g, B, vol, r = _setup(ora)
    vol = np.round(vol * 64) / 64
    data = r.uniform(0, 2, (g.P,) + g.det + (4,)).astype(np.float32)
    w = r.uniform(0.5, 1.5, data.shape).astype(np.float32)
    L0, grad, _ = ora.loss_gradient(g, B, vol.astype(np.float32), data, w)
    h = 2.0 ** -7
    for t in range(3):
        dirn = np.round(r.standard_normal(vol.shape) * 8) / 8
        Lp = ora.loss_gradient(g, B, (vol + h * dirn).astype(np.float32), data, w)[0]
        Lm = ora.loss_gradient(g, B, (vol - h * dirn).astype(np.float32), data, w)[0]
        fd = (Lp - Lm) / (2 * h)                                           # exact for a quadratic
        an = float(np.sum(grad * dirn))
        assert abs(fd - an) < 1e-9 * max(1.0, abs(an))


def test_zero_residual_and_zero_weights(ora):
    g, B, vol, r = _setup(ora)
    I = ora.forward(g, B, vol)
    # data = model exactly is not representable in fp32; use weights = 0 instead for the exact-zero case
    data = I.astype(np.float32)
    L, grad, _ = ora.loss_gradient(g, B, vol, data, None)
    assert L < 1e-10 and np.abs(grad).max() < 1e-4
    w = np.ones(data.shape, np.float32)
    w[1, 2:5] = 0
    d2 = data.copy()
    d2[1, 2:5] += 1000.0                                                   # garbage under the mask
    L2, grad2, _ = ora.loss_gradient(g, B, vol, d2, w)
    L3, grad3, _ = ora.loss_gradient(g, B, vol, data, w)
    assert L2 == L3 and np.array_equal(grad2, grad3)
    Lz, gz, _ = ora.loss_gradient(g, B, vol, d2, np.zeros_like(w))
    assert Lz == 0.0 and np.abs(gz).max() == 0.0


def test_gradient_voxels_matches_full(ora):
    g, B, vol, r = _setup(ora)
    data = r.uniform(0, 2, (g.P,) + g.det + (4,)).astype(np.float32)
    w = r.uniform(0.5, 1.5, data.shape).astype(np.float32)
    _, grad, _ = ora.loss_gradient(g, B, vol, data, w)
    xyz = np.array([[0, 0, 0], [2, 3, 1], [4, 5, 3]], dtype=np.int32)
    got = ora.gradient_voxels(g, B, vol, data, w, xyz)
    assert np.abs(got - grad[xyz[:, 0], xyz[:, 1], xyz[:, 2]]).max() < 1e-11


def test_forward_rays_matches_full(ora):
    g, B, vol, _ = _setup(ora)
    I = ora.forward(g, B, vol)
    sjk = np.array([[0, 0, 0], [3, 6, 5], [2, 3, 3]], dtype=np.int32)
    assert np.abs(ora.forward_rays(g, B, vol, sjk) - I[sjk[:, 0], sjk[:, 1], sjk[:, 2]]).max() < 1e-13


def test_huber_loss_limits_and_gradient(ora):
    """NEXT-4: Huber = squared loss for delta above every |r|; linear growth delta(|r| - delta/2) far
    out; gradient checked by finite differences (rho is C^1)."""
    r = np.random.default_rng(12)
    shape, det, P, K, D = (6, 5, 7), (8, 7), 4, 3, 4
    g = ora.Geometry(shape, det, r.uniform(0, 6.28, P), r.uniform(-0.5, 0.5, P))
    B = r.standard_normal((P, K, D))
    c = r.standard_normal(shape + (K,)).astype(np.float32)
    data = ora.forward(g, B, c) + r.standard_normal((P,) + det + (D,)) * 3.0
    w = r.uniform(0.5, 1.5, (P,) + det + (D,))
    L2, g2, wr2 = ora.loss_gradient(g, B, c, data, w)
    Lh, gh, wpsi = ora.huber_loss_gradient(g, B, c, data, 1e9, w)
    assert abs(Lh - L2) < 1e-9 * L2 and np.abs(gh - g2).max() < 1e-9 and np.abs(wpsi - wr2).max() < 1e-12
    delta = 1.0
    Lh, gh, wpsi = ora.huber_loss_gradient(g, B, c, data, delta, w)
    res = ora.forward(g, B, c) - data
    big = np.abs(res) > delta
    assert big.any() and (~big).any() and np.abs(wpsi).max() <= 1.5 * delta + 1e-12
    assert abs(Lh - (np.sum(w[~big] * 0.5 * res[~big] ** 2) + np.sum(w[big] * delta * (np.abs(res[big]) - 0.5 * delta)))) < 1e-9 * Lh
    d = r.standard_normal(c.shape).astype(np.float32)
    h = 1e-3
    fd = (ora.huber_loss_gradient(g, B, c + h * d, data, delta, w)[0] - ora.huber_loss_gradient(g, B, c - h * d, data, delta, w)[0]) / (2 * h)
    assert abs(fd - np.sum(gh * d)) < 2e-4 * abs(fd)
