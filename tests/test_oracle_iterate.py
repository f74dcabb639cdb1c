"""Pins for the oracle's regularised iteration with the relative-change stop rule (reading S25) and
for the sparse approximation of the basis matrix (reading S26) — CPU only."""
import math

import numpy as np


def _axis_problem(ora, X=3, Y=4, Z=5, seed=0):
    """One projection along z (alpha = beta = 0), K = D = 1, B = 1: every ray (j, k) sums the Z voxels of the column
    (x = k, y = j) with weight 1 and the columns are disjoint, so A A^T = Z I and the iteration decouples per column."""
    g = ora.Geometry((X, Y, Z), (Y, X), [0.0], [0.0])
    B = np.ones((1, 1, 1), dtype=np.float32)
    d = np.random.default_rng(seed).uniform(1.0, 2.0, (1, Y, X, 1)).astype(np.float32)
    return g, B, d


def test_iterate_matches_closed_form_on_decoupled_columns(ora):
    """Plain gradient descent (m = 0) with an L2 term from c = 0: a column's common value gamma obeys
    gamma_{k+1} = gamma_k (1 - eta (Z + mu)) + eta d, so L_k = sum_rays 1/2 (Z gamma_k - d)^2 + mu/2 Z gamma_k^2 and the
    stop index follows from that sequence alone."""
    g, B, d = _axis_problem(ora)
    Z, mu, eta, tol = g.shape[2], 0.7, 0.11, 1e-6
    d64 = d.astype(np.float64)[0, :, :, 0]
    gam = np.zeros_like(d64)
    want = []
    for k in range(200):
        want.append(float(np.sum(0.5 * (Z * gam - d64) ** 2 + 0.5 * float(np.float32(mu)) * Z * gam ** 2)))
        gam = gam * (1.0 - float(np.float32(eta)) * (Z + float(np.float32(mu)))) + float(np.float32(eta)) * d64
        if k >= 1 and abs(want[-1] - want[-2]) <= tol * abs(want[-1]):
            break
    c, v, losses = ora.iterate(g, B, d, None, np.zeros(g.shape + (1,), np.float32), eta, 0.0, 0.0, mu, 200, tol)
    assert len(losses) == len(want) and 5 < len(want) < 200          # same stop index, and the rule did fire
    assert np.allclose(losses, want, rtol=2e-6)                        # fp32 state of the iterate only
    assert np.abs(c[..., 0] - gam.T[:, :, None]).max() < 1e-6          # volume is [x][y][z]; ray (j, k) = (y, x)
    # fixed point of the recursion: gamma* = d / (Z + mu)
    assert np.abs(c[..., 0] - (d64 / (Z + float(np.float32(mu)))).T[:, :, None]).max() < 1e-3


def test_iterate_loss_monotone_and_check_every(ora):
    """consistent data, no regulariser, step below 1/||A||^2: the loss never increases; with check_every = 4 the stop
    can only fall on a multiple of 4."""
    r = np.random.default_rng(3)
    g = ora.Geometry((6, 5, 7), (8, 8), [0.0, 0.8, 2.1], [0.0, 0.3, -0.4], j_offsets=[0.2, -0.3, 0.1], k_offsets=[0.0, 0.4, -0.2])
    c = np.arange(4) + 0.0
    B = ora.basis_matrix(g, 2, c * math.pi / 4, (c + 1) * math.pi / 4).astype(np.float32)
    K = B.shape[1]
    truth = r.uniform(0, 1, g.shape + (K,)).astype(np.float32)
    data = ora.forward(g, B, truth).astype(np.float32)
    absB = np.abs(B)
    lip = ora.forward(g, absB, np.ones(g.shape + (K,), np.float32)).max() * ora.adjoint(g, absB, np.ones((g.P,) + g.det + (4,)), form="scatter").max()
    # (the relative change per iteration falls from 27 % to 10 % over the first 15 iterations with this safe step)
    _, _, losses = ora.iterate(g, B, data, None, np.zeros_like(truth), 1.0 / lip, 0.0, 0.0, 0.0, 40, 0.12, check_every=4)
    assert all(b <= a * (1 + 1e-12) for a, b in zip(losses, losses[1:]))
    assert len(losses) % 4 == 0 and len(losses) < 40
    _, _, l1 = ora.iterate(g, B, data, None, np.zeros_like(truth), 1.0 / lip, 0.0, 0.0, 0.0, 40, 0.12, check_every=1)
    assert len(losses) - 4 < len(l1) <= len(losses) and np.allclose(l1, losses[:len(l1)], rtol=1e-12)
    assert abs(l1[-1] - l1[-2]) <= 0.12 * l1[-1] < abs(l1[-2] - l1[-3])      # first iteration at which the rule holds
    # momentum and a Laplacian term change the path but still descend overall
    _, _, l2 = ora.iterate(g, B, data, None, np.zeros_like(truth), 1.0 / (lip + 144 * 0.05 * lip), 0.5, 0.05 * lip, 0.0, 25, 0.0)
    assert len(l2) == 25 and l2[-1] < 0.5 * l2[0]


def test_sparsify_basis(ora):
    r = np.random.default_rng(5)
    B = r.standard_normal((3, 9, 4)).astype(np.float32)
    assert np.array_equal(ora.sparsify_basis(B, 9), B) and np.array_equal(ora.sparsify_basis(B, 50), B)
    for n in (1, 2, 5):
        S = ora.sparsify_basis(B, n)
        assert np.all((S != 0).sum(axis=1) == n)                       # n survivors in every (s, c) column
        assert np.all((S == 0) | (S == B))                              # survivors keep their value
        for s in range(3):
            for c in range(4):                                          # ... and are the largest ones
                keep = np.abs(B[s, :, c])[S[s, :, c] != 0].min()
                drop = np.abs(B[s, :, c])[S[s, :, c] == 0].max()
                assert keep >= drop
        assert np.array_equal(ora.sparsify_basis(S, n), S)             # idempotent
    # ties: the lowest index wins
    T = np.ones((1, 4, 1), dtype=np.float32)
    assert np.array_equal(ora.sparsify_basis(T, 2)[0, :, 0], [1, 1, 0, 0])
    # an NN basis has at most n_quad non-zeros per column (one indicator per quadrature point): keeping that many is exact
    g = ora.Geometry((4, 4, 4), (4, 4), [0.3, 1.1], [0.2, -0.5])
    from paper_2504_16446_b200 import synth
    c = np.arange(8) + 0.0
    Bnn = ora.basis_matrix_grid(g, synth.grid_directions(40), "nn", c * math.pi / 8, (c + 1) * math.pi / 8, n_quad=4)
    assert ((Bnn != 0).sum(axis=1) <= 4).all() and np.array_equal(ora.sparsify_basis(Bnn, 4), Bnn)
    # forward model with the sparse matrix = forward model of the dense one restricted to the survivors (linearity)
    vol = r.uniform(0, 1, (4, 4, 4, 40)).astype(np.float32)
    S1 = ora.sparsify_basis(Bnn, 1)
    assert np.abs(ora.forward(g, S1, vol) + ora.forward(g, Bnn - S1, vol) - ora.forward(g, Bnn, vol)).max() < 1e-12
