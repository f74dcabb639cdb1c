"""Pins of the oracle's derived quantities (NEXT-4; Eq. 10-12)."""
import math

import numpy as np


def coeffs_of_squared_cosine(ora, n, ell_max):
    """(q.n)^2 = 1/3 + (2/3) P_2(q.n) = 1/3 + (2/15) sum_m Y_2m(q) Y_2m(n)  (addition theorem, 4pi-normalised Y)."""
    idx = ora.sh_index(ell_max)
    c = np.zeros(len(idx))
    c[0] = 1.0 / 3.0
    for i, (l, m) in enumerate(idx):
        if l == 2:
            c[i] = (2.0 / 15.0) * ora.real_sh(2, m, np.asarray(n, float))
    return c


def test_isotropic_and_squared_cosine_closed_forms(ora):
    iso = np.zeros(15); iso[0] = 2.5
    d = ora.derived_quantities(iso, 4)
    assert abs(d["mean"] - 2.5) < 1e-13 and np.abs(d["M"] - 2.5 / 3 * np.eye(3)).max() < 1e-13 and abs(d["fa"]) < 1e-6
    n = np.array([0.36, -0.48, 0.8])
    d = ora.derived_quantities(coeffs_of_squared_cosine(ora, n, 4), 4)
    assert abs(d["mean"] - 1.0 / 3.0) < 1e-13                         # <(q.n)^2> = 1/3
    assert np.abs(d["M"] - (np.eye(3) + 2.0 * np.outer(n, n)) / 15.0).max() < 1e-13    # <q_i q_j (q.n)^2>
    assert np.allclose(d["eig"], [3 / 15, 1 / 15, 1 / 15], atol=1e-13)
    assert abs(abs(d["vec"][0] @ n) - 1.0) < 1e-12                     # main orientation = n (up to sign)
    assert abs(d["fa"] - math.sqrt(8.0 / 22.0)) < 1e-12


def test_high_orders_do_not_enter_and_batching(ora):
    r = np.random.default_rng(3)
    c = r.standard_normal((4, 5, 45))
    d8 = ora.derived_quantities(c, 8)
    c2 = c[..., :6]
    d2 = ora.derived_quantities(c2, 2)
    assert np.abs(d8["M"] - d2["M"]).max() < 1e-12 and np.abs(d8["mean"] - c[..., 0]).max() < 1e-12
    assert d8["eig"].shape == (4, 5, 3) and np.all(np.diff(d8["eig"], axis=-1) <= 1e-15)
    for i in range(3):                                                # M v = lambda v
        v = d8["vec"][..., i, :]
        assert np.abs(np.einsum("...ij,...j->...i", d8["M"], v) - d8["eig"][..., i:i + 1] * v).max() < 1e-12
    assert np.all((d8["fa"] >= 0) & (d8["fa"] <= math.sqrt(1.5) + 1e-12))   # <= 1 only for a non-negative RSM
    assert ora.derived_quantities(np.zeros(6), 2)["fa"] == 0.0
