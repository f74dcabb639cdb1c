"""CPU-only checks of the C-ABI library: it loads, exports every symbol include/mm.h declares, validates its
arguments, and its HOST parts (geometry table, SH basis-matrix helper) agree with the independently written
oracle.  No compute call is made (there is no GPU here); device calls must fail loudly, never fall back."""
import ctypes
import math
import os
import re

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)


@pytest.fixture(scope="module")
def mm():
    from paper_2504_16446_b200 import build, mm as binding
    build.build()
    binding.load()
    return binding


def _segs(D):
    c = np.arange(D)
    return c * math.pi / D, (c + 1) * math.pi / D


def test_exports_every_declared_symbol(mm):
    hdr = open(os.path.join(ROOT, "include", "mm.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(mm_[a-z0-9_]+)\s*\(", hdr))
    assert {"mm_geometry_create", "mm_john_forward", "mm_john_adjoint", "mm_basis_forward", "mm_basis_adjoint",
            "mm_loss_gradient"} <= declared                      # BASELINE.json north_star's list
    L = ctypes.CDLL(mm.LIB_PATH)
    for name in declared:
        assert hasattr(L, name), name
    assert declared == set(mm.SYMBOLS)


def test_table1_golden(mm):
    rows = {}
    with open(os.path.join(HERE, "golden", "table1_standard_geometry.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            t = line.split()
            rows[t[0]] = np.array([float(v) for v in t[1:4]])
    g = mm.Geometry((4, 5, 6), (5, 4), [0.0], [0.0])
    d, js, ks, m, w = g.get(0)
    assert np.allclose(d, rows["p"], atol=1e-15) and np.allclose(js, rows["j"], atol=1e-15)
    assert np.allclose(ks, rows["k"], atol=1e-15)
    assert m == 2 and w == 1.0


def test_geometry_matches_oracle(mm, ora):
    r = np.random.default_rng(5)
    P = 40
    rot = r.uniform(0, 2 * math.pi, P)
    tilt = r.uniform(-math.pi / 4, math.pi / 4, P)
    rot[:4] = [math.pi / 4, 0.0, 3 * math.pi / 4, math.pi / 2]             # ties of reading S8
    tilt[:4] = [0.0, math.pi / 4, 0.3, 0.0]
    go = ora.Geometry((9, 7, 8), (6, 10), rot, tilt)
    gm = mm.Geometry((9, 7, 8), (6, 10), rot, tilt)
    for s in range(P):
        a, b = go.get(s), gm.get(s)
        for x, y in zip(a[:3], b[:3]):
            assert np.abs(x - y).max() < 1e-14
        assert a[3] == b[3] and abs(a[4] - b[4]) < 1e-13
    # non-standard (rotated) lab vectors
    vecs = {"p": (1.0, 0.0, 0.0), "j": (0.0, 0.0, 1.0), "k": (0.0, 1.0, 0.0), "inner_axis": (0.0, 0.0, 1.0),
            "outer_axis": (0.0, 1.0, 0.0)}
    go = ora.Geometry((5, 5, 5), (5, 5), rot[:8], tilt[:8], vecs=vecs)
    gm = mm.Geometry((5, 5, 5), (5, 5), rot[:8], tilt[:8], vecs=vecs)
    for s in range(8):
        a, b = go.get(s), gm.get(s)
        for x, y in zip(a[:3], b[:3]):
            assert np.abs(x - y).max() < 1e-14
        assert a[3] == b[3]


@pytest.mark.parametrize("ell,D", [(0, 4), (2, 8), (4, 8), (8, 8), (6, 16)])
def test_sh_matrix_matches_oracle(mm, ora, ell, D):
    r = np.random.default_rng(ell)
    P = 12
    rot, tilt = r.uniform(0, 2 * math.pi, P), r.uniform(0, math.pi / 4, P)
    rot[0] = tilt[0] = 0.0
    go = ora.Geometry((4, 4, 4), (4, 4), rot, tilt)
    gm = mm.Geometry((4, 4, 4), (4, 4), rot, tilt)
    s0, s1 = _segs(D)
    Bo = ora.basis_matrix(go, ell, s0, s1, n_quad=48)
    Bm = mm.mm_basis_sh_matrix(gm, ell, s0, s1)
    assert Bm.shape == Bo.shape and Bm.dtype == np.float32
    assert np.abs(Bm - Bo).max() < 4e-7 * max(1.0, np.abs(Bo).max())          # fp32 rounding of the output only
    assert np.allclose(Bm[:, 0, :], 1.0)                                       # Y_00 = 1 (reading S14)
    # uneven, partly reversed and zero-width segments
    s0 = np.array([0.1, 2.0, 0.7, 1.3])
    s1 = np.array([0.9, 1.1, 0.7 + 1e-15, 4.0])
    Bo = ora.basis_matrix(go, ell, s0, s1, n_quad=64)
    Bm = mm.mm_basis_sh_matrix(gm, ell, s0, s1)
    assert np.abs(Bm - Bo).max() < 4e-7 * max(1.0, np.abs(Bo).max())


def test_argument_validation(mm):
    with pytest.raises(mm.MMError, match="MM_ERR_SHAPE"):
        mm.Geometry((0, 4, 4), (4, 4), [0.0], [0.0])
    with pytest.raises(mm.MMError, match="MM_ERR_SHAPE"):
        mm.Geometry((4, 4, 4), (4, 0), [0.0], [0.0])
    with pytest.raises(mm.MMError, match="MM_ERR_VALUE"):
        mm.Geometry((4, 4, 4), (4, 4), [float("nan")], [0.0])
    with pytest.raises(mm.MMError, match="MM_ERR_VALUE"):
        mm.Geometry((4, 4, 4), (4, 4), [0.0], [0.0], vecs={"p": (0.0, 0.0, 2.0)})
    with pytest.raises(mm.MMError, match="MM_ERR_VALUE"):
        mm.Geometry((4, 4, 4), (4, 4), [0.0], [0.0], vecs={"p": (0.0, 1.0, 0.0)})     # p parallel to j
    L = mm.load()
    assert L.mm_geometry_create(None, None) == 1
    assert L.mm_geometry_destroy(None) == 0
    g = mm.Geometry((4, 4, 4), (4, 4), [0.0], [0.0])
    with pytest.raises(mm.MMError, match="MM_ERR_SHAPE"):
        g.get(3)
    with pytest.raises(mm.MMError, match="MM_ERR_SHAPE"):
        mm.mm_basis_sh_matrix(g, 3, *_segs(4))
    assert L.mm_john_forward(None, None, 1, 1, None, None) == 1
    assert L.mm_status_string(5) == b"MM_ERR_CUDA"


def test_device_calls_fail_loudly_without_gpu(mm):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    g = mm.Geometry((4, 4, 4), (4, 4), [0.0], [0.0])
    L = mm.load()
    dummy = ctypes.c_void_p(16)
    st = L.mm_john_forward(g._h, dummy, 4, 4, dummy, None)
    assert st == 5 and b"no CPU fallback" in L.mm_last_error()
    st = L.mm_loss_gradient(g._h, dummy, dummy, 4, 4, 4, dummy, None, dummy, dummy, dummy, None)
    assert st == 5
    assert L.mm_launch_count() == 0


@pytest.mark.parametrize("kind,name,sigma", [(1, "nn", 0.0), (2, "gk", 0.35)])
def test_grid_basis_matrix_matches_oracle(mm, ora, kind, name, sigma):
    """NEXT-2: the library's NN / GK basis-matrix helper against the oracle's (independent code, same quadrature)."""
    from paper_2504_16446_b200 import synth
    r = np.random.default_rng(17)
    P = 11
    rot, tilt = r.uniform(0, 2 * math.pi, P), r.uniform(-0.7, 0.7, P)
    gm = mm.Geometry((5, 6, 7), (6, 5), rot, tilt)
    go = ora.Geometry((5, 6, 7), (6, 5), rot, tilt)
    dirs = synth.grid_directions(18) * r.uniform(0.5, 2.0, (18, 1))      # the helper normalises
    s0, s1 = _segs(8)
    got = mm.mm_basis_grid_matrix(gm, kind, dirs, s0, s1, sigma=sigma, n_quad=12)
    want = ora.basis_matrix_grid(go, dirs, name, s0, s1, sigma=sigma or None, n_quad=12)
    assert got.shape == want.shape == (P, 18, 8)
    if name == "nn":
        # an indicator can flip where two directions are equidistant to 1e-16: allow one quadrature point in a few entries
        diff = np.abs(got - want)
        assert diff.max() <= 1.0 / 12 + 1e-6 and (diff > 1e-6).mean() < 0.01
        assert np.allclose(got.sum(axis=1), 1.0, atol=1e-6)
    else:
        assert np.abs(got - want).max() < 1e-6


def test_grid_basis_matrix_rejects_bad_arguments(mm):
    gm = mm.Geometry((4, 4, 4), (4, 4), [0.0], [0.0])
    s0, s1 = _segs(4)
    with pytest.raises(mm.MMError):
        mm.mm_basis_grid_matrix(gm, 2, np.eye(3), s0, s1, sigma=0.0)          # GK needs sigma > 0
    with pytest.raises(mm.MMError):
        mm.mm_basis_grid_matrix(gm, 7, np.eye(3), s0, s1, sigma=1.0)          # unknown kind
    with pytest.raises(mm.MMError):
        mm.mm_basis_grid_matrix(gm, 1, np.zeros((2, 3)), s0, s1)              # zero direction


def test_sh_matrix_full_two_theta_matches_oracle(mm, ora):
    """NEXT-4: full scattering vector of Eq. 1 (first line) in the SH basis-matrix helper, WAXS-style segments."""
    r = np.random.default_rng(23)
    P = 9
    rot, tilt = r.uniform(0, 2 * math.pi, P), r.uniform(-0.7, 0.7, P)
    gm = mm.Geometry((5, 6, 7), (6, 5), rot, tilt)
    go = ora.Geometry((5, 6, 7), (6, 5), rot, tilt)
    c = np.arange(12)
    s0, s1 = c * 2 * math.pi / 12, (c + 1) * 2 * math.pi / 12
    for tt in (0.0, 0.35, 1.2):
        got = mm.mm_basis_sh_matrix(gm, 6, s0, s1, two_theta=tt)
        assert np.abs(got - ora.basis_matrix(go, 6, s0, s1, two_theta=tt)).max() < 1e-6
    assert np.array_equal(mm.mm_basis_sh_matrix(gm, 6, s0, s1, two_theta=0.0), mm.mm_basis_sh_matrix(gm, 6, s0, s1))


def test_host_workspace_release_with_nothing_allocated(mm):
    """mm_host_workspace_release is a no-op (MM_OK) before any host call and needs no device."""
    mm.mm_host_workspace_release()
    mm.mm_host_workspace_release()


def test_sparsify_and_plan_match_the_oracle(ora, mm):
    """NEXT-2 host parts (reading S26): mm_basis_sparsify == oracle.sparsify_basis bit for bit, incl. ties;
    the plan's channel lists are the rows of B with a non-zero entry."""
    from paper_2504_16446_b200 import synth
    r = np.random.default_rng(8)
    B = r.standard_normal((4, 11, 5)).astype(np.float32)
    B[1, 3] = B[1, 7]                                                  # equal magnitudes: lowest index first
    for n in (1, 2, 6, 11, 40):
        assert np.array_equal(mm.mm_basis_sparsify(B, n), ora.sparsify_basis(B, n))
    g = mm.Geometry((4, 4, 4), (4, 4), [0.3, 1.1, 2.0], [0.2, -0.5, 0.0])
    Bnn = mm.mm_basis_grid_matrix(g, mm.MM_BASIS_NN, synth.grid_directions(60), *_segs(8), n_quad=4)
    plan = mm.SparsePlan(g, Bnn)
    want = (np.abs(Bnn).sum(axis=2) > 0).sum(axis=1)
    assert np.array_equal(plan.counts, want) and plan.max_active == want.max() and abs(plan.mean_active - want.mean()) < 1e-12
    assert plan.max_active <= 8 * 4 < 60                               # at most one direction per quadrature point
    one = mm.SparsePlan(g, mm.mm_basis_sparsify(Bnn, 1))
    assert one.max_active <= 8
