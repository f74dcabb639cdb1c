"""GPU parity: every C-ABI device call against the fp64 CPU oracle on the same seeded inputs (run with -m gpu).

Error metric (reading S18, BASELINE.json north_star): E_inf = max|gpu - oracle| / max|oracle| over the
whole output array <= 1e-5 for projections, sinograms and gradients; |L_gpu - L_ora| / |L_ora| <= 1e-4 for the loss.
"""
import math

import numpy as np
import pytest

from paper_2504_16446_b200 import synth

pytestmark = pytest.mark.gpu

TOL = 1e-5
TOL_LOSS = 1e-4


@pytest.fixture(scope="module")
def mm():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2504_16446_b200 import mm as binding
    binding.load()           # raises if libmm.so is missing: no fallback
    return binding


def einf(got, want):
    want = np.asarray(want, dtype=np.float64)
    got = np.asarray(got, dtype=np.float64)
    den = np.abs(want).max()
    return np.abs(got - want).max() / (den if den > 0 else 1.0)


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


class Case:
    """seeded inputs for one geometry, usable by both sides"""

    def __init__(self, shape, det, rot, tilt, K, ldk, D, seed=0, joff=None, koff=None, vecs=None, a=1.0, b=1.0,
                 vol=None, B=None, weights="uniform"):
        r = np.random.default_rng(seed)
        self.shape, self.det, self.K, self.ldk, self.D = tuple(shape), tuple(det), K, ldk, D
        self.rot, self.tilt = np.asarray(rot, dtype=np.float64), np.asarray(tilt, dtype=np.float64)
        self.P = self.rot.size
        self.kw = dict(j_offsets=joff, k_offsets=koff, vecs=vecs, voxel_size=a, pixel_size=b)
        if vol is None:
            vol = r.standard_normal(self.shape + (ldk,)).astype(np.float32)
        self.vol = vol                                               # pad channels hold garbage on purpose
        self.B = (r.standard_normal((self.P, K, D)).astype(np.float32) if B is None else B)
        sh = (self.P,) + self.det
        self.y = r.standard_normal(sh + (ldk,)).astype(np.float32)  # K-channel projections for the adjoint
        self.sino = r.standard_normal(sh + (D,)).astype(np.float32)
        self.data = r.standard_normal(sh + (D,)).astype(np.float32)
        if weights == "uniform":
            self.w = r.uniform(0.5, 1.5, sh + (D,)).astype(np.float32)
        elif weights == "mask":
            self.w = np.ascontiguousarray(np.broadcast_to((r.uniform(size=sh) >= 0.05).astype(np.float32)[..., None], sh + (D,)))
        else:
            self.w = None

    def geoms(self, ora, mm):
        return (ora.Geometry(self.shape, self.det, self.rot, self.tilt, **self.kw),
                mm.Geometry(self.shape, self.det, self.rot, self.tilt, **self.kw))


def cfg_case(name, shape, det, n_rot, seed, joff=False, weights="uniform"):
    cfg = synth.get_config(name, shape=shape, det=det, n_rot=n_rot)
    rot, tilt = synth.angles(cfg)
    ldk = synth.ldk_for(cfg.K)
    vol = synth.make_volume(cfg, ldk)
    r = np.random.default_rng(seed)
    jo = r.uniform(-1.5, 1.5, cfg.P) if joff else None
    ko = r.uniform(-1.5, 1.5, cfg.P) if joff else None
    return cfg, Case(cfg.shape, cfg.det, rot, tilt, cfg.K, ldk, cfg.D, seed=seed, joff=jo, koff=ko, vol=vol, weights=weights)


def run_all_ops(ora, mm, c, check_fused_composition=True, sh_basis=None):
    """all device calls on case c vs the oracle; returns dict of errors"""
    import torch
    go, gm = c.geoms(ora, mm)
    K, ldk, D = c.K, c.ldk, c.D
    B = c.B
    if sh_basis is not None:
        B = mm.mm_basis_sh_matrix(gm, sh_basis, *synth.segments(D))
        assert einf(B, ora.basis_matrix(go, sh_basis, *synth.segments(D))) < 1e-6
    dB, dvol = dev(B), dev(c.vol)
    errs = {}
    # --- John forward (a3)
    proj = torch.full(gm.proj_shape(ldk), float("nan"), device="cuda")
    mm.mm_john_forward(gm, dvol, K, proj)
    want = ora.john_forward(go, c.vol, K)
    got = proj.cpu().numpy()
    errs["john_forward"] = einf(got[..., :K], want)
    assert np.all(got[..., K:] == 0.0)                                   # pad channels written as 0
    # --- John adjoint (a7)
    dy = dev(c.y)
    vout = torch.full(gm.vol_shape(ldk), float("nan"), device="cuda")
    mm.mm_john_adjoint(gm, dy, K, vout)
    want = ora.john_adjoint(go, c.y[..., :K].astype(np.float64), form="scatter")
    got = vout.cpu().numpy()
    errs["john_adjoint"] = einf(got[..., :K], want)
    assert np.all(got[..., K:] == 0.0)
    # --- basis maps (a4, a6)
    sino = torch.empty(gm.proj_shape(D), device="cuda")
    mm.mm_basis_forward(gm, dB, dy, K, sino)
    errs["basis_forward"] = einf(sino.cpu().numpy(), ora.basis_forward(B, c.y[..., :K]))
    dsino = dev(c.sino)
    pr = torch.full(gm.proj_shape(ldk), float("nan"), device="cuda")
    mm.mm_basis_adjoint(gm, dB, dsino, K, pr)
    got = pr.cpu().numpy()
    errs["basis_adjoint"] = einf(got[..., :K], ora.basis_adjoint(B, c.sino))
    assert np.all(got[..., K:] == 0.0)
    # --- fused forward model and its transpose
    model = torch.empty(gm.proj_shape(D), device="cuda")
    mm.mm_forward(gm, dB, dvol, K, model)
    want_model = ora.forward(go, B, c.vol[..., :K])
    errs["forward"] = einf(model.cpu().numpy(), want_model)
    vout2 = torch.full(gm.vol_shape(ldk), float("nan"), device="cuda")
    mm.mm_adjoint(gm, dB, dsino, K, vout2)
    want = ora.adjoint(go, B, c.sino, form="scatter")
    got = vout2.cpu().numpy()
    errs["adjoint"] = einf(got[..., :K], want)
    assert np.all(got[..., K:] == 0.0)
    # --- NEXT-1: the paper's bilinear back-projection, K-channel and fused with basis^T
    vb = torch.full(gm.vol_shape(ldk), float("nan"), device="cuda")
    mm.mm_john_backproject(gm, dy, K, vb)
    got = vb.cpu().numpy()
    errs["john_backproject"] = einf(got[..., :K], ora.john_backproject_bilinear(go, c.y[..., :K]))
    assert np.all(got[..., K:] == 0.0)
    vb.fill_(float("nan"))
    mm.mm_backproject(gm, dB, dsino, K, vb)
    got = vb.cpu().numpy()
    errs["backproject"] = einf(got[..., :K], ora.backproject_bilinear(go, B, c.sino))
    assert np.all(got[..., K:] == 0.0)
    # --- fused gradient (a8)
    scale = float(np.abs(want_model).max())
    data = (want_model + 0.1 * scale * c.data).astype(np.float32)          # data near the model: no giant residuals
    grad = torch.full(gm.vol_shape(ldk), float("nan"), device="cuda")
    loss = torch.full((1,), float("nan"), device="cuda", dtype=torch.float64)
    wr = torch.empty(gm.proj_shape(D), device="cuda")
    dw = None if c.w is None else dev(c.w)
    mm.mm_loss_gradient(gm, dB, dvol, K, dev(data), dw, grad, loss, wr)
    L, want_grad, want_wr = ora.loss_gradient(go, B, c.vol[..., :K], data, c.w, form="scatter")
    errs["wr"] = np.abs(wr.cpu().numpy() - want_wr).max() / scale          # residuals cancel: scale by the model
    got = grad.cpu().numpy()
    errs["grad"] = einf(got[..., :K], want_grad)
    errs["loss"] = abs(loss.item() - L) / abs(L)
    assert np.all(got[..., K:] == 0.0)
    if check_fused_composition:
        # fused == composition of the standalone calls, on the GPU
        mm.mm_john_forward(gm, dvol, K, proj)
        mm.mm_basis_forward(gm, dB, proj, K, sino)
        assert einf(sino.cpu().numpy(), model.cpu().numpy()) < 3e-6
        mm.mm_basis_adjoint(gm, dB, wr, K, pr)
        mm.mm_john_adjoint(gm, pr, K, vout)
        assert einf(vout.cpu().numpy()[..., :K], got[..., :K]) < 1e-5    # two fp32 paths, each within TOL of the oracle
    return errs


def assert_errs(errs):
    print("parity errors:", {k: float("%.2e" % v) for k, v in errs.items()})
    for k, v in errs.items():
        assert v <= (TOL_LOSS if k == "loss" else TOL), (k, v, errs)


def test_c1_full(ora, mm):
    """BASELINE.json config 1 at full size (32^3, K=6, 60 projections at tilt 0, includes the 45-degree tie)."""
    cfg, c = cfg_case("C1", None, None, None, seed=1, weights=None)
    assert_errs(run_all_ops(ora, mm, c, sh_basis=cfg.ell_max))


def test_c2_shrunk_masked_ragged(ora, mm):
    """config 2 recipe (K=15, six tilts, 5% masked pixels) on a ragged grid spanning several tiles."""
    cfg, c = cfg_case("C2", (40, 36, 44), (45, 50), 6, seed=2, weights="mask")
    assert_errs(run_all_ops(ora, mm, c, sh_basis=cfg.ell_max))


def test_c3_shrunk_offsets(ora, mm):
    """config 3 recipe (K=45 -> ldk 48, eight tilts up to 45 degrees incl. y-major projections), sub-pixel offsets."""
    cfg, c = cfg_case("C3", (30, 26, 34), (37, 41), 5, seed=3, joff=True)
    assert_errs(run_all_ops(ora, mm, c, sh_basis=cfg.ell_max))


def test_c4_shrunk_plate(ora, mm):
    """config 4 recipe (non-cubic plate, K=28, D=16, weights U[0.5,1.5])."""
    cfg, c = cfg_case("C4", (20, 40, 40), (44, 44), 4, seed=4)
    assert_errs(run_all_ops(ora, mm, c, sh_basis=cfg.ell_max))


def test_c5_shrunk(ora, mm):
    """config 5 recipe (ellipsoid density, nine tilts) on 48^3."""
    cfg, c = cfg_case("C5", (48, 48, 48), (48, 48), 4, seed=5, weights=None)
    assert_errs(run_all_ops(ora, mm, c, sh_basis=cfg.ell_max))


@pytest.mark.parametrize("K,ldk,D", [(7, 7, 5), (1, 1, 1), (3, 4, 8), (33, 36, 12), (70, 72, 9), (130, 132, 4), (20, 21, 32)])
def test_odd_channel_counts(ora, mm, K, ldk, D):
    """scalar (unaligned ldk) path, K not a multiple of 4, D not a multiple of 4, channel chunking (K > 48)."""
    r = np.random.default_rng(K)
    P = 7
    c = Case((11, 9, 13), (12, 14), r.uniform(0, 2 * math.pi, P), r.uniform(-0.7, 0.7, P), K, ldk, D, seed=K,
             joff=r.uniform(-1, 1, P), koff=r.uniform(-1, 1, P))
    assert_errs(run_all_ops(ora, mm, c))


def test_rotated_lab_frame_and_size_ratio(ora, mm):
    """non-standard Table I vectors (voxel gather window wider than in the standard geometry) and a != b."""
    r = np.random.default_rng(11)
    P = 9
    rot, tilt = r.uniform(0, 2 * math.pi, P), r.uniform(-0.6, 0.6, P)
    s = math.sqrt(0.5)
    vecs = {"p": (0.0, 0.0, 1.0), "j": (s, s, 0.0), "k": (s, -s, 0.0), "inner_axis": (0.0, 1.0, 0.0), "outer_axis": (1.0, 0.0, 0.0)}
    assert_errs(run_all_ops(ora, mm, Case((12, 10, 14), (16, 15), rot, tilt, 6, 8, 8, seed=12, vecs=vecs)))
    assert_errs(run_all_ops(ora, mm, Case((12, 10, 14), (20, 22), rot, tilt, 6, 8, 8, seed=13, a=1.0, b=0.7)))
    assert_errs(run_all_ops(ora, mm, Case((12, 10, 14), (9, 8), rot, tilt, 6, 8, 8, seed=14, a=0.8, b=1.3)))
    vecs = {"p": (1.0, 0.0, 0.0), "j": (0.0, 0.0, 1.0), "k": (0.0, 1.0, 0.0), "inner_axis": (0.0, 0.0, 1.0), "outer_axis": (0.0, 1.0, 0.0)}
    assert_errs(run_all_ops(ora, mm, Case((12, 10, 14), (16, 15), rot, tilt, 6, 8, 8, seed=15, vecs=vecs)))


def test_degenerate_shapes(ora, mm):
    """single voxel, single pixel, single projection, detector much larger / smaller than the sample, thin axes."""
    for shape, det in [((1, 1, 1), (1, 1)), ((1, 1, 1), (5, 4)), ((6, 1, 5), (3, 9)), ((2, 7, 1), (8, 2)),
                       ((5, 5, 5), (17, 19)), ((9, 9, 9), (2, 3)), ((1, 8, 8), (8, 8))]:
        for rot, tilt in [([0.0], [0.0]), ([0.5, math.pi / 4, 2.0], [0.2, 0.0, math.pi / 4])]:
            c = Case(shape, det, rot, tilt, 4, 4, 8, seed=len(rot) + shape[0])
            errs = run_all_ops(ora, mm, c)
            assert_errs(errs)


def test_far_offsets_empty_rays(ora, mm):
    """offsets that push every ray off the sample: all outputs exactly zero, nothing read out of bounds."""
    import torch
    c = Case((6, 6, 6), (5, 5), [0.3, 1.0], [0.1, 0.4], 4, 4, 8, seed=3, joff=[100.0, -80.0], koff=[50.0, 60.0])
    go, gm = c.geoms(ora, mm)
    proj = torch.full(gm.proj_shape(4), float("nan"), device="cuda")
    mm.mm_john_forward(gm, dev(c.vol), 4, proj)
    assert torch.all(proj == 0).item()
    assert np.all(ora.john_forward(go, c.vol, 4) == 0)
    vout = torch.full(gm.vol_shape(4), float("nan"), device="cuda")
    mm.mm_john_adjoint(gm, dev(c.y), 4, vout)
    assert torch.all(vout == 0).item()


def test_gpu_dot_product_identity(mm):
    """<A x, y> = <x, A^T y> for the GPU pair itself (fused and K-channel), on a multi-tilt geometry with ties."""
    import torch
    cfg = synth.get_config("C3", shape=(28, 24, 30), det=(33, 35), n_rot=4)
    rot, tilt = synth.angles(cfg)
    r = np.random.default_rng(7)
    gm = mm.Geometry(cfg.shape, cfg.det, rot, tilt, j_offsets=r.uniform(-1, 1, cfg.P), k_offsets=r.uniform(-1, 1, cfg.P))
    K, ldk, D = cfg.K, 48, cfg.D
    torch.manual_seed(7)
    x = torch.randn(gm.vol_shape(ldk), device="cuda")
    x[..., K:] = 0
    y = torch.randn(gm.proj_shape(ldk), device="cuda")
    y[..., K:] = 0
    Ax = torch.empty_like(y)
    ATy = torch.empty_like(x)
    mm.mm_john_forward(gm, x, K, Ax)
    mm.mm_john_adjoint(gm, y, K, ATy)
    # white-noise inner products cancel, so the scale of the comparison is |Ax||y| (Cauchy-Schwarz), not |<Ax,y>|
    lhs, rhs = (Ax.double() * y.double()).sum().item(), (x.double() * ATy.double()).sum().item()
    assert abs(lhs - rhs) <= 1e-5 * (Ax.double().norm() * y.double().norm()).item(), (lhs, rhs)
    B = dev(mm.mm_basis_sh_matrix(gm, cfg.ell_max, *synth.segments(D)))
    ys = torch.randn(gm.proj_shape(D), device="cuda")
    Axs = torch.empty_like(ys)
    mm.mm_forward(gm, B, x, K, Axs)
    mm.mm_adjoint(gm, B, ys, K, ATy)
    lhs, rhs = (Axs.double() * ys.double()).sum().item(), (x.double() * ATy.double()).sum().item()
    assert abs(lhs - rhs) <= 1e-5 * (Axs.double().norm() * ys.double().norm()).item(), (lhs, rhs)
    # non-cancelling case: x, y >= 0 (and the John transform has non-negative entries), so <Ax,y> is a sum of
    # non-negative terms and the identity must hold to 1e-5 of the inner product itself
    xp, yp = x.abs(), y.abs()
    mm.mm_john_forward(gm, xp, K, Ax)
    mm.mm_john_adjoint(gm, yp, K, ATy)
    lhs, rhs = (Ax.double() * yp.double()).sum().item(), (xp.double() * ATy.double()).sum().item()
    assert lhs > 0 and abs(lhs - rhs) <= 1e-5 * lhs, (lhs, rhs)
    # same through the fused pair with |B| (A = P (x) |B| is then non-negative too)
    absB = B.abs()
    mm.mm_forward(gm, absB, xp, K, Axs)
    mm.mm_adjoint(gm, absB, ys.abs(), K, ATy)
    lhs, rhs = (Axs.double() * ys.abs().double()).sum().item(), (xp.double() * ATy.double()).sum().item()
    assert lhs > 0 and abs(lhs - rhs) <= 1e-5 * lhs, (lhs, rhs)


def test_zero_residual_and_zero_weight(mm):
    """data = A c (rounded to fp32, as any data is) gives L ~ 0, grad ~ 0: the residual is that rounding and nothing
    else, because the model value is kept unrounded until the subtraction; zero-weight pixels do not
    contribute whatever they hold (reading S11)."""
    import torch
    cfg = synth.get_config("C2", shape=(20, 20, 20), det=(22, 22), n_rot=3)
    rot, tilt = synth.angles(cfg)
    gm = mm.Geometry(cfg.shape, cfg.det, rot, tilt)
    K, ldk, D = cfg.K, 16, cfg.D
    hB = mm.mm_basis_sh_matrix(gm, cfg.ell_max, *synth.segments(D))
    B = dev(hB)
    vol = dev(synth.make_volume(cfg, ldk))
    model = torch.empty(gm.proj_shape(D), device="cuda")
    mm.mm_forward(gm, B, vol, K, model)
    grad = torch.empty(gm.vol_shape(ldk), device="cuda")
    loss = torch.zeros(1, device="cuda", dtype=torch.float64)
    wr = torch.empty_like(model)
    mm.mm_loss_gradient(gm, B, vol, K, model, None, grad, loss, wr)
    u = 2.0 ** -24
    assert torch.all(wr.abs() <= 1.01 * u * model.abs()).item()
    assert loss.item() <= 0.5 * float((u * model.double()).pow(2).sum())
    bound = torch.empty_like(grad)
    mm.mm_adjoint(gm, dev(np.abs(hB)), model.abs(), K, bound)             # |A|^T |model| bounds |A^T wr| / u entrywise
    assert torch.all(grad.abs() <= 1.01 * u * bound + 1e-30).item()
    w = (torch.rand(gm.proj_shape(D), device="cuda") > 0.5).float()
    junk = model + 1e6 * (1 - w) * torch.randn_like(model)               # garbage where the weight is 0
    g1, l1, w1 = torch.empty_like(grad), torch.zeros_like(loss), torch.empty_like(wr)
    mm.mm_loss_gradient(gm, B, vol, K, model, w, g1, l1, w1)
    mm.mm_loss_gradient(gm, B, vol, K, junk, w, grad, loss, wr)
    # (the loss is summed with fp64 atomics in no fixed order: equal to rounding, not bit for bit)
    assert abs(loss.item() - l1.item()) <= 1e-12 * l1.item() and torch.equal(grad, g1) and torch.equal(wr, w1)


def test_host_entry_point_matches_device_path(ora, mm):
    import torch
    cfg, c = cfg_case("C2", (24, 22, 26), (27, 30), 3, seed=9)
    go, gm = c.geoms(ora, mm)
    B = mm.mm_basis_sh_matrix(gm, cfg.ell_max, *synth.segments(c.D))
    data = synth.surrogate_model(cfg)
    h_grad = np.full(gm.vol_shape(c.ldk), np.nan, dtype=np.float32)
    L = mm.mm_loss_gradient_host(gm, B, c.vol, c.K, data, c.w, h_grad)
    grad = torch.empty(gm.vol_shape(c.ldk), device="cuda")
    loss = torch.zeros(1, device="cuda", dtype=torch.float64)
    wr = torch.empty(gm.proj_shape(c.D), device="cuda")
    mm.mm_loss_gradient(gm, dev(B), dev(c.vol), c.K, dev(data), dev(c.w), grad, loss, wr)
    assert abs(L - loss.item()) <= 1e-12 * abs(L)
    assert np.array_equal(h_grad, grad.cpu().numpy())
    Lo, go_grad, _ = ora.loss_gradient(go, B, c.vol[..., :c.K], data, c.w, form="scatter")
    assert abs(L - Lo) <= TOL_LOSS * abs(Lo) and einf(h_grad[..., :c.K], go_grad) <= TOL


def test_host_entry_point_arena_regrows_and_releases(ora, mm):
    """The library-owned device arena of mm_loss_gradient_host is reused, regrown for a larger problem and freed by
    mm_host_workspace_release; every call equals the device path bit for bit (8 voxel ranges, ragged last one)."""
    import torch
    for n, (shape, det, seed) in enumerate((((12, 10, 14), (15, 17), 3), ((33, 31, 29), (37, 35), 4), ((12, 10, 14), (15, 17), 3))):
        cfg, c = cfg_case("C3", shape, det, 4, seed=seed)
        _, gm = c.geoms(ora, mm)
        B = mm.mm_basis_sh_matrix(gm, cfg.ell_max, *synth.segments(c.D))
        data = synth.surrogate_model(cfg)
        h_grad = np.full(gm.vol_shape(c.ldk), np.nan, dtype=np.float32)
        L = mm.mm_loss_gradient_host(gm, B, c.vol, c.K, data, c.w, h_grad)
        grad = torch.empty(gm.vol_shape(c.ldk), device="cuda")
        loss = torch.zeros(1, device="cuda", dtype=torch.float64)
        wr = torch.empty(gm.proj_shape(c.D), device="cuda")
        mm.mm_loss_gradient(gm, dev(B), dev(c.vol), c.K, dev(data), dev(c.w), grad, loss, wr)
        assert abs(L - loss.item()) <= 1e-12 * abs(L)
        assert np.array_equal(h_grad, grad.cpu().numpy())
        if n == 1:
            mm.mm_host_workspace_release()
    mm.mm_host_workspace_release()
    mm.mm_host_workspace_release()          # idempotent


def test_gd_iterations_c4_recipe(ora, mm):
    """config 4's timed loop (gradient + fixed-step update) on a shrunk plate: trajectory parity."""
    import torch
    cfg, c = cfg_case("C4", (12, 24, 24), (26, 26), 3, seed=21)
    go, gm = c.geoms(ora, mm)
    K, ldk, D = c.K, c.ldk, c.D
    B = mm.mm_basis_sh_matrix(gm, cfg.ell_max, *synth.segments(D))
    data = synth.poisson_data(ora.forward(go, B, c.vol[..., :K]), cfg.counts, cfg.seed)
    # eta = 1 / (max w * ||A||_1 ||A||_inf) from |B| and all-ones inputs (DESIGN.md input recipe), oracle side
    absB = np.abs(B)
    rows = ora.forward(go, absB, np.ones(c.shape + (K,), np.float32)).max()
    cols = ora.adjoint(go, absB, np.ones((c.P,) + c.det + (D,)), form="scatter").max()
    eta = 1.0 / (float(c.w.max()) * rows * cols)
    x_o = np.zeros(c.shape + (K,), dtype=np.float32)
    x_g = torch.zeros(gm.vol_shape(ldk), device="cuda")
    dB, dd, dw = dev(B), dev(data), dev(c.w)
    grad = torch.empty_like(x_g)
    loss = torch.zeros(1, device="cuda", dtype=torch.float64)
    wr = torch.empty(gm.proj_shape(D), device="cuda")
    for it in range(5):
        mm.mm_loss_gradient(gm, dB, x_g, K, dd, dw, grad, loss, wr)
        mm.mm_axpy(x_g, grad, eta)
        Lo, g_o, _ = ora.loss_gradient(go, B, x_o, data, c.w, form="scatter")
        if it == 0:
            assert einf(grad.cpu().numpy()[..., :K], g_o) <= TOL
        assert abs(loss.item() - Lo) <= TOL_LOSS * abs(Lo)
        x_o = (x_o.astype(np.float64) - np.float32(eta).astype(np.float64) * g_o).astype(np.float32)
    assert einf(x_g.cpu().numpy()[..., :K], x_o) <= 1e-4


def test_c5_full_size_sampled(ora, mm):
    """BASELINE.json config 5 at FULL size (256^3, K=45, 360 projections, 256^2 detector, D=8), in the launch
    configuration bench.py times (ldk = 48, unit weights).  The oracle cannot run the whole problem in test time, so
    parity is checked on sampled outputs it computes one by one: rays of the model sinogram / weighted residual
    (forward_rays) and voxels of the gradient (gradient_voxels, from scratch through the voxel's column of A).
    Errors are scaled by the maximum of the whole GPU array (the oracle's maximum is not available at this size;
    the two agree to the tolerance being tested).  Data is synth.surrogate_model: made by neither implementation."""
    import torch
    cfg = synth.get_config("C5")
    rot, tilt = synth.angles(cfg)
    K, D, ldk = cfg.K, cfg.D, synth.ldk_for(cfg.K)
    vol = synth.make_volume(cfg, ldk)
    gm = mm.Geometry(cfg.shape, cfg.det, rot, tilt)
    go = ora.Geometry(cfg.shape, cfg.det, rot, tilt)
    B = mm.mm_basis_sh_matrix(gm, cfg.ell_max, *synth.segments(D))
    data = synth.surrogate_model(cfg, level=float(np.abs(vol[..., 0]).max()) * 100.0)
    dB, dvol, ddata = dev(B), dev(vol), dev(data)
    model = torch.empty(gm.proj_shape(D), device="cuda")
    mm.mm_forward(gm, dB, dvol, K, model)
    grad = torch.full(gm.vol_shape(ldk), float("nan"), device="cuda")
    loss = torch.zeros(1, device="cuda", dtype=torch.float64)
    wr = torch.empty(gm.proj_shape(D), device="cuda")
    mm.mm_loss_gradient(gm, dB, dvol, K, ddata, None, grad, loss, wr)
    torch.cuda.synchronize()
    r = np.random.default_rng(55)
    # --- sampled rays: every tilt, rays through the sample and near the detector edge
    sjk = np.stack([r.integers(0, cfg.P, 240), r.integers(0, cfg.det[0], 240), r.integers(0, cfg.det[1], 240)], axis=1)
    sjk[:40, 1] = r.integers(96, 160, 40); sjk[:40, 2] = r.integers(96, 160, 40)       # central rays for sure
    want = ora.forward_rays(go, B, vol, sjk)
    idx = tuple(torch.from_numpy(sjk[:, i].astype(np.int64)).cuda() for i in range(3))
    got = model[idx].cpu().numpy()
    scale = float(model.abs().max())
    assert np.abs(want).max() > 0.05 * scale                       # the sample is not all background
    assert np.abs(got - want).max() / scale <= TOL
    got_wr = wr[idx].cpu().numpy()
    assert np.abs(got_wr - (want - data[sjk[:, 0], sjk[:, 1], sjk[:, 2]])).max() / scale <= TOL
    # --- loss: fp64 reduction of the GPU's own residuals (the residuals themselves are checked above)
    L64 = 0.5 * float((wr.double() ** 2).sum())
    assert abs(loss.item() - L64) <= TOL_LOSS * L64
    # --- sampled voxels of the gradient: interior, faces, corners
    xyz = np.concatenate([r.integers(64, 192, (10, 3)), r.integers(0, 256, (6, 3)),
                          np.array([[0, 0, 0], [255, 255, 255], [0, 128, 255], [128, 0, 17]])]).astype(np.int32)
    want_g = ora.gradient_voxels(go, B, vol, data, None, xyz)
    gi = tuple(torch.from_numpy(xyz[:, i].astype(np.int64)).cuda() for i in range(3))
    got_g = grad[gi].cpu().numpy()
    gscale = float(grad[..., :K].abs().max())
    assert np.abs(got_g[:, :K] - want_g).max() / gscale <= TOL
    assert np.all(got_g[:, K:] == 0.0)
    assert not torch.isnan(grad).any().item()
    # --- NEXT-1 at full size: the paper's bilinear back-projection of the weighted residual, same sampled voxels
    mm.mm_backproject(gm, dB, wr, K, grad)
    # (projection by projection: back-project the D channels, then apply that projection's B^T — the K-channel
    # sinogram of the whole problem would not fit the oracle's budget)
    wr_h = wr.cpu().numpy()
    want_b = np.zeros((xyz.shape[0], K))
    for s in range(cfg.P):
        g1 = ora.Geometry(cfg.shape, cfg.det, rot[s:s + 1], tilt[s:s + 1])
        want_b += ora.john_backproject_bilinear_voxels(g1, wr_h[s:s + 1].astype(np.float64), xyz) @ B[s].astype(np.float64).T
    got_b = grad[gi].cpu().numpy()
    assert np.abs(got_b[:, :K] - want_b).max() / float(grad[..., :K].abs().max()) <= TOL


@pytest.mark.parametrize("K,ldk,D,P", [(13, 16, 8, 7), (13, 16, 16, 5), (30, 32, 8, 19), (45, 48, 16, 9), (60, 64, 8, 17),
                                        (61, 64, 16, 33), (90, 92, 8, 9), (120, 128, 16, 7), (162, 164, 8, 11),
                                        (250, 252, 8, 5), (200, 200, 16, 4)])
def test_tensor_core_adjoint_instantiations(ora, mm, K, ldk, D, P):
    """every (D, accumulator width) instantiation of the tcgen05 adjoint, with projection counts that leave a
    short last chunk (P odd), fewer chunks than one accumulation window, and more than two windows."""
    r = np.random.default_rng(100 * K + D)
    c = Case((19, 17, 21), (24, 22), r.uniform(0, 2 * math.pi, P), r.uniform(-0.75, 0.75, P), K, ldk, D, seed=K + D,
             joff=r.uniform(-1, 1, P), koff=r.uniform(-1, 1, P))
    assert_errs(run_all_ops(ora, mm, c))


@pytest.mark.parametrize("matched", [False, True])
def test_sirt_iterations(ora, mm, matched):
    """SIRT/MITRA as preconditioned weighted least squares (reading S19), composed from the C-ABI
    calls: W = 1/(|A| 1), C = 1/(|A|' 1) by mm_forward / back-projector on ones + mm_reciprocal, then per iteration
    mm_residual_loss -> mm_backproject (the paper's pair) or mm_adjoint (matched pair) -> mm_axpy_precond."""
    import torch
    cfg, c = cfg_case("C2", (22, 20, 24), (26, 25), 3, seed=31, joff=True, weights=None)
    go, gm = c.geoms(ora, mm)
    K, ldk, D = c.K, c.ldk, c.D
    B = mm.mm_basis_sh_matrix(gm, cfg.ell_max, *synth.segments(D))
    data = synth.poisson_data(ora.forward(go, B, c.vol[..., :K]), cfg.counts, cfg.seed)
    W_o, C_o = ora.sirt_preconditioners(go, B, matched=matched)
    back = mm.mm_adjoint if matched else mm.mm_backproject
    dB, dabsB, dd = dev(B), dev(np.abs(B)), dev(data)
    W = torch.empty(gm.proj_shape(D), device="cuda")
    ones_v = torch.ones(gm.vol_shape(ldk), device="cuda")
    mm.mm_forward(gm, dabsB, ones_v, K, W)
    mm.mm_reciprocal(W, 1e-6)
    Cp = torch.empty(gm.vol_shape(ldk), device="cuda")
    back(gm, dabsB, torch.ones(gm.proj_shape(D), device="cuda"), K, Cp)
    mm.mm_reciprocal(Cp, 1e-6)
    assert einf(W.cpu().numpy(), W_o) <= TOL and einf(Cp.cpu().numpy()[..., :K], C_o) <= TOL
    x_g = torch.zeros(gm.vol_shape(ldk), device="cuda")
    x_o = np.zeros(c.shape + (K,), dtype=np.float32)
    wr = torch.empty(gm.proj_shape(D), device="cuda")
    bp = torch.empty_like(x_g)
    loss = torch.zeros(1, device="cuda", dtype=torch.float64)
    losses = []
    for it in range(4):
        mm.mm_residual_loss(gm, dB, x_g, K, dd, W, wr, loss)
        back(gm, dB, wr, K, bp)
        mm.mm_axpy_precond(x_g, bp, Cp, 1.0)
        x_new, L_o = ora.sirt_step(go, B, x_o, data, W_o, C_o, matched=matched)
        assert abs(loss.item() - L_o) <= TOL_LOSS * abs(L_o)
        losses.append(L_o)
        x_o = x_new.astype(np.float32)
    assert einf(x_g.cpu().numpy()[..., :K], x_o) <= 1e-4            # errors compound over the iterations
    assert losses[-1] < losses[0]


@pytest.mark.parametrize("kind,K", [("gk", 18), ("nn", 18), ("gk", 50)])
def test_grid_basis_sets_through_the_same_kernels(ora, mm, kind, K):
    """NEXT-2: GK / NN basis sets only change the B matrix; every device call is checked with
    B built by the library's helper (K = 18 and 50 as in the paper's Table V; ldk 20 and 52)."""
    r = np.random.default_rng(K)
    P = 10
    ldk = synth.ldk_for(K)
    c = Case((18, 16, 20), (22, 21), r.uniform(0, 2 * math.pi, P), r.uniform(-0.7, 0.7, P), K, ldk, 8, seed=K)
    _, gm = c.geoms(ora, mm)
    c.B = mm.mm_basis_grid_matrix(gm, mm.MM_BASIS_GK if kind == "gk" else mm.MM_BASIS_NN, synth.grid_directions(K),
                                  *synth.segments(8), sigma=0.3, n_quad=8)
    assert_errs(run_all_ops(ora, mm, c))


@pytest.mark.parametrize("K,ldk,shape", [(6, 8, (17, 13, 19)), (5, 5, (9, 1, 7)), (45, 48, (12, 14, 10)), (1, 1, (1, 1, 1))])
def test_laplacian(ora, mm, K, ldk, shape):
    """NEXT-3: zero-padded 7-point Laplacian of every channel (reading S21), float4 and scalar paths."""
    import torch
    gm = mm.Geometry(shape, (4, 4), [0.0], [0.0])
    v = np.random.default_rng(K).standard_normal(shape + (ldk,)).astype(np.float32)
    out = torch.full(gm.vol_shape(ldk), float("nan"), device="cuda")
    mm.mm_laplacian(gm, dev(v), K, out)
    got = out.cpu().numpy()
    want = ora.laplacian(v[..., :K])
    assert np.abs(got[..., :K] - want).max() <= 1e-5 * max(1.0, np.abs(want).max()) and np.all(got[..., K:] == 0.0)


def test_regularised_nesterov_iterations(ora, mm):
    """a device-resident MITRA/SIGTT-style loop: data term + Laplacian + L2 regularisers,
    Nesterov momentum, composed from the C-ABI calls; trajectory and losses against the oracle."""
    import torch
    cfg, c = cfg_case("C2", (18, 16, 20), (22, 21), 3, seed=41, weights=None)
    go, gm = c.geoms(ora, mm)
    K, ldk, D = c.K, c.ldk, c.D
    B = mm.mm_basis_sh_matrix(gm, cfg.ell_max, *synth.segments(D))
    data = synth.poisson_data(ora.forward(go, B, c.vol[..., :K]), cfg.counts, cfg.seed)
    absB = np.abs(B)
    lip = float(ora.forward(go, absB, np.ones(c.shape + (K,), np.float32)).max() *
                ora.adjoint(go, absB, np.ones((c.P,) + c.det + (D,)), form="scatter").max())
    mu_lap, mu_l2, mom = 1e-3 * lip, 1e-4 * lip, 0.8
    eta = 1.0 / (lip + 144.0 * mu_lap + mu_l2)                       # ||Lap||^2 <= 12^2
    dB, dd = dev(B), dev(data)
    n = int(np.prod(gm.vol_shape(ldk)))
    x = torch.zeros(gm.vol_shape(ldk), device="cuda"); v = torch.zeros_like(x)
    look, grad, l1, l2 = (torch.empty_like(x) for _ in range(4))
    wr = torch.empty(gm.proj_shape(D), device="cuda")
    loss = torch.zeros(1, device="cuda", dtype=torch.float64)
    x_o = np.zeros(c.shape + (K,)); v_o = np.zeros_like(x_o)
    for it in range(4):
        # look-ahead point c + m v (torch only moves memory here: a copy and the library's own axpy)
        look.copy_(x); mm.mm_axpy(look, v, -mom)
        mm.mm_loss_gradient(gm, dB, look, K, dd, None, grad, loss, wr)
        mm.mm_laplacian(gm, look, K, l1); mm.mm_laplacian(gm, l1, K, l2)
        mm.mm_axpy(grad, l2, -mu_lap); mm.mm_axpy(grad, look, -mu_l2)
        mm.mm_nesterov_step(x, v, grad, eta, mom)
        look_o = (x_o + np.float32(mom) * v_o).astype(np.float32)
        L_o, g_o, _ = ora.loss_gradient(go, B, look_o, data, None, form="scatter")
        g_o = g_o + np.float32(mu_lap) * ora.laplacian_regulariser(look_o)[1] + np.float32(mu_l2) * ora.l2_regulariser(look_o)[1]
        x_o, v_o = ora.nesterov_step(x_o, v_o, g_o, np.float32(eta), np.float32(mom))
        assert abs(loss.item() - L_o) <= TOL_LOSS * abs(L_o)
        if it == 0:
            assert einf(grad.cpu().numpy()[..., :K], g_o) <= TOL
    assert einf(x.cpu().numpy()[..., :K], x_o) <= 1e-4 and einf(v.cpu().numpy()[..., :K], v_o) <= 1e-4


@pytest.mark.parametrize("weights", ["uniform", None])
def test_huber_loss_gradient(ora, mm, weights):
    """NEXT-4 (reading S23): Huber-regressor loss, clipped weighted residual and gradient; a threshold
    that clips about a third of the residuals, and a huge one that must reproduce mm_loss_gradient bit for bit."""
    import torch
    cfg, c = cfg_case("C3", (20, 18, 22), (25, 24), 2, seed=51, joff=True, weights=weights)
    go, gm = c.geoms(ora, mm)
    K, ldk, D = c.K, c.ldk, c.D
    B = mm.mm_basis_sh_matrix(gm, cfg.ell_max, *synth.segments(D))
    model = ora.forward(go, B, c.vol[..., :K])
    scale = float(np.abs(model).max())
    data = (model + 0.05 * scale * c.data).astype(np.float32)
    delta = 0.05 * scale                                            # |noise| > delta for ~32 % of the samples
    dB, dvol, dd = dev(B), dev(c.vol), dev(data)
    dw = None if c.w is None else dev(c.w)
    grad = torch.full(gm.vol_shape(ldk), float("nan"), device="cuda")
    wr = torch.empty(gm.proj_shape(D), device="cuda")
    loss = torch.zeros(1, device="cuda", dtype=torch.float64)
    mm.mm_loss_gradient_huber(gm, dB, dvol, K, dd, dw, delta, grad, loss, wr)
    L, g_o, wpsi = ora.huber_loss_gradient(go, B, c.vol[..., :K], data, delta, c.w, form="scatter")
    clipped = np.isclose(np.abs(wpsi), delta * (1.0 if c.w is None else c.w))
    assert 0.15 < clipped.mean() < 0.5
    assert abs(loss.item() - L) <= TOL_LOSS * L
    assert np.abs(wr.cpu().numpy() - wpsi).max() / scale <= TOL
    got = grad.cpu().numpy()
    assert einf(got[..., :K], g_o) <= TOL and np.all(got[..., K:] == 0.0)
    g2, wr2, loss2 = torch.empty_like(grad), torch.empty_like(wr), torch.zeros_like(loss)
    mm.mm_loss_gradient_huber(gm, dB, dvol, K, dd, dw, 1e30, grad, loss, wr)
    mm.mm_loss_gradient(gm, dB, dvol, K, dd, dw, g2, loss2, wr2)
    assert torch.equal(grad, g2) and torch.equal(wr, wr2) and abs(loss.item() - loss2.item()) <= 1e-12 * loss2.item()


@pytest.mark.parametrize("name,shape", [("C3", (14, 12, 16)), ("C1", (9, 11, 7))])
def test_derived_quantities(ora, mm, name, shape):
    """NEXT-4 (Eq. 10-12): mean, second-moment tensor, eigen-decomposition and FA of an SH volume.
    Eigenvectors are unique only up to sign and only where the eigenvalue is isolated: compared as |v.v_ref| there,
    and checked to be valid (M v = lambda v, unit length) everywhere."""
    import torch
    cfg = synth.get_config(name, shape=shape, det=(8, 8), n_rot=2)
    K, ldk = cfg.K, synth.ldk_for(cfg.K)
    vol = synth.make_volume(cfg, ldk)
    vol[..., K:] = 7.0                                                 # pad channels must be ignored
    vol[0, 0, 0, :K] = 0.0                                             # an empty voxel: M = 0, FA = 0
    vol[1, 1, 1, :K] = 0.0; vol[1, 1, 1, 0] = 2.0                      # an isotropic voxel: degenerate eigenvalues
    # an exactly fibre-symmetric voxel about an oblique axis n: c_2m = Y_2m(n) (closed forms, 4pi-normalised) gives
    # M = a I + b n n^T, a repeated eigenvalue whose plane contains no coordinate axis
    nx, ny, nz = 0.48, -0.6, 0.64
    s15, s5 = math.sqrt(15.0), math.sqrt(5.0)
    vol[2, 2, 2, :K] = 0.0; vol[2, 2, 2, 0] = 1.0
    vol[2, 2, 2, 1:6] = [s15 * nx * ny, s15 * ny * nz, 0.5 * s5 * (3 * nz * nz - 1), s15 * nx * nz, 0.5 * s15 * (nx * nx - ny * ny)]
    gm = mm.Geometry(cfg.shape, cfg.det, [0.0], [0.0])
    mean = torch.empty(cfg.shape, device="cuda"); fa = torch.empty(cfg.shape, device="cuda")
    mom = torch.empty(cfg.shape + (6,), device="cuda"); eig = torch.empty(cfg.shape + (3,), device="cuda")
    vec = torch.empty(cfg.shape + (3, 3), device="cuda")
    mm.mm_derived_quantities(gm, dev(vol), K, mean, mom, eig, vec, fa)
    d = ora.derived_quantities(vol[..., :K], cfg.ell_max)
    scale = float(np.abs(d["M"]).max())
    assert np.abs(mean.cpu().numpy() - d["mean"]).max() <= TOL * np.abs(d["mean"]).max()
    m = mom.cpu().numpy()
    Mg = np.stack([np.stack([m[..., 0], m[..., 3], m[..., 4]], -1), np.stack([m[..., 3], m[..., 1], m[..., 5]], -1),
                   np.stack([m[..., 4], m[..., 5], m[..., 2]], -1)], -2)
    assert np.abs(Mg - d["M"]).max() <= TOL * scale
    e = eig.cpu().numpy()
    assert np.abs(e - d["eig"]).max() <= TOL * scale
    v = vec.cpu().numpy().astype(np.float64)
    assert np.abs(np.linalg.norm(v, axis=-1) - 1.0).max() < 1e-5
    gram = np.einsum("...ij,...kj->...ik", v, v)
    assert np.abs(gram - np.eye(3)).max() < 1e-5                          # an orthonormal frame at every voxel, degenerate or not
    assert np.abs(np.abs(v[2, 2, 2] @ np.array([nx, ny, nz])) - np.array([1.0, 0.0, 0.0])).max() < 1e-5   # fibre axis first, the rest orthogonal
    resid = np.einsum("...ij,...kj->...ki", d["M"], v) - d["eig"][..., :, None] * v
    assert np.abs(resid).max() <= 1e-4 * scale                          # valid eigenvectors everywhere
    g01, g12 = np.abs(d["eig"][..., 0] - d["eig"][..., 1]), np.abs(d["eig"][..., 1] - d["eig"][..., 2])
    isolated = [g01 > 1e-2 * scale, np.minimum(g01, g12) > 1e-2 * scale, g12 > 1e-2 * scale]
    filled = np.abs(d["eig"]).max(axis=-1) > 1e-3 * scale
    assert filled.any() and isolated[0][filled].mean() > 0.5      # axially symmetric synthetic ODFs: main axis isolated
    for i in range(3):
        if isolated[i].any():
            assert np.abs(np.abs(np.sum(v[..., i, :] * d["vec"][..., i, :], axis=-1))[isolated[i]] - 1.0).max() < 1e-3
    big = np.abs(d["eig"]).max(axis=-1) > 1e-3 * scale
    assert np.abs(fa.cpu().numpy() - d["fa"])[big].max() <= 1e-4
    assert fa[0, 0, 0].item() == 0.0 and abs(fa[1, 1, 1].item()) < 1e-6


@pytest.mark.parametrize("K,ldk,shape", [(6, 8, (13, 11, 15)), (5, 5, (7, 1, 9)), (45, 48, (10, 12, 8))])
def test_l1_huber_tv_regularisers(ora, mm, K, ldk, shape):
    """NEXT-3 (reading S24): value and gradient of L1Norm, HuberNorm and TotalVariation."""
    import torch
    gm = mm.Geometry(shape, (4, 4), [0.0], [0.0])
    v = np.random.default_rng(K).standard_normal(shape + (ldk,)).astype(np.float32)
    dv = dev(v)
    for kind, fn in [(mm.MM_REG_L1, lambda c: ora.l1_regulariser(c)), (mm.MM_REG_HUBER, lambda c: ora.huber_norm_regulariser(c, 0.4)),
                     (mm.MM_REG_TV, lambda c: ora.total_variation_regulariser(c, 0.4))]:
        grad = torch.full(gm.vol_shape(ldk), float("nan"), device="cuda")
        val = torch.full((1,), float("nan"), device="cuda", dtype=torch.float64)
        mm.mm_regulariser(gm, kind, dv, K, 0.4, grad, val)
        R, g_o = fn(v[..., :K])
        got = grad.cpu().numpy()
        assert abs(val.item() - R) <= 1e-5 * R
        assert np.abs(got[..., :K] - g_o).max() <= 2e-5 * max(1.0, np.abs(g_o).max()) and np.all(got[..., K:] == 0.0)


@pytest.mark.parametrize("momentum,mu_lap,mu_l2,check_every", [(0.0, 0.0, 0.0, 1), (0.7, 1e-3, 1e-4, 1), (0.5, 0.0, 2e-4, 3)])
def test_device_resident_iteration_with_stop_rule(ora, mm, momentum, mu_lap, mu_l2, check_every):
    """NEXT-3: mm_iterate = the whole regularised Nesterov loop on the device with the relative-change stop rule
    (reading S25) against the oracle's `iterate`: same stop iteration, same loss history,
    same iterate; pad channels untouched; nothing but a 4-byte flag crosses the bus inside the loop."""
    import torch
    cfg, c = cfg_case("C2", (18, 16, 20), (22, 21), 3, seed=61, weights="mask")
    go, gm = c.geoms(ora, mm)
    K, ldk, D = c.K, c.ldk, c.D
    B = mm.mm_basis_sh_matrix(gm, cfg.ell_max, *synth.segments(D))
    data = synth.poisson_data(ora.forward(go, B, c.vol[..., :K]), cfg.counts, cfg.seed)
    absB = np.abs(B)
    lip = float(ora.forward(go, absB, np.ones(c.shape + (K,), np.float32)).max() *
                ora.adjoint(go, absB, np.ones((c.P,) + c.det + (D,)), form="scatter").max())
    mu_lap, mu_l2 = mu_lap * lip, mu_l2 * lip
    eta = 1.0 / (lip + 144.0 * mu_lap + mu_l2)
    max_iter = 30
    start = np.zeros(c.shape + (K,), np.float32)
    # tolerance placed between two consecutive relative changes of the (oracle) loss history, so that the rule must fire
    # at a known check well inside the budget and no fp32-vs-fp64 difference can flip the decision
    _, _, L_all = ora.iterate(go, B, data, c.w, start, eta, momentum, mu_lap, mu_l2, max_iter, 0.0)
    rel = [abs(a - b) / b for a, b in zip(L_all[:-1], L_all[1:])]         # rel[k-1] is what the check after iteration k sees
    k_stop = next(k for k in range(12, max_iter) if (k + 1) % check_every == 0)
    tol = math.sqrt(rel[k_stop - 1] * rel[k_stop - 2])
    assert rel[k_stop - 1] < 0.99 * tol and all(r > 1.01 * tol for r in rel[:k_stop - 1])
    c_o, v_o, L_o = ora.iterate(go, B, data, c.w, start, eta, momentum, mu_lap, mu_l2, max_iter, tol, check_every=check_every)
    assert len(L_o) == k_stop + 1
    x = torch.zeros(gm.vol_shape(ldk), device="cuda"); v = torch.zeros_like(x)
    x[..., K:] = 7.0                                                      # pad channels: ignored and left alone
    losses = torch.full((max_iter,), float("nan"), device="cuda", dtype=torch.float64)
    n0 = mm.mm_launch_count()
    n = mm.mm_iterate(gm, dev(B), K, dev(data), dev(c.w), x, v, losses, eta, momentum, mu_lap, mu_l2, max_iter, tol, check_every)
    torch.cuda.synchronize()
    assert n == len(L_o)
    got = losses.cpu().numpy()
    assert np.all(np.isnan(got[n:])) and np.abs(got[:n] - np.array(L_o)).max() <= TOL_LOSS * max(L_o)
    assert einf(x.cpu().numpy()[..., :K], c_o) <= 1e-4 and einf(v.cpu().numpy()[..., :K], v_o) <= 1e-4
    assert torch.all(x[..., K:] == 7.0).item() and torch.all(v[..., K:] == 0.0).item()
    assert mm.mm_launch_count() - n0 >= 5 * n                            # kernels ran; the loop is the library's
    # tol <= 0: runs max_iter iterations without a single synchronisation
    x2 = torch.zeros_like(x); v2 = torch.zeros_like(x)
    l6 = torch.full((6,), float("nan"), device="cuda", dtype=torch.float64)
    assert mm.mm_iterate(gm, dev(B), K, dev(data), dev(c.w), x2, v2, l6, eta, momentum, mu_lap, mu_l2, 6, 0.0, 1) == 6
    _, _, L6 = ora.iterate(go, B, data, c.w, np.zeros(c.shape + (K,), np.float32), eta, momentum, mu_lap, mu_l2, 6, 0.0)
    torch.cuda.synchronize()
    assert np.abs(l6.cpu().numpy() - np.array(L6)).max() <= TOL_LOSS * max(L6)


@pytest.mark.parametrize("kind,K,n_keep", [("nn", 162, None), ("nn", 50, None), ("gk", 50, 2), ("gk", 18, 1), ("sh", 45, 3)])
def test_sparse_forward_and_gradient(ora, mm, kind, K, n_keep):
    """NEXT-2 (reading S26): the forward model and the fused gradient with a sparse reciprocal-space map —
    an NN basis as it is (K = 162, 50: Table V's sizes) or a GK / SH basis thresholded to n_keep coefficients per
    segment — against the oracle with the same sparse matrix, and against the library's dense calls."""
    import torch
    r = np.random.default_rng(K + (n_keep or 0))
    P, D = 9, 8
    ldk = synth.ldk_for(K)
    c = Case((17, 15, 19), (21, 20), r.uniform(0, 2 * math.pi, P), r.uniform(-0.7, 0.7, P), K, ldk, D, seed=K,
             joff=r.uniform(-1, 1, P), koff=r.uniform(-1, 1, P))
    go, gm = c.geoms(ora, mm)
    if kind == "sh":
        B = mm.mm_basis_sh_matrix(gm, 8, *synth.segments(D))
    else:
        B = mm.mm_basis_grid_matrix(gm, mm.MM_BASIS_GK if kind == "gk" else mm.MM_BASIS_NN, synth.grid_directions(K),
                                    *synth.segments(D), sigma=0.3, n_quad=8)
    if n_keep is not None:
        B = mm.mm_basis_sparsify(B, n_keep)
        assert np.array_equal(B, ora.sparsify_basis(B, n_keep)) and ((B != 0).sum(axis=1) <= n_keep).all()
    plan = mm.SparsePlan(gm, B)
    assert plan.max_active < K and plan.max_active <= D * (n_keep or 8)
    dB, dvol = dev(B), dev(c.vol)
    model = torch.full(gm.proj_shape(D), float("nan"), device="cuda")
    launches = mm.mm_launch_count()
    mm.mm_forward_sparse(gm, plan, dB, dvol, K, model)
    launches = mm.mm_launch_count() - launches
    # <= 32 active channels: the march on channel-planar copies (transposes + march); more: the record-layout kernel
    assert launches >= 2 if plan.max_active <= 32 else launches == 1
    want_model = ora.forward(go, B, c.vol[..., :K])
    scale = float(np.abs(want_model).max())
    assert einf(model.cpu().numpy(), want_model) <= TOL
    dense = torch.empty_like(model)
    mm.mm_forward(gm, dB, dvol, K, dense)
    assert einf(dense.cpu().numpy(), model.cpu().numpy()) <= 2e-6
    data = (want_model + 0.05 * scale * c.data).astype(np.float32)
    grad = torch.full(gm.vol_shape(ldk), float("nan"), device="cuda")
    loss = torch.full((1,), float("nan"), device="cuda", dtype=torch.float64)
    wr = torch.full(gm.proj_shape(D), float("nan"), device="cuda")
    mm.mm_loss_gradient_sparse(gm, plan, dB, dvol, K, dev(data), dev(c.w), grad, loss, wr)
    L, g_o, wr_o = ora.loss_gradient(go, B, c.vol[..., :K], data, c.w, form="scatter")
    got = grad.cpu().numpy()
    assert np.abs(wr.cpu().numpy() - wr_o).max() / scale <= TOL and abs(loss.item() - L) <= TOL_LOSS * L
    assert einf(got[..., :K], g_o) <= TOL and np.all(got[..., K:] == 0.0)


def test_sparse_planar_all_major_axes(ora, mm):
    """the channel-planar sparse march with all three major axes in one geometry (tilts up to 63 degrees make y the
    major axis of some projections: copy Z marched along y, besides x on copy Z and z on copy X), a ragged detector
    (tiles of 32 x 4 rays with tails) and non-cubic volume"""
    import torch
    r = np.random.default_rng(77)
    K, D, P = 50, 8, 14
    ldk = synth.ldk_for(K)
    tilts = np.concatenate([r.uniform(-1.1, 1.1, P - 4), [1.05, -1.0, 0.0, 0.79]])
    c = Case((13, 18, 11), (37, 9), r.uniform(0, 2 * math.pi, P), tilts, K, ldk, D, seed=78,
             joff=r.uniform(-1, 1, P), koff=r.uniform(-1, 1, P))
    go, gm = c.geoms(ora, mm)
    majors = {go.get(s)[3] for s in range(P)}
    assert majors == {0, 1, 2}
    B = mm.mm_basis_grid_matrix(gm, mm.MM_BASIS_NN, synth.grid_directions(K), *synth.segments(D), sigma=0.3, n_quad=8)
    plan = mm.SparsePlan(gm, B)
    assert plan.max_active <= 32
    dB, dvol = dev(B), dev(c.vol)
    model = torch.full(gm.proj_shape(D), float("nan"), device="cuda")
    launches = mm.mm_launch_count()
    mm.mm_forward_sparse(gm, plan, dB, dvol, K, model)
    assert mm.mm_launch_count() - launches == 3                       # two transposes + the march
    want = ora.forward(go, B, c.vol[..., :K])
    assert einf(model.cpu().numpy(), want) <= TOL
    data = (want + 0.05 * float(np.abs(want).max()) * c.data).astype(np.float32)
    grad = torch.full(gm.vol_shape(ldk), float("nan"), device="cuda")
    loss = torch.full((1,), float("nan"), device="cuda", dtype=torch.float64)
    wr = torch.full(gm.proj_shape(D), float("nan"), device="cuda")
    mm.mm_loss_gradient_sparse(gm, plan, dB, dvol, K, dev(data), dev(c.w), grad, loss, wr)
    L, g_o, wr_o = ora.loss_gradient(go, B, c.vol[..., :K], data, c.w, form="scatter")
    assert np.abs(wr.cpu().numpy() - wr_o).max() / float(np.abs(want).max()) <= TOL and abs(loss.item() - L) <= TOL_LOSS * L
    assert einf(grad.cpu().numpy()[..., :K], g_o) <= TOL


def test_boundary_errors_and_workspace_release(ora, mm):
    """robustness at the boundary: unsupported channel strides are refused (not half-written), the scratch pool can be
    released and refills, and the result after a release is bit-identical."""
    import torch
    gm = mm.Geometry((8, 8, 8), (8, 8), [0.2, 1.0], [0.0, 0.3])
    big = torch.zeros(gm.vol_shape(260), device="cuda")
    with pytest.raises(mm.MMError, match="not supported"):
        mm.mm_john_forward(gm, big, 200, torch.zeros(gm.proj_shape(260), device="cuda"))
    cfg, c = cfg_case("C3", (12, 10, 14), (15, 17), 2, seed=71)
    go, gm = c.geoms(ora, mm)
    B = dev(mm.mm_basis_sh_matrix(gm, cfg.ell_max, *synth.segments(c.D)))
    data = dev(synth.surrogate_model(cfg))
    out = []
    for rep in range(2):
        grad = torch.full(gm.vol_shape(c.ldk), float("nan"), device="cuda")
        loss = torch.zeros(1, device="cuda", dtype=torch.float64)
        wr = torch.empty(gm.proj_shape(c.D), device="cuda")
        mm.mm_loss_gradient(gm, B, dev(c.vol), c.K, data, dev(c.w), grad, loss, wr)     # ldk = 48: pooled copy + pooled operand tiles
        torch.cuda.synchronize()
        out.append((grad.clone(), wr.clone()))
        mm.mm_workspace_release()
    assert torch.equal(out[0][0], out[1][0]) and torch.equal(out[0][1], out[1][1]) and not torch.isnan(out[0][0]).any().item()
