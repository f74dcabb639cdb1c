"""oracle/oracle.py — CPU ORACLE of the tensor-tomography gradient path.  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` legs may import this.
It shares no code with the CUDA library and never imports the package's binding.

What is here (numpy, fp64) and what it follows:
  real_sh / sh_index   real spherical harmonics, textbook definition                PAPER.md:236-238, reading S14
  q_hat                small-angle scattering direction, Eq. 1 second line
  basis_matrix         segment average B_{sc,i}, Eq. 3, Gauss-Legendre quadrature
  basis_forward/adjoint Eq. 6 reciprocal-space map and its transpose
  forward / adjoint    A = (basis map) o (John transform), Eq. 6-8, and A^T
  loss_gradient        r = Ac - I (Eq. 13), L = 1/2 sum w r^2, grad = A^T (w r)     PAPER.md:101, 324, readings S10, S11
  john_backproject_bilinear / backproject_bilinear  the paper's own unmatched adjoint  PAPER.md:314 (NEXT-1)
  basis_matrix_grid    NN indicator / GK Gaussian-kernel basis sets on a grid of orientations   PAPER.md:240-246 (NEXT-2)
  laplacian / laplacian_regulariser / l2_regulariser / nesterov_step   regularisers, momentum   PAPER.md:336-340 (NEXT-3)
  iterate              regularised Nesterov iteration with the relative-change stop rule   PAPER.md:262-264, 270-272 (NEXT-3, reading S25)
  sparsify_basis       sparse approximation of the reciprocal-space map   PAPER.md:274 (NEXT-2, reading S26)
  l1_regulariser / huber_norm_regulariser / total_variation_regulariser   PAPER.md:336-338 (NEXT-3, reading S24)
  derived_quantities   mean, second-moment tensor, eigen-decomposition, FA   PAPER.md:198-224, Eq. 10-12 (NEXT-4)
  huber_loss_gradient  Huber-regressor loss and its gradient   PAPER.md:334 (NEXT-4, reading S23)
  sirt_preconditioners / sirt_step   SIRT/MITRA as preconditioned weighted least squares  PAPER.md:258-262, reading S19
The John transform itself (Joseph's method) is oracle/ora.c, loaded with ctypes.

Pins: tests/test_oracle_sh.py, tests/test_oracle_john.py, tests/test_oracle_model.py (all CPU).
"""
from __future__ import annotations

import ctypes
import math
import os
import subprocess

import numpy as np
from numpy.polynomial import legendre as _leg

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libora.so")
_lib = None

STANDARD_VECS = {            # Table I, PAPER.md:27-37 (row 2 garbled: reading S1, j = +y, k = +x)
    "p": (0.0, 0.0, 1.0), "j": (0.0, 1.0, 0.0), "k": (1.0, 0.0, 0.0),
    "q0": (1.0, 0.0, 0.0), "q90": (0.0, 1.0, 0.0),
    "inner_axis": (0.0, 1.0, 0.0), "outer_axis": (1.0, 0.0, 0.0),
}


def build(force: bool = False) -> str:
    """compile oracle/ora.c -> oracle/libora.so (gcc -O2, OpenMP on the embarrassingly parallel loops)."""
    src = os.path.join(_HERE, "ora.c")
    if force or not os.path.exists(_LIB_PATH) or os.path.getmtime(_LIB_PATH) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-o", _LIB_PATH, src, "-lm"])
    return _LIB_PATH


def _load():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB_PATH)
        dp, fp, ip = (ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_float), ctypes.POINTER(ctypes.c_int32))
        L.ora_geom_create.restype = ctypes.c_void_p
        L.ora_geom_create.argtypes = [ctypes.c_int] * 6 + [dp, dp, dp, dp, dp, ctypes.c_double, ctypes.c_double]
        L.ora_geom_destroy.argtypes = [ctypes.c_void_p]
        L.ora_geom_get.argtypes = [ctypes.c_void_p, ctypes.c_int, dp, dp, dp, ctypes.POINTER(ctypes.c_int), dp]
        L.ora_john_forward.argtypes = [ctypes.c_void_p, fp, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, dp, ctypes.c_int]
        L.ora_john_forward_rays.argtypes = [ctypes.c_void_p, fp, ctypes.c_int, ctypes.c_int, ctypes.c_long, ip, dp, ctypes.c_int]
        L.ora_john_adjoint_scatter.argtypes = [ctypes.c_void_p, dp, ctypes.c_int, dp]
        L.ora_john_adjoint_gather.argtypes = [ctypes.c_void_p, dp, ctypes.c_int, dp, ctypes.c_int]
        L.ora_john_adjoint_voxels.argtypes = [ctypes.c_void_p, dp, ctypes.c_int, ctypes.c_long, ip, dp, ctypes.c_int]
        L.ora_voxel_taps.restype = ctypes.c_long
        L.ora_voxel_taps.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int, dp, ctypes.c_long]
        L.ora_dense_matrix.argtypes = [ctypes.c_void_p, ctypes.c_int, dp]
        L.ora_john_backproject_bilinear.argtypes = [ctypes.c_void_p, dp, ctypes.c_int, dp, ctypes.c_int]
        L.ora_john_backproject_bilinear_voxels.argtypes = [ctypes.c_void_p, dp, ctypes.c_int, ctypes.c_long, ip, dp]
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _fp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_float))


def _ip(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))


def default_threads() -> int:
    return len(os.sched_getaffinity(0))


# ------------------------------------------------------------------------------------------------
# geometry + John transform (C)
# ------------------------------------------------------------------------------------------------
class Geometry:
    """Per-projection geometry (A0).  rotations/tilts in radians; offsets in pixels; vecs overrides Table I."""

    def __init__(self, volume_shape, det_shape, rotations, tilts, j_offsets=None, k_offsets=None, vecs=None,
                 voxel_size=1.0, pixel_size=1.0):
        L = _load()
        self.shape = tuple(int(v) for v in volume_shape)
        self.det = tuple(int(v) for v in det_shape)
        self.rot = np.ascontiguousarray(rotations, dtype=np.float64)
        self.tilt = np.ascontiguousarray(tilts, dtype=np.float64)
        self.P = int(self.rot.size)
        self.joff = np.zeros(self.P) if j_offsets is None else np.ascontiguousarray(j_offsets, dtype=np.float64)
        self.koff = np.zeros(self.P) if k_offsets is None else np.ascontiguousarray(k_offsets, dtype=np.float64)
        v = dict(STANDARD_VECS)
        if vecs:
            v.update(vecs)
        self.vecs = {k: np.asarray(val, dtype=np.float64) for k, val in v.items()}
        flat = np.concatenate([self.vecs[n] for n in ("p", "j", "k", "inner_axis", "outer_axis")]).astype(np.float64)
        self.a, self.b = float(voxel_size), float(pixel_size)
        self._h = L.ora_geom_create(*self.shape, *self.det, self.P, _dp(self.rot), _dp(self.tilt), _dp(self.joff),
                                    _dp(self.koff), _dp(flat), self.a, self.b)

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.ora_geom_destroy(self._h)
            self._h = None

    def get(self, s):
        d, js, ks = np.zeros(3), np.zeros(3), np.zeros(3)
        m, w = ctypes.c_int(), ctypes.c_double()
        _load().ora_geom_get(self._h, int(s), _dp(d), _dp(js), _dp(ks), ctypes.byref(m), ctypes.byref(w))
        return d, js, ks, m.value, w.value

    def rotation_matrix(self, s):
        """R_s = R_beta(beta_s) R_alpha(alpha_s), PAPER.md:46 (numpy restatement used by the basis builder)."""
        return _rodrigues(self.vecs["outer_axis"], self.tilt[s]) @ _rodrigues(self.vecs["inner_axis"], self.rot[s])


def _rodrigues(n, theta):
    n = np.asarray(n, dtype=np.float64)
    Kx = np.array([[0, -n[2], n[1]], [n[2], 0, -n[0]], [-n[1], n[0], 0]])
    return np.eye(3) * math.cos(theta) + math.sin(theta) * Kx + (1 - math.cos(theta)) * np.outer(n, n)


def _vol32(vol, K):
    vol = np.ascontiguousarray(vol, dtype=np.float32)
    assert vol.ndim == 4 and vol.shape[3] >= K
    return vol, vol.shape[3]


def john_forward(g: Geometry, vol, K, s0=0, s1=None, threads=None):
    """proj[s1-s0][J][Kd][K] float64 = Joseph line integrals of the K-channel volume (A1)."""
    s1 = g.P if s1 is None else s1
    vol, ldk = _vol32(vol, K)
    assert vol.shape[:3] == g.shape
    out = np.empty((s1 - s0,) + g.det + (K,), dtype=np.float64)
    _load().ora_john_forward(g._h, _fp(vol), K, ldk, s0, s1, _dp(out), threads or default_threads())
    return out


def john_forward_rays(g: Geometry, vol, K, sjk, threads=None):
    vol, ldk = _vol32(vol, K)
    sjk = np.ascontiguousarray(sjk, dtype=np.int32).reshape(-1, 3)
    out = np.empty((sjk.shape[0], K), dtype=np.float64)
    _load().ora_john_forward_rays(g._h, _fp(vol), K, ldk, sjk.shape[0], _ip(sjk), _dp(out), threads or default_threads())
    return out


def john_adjoint(g: Geometry, y, form="gather", threads=None):
    """out[X][Y][Z][K] float64 = exact transpose of john_forward applied to y[P][J][Kd][K] (A2)."""
    y = np.ascontiguousarray(y, dtype=np.float64)
    K = y.shape[-1]
    assert y.shape == (g.P,) + g.det + (K,)
    out = np.empty(g.shape + (K,), dtype=np.float64)
    if form == "scatter":
        _load().ora_john_adjoint_scatter(g._h, _dp(y), K, _dp(out))
    else:
        _load().ora_john_adjoint_gather(g._h, _dp(y), K, _dp(out), threads or default_threads())
    return out


def john_backproject_bilinear(g: Geometry, y, threads=None):
    """out[X][Y][Z][K] float64: the paper's own (unmatched) adjoint, PAPER.md:314 — voxel-driven bilinear
    interpolation of the projection y[P][J][Kd][K] at the voxel's detector position, weighted by w_s (NEXT-1)."""
    y = np.ascontiguousarray(y, dtype=np.float64)
    K = y.shape[-1]
    assert y.shape == (g.P,) + g.det + (K,)
    out = np.empty(g.shape + (K,), dtype=np.float64)
    _load().ora_john_backproject_bilinear(g._h, _dp(y), K, _dp(out), threads or default_threads())
    return out


def john_backproject_bilinear_voxels(g: Geometry, y, xyz):
    """john_backproject_bilinear at sampled voxels xyz[n][3] -> [n][K]."""
    y = np.ascontiguousarray(y, dtype=np.float64)
    K = y.shape[-1]
    xyz = np.ascontiguousarray(xyz, dtype=np.int32).reshape(-1, 3)
    out = np.empty((xyz.shape[0], K), dtype=np.float64)
    _load().ora_john_backproject_bilinear_voxels(g._h, _dp(y), K, xyz.shape[0], _ip(xyz), _dp(out))
    return out


def backproject_bilinear(g: Geometry, B, sino, threads=None):
    """basis^T (Eq. 6 transposed) followed by the paper's bilinear back-projection."""
    return john_backproject_bilinear(g, basis_adjoint(B, sino), threads=threads)


def john_adjoint_voxels(g: Geometry, y, xyz, threads=None):
    y = np.ascontiguousarray(y, dtype=np.float64)
    K = y.shape[-1]
    xyz = np.ascontiguousarray(xyz, dtype=np.int32).reshape(-1, 3)
    out = np.empty((xyz.shape[0], K), dtype=np.float64)
    _load().ora_john_adjoint_voxels(g._h, _dp(y), K, xyz.shape[0], _ip(xyz), _dp(out), threads or default_threads())
    return out


def voxel_taps(g: Geometry, x, y, z):
    """rows (s, j, k, P_{sjk,xyz}) of the non-zero entries of the John matrix in the column of voxel (x,y,z)."""
    cap = 64 * g.P
    buf = np.empty((cap, 4), dtype=np.float64)
    n = _load().ora_voxel_taps(g._h, int(x), int(y), int(z), _dp(buf), cap)
    assert n <= cap
    return buf[:n].copy()


def dense_john_matrix(g: Geometry, s):
    """[J*Kd][X*Y*Z] dense P_s from the closed form Lambda*Lambda (tiny problems only)."""
    nv = g.shape[0] * g.shape[1] * g.shape[2]
    mat = np.empty((g.det[0] * g.det[1], nv), dtype=np.float64)
    _load().ora_dense_matrix(g._h, int(s), _dp(mat))
    return mat


# ------------------------------------------------------------------------------------------------
# real spherical harmonics and the segment-integrated basis matrix (numpy)
# ------------------------------------------------------------------------------------------------
def sh_index(ell_max: int):
    """[(l, m)] for even l <= ell_max, l ascending then m = -l..l (reading S14)."""
    return [(l, m) for l in range(0, ell_max + 1, 2) for m in range(-l, l + 1)]


def real_sh(l: int, m: int, n):
    """Real spherical harmonic Y_lm at unit vectors n[..., 3], 4pi-normalised (sphere mean of Y^2 = 1, Y_00 = 1),
    no Condon-Shortley phase:  Y_lm = N_l|m| P_l^|m|(cos th) * {sqrt2 cos(m ph) | 1 | sqrt2 sin(|m| ph)} for
    m > 0 | m = 0 | m < 0, with P_l^m(x) = (1-x^2)^(m/2) d^m/dx^m P_l(x), N_lm = sqrt((2l+1)(l-m)!/(l+m)!)."""
    n = np.asarray(n, dtype=np.float64)
    ct = np.clip(n[..., 2], -1.0, 1.0)
    ph = np.arctan2(n[..., 1], n[..., 0])
    am = abs(m)
    plm = (1.0 - ct * ct) ** (0.5 * am) * _leg.Legendre.basis(l).deriv(am)(ct)
    norm = math.sqrt((2 * l + 1) * math.factorial(l - am) / math.factorial(l + am))
    if m > 0:
        return math.sqrt(2.0) * norm * plm * np.cos(m * ph)
    if m < 0:
        return math.sqrt(2.0) * norm * plm * np.sin(am * ph)
    return norm * plm


def q_hat(g: Geometry, phi, two_theta=0.0):
    """lab-frame scattering direction, Eq. 1:
        q(phi) = cos(2theta/2) (cos(phi) q0 + sin(phi) q90) - sin(2theta/2) p;
    two_theta = 0 is the small-angle second line, cos(phi) q0 + sin(phi) q90 (reading S13, the SAXS default)."""
    phi = np.asarray(phi, dtype=np.float64)
    inplane = np.cos(phi)[..., None] * g.vecs["q0"] + np.sin(phi)[..., None] * g.vecs["q90"]
    return math.cos(0.5 * two_theta) * inplane - math.sin(0.5 * two_theta) * g.vecs["p"]


def basis_matrix(g: Geometry, ell_max: int, seg_start, seg_end, n_quad: int = 32, rule: str = "gauss", two_theta: float = 0.0):
    """B[P][K][D] float64: B[s][i][c] = mean over [start_c, end_c] of Y_i(R_s^T q(phi))  (Eq. 3).
    rule = 'gauss' (Gauss-Legendre, n_quad nodes), 'simpson' (composite, n_quad panels) or 'central'
    (the central-angle approximation the paper mentions)."""
    seg_start = np.asarray(seg_start, dtype=np.float64)
    seg_end = np.asarray(seg_end, dtype=np.float64)
    D = seg_start.size
    idx = sh_index(ell_max)
    B = np.zeros((g.P, len(idx), D), dtype=np.float64)
    if rule == "gauss":
        xs, ws = _leg.leggauss(n_quad)
        ws = ws / 2.0                                   # weights of the mean over [-1,1]
    elif rule == "simpson":
        xs = np.linspace(-1.0, 1.0, 2 * n_quad + 1)
        ws = np.ones_like(xs)
        ws[1:-1:2] = 4.0
        ws[2:-1:2] = 2.0
        ws /= ws.sum()
    elif rule == "central":
        xs, ws = np.zeros(1), np.ones(1)
    else:
        raise ValueError(rule)
    for s in range(g.P):
        Rt = g.rotation_matrix(s).T
        for c in range(D):
            phi = 0.5 * (seg_start[c] + seg_end[c]) + 0.5 * (seg_end[c] - seg_start[c]) * xs
            qs = q_hat(g, phi, two_theta) @ Rt.T        # rows: R_s^T q(phi)
            for i, (l, m) in enumerate(idx):
                B[s, i, c] = np.dot(ws, real_sh(l, m, qs))
    return B


def basis_forward(B, proj):
    """Imod[s,j,k,c] = sum_i B[s][i][c] proj[s,j,k,i]   (Eq. 6, inner sum)."""
    return np.einsum("sjki,sic->sjkc", np.asarray(proj, dtype=np.float64), np.asarray(B, dtype=np.float64))


def basis_adjoint(B, sino):
    """g[s,j,k,i] = sum_c B[s][i][c] sino[s,j,k,c]   (transpose of Eq. 6's inner sum)."""
    return np.einsum("sjkc,sic->sjki", np.asarray(sino, dtype=np.float64), np.asarray(B, dtype=np.float64))


# ------------------------------------------------------------------------------------------------
# forward model, adjoint, loss and gradient
# ------------------------------------------------------------------------------------------------
def forward(g: Geometry, B, vol, threads=None, chunk=16):
    """I = A c (Eq. 6-7): John transform of every coefficient channel, then the per-projection basis map."""
    B = np.asarray(B, dtype=np.float64)
    K, D = B.shape[1], B.shape[2]
    out = np.empty((g.P,) + g.det + (D,), dtype=np.float64)
    for s0 in range(0, g.P, chunk):
        s1 = min(g.P, s0 + chunk)
        out[s0:s1] = basis_forward(B[s0:s1], john_forward(g, vol, K, s0, s1, threads))
    return out


def adjoint(g: Geometry, B, sino, form="gather", threads=None):
    """A^T y = John^T (basis^T y), the exact transpose of `forward`."""
    return john_adjoint(g, basis_adjoint(B, sino), form=form, threads=threads)


def loss_gradient(g: Geometry, B, vol, data, weights=None, form="gather", threads=None, model=None):
    """r = A c - I (Eq. 13); L = 1/2 sum w r^2 (Eq. 9 with a = 2, readings S10/S11); grad = A^T (w r).
    Returns (L, grad[X][Y][Z][K], wr[P][J][Kd][D]).  `model`: forward(g, B, vol) if the caller already holds it
    (the large parity cases draw their data from it and must not pay for the forward twice)."""
    r = (forward(g, B, vol, threads) if model is None else np.asarray(model, dtype=np.float64)) - np.asarray(data, dtype=np.float64)
    w = np.ones_like(r) if weights is None else np.asarray(weights, dtype=np.float64)
    wr = w * r
    L = 0.5 * float(np.sum(wr * r))
    return L, adjoint(g, B, wr, form=form, threads=threads), wr


def forward_rays(g: Geometry, B, vol, sjk, threads=None):
    """I[s,j,k,:] for sampled rays sjk[n][3] -> [n][D]."""
    B = np.asarray(B, dtype=np.float64)
    sjk = np.asarray(sjk, dtype=np.int32).reshape(-1, 3)
    p = john_forward_rays(g, vol, B.shape[1], sjk, threads)
    return np.einsum("ni,nic->nc", p, B[sjk[:, 0]])


def gradient_voxels(g: Geometry, B, vol, data, weights, xyz, threads=None):
    """grad[x, :] of loss_gradient at sampled voxels xyz[n][3], computed from scratch one voxel at a time:
    the voxel's column of the John matrix (voxel_taps) names the rays that see it; those rays are traced,
    mapped, compared with the data, and their weighted residuals brought back through B^T and the column."""
    B = np.asarray(B, dtype=np.float64)
    xyz = np.asarray(xyz, dtype=np.int32).reshape(-1, 3)
    out = np.zeros((xyz.shape[0], B.shape[1]), dtype=np.float64)
    for q, (x, y, z) in enumerate(xyz):
        taps = voxel_taps(g, x, y, z)
        if taps.shape[0] == 0:
            continue
        sjk = taps[:, :3].astype(np.int32)
        imod = forward_rays(g, B, vol, sjk, threads)
        s, j, k = sjk[:, 0], sjk[:, 1], sjk[:, 2]
        r = imod - np.asarray(data[s, j, k], dtype=np.float64)
        wr = r if weights is None else r * np.asarray(weights[s, j, k], dtype=np.float64)
        out[q] = np.einsum("n,nic,nc->i", taps[:, 3], B[s], wr)
    return out


# ------------------------------------------------------------------------------------------------
# NEXT-1 (second half): SIRT / MITRA as preconditioned weighted least squares
# ------------------------------------------------------------------------------------------------
def sirt_preconditioners(g: Geometry, B, matched=False, floor=1e-6, threads=None):
    """(W[P][J][Kd][D], C[X][Y][Z][K]) of the SIRT/MITRA iteration ("the weight-preconditioner approach
    ... can also be extended to the RSM").  The paper gives no formula; reading S19: the classical SIRT
    choice on the entrywise absolute value of the system matrix, |A|_s = P_s (x) |B_s| (P >= 0):
        W = 1 / (|A| 1)   (inverse row sums),      C = 1 / (|A|' 1)   (inverse column sums),
    with |A|' the back-projector the iteration itself uses (exact transpose if matched, else the paper's bilinear
    one), and 0 where a sum does not exceed `floor` (rays that miss the sample, voxels no ray sees)."""
    absB = np.abs(np.asarray(B, dtype=np.float64))
    K, D = absB.shape[1], absB.shape[2]
    rows = forward(g, absB, np.ones(g.shape + (K,), dtype=np.float32), threads)
    ones = np.ones((g.P,) + g.det + (D,), dtype=np.float64)
    cols = adjoint(g, absB, ones, form="scatter") if matched else backproject_bilinear(g, absB, ones, threads)
    W = np.where(rows > floor, 1.0 / np.maximum(rows, floor), 0.0)
    C = np.where(cols > floor, 1.0 / np.maximum(cols, floor), 0.0)
    return W, C


def sirt_step(g: Geometry, B, vol, data, W, C, matched=False, threads=None):
    """one iteration  c <- c - C (.) A'( W (.) (A c - I) )  (ref. 45); returns (c_new, L) with
    L = 1/2 sum W r^2 evaluated at the incoming c."""
    r = forward(g, B, np.asarray(vol, dtype=np.float32), threads) - np.asarray(data, dtype=np.float64)
    wr = W * r
    back = adjoint(g, B, wr, form="scatter") if matched else backproject_bilinear(g, B, wr, threads)
    return np.asarray(vol, dtype=np.float64) - C * back, 0.5 * float(np.sum(wr * r))


# ------------------------------------------------------------------------------------------------
# NEXT-2: basis sets defined by a grid of orientations
# ------------------------------------------------------------------------------------------------
def basis_matrix_grid(g: Geometry, dirs, kind, seg_start, seg_end, sigma=None, n_quad=16):
    """B[P][K][D] float64 for the K basis functions attached to the unit vectors dirs[K][3] (sample frame):
      kind "nn"  nearest-neighbour indicator functions: B_i(q) = 1 if g_i is the grid direction
                 closest to the line through q (largest |q.g_i|, lowest index on ties), else 0;
      kind "gk"  Gaussian kernels ("Bunge normal distribution"): B_i(q) = exp(-theta_i^2 / (2 sigma^2)),
                 theta_i = arccos|q.g_i| the angle between the lines through q and g_i (reading S20: the RSM of
                 SAXS is even in q, so distances are between lines, not vectors).
    Eq. 3 by the midpoint rule with n_quad points per segment ("standard quadrature", PAPER.md:68;
    n_quad = 1 is the central-angle approximation of PAPER.md:316)."""
    dirs = np.asarray(dirs, dtype=np.float64)
    dirs = dirs / np.linalg.norm(dirs, axis=1, keepdims=True)
    seg_start = np.asarray(seg_start, dtype=np.float64)
    seg_end = np.asarray(seg_end, dtype=np.float64)
    K, D = dirs.shape[0], seg_start.size
    B = np.zeros((g.P, K, D), dtype=np.float64)
    t = (np.arange(n_quad) + 0.5) / n_quad
    for s in range(g.P):
        Rt = g.rotation_matrix(s).T
        for c in range(D):
            phi = seg_start[c] + (seg_end[c] - seg_start[c]) * t
            qs = q_hat(g, phi) @ Rt.T                                  # rows R_s^T q(phi)
            cosang = np.abs(qs @ dirs.T)                               # [n_quad][K]
            if kind == "nn":
                hit = np.zeros_like(cosang)
                hit[np.arange(n_quad), np.argmax(cosang, axis=1)] = 1.0
                B[s, :, c] = hit.mean(axis=0)
            elif kind == "gk":
                theta = np.arccos(np.minimum(cosang, 1.0))
                B[s, :, c] = np.exp(-theta ** 2 / (2.0 * sigma ** 2)).mean(axis=0)
            else:
                raise ValueError(kind)
    return B


# ------------------------------------------------------------------------------------------------
# NEXT-3: regulariser gradients and momentum
# ------------------------------------------------------------------------------------------------
def laplacian(vol):
    """finite-difference Laplacian of every channel of vol[X][Y][Z][K] ("finite-difference Laplacian
    operator of the tensor field"): 7-point stencil, unit spacing, neighbours outside the volume count as 0
    (reading S21: the paper does not state the boundary rule; zero padding is the one the forward model uses)."""
    v = np.asarray(vol, dtype=np.float64)
    out = -6.0 * v
    for ax in range(3):
        lo = [slice(None)] * 4
        hi = [slice(None)] * 4
        lo[ax], hi[ax] = slice(0, -1), slice(1, None)
        out[tuple(lo)] += v[tuple(hi)]
        out[tuple(hi)] += v[tuple(lo)]
    return out


def laplacian_regulariser(vol):
    """(R, grad): R = 1/2 ||Lap c||^2, grad = Lap^T Lap c = Lap(Lap c) (the zero-padded stencil is symmetric)."""
    l = laplacian(vol)
    return 0.5 * float(np.sum(l * l)), laplacian(l)


def l2_regulariser(vol):
    """(R, grad) of the L2Norm regulariser: R = 1/2 ||c||^2, grad = c."""
    v = np.asarray(vol, dtype=np.float64)
    return 0.5 * float(np.sum(v * v)), v.copy()


def nesterov_step(c, v, grad_at_lookahead, eta, momentum):
    """GradientDescent with Nesterov accelerated momentum; reading S22, the usual form:
        v <- m v - eta g(c + m v);   c <- c + v.   Returns (c_new, v_new); the caller evaluates g at c + m v."""
    v_new = momentum * np.asarray(v, dtype=np.float64) - eta * np.asarray(grad_at_lookahead, dtype=np.float64)
    return np.asarray(c, dtype=np.float64) + v_new, v_new


def iterate(g: Geometry, B, data, weights, c0, eta, momentum, mu_laplacian, mu_l2, max_iter, tol, check_every=1, threads=None):
    """A regularised gradient iteration that runs until the relative change of the loss drops below `tol`
    ("a stop criterion based on the relative change of the loss function"; PAPER.md:262 MITRA: arbitrary
    regularisers + Nesterov momentum; the asynchronous pipelines keep this loop on the GPU).
    Reading S25 (the paper gives no formulas): iteration k = 0, 1, ... evaluates everything at the look-ahead point
    y_k = c_k + m v_k (reading S22),
        L_k = 1/2 sum w r(y_k)^2 + mu_lap/2 ||Lap y_k||^2 + mu_l2/2 ||y_k||^2,      g_k = grad of that at y_k,
        v_{k+1} = m v_k - eta g_k,   c_{k+1} = c_k + v_{k+1}                           (fp32 state, as the device holds it),
    and after the update of every `check_every`-th iteration (k + 1 a multiple of check_every, k >= 1) stops if
        |L_k - L_{k-1}| <= tol |L_k|.
    Returns (c, v, [L_0 .. L_last])."""
    c = np.asarray(c0, dtype=np.float32).copy()
    v = np.zeros_like(c)
    m32, eta32 = np.float32(momentum), np.float32(eta)
    losses = []
    for k in range(int(max_iter)):
        look = (c.astype(np.float64) + float(m32) * v.astype(np.float64)).astype(np.float32)
        L, grad, _ = loss_gradient(g, B, look, data, weights, form="scatter", threads=threads)
        if mu_laplacian:
            R, gr = laplacian_regulariser(look)
            L, grad = L + float(np.float32(mu_laplacian)) * R, grad + float(np.float32(mu_laplacian)) * gr
        if mu_l2:
            R, gr = l2_regulariser(look)
            L, grad = L + float(np.float32(mu_l2)) * R, grad + float(np.float32(mu_l2)) * gr
        losses.append(L)
        c64, v64 = nesterov_step(c, v, grad, float(eta32), float(m32))
        c, v = c64.astype(np.float32), v64.astype(np.float32)
        if k >= 1 and (k + 1) % int(check_every) == 0 and abs(losses[-1] - losses[-2]) <= tol * abs(losses[-1]):
            break
    return c, v, losses


# ------------------------------------------------------------------------------------------------
# NEXT-2 (second half): sparse approximation of the reciprocal-space map
# ------------------------------------------------------------------------------------------------
def sparsify_basis(B, n_keep):
    """The "sparse approximation to the reciprocal-space mapping" of the sparse pipelines ("... such as
    only mapping one basis function to each segment").  Reading S26 (no formula in the paper): for every projection s
    and segment c keep the n_keep coefficients B[s][i][c] of largest magnitude (lowest i first among equals) and set
    the others to zero.  The sparse forward model, adjoint and gradient are `forward`, `adjoint`, `loss_gradient` with
    this matrix; n_keep >= K changes nothing."""
    B = np.asarray(B)
    P, K, D = B.shape
    n_keep = int(n_keep)
    if n_keep >= K:
        return B.copy()
    out = np.zeros_like(B)
    for s in range(P):
        for c in range(D):
            col = np.abs(B[s, :, c].astype(np.float64))
            order = sorted(range(K), key=lambda i: (-col[i], i))[:n_keep]
            for i in order:
                out[s, i, c] = B[s, i, c]
    return out


# ------------------------------------------------------------------------------------------------
# NEXT-4: robust regression, PAPER.md:334 (HuberLoss)
# ------------------------------------------------------------------------------------------------
def huber_loss_gradient(g: Geometry, B, vol, data, delta, weights=None, form="gather", threads=None):
    """Huber regressor on the residual r = A c - I (ref. 53; reading S23, the textbook form):
        rho(r) = 1/2 r^2 if |r| <= delta, else delta (|r| - delta/2);   L = sum w rho(r);
        grad = A^T (w psi(r)),  psi(r) = rho'(r) = clip(r, -delta, delta).
    Returns (L, grad[X][Y][Z][K], w psi[P][J][Kd][D])."""
    r = forward(g, B, vol, threads) - np.asarray(data, dtype=np.float64)
    w = np.ones_like(r) if weights is None else np.asarray(weights, dtype=np.float64)
    a = np.abs(r)
    rho = np.where(a <= delta, 0.5 * r * r, delta * (a - 0.5 * delta))
    wpsi = w * np.clip(r, -delta, delta)
    return float(np.sum(w * rho)), adjoint(g, B, wpsi, form=form, threads=threads), wpsi


# ------------------------------------------------------------------------------------------------
# NEXT-4: derived quantities, PAPER.md:198-224 (Eq. 10-12)
# ------------------------------------------------------------------------------------------------
def derived_quantities(coeffs, ell_max, n_theta=None):
    """For SH coefficients coeffs[..., K] (even l <= ell_max): the definitions written out on a sphere quadrature
    (Gauss-Legendre in cos(theta) x uniform phi, exact for polynomials of degree <= ell_max + 2):
        mean  = <f>_q                                   Eq. 10
        M_ij  = <q_i q_j f(q)>_q                        Eq. 11   (returned as [..., 3, 3])
        eig   = eigenvalues of M, descending; vec = their eigenvectors (rows, sign arbitrary)
        FA    = sqrt((l1-l2)^2 + (l2-l3)^2 + (l3-l1)^2) / sqrt(2 (l1^2 + l2^2 + l3^2)),  0 when M = 0     Eq. 12
    Returns dict(mean, M, eig, vec, fa)."""
    c = np.asarray(coeffs, dtype=np.float64)
    nt = n_theta or (ell_max + 4)
    xs, ws = _leg.leggauss(nt)
    nphi = 2 * (ell_max + 4)
    ph = 2.0 * math.pi * np.arange(nphi) / nphi
    st = np.sqrt(1.0 - xs * xs)
    q = np.stack([st[:, None] * np.cos(ph)[None, :], st[:, None] * np.sin(ph)[None, :], np.repeat(xs[:, None], nphi, 1)], -1)
    w = np.repeat((ws / 2.0)[:, None], nphi, 1) / nphi                 # weights of the sphere mean
    Y = np.stack([real_sh(l, m, q) for (l, m) in sh_index(ell_max)], axis=-1)      # [nt][nphi][K]
    f = np.tensordot(c, Y, axes=([-1], [-1]))                          # [..., nt, nphi]
    mean = np.tensordot(f, w, axes=([-2, -1], [0, 1]))
    M = np.einsum("...tp,tp,tpi,tpj->...ij", f, w, q, q)
    evals, evecs = np.linalg.eigh(M)
    eig = evals[..., ::-1]
    vec = np.swapaxes(evecs, -1, -2)[..., ::-1, :]
    num = np.sqrt((eig[..., 0] - eig[..., 1]) ** 2 + (eig[..., 1] - eig[..., 2]) ** 2 + (eig[..., 2] - eig[..., 0]) ** 2)
    den = np.sqrt(2.0 * np.sum(eig * eig, axis=-1))
    fa = np.where(den > 0, num / np.where(den > 0, den, 1.0), 0.0)
    return {"mean": mean, "M": M, "eig": eig, "vec": vec, "fa": fa}


def _huber(t, delta):
    """Huber function of PAPER.md:336-338 ("acts as an L1 norm for large values and an L2 norm for small values"),
    reading S24: h(t) = t^2 / (2 delta) for |t| <= delta, |t| - delta/2 beyond (slope 1 far out, C^1)."""
    a = np.abs(t)
    return np.where(a <= delta, t * t / (2.0 * delta), a - 0.5 * delta)


def l1_regulariser(vol):
    """(R, grad) of L1Norm: R = sum |c|, grad = sign(c) (0 at 0)."""
    v = np.asarray(vol, dtype=np.float64)
    return float(np.sum(np.abs(v))), np.sign(v)


def huber_norm_regulariser(vol, delta):
    """(R, grad) of HuberNorm: R = sum h(c), grad = clip(c / delta, -1, 1)."""
    v = np.asarray(vol, dtype=np.float64)
    return float(np.sum(_huber(v, delta))), np.clip(v / delta, -1.0, 1.0)


def total_variation_regulariser(vol, delta):
    """(R, grad) of TotalVariation ("the Huber norm of the spatial gradient for each basis-set mode"),
    reading S24: forward differences d_a c[x] = c[x + e_a] - c[x] (0 across the last face), per voxel and channel
    n = sqrt(sum_a (d_a c)^2), R = sum h(n); grad = D^T ( h'(n) d c / n ) with h'(n)/n = 1 / max(n, delta)."""
    v = np.asarray(vol, dtype=np.float64)
    d = np.zeros((3,) + v.shape)
    for ax in range(3):
        lo = [slice(None)] * 4
        hi = [slice(None)] * 4
        lo[ax], hi[ax] = slice(0, -1), slice(1, None)
        d[(ax,) + tuple(lo)] = v[tuple(hi)] - v[tuple(lo)]
    n = np.sqrt(np.sum(d * d, axis=0))
    R = float(np.sum(_huber(n, delta)))
    p = d / np.maximum(n, delta)
    g = np.zeros_like(v)
    for ax in range(3):
        lo = [slice(None)] * 4
        hi = [slice(None)] * 4
        lo[ax], hi[ax] = slice(0, -1), slice(1, None)
        g[tuple(lo)] -= p[(ax,) + tuple(lo)]
        g[tuple(hi)] += p[(ax,) + tuple(lo)]
    return R, g
