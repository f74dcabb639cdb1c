"""Seeded synthetic inputs for the tensor-tomography hot path.

This module is the ONLY code shared by the CUDA path's callers (tests, bench.py) and the oracle's callers.
It holds no step of the method itself (no John transform, no basis matrix, no loss): it only draws the
arrays both sides consume — angles, volumes of SH coefficients, weights, noisy data from a caller-supplied
model sinogram.  The band-limited ODF recipe needs real spherical harmonics of the fibre axis; the small
evaluator below is private to the input recipe and is imported by neither `oracle/` nor the CUDA library.

The paper's only workload is the public trabecular-bone data set (247 x 65 x 55 x 8,
PAPER.md:354) which is not available here; BASELINE.json's five configs stand in for it.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace

import numpy as np

__all__ = ["Config", "CONFIGS", "get_config", "angles", "segments", "n_coeffs", "make_volume",
           "make_weights", "poisson_data", "surrogate_model", "pad_channels", "ldk_for", "grid_directions"]


@dataclass(frozen=True)
class Config:
    name: str
    shape: tuple            # (X, Y, Z)
    ell_max: int
    tilts_deg: tuple        # outer angles beta
    n_rot: int              # rotations per tilt
    det: tuple              # (J, Kd)
    D: int
    counts: float = 1e3
    field_kind: str = "smooth"      # smooth | voronoi
    density: str = "ball"           # ball | plate | ellipsoids
    weights: str = "unit"           # unit | mask5 | uniform
    seed: int = 1000
    gd_iters: int = 1

    @property
    def K(self):
        return n_coeffs(self.ell_max)

    @property
    def P(self):
        return len(self.tilts_deg) * self.n_rot

    @property
    def n_voxels(self):
        return self.shape[0] * self.shape[1] * self.shape[2]

    @property
    def vcp(self):
        """voxel-channel-projections N*K*P: the unit of BASELINE.json's throughput metric."""
        return self.n_voxels * self.K * self.P


def n_coeffs(ell_max: int) -> int:
    return (ell_max + 1) * (ell_max + 2) // 2


def ldk_for(K: int) -> int:
    """channel stride (floats) used by the fast paths: next multiple of 4, or of 8 (32-byte lanes) from K > 20."""
    return (K + 7) // 8 * 8 if K > 20 else (K + 3) // 4 * 4


CONFIGS = {
    "C1": Config("C1", (32, 32, 32), 2, (0.0,), 60, (32, 32), 8, 1e3, seed=1001),
    "C2": Config("C2", (64, 64, 64), 4, (0.0, 9.0, 18.0, 27.0, 36.0, 45.0), 40, (64, 64), 8, 1e3,
                 weights="mask5", seed=1002),
    "C3": Config("C3", (100, 100, 100), 8, tuple(45.0 * t / 7 for t in range(8)), 40, (100, 100), 8, 1e3,
                 field_kind="voronoi", seed=1003),
    "C4": Config("C4", (80, 160, 160), 6, tuple(5.0 * t for t in range(10)), 50, (160, 160), 16, 1e3,
                 density="plate", weights="uniform", seed=1004, gd_iters=20),
    "C5": Config("C5", (256, 256, 256), 8, tuple(5.625 * t for t in range(9)), 40, (256, 256), 8, 1e4,
                 density="ellipsoids", seed=1005),
}


def get_config(name: str, shape=None, det=None, n_rot=None, tilts_deg=None) -> Config:
    """A BASELINE.json config, optionally shrunk (same recipe, smaller grid) for oracle-sized tests."""
    c = CONFIGS[name]
    kw = {}
    if shape is not None:
        kw["shape"] = tuple(shape)
    if det is not None:
        kw["det"] = tuple(det)
    if n_rot is not None:
        kw["n_rot"] = int(n_rot)
    if tilts_deg is not None:
        kw["tilts_deg"] = tuple(tilts_deg)
    return replace(c, **kw) if kw else c


def angles(cfg: Config):
    """(rotations alpha_s, tilts beta_s) in radians, [P] float64.  Rotations are uniform in [0,180) at
    tilt 0 and in [0,360) at tilt > 0 (BASELINE.json configs 2-5); s = tilt-major, rotation-minor."""
    rot, tilt = [], []
    for b in cfg.tilts_deg:
        span = 180.0 if b == 0.0 else 360.0
        for i in range(cfg.n_rot):
            rot.append(span * i / cfg.n_rot)
            tilt.append(b)
    return np.deg2rad(np.array(rot, dtype=np.float64)), np.deg2rad(np.array(tilt, dtype=np.float64))


def segments(D: int):
    """D azimuthal segments tiling [0, pi) (SAXS: 180 degrees): start, end in radians."""
    c = np.arange(D, dtype=np.float64)
    return c * math.pi / D, (c + 1) * math.pi / D


# ----------------------------------------------------------------------------------------------
# private helpers of the input recipe
# ----------------------------------------------------------------------------------------------
def _gauss_filter_periodic(a: np.ndarray, sigma: float) -> np.ndarray:
    """separable periodic Gaussian filter via FFT (float64 in, float64 out)."""
    f = np.fft.rfftn(a)
    for ax, n in enumerate(a.shape):
        k = np.fft.rfftfreq(n) if ax == a.ndim - 1 else np.fft.fftfreq(n)
        g = np.exp(-2.0 * (math.pi * sigma * k) ** 2)
        sh = [1] * a.ndim
        sh[ax] = g.size
        f *= g.reshape(sh)
    return np.fft.irfftn(f, s=a.shape)


def _real_sh_even(n: np.ndarray, ell_max: int, scale_l) -> np.ndarray:
    """[..., K] float32: scale_l[l] * Y_lm(n) for even l <= ell_max, order l ascending, m = -l..l,
    4pi-normalised real harmonics (m<0 ~ sin|m|phi, m>0 ~ cos m phi).  Input-recipe use only."""
    x, y, z = n[..., 0], n[..., 1], n[..., 2]
    out = np.empty(n.shape[:-1] + (n_coeffs(ell_max),), dtype=np.float32)
    # A_m + i B_m = (x + i y)^m
    A = [np.ones_like(x)]
    Bm = [np.zeros_like(x)]
    for m in range(1, ell_max + 1):
        A.append(A[-1] * x - Bm[-1] * y)
        Bm.append(Bm[-1] * x + A[-2] * y)
    col = {}
    idx = 0
    for l in range(0, ell_max + 1, 2):
        for m in range(-l, l + 1):
            col[(l, m)] = idx
            idx += 1
    for m in range(0, ell_max + 1):
        # Pt_l^m(z) = d^m/dz^m P_l(z), upward recurrence in l
        pmm = 1.0
        for i in range(1, m + 1):
            pmm *= (2 * i - 1)
        p_prev = np.full_like(z, pmm)          # l = m
        p_cur = (2 * m + 1) * z * p_prev       # l = m+1
        for l in range(m, ell_max + 1):
            if l == m:
                pl = p_prev
            elif l == m + 1:
                pl = p_cur
            else:
                pl = ((2 * l - 1) * z * p_cur - (l + m - 1) * p_prev) / (l - m)
                p_prev, p_cur = p_cur, pl
            if l % 2:
                continue
            norm = math.sqrt((2 * l + 1) * math.factorial(l - m) / math.factorial(l + m)) * scale_l[l]
            if m == 0:
                out[..., col[(l, 0)]] = norm * pl
            else:
                out[..., col[(l, m)]] = (math.sqrt(2.0) * norm) * pl * A[m]
                out[..., col[(l, -m)]] = (math.sqrt(2.0) * norm) * pl * Bm[m]
    return out


def _orientation(cfg: Config, rng: np.random.Generator) -> np.ndarray:
    shape = cfg.shape
    sigma = max(shape) / 8.0
    noise = np.stack([_gauss_filter_periodic(rng.standard_normal(shape), sigma) for _ in range(3)], axis=-1)
    noise /= max(float(np.sqrt((noise ** 2).sum(-1).mean())), 1e-30)       # unit rms length
    if cfg.field_kind == "voronoi":
        seeds = rng.uniform(0.0, 1.0, size=(4, 3)) * np.array(shape)
        axes = rng.standard_normal((4, 3))
        axes /= np.linalg.norm(axes, axis=1, keepdims=True)
        gx, gy, gz = np.meshgrid(*[np.arange(n, dtype=np.float64) for n in shape], indexing="ij")
        d2 = np.stack([(gx - s[0]) ** 2 + (gy - s[1]) ** 2 + (gz - s[2]) ** 2 for s in seeds], axis=-1)
        cell = d2.argmin(-1)
        vec = axes[cell] + 0.3 * noise
    else:
        vec = noise
    nrm = np.linalg.norm(vec, axis=-1, keepdims=True)
    vec = np.where(nrm > 1e-12, vec / np.maximum(nrm, 1e-12), np.array([0.0, 0.0, 1.0]))
    return vec


def _density(cfg: Config, rng: np.random.Generator) -> np.ndarray:
    X, Y, Z = cfg.shape
    gx, gy, gz = np.meshgrid(np.arange(X) - (X - 1) / 2, np.arange(Y) - (Y - 1) / 2,
                             np.arange(Z) - (Z - 1) / 2, indexing="ij")
    if cfg.density == "ball":
        rho = rng.uniform(0.0, 1.0, size=cfg.shape)
        rho[gx ** 2 + gy ** 2 + gz ** 2 > (0.45 * min(cfg.shape)) ** 2] = 0.0
    elif cfg.density == "plate":
        rho = rng.uniform(0.0, 1.0, size=cfg.shape)
        rho[rng.uniform(size=cfg.shape) < 0.10] = 0.0
    elif cfg.density == "ellipsoids":
        rho = np.zeros(cfg.shape, dtype=np.float64)
        n = float(min(cfg.shape))
        for _ in range(50):
            ctr = rng.uniform(-0.3, 0.3, size=3) * np.array(cfg.shape)
            semi = rng.uniform(0.05, 0.2, size=3) * n
            q, _r = np.linalg.qr(rng.standard_normal((3, 3)))
            amp = rng.uniform(0.2, 1.0)
            px, py, pz = gx - ctr[0], gy - ctr[1], gz - ctr[2]
            u = (q[0, 0] * px + q[1, 0] * py + q[2, 0] * pz) / semi[0]
            v = (q[0, 1] * px + q[1, 1] * py + q[2, 1] * pz) / semi[1]
            w = (q[0, 2] * px + q[1, 2] * py + q[2, 2] * pz) / semi[2]
            rho += amp * ((u * u + v * v + w * w) <= 1.0)
        np.clip(rho, 0.0, 1.0, out=rho)
    else:
        raise ValueError(cfg.density)
    return rho


def make_volume(cfg: Config, ldk: int | None = None) -> np.ndarray:
    """Coefficient volume c[X][Y][Z][ldk] float32 (pad channels zero): c_lm(x) = rho(x) a_l Y_lm(n(x)),
    a_l = exp(-0.1 l(l+1)) — a band-limited ODF peaked on the fibre axis n(x) (BASELINE.json configs)."""
    rng = np.random.Generator(np.random.PCG64(cfg.seed))
    n = _orientation(cfg, rng)                      # draw order: orientation noise -> density
    rho = _density(cfg, rng)
    a_l = {l: math.exp(-0.1 * l * (l + 1)) for l in range(0, cfg.ell_max + 1)}
    K = cfg.K
    ldk = K if ldk is None else ldk
    vol = np.zeros(cfg.shape + (ldk,), dtype=np.float32)
    X = cfg.shape[0]
    step = max(1, (1 << 21) // (cfg.shape[1] * cfg.shape[2]))       # chunk over x to bound temporaries
    for x0 in range(0, X, step):
        sl = slice(x0, min(X, x0 + step))
        y = _real_sh_even(n[sl], cfg.ell_max, a_l)
        vol[sl, :, :, :K] = y * rho[sl][..., None].astype(np.float32)
    return vol


def make_weights(cfg: Config) -> np.ndarray:
    """weights[P][J][Kd][D] float32: unit, 5% of pixels (s,j,k) masked, or U[0.5,1.5] per pixel."""
    rng = np.random.Generator(np.random.PCG64(cfg.seed + 500))
    shp = (cfg.P,) + tuple(cfg.det)
    if cfg.weights == "unit":
        w = np.ones(shp, dtype=np.float32)
    elif cfg.weights == "mask5":
        w = (rng.uniform(size=shp) >= 0.05).astype(np.float32)
    elif cfg.weights == "uniform":
        w = rng.uniform(0.5, 1.5, size=shp).astype(np.float32)
    else:
        raise ValueError(cfg.weights)
    return np.ascontiguousarray(np.broadcast_to(w[..., None], shp + (cfg.D,)))


def poisson_data(model: np.ndarray, counts: float, seed: int) -> np.ndarray:
    """data = Poisson(s * max(model,0)) / s with s = counts / mean(model[model>0]); float32, same shape.
    `model` is a caller-supplied noise-free sinogram (who computes it is the caller's business)."""
    rng = np.random.Generator(np.random.PCG64(seed + 900))
    m = np.maximum(np.asarray(model, dtype=np.float64), 0.0)
    pos = m[m > 0]
    s = counts / float(pos.mean()) if pos.size else 1.0
    return (rng.poisson(m * s) / s).astype(np.float32)


def surrogate_model(cfg: Config, level: float = 1.0) -> np.ndarray:
    """A forward-model-free positive, smooth model sinogram [P][J][Kd][D] (float32) for full-size parity
    runs whose data must not come from either implementation: a raised-cosine 'shadow' of the sample on
    the detector times a per-segment azimuthal modulation.  Pure arithmetic on index grids."""
    J, Kd = cfg.det
    jj = (np.arange(J) - (J - 1) / 2) / (0.5 * J)
    kk = (np.arange(Kd) - (Kd - 1) / 2) / (0.5 * Kd)
    r2 = jj[:, None] ** 2 + kk[None, :] ** 2
    shadow = np.sqrt(np.maximum(0.81 - r2, 0.0)).astype(np.float32)
    s = np.arange(cfg.P, dtype=np.float32)
    c = np.arange(cfg.D, dtype=np.float32)
    mod = 1.0 + 0.3 * np.cos(2.0 * (math.pi * (c[None, :] + 0.5) / cfg.D - 0.05 * s[:, None]))
    out = level * shadow[None, :, :, None] * mod[:, None, None, :].astype(np.float32)
    return np.ascontiguousarray(out, dtype=np.float32)


def grid_directions(n: int) -> np.ndarray:
    """n unit vectors spread over the upper half sphere (Fibonacci spiral) — a stand-in for the orientation grid
    that defines an NN or GK basis set (the grid is an input of the method)."""
    i = np.arange(n) + 0.5
    z = i / n
    ph = i * math.pi * (3.0 - math.sqrt(5.0))
    rr = np.sqrt(1.0 - z * z)
    return np.stack([rr * np.cos(ph), rr * np.sin(ph), z], axis=1)


def pad_channels(a: np.ndarray, ldk: int) -> np.ndarray:
    """zero-pad the last axis to ldk."""
    if a.shape[-1] == ldk:
        return np.ascontiguousarray(a)
    out = np.zeros(a.shape[:-1] + (ldk,), dtype=a.dtype)
    out[..., : a.shape[-1]] = a
    return out
