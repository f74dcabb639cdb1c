"""Thin Python binding of the C ABI in include/mm.h (ctypes; argument marshalling only).

Every function here has the name of the C entry point it calls and does nothing but check tensor
shapes/dtypes/devices, pass `data_ptr()`s and the current CUDA stream, and turn a non-zero mm_status into an
exception.  All arithmetic of the method runs in the CUDA kernels of libmm.so; there is no CPU fallback:
if the library is missing, `load()` raises.  PyTorch is used only to own device memory and streams.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("MM_LIB_PATH") or os.path.join(_HERE, "libmm.so")     # MM_LIB_PATH: an alternative build (kernel experiments)
_lib = None

SYMBOLS = ["mm_geometry_create", "mm_geometry_destroy", "mm_geometry_get", "mm_basis_sh_matrix", "mm_basis_sh_matrix_2theta", "mm_basis_grid_matrix",
           "mm_john_forward", "mm_john_adjoint", "mm_basis_forward", "mm_basis_adjoint", "mm_forward",
           "mm_adjoint", "mm_adjoint_noalloc", "mm_john_backproject", "mm_backproject", "mm_loss_gradient", "mm_loss_gradient_huber", "mm_residual_loss", "mm_reciprocal",
           "mm_axpy_precond", "mm_basis_sparsify", "mm_sparse_plan_create", "mm_sparse_plan_destroy", "mm_sparse_plan_info", "mm_forward_sparse", "mm_loss_gradient_sparse", "mm_iterate", "mm_workspace_release", "mm_laplacian", "mm_regulariser", "mm_nesterov_step", "mm_derived_quantities", "mm_axpy", "mm_loss_gradient_host", "mm_host_workspace_release", "mm_launch_count", "mm_set_phase_event",
           "mm_status_string", "mm_last_error"]


class MMError(RuntimeError):
    pass


class _Desc(ctypes.Structure):
    _fields_ = [("volume_shape", ctypes.c_int32 * 3), ("det_shape", ctypes.c_int32 * 2), ("n_proj", ctypes.c_int32),
                ("rotations", ctypes.POINTER(ctypes.c_double)), ("tilts", ctypes.POINTER(ctypes.c_double)),
                ("j_offsets", ctypes.POINTER(ctypes.c_double)), ("k_offsets", ctypes.POINTER(ctypes.c_double)),
                ("p_dir", ctypes.c_double * 3), ("j_dir", ctypes.c_double * 3), ("k_dir", ctypes.c_double * 3),
                ("q0_dir", ctypes.c_double * 3), ("q90_dir", ctypes.c_double * 3),
                ("inner_axis", ctypes.c_double * 3), ("outer_axis", ctypes.c_double * 3),
                ("voxel_size", ctypes.c_double), ("pixel_size", ctypes.c_double)]


class _IterParams(ctypes.Structure):
    _fields_ = [("eta", ctypes.c_float), ("momentum", ctypes.c_float), ("mu_laplacian", ctypes.c_float), ("mu_l2", ctypes.c_float),
                ("max_iter", ctypes.c_int32), ("check_every", ctypes.c_int32), ("tol", ctypes.c_double)]


def load():
    """dlopen libmm.so (built by `python -m paper_2504_16446_b200.build`).  Raises if it is not there."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise MMError(f"{LIB_PATH} not found: build it with `python -m paper_2504_16446_b200.build` "
                      "(there is no CPU fallback)")
    L = ctypes.CDLL(LIB_PATH)
    vp, i32, i64, dp = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.POINTER(ctypes.c_double)
    L.mm_geometry_create.argtypes = [ctypes.POINTER(_Desc), ctypes.POINTER(vp)]
    L.mm_geometry_destroy.argtypes = [vp]
    L.mm_geometry_get.argtypes = [vp, i32, dp, dp, dp, ctypes.POINTER(i32), dp]
    L.mm_basis_sh_matrix.argtypes = [vp, i32, i32, dp, dp, vp]
    L.mm_basis_sh_matrix_2theta.argtypes = [vp, i32, ctypes.c_double, i32, dp, dp, vp]
    L.mm_basis_grid_matrix.argtypes = [vp, i32, i32, dp, ctypes.c_double, i32, dp, dp, i32, vp]
    L.mm_john_forward.argtypes = [vp, vp, i32, i32, vp, vp]
    L.mm_john_adjoint.argtypes = [vp, vp, i32, i32, vp, vp]
    L.mm_basis_forward.argtypes = [vp, vp, vp, i32, i32, i32, vp, vp]
    L.mm_basis_adjoint.argtypes = [vp, vp, vp, i32, i32, i32, vp, vp]
    L.mm_forward.argtypes = [vp, vp, vp, i32, i32, i32, vp, vp]
    L.mm_adjoint.argtypes = [vp, vp, vp, i32, i32, i32, vp, vp]
    L.mm_adjoint_noalloc.argtypes = [vp, vp, vp, i32, i32, i32, vp, vp]
    L.mm_john_backproject.argtypes = [vp, vp, i32, i32, vp, vp]
    L.mm_backproject.argtypes = [vp, vp, vp, i32, i32, i32, vp, vp]
    L.mm_loss_gradient.argtypes = [vp, vp, vp, i32, i32, i32, vp, vp, vp, vp, vp, vp]
    L.mm_axpy.argtypes = [vp, vp, ctypes.c_float, i64, vp]
    L.mm_residual_loss.argtypes = [vp, vp, vp, i32, i32, i32, vp, vp, vp, vp, vp]
    L.mm_loss_gradient_huber.argtypes = [vp, vp, vp, i32, i32, i32, vp, vp, ctypes.c_float, vp, vp, vp, vp]
    L.mm_reciprocal.argtypes = [vp, i64, ctypes.c_float, vp]
    L.mm_laplacian.argtypes = [vp, vp, i32, i32, vp, vp]
    L.mm_regulariser.argtypes = [vp, i32, vp, i32, i32, ctypes.c_float, vp, vp, vp]
    L.mm_derived_quantities.argtypes = [vp, vp, i32, i32, vp, vp, vp, vp, vp, vp]
    L.mm_nesterov_step.argtypes = [vp, vp, vp, ctypes.c_float, ctypes.c_float, i64, vp]
    L.mm_axpy_precond.argtypes = [vp, vp, vp, ctypes.c_float, i64, vp]
    L.mm_loss_gradient_host.argtypes = [vp, vp, vp, i32, i32, i32, vp, vp, vp, vp]
    L.mm_host_workspace_release.argtypes = []
    L.mm_workspace_release.argtypes = []
    L.mm_basis_sparsify.argtypes = [vp, i32, i32, i32, i32, vp]
    L.mm_sparse_plan_create.argtypes = [vp, vp, i32, i32, ctypes.POINTER(vp)]
    L.mm_sparse_plan_destroy.argtypes = [vp]
    L.mm_sparse_plan_info.argtypes = [vp, ctypes.POINTER(i32), dp, vp]
    L.mm_forward_sparse.argtypes = [vp, vp, vp, vp, i32, i32, i32, vp, vp]
    L.mm_loss_gradient_sparse.argtypes = [vp, vp, vp, vp, i32, i32, i32, vp, vp, vp, vp, vp, vp]
    L.mm_iterate.argtypes = [vp, vp, i32, i32, i32, vp, vp, ctypes.POINTER(_IterParams), vp, vp, vp, ctypes.POINTER(i32), vp]
    L.mm_set_phase_event.argtypes = [vp]
    L.mm_launch_count.restype = i64
    L.mm_launch_count.argtypes = []
    L.mm_status_string.restype = ctypes.c_char_p
    L.mm_status_string.argtypes = [ctypes.c_int]
    L.mm_last_error.restype = ctypes.c_char_p
    L.mm_last_error.argtypes = []
    for name in SYMBOLS:
        if name not in ("mm_launch_count", "mm_status_string", "mm_last_error"):
            getattr(L, name).restype = ctypes.c_int
    _lib = L
    return L


def _check(status: int, who: str):
    if status != 0:
        L = load()
        raise MMError(f"{who}: {L.mm_status_string(status).decode()}: {L.mm_last_error().decode()}")


def _stream(stream):
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))


def _dev(t, shape, who, dtype=None):
    import torch
    dtype = dtype or torch.float32
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise MMError(f"{who}: expected a contiguous CUDA {dtype} tensor")
    if tuple(t.shape) != tuple(shape):
        raise MMError(f"{who}: expected shape {tuple(shape)}, got {tuple(t.shape)}")
    return ctypes.c_void_p(t.data_ptr())


class Geometry:
    """Owner of an mm_geometry handle (mm_geometry_create / mm_geometry_destroy)."""

    def __init__(self, volume_shape, det_shape, rotations, tilts, j_offsets=None, k_offsets=None, vecs=None,
                 voxel_size=0.0, pixel_size=0.0):
        L = load()
        self.shape = tuple(int(v) for v in volume_shape)
        self.det = tuple(int(v) for v in det_shape)
        rot = np.ascontiguousarray(rotations, dtype=np.float64)
        tilt = np.ascontiguousarray(tilts, dtype=np.float64)
        self.P = int(rot.size)
        d = _Desc()
        d.volume_shape[:] = self.shape
        d.det_shape[:] = self.det
        d.n_proj = self.P
        dp = ctypes.POINTER(ctypes.c_double)
        keep = [rot, tilt]
        d.rotations = rot.ctypes.data_as(dp)
        d.tilts = tilt.ctypes.data_as(dp)
        for name, arr in (("j_offsets", j_offsets), ("k_offsets", k_offsets)):
            if arr is not None:
                a = np.ascontiguousarray(arr, dtype=np.float64)
                keep.append(a)
                setattr(d, name, a.ctypes.data_as(dp))
        for key, fld in (("p", "p_dir"), ("j", "j_dir"), ("k", "k_dir"), ("q0", "q0_dir"), ("q90", "q90_dir"),
                         ("inner_axis", "inner_axis"), ("outer_axis", "outer_axis")):
            if vecs and key in vecs:
                getattr(d, fld)[:] = [float(x) for x in vecs[key]]
        d.voxel_size, d.pixel_size = float(voxel_size), float(pixel_size)
        h = ctypes.c_void_p()
        _check(L.mm_geometry_create(ctypes.byref(d), ctypes.byref(h)), "mm_geometry_create")
        self._h = h

    def __del__(self):
        if getattr(self, "_h", None) is not None and _lib is not None:
            _lib.mm_geometry_destroy(self._h)
            self._h = None

    def get(self, s):
        d, js, ks = np.zeros(3), np.zeros(3), np.zeros(3)
        m, w = ctypes.c_int32(), ctypes.c_double()
        dp = ctypes.POINTER(ctypes.c_double)
        _check(load().mm_geometry_get(self._h, int(s), d.ctypes.data_as(dp), js.ctypes.data_as(dp),
                                      ks.ctypes.data_as(dp), ctypes.byref(m), ctypes.byref(w)), "mm_geometry_get")
        return d, js, ks, m.value, w.value

    def vol_shape(self, ldk):
        return self.shape + (int(ldk),)

    def proj_shape(self, ldk):
        return (self.P,) + self.det + (int(ldk),)


def mm_basis_sh_matrix(g: Geometry, ell_max: int, seg_start, seg_end, two_theta: float | None = None) -> np.ndarray:
    """host helper: B[P][K][D] float32 (numpy); two_theta (radians) selects mm_basis_sh_matrix_2theta."""
    s0 = np.ascontiguousarray(seg_start, dtype=np.float64)
    s1 = np.ascontiguousarray(seg_end, dtype=np.float64)
    D = int(s0.size)
    K = (ell_max + 1) * (ell_max + 2) // 2
    out = np.empty((g.P, K, D), dtype=np.float32)
    dp = ctypes.POINTER(ctypes.c_double)
    if two_theta is None:
        _check(load().mm_basis_sh_matrix(g._h, int(ell_max), D, s0.ctypes.data_as(dp), s1.ctypes.data_as(dp),
                                         ctypes.c_void_p(out.ctypes.data)), "mm_basis_sh_matrix")
    else:
        _check(load().mm_basis_sh_matrix_2theta(g._h, int(ell_max), float(two_theta), D, s0.ctypes.data_as(dp),
                                                s1.ctypes.data_as(dp), ctypes.c_void_p(out.ctypes.data)),
               "mm_basis_sh_matrix_2theta")
    return out


MM_BASIS_NN, MM_BASIS_GK = 1, 2


def mm_basis_grid_matrix(g: Geometry, kind: int, dirs, seg_start, seg_end, sigma: float = 0.0, n_quad: int = 16) -> np.ndarray:
    """host helper: B[P][n_dirs][D] float32 (numpy) for the NN / GK basis set on the grid directions dirs[n][3]."""
    d = np.ascontiguousarray(dirs, dtype=np.float64).reshape(-1, 3)
    s0 = np.ascontiguousarray(seg_start, dtype=np.float64)
    s1 = np.ascontiguousarray(seg_end, dtype=np.float64)
    out = np.empty((g.P, d.shape[0], s0.size), dtype=np.float32)
    dp = ctypes.POINTER(ctypes.c_double)
    _check(load().mm_basis_grid_matrix(g._h, int(kind), d.shape[0], d.ctypes.data_as(dp), float(sigma), int(s0.size),
                                       s0.ctypes.data_as(dp), s1.ctypes.data_as(dp), int(n_quad),
                                       ctypes.c_void_p(out.ctypes.data)), "mm_basis_grid_matrix")
    return out


def mm_john_forward(g: Geometry, vol, K: int, proj, stream=None):
    ldk = vol.shape[-1]
    _check(load().mm_john_forward(g._h, _dev(vol, g.vol_shape(ldk), "vol"), K, ldk,
                                  _dev(proj, g.proj_shape(ldk), "proj"), _stream(stream)), "mm_john_forward")
    return proj


def mm_john_adjoint(g: Geometry, proj, K: int, vol_out, stream=None):
    ldk = proj.shape[-1]
    _check(load().mm_john_adjoint(g._h, _dev(proj, g.proj_shape(ldk), "proj"), K, ldk,
                                  _dev(vol_out, g.vol_shape(ldk), "vol_out"), _stream(stream)), "mm_john_adjoint")
    return vol_out


def mm_basis_forward(g: Geometry, B, proj, K: int, sino, stream=None):
    ldk, D = proj.shape[-1], B.shape[-1]
    _check(load().mm_basis_forward(g._h, _dev(B, (g.P, K, D), "B"), _dev(proj, g.proj_shape(ldk), "proj"), K, ldk, D,
                                   _dev(sino, g.proj_shape(D), "sino"), _stream(stream)), "mm_basis_forward")
    return sino


def mm_basis_adjoint(g: Geometry, B, sino, K: int, proj, stream=None):
    ldk, D = proj.shape[-1], B.shape[-1]
    _check(load().mm_basis_adjoint(g._h, _dev(B, (g.P, K, D), "B"), _dev(sino, g.proj_shape(D), "sino"), K, ldk, D,
                                   _dev(proj, g.proj_shape(ldk), "proj"), _stream(stream)), "mm_basis_adjoint")
    return proj


def mm_forward(g: Geometry, B, vol, K: int, sino, stream=None):
    ldk, D = vol.shape[-1], B.shape[-1]
    _check(load().mm_forward(g._h, _dev(B, (g.P, K, D), "B"), _dev(vol, g.vol_shape(ldk), "vol"), K, ldk, D,
                             _dev(sino, g.proj_shape(D), "sino"), _stream(stream)), "mm_forward")
    return sino


def mm_adjoint(g: Geometry, B, sino, K: int, vol_out, stream=None):
    ldk, D = vol_out.shape[-1], B.shape[-1]
    _check(load().mm_adjoint(g._h, _dev(B, (g.P, K, D), "B"), _dev(sino, g.proj_shape(D), "sino"), K, ldk, D,
                             _dev(vol_out, g.vol_shape(ldk), "vol_out"), _stream(stream)), "mm_adjoint")
    return vol_out


ADJOINT_NOALLOC_MAX_BYTES = 4 << 20            # MM_ADJOINT_NOALLOC_MAX_BYTES of include/mm.h


def mm_adjoint_noalloc(g: Geometry, B, sino, K: int, vol_out, stream=None):
    """mm_adjoint without any allocation: operand scratch in the library's static device array (include/mm.h)."""
    ldk, D = vol_out.shape[-1], B.shape[-1]
    _check(load().mm_adjoint_noalloc(g._h, _dev(B, (g.P, K, D), "B"), _dev(sino, g.proj_shape(D), "sino"), K, ldk, D,
                                     _dev(vol_out, g.vol_shape(ldk), "vol_out"), _stream(stream)), "mm_adjoint_noalloc")
    return vol_out


def mm_john_backproject(g: Geometry, proj, K: int, vol_out, stream=None):
    ldk = proj.shape[-1]
    _check(load().mm_john_backproject(g._h, _dev(proj, g.proj_shape(ldk), "proj"), K, ldk,
                                      _dev(vol_out, g.vol_shape(ldk), "vol_out"), _stream(stream)), "mm_john_backproject")
    return vol_out


def mm_backproject(g: Geometry, B, sino, K: int, vol_out, stream=None):
    ldk, D = vol_out.shape[-1], B.shape[-1]
    _check(load().mm_backproject(g._h, _dev(B, (g.P, K, D), "B"), _dev(sino, g.proj_shape(D), "sino"), K, ldk, D,
                                 _dev(vol_out, g.vol_shape(ldk), "vol_out"), _stream(stream)), "mm_backproject")
    return vol_out


def mm_loss_gradient(g: Geometry, B, vol, K: int, data, weights, grad, loss, wr_workspace, stream=None):
    """loss: CUDA float64 tensor with one element (device scalar, overwritten)."""
    import torch
    ldk, D = vol.shape[-1], B.shape[-1]
    w = ctypes.c_void_p(None) if weights is None else _dev(weights, g.proj_shape(D), "weights")
    _check(load().mm_loss_gradient(g._h, _dev(B, (g.P, K, D), "B"), _dev(vol, g.vol_shape(ldk), "vol"), K, ldk, D,
                                   _dev(data, g.proj_shape(D), "data"), w, _dev(grad, g.vol_shape(ldk), "grad"),
                                   _dev(loss, (1,), "loss", torch.float64),
                                   _dev(wr_workspace, g.proj_shape(D), "wr_workspace"), _stream(stream)),
           "mm_loss_gradient")
    return grad, loss


def mm_loss_gradient_huber(g: Geometry, B, vol, K: int, data, weights, delta: float, grad, loss, wr_workspace, stream=None):
    import torch
    ldk, D = vol.shape[-1], B.shape[-1]
    w = ctypes.c_void_p(None) if weights is None else _dev(weights, g.proj_shape(D), "weights")
    _check(load().mm_loss_gradient_huber(g._h, _dev(B, (g.P, K, D), "B"), _dev(vol, g.vol_shape(ldk), "vol"), K, ldk, D,
                                         _dev(data, g.proj_shape(D), "data"), w, float(delta),
                                         _dev(grad, g.vol_shape(ldk), "grad"), _dev(loss, (1,), "loss", torch.float64),
                                         _dev(wr_workspace, g.proj_shape(D), "wr_workspace"), _stream(stream)),
           "mm_loss_gradient_huber")
    return grad, loss


def mm_residual_loss(g: Geometry, B, vol, K: int, data, weights, wr, loss, stream=None):
    import torch
    ldk, D = vol.shape[-1], B.shape[-1]
    w = ctypes.c_void_p(None) if weights is None else _dev(weights, g.proj_shape(D), "weights")
    _check(load().mm_residual_loss(g._h, _dev(B, (g.P, K, D), "B"), _dev(vol, g.vol_shape(ldk), "vol"), K, ldk, D,
                                   _dev(data, g.proj_shape(D), "data"), w, _dev(wr, g.proj_shape(D), "wr"),
                                   _dev(loss, (1,), "loss", torch.float64), _stream(stream)), "mm_residual_loss")
    return wr, loss


def mm_reciprocal(x, floor: float, stream=None):
    _check(load().mm_reciprocal(_dev(x, x.shape, "x"), x.numel(), float(floor), _stream(stream)), "mm_reciprocal")
    return x


def mm_axpy_precond(c, grad, pre, eta: float, stream=None):
    _check(load().mm_axpy_precond(_dev(c, c.shape, "c"), _dev(grad, c.shape, "grad"), _dev(pre, c.shape, "pre"), float(eta),
                                  c.numel(), _stream(stream)), "mm_axpy_precond")
    return c


def mm_laplacian(g: Geometry, vol, K: int, vol_out, stream=None):
    ldk = vol.shape[-1]
    _check(load().mm_laplacian(g._h, _dev(vol, g.vol_shape(ldk), "vol"), K, ldk, _dev(vol_out, g.vol_shape(ldk), "vol_out"),
                               _stream(stream)), "mm_laplacian")
    return vol_out


def mm_derived_quantities(g: Geometry, vol, K: int, mean=None, moments=None, eigenvalues=None, eigenvectors=None, fa=None,
                          stream=None):
    ldk = vol.shape[-1]
    n = g.shape
    opt = lambda t, shp, who: ctypes.c_void_p(None) if t is None else _dev(t, shp, who)
    _check(load().mm_derived_quantities(g._h, _dev(vol, g.vol_shape(ldk), "vol"), K, ldk, opt(mean, n, "mean"),
                                        opt(moments, n + (6,), "moments"), opt(eigenvalues, n + (3,), "eigenvalues"),
                                        opt(eigenvectors, n + (3, 3), "eigenvectors"), opt(fa, n, "fa"), _stream(stream)),
           "mm_derived_quantities")


MM_REG_L1, MM_REG_HUBER, MM_REG_TV = 1, 2, 3


def mm_regulariser(g: Geometry, kind: int, vol, K: int, delta: float, grad_out, value=None, stream=None):
    """value: CUDA float64 tensor with one element (overwritten) or None."""
    import torch
    ldk = vol.shape[-1]
    v = ctypes.c_void_p(None) if value is None else _dev(value, (1,), "value", torch.float64)
    _check(load().mm_regulariser(g._h, int(kind), _dev(vol, g.vol_shape(ldk), "vol"), K, ldk, float(delta),
                                 _dev(grad_out, g.vol_shape(ldk), "grad_out"), v, _stream(stream)), "mm_regulariser")
    return grad_out


def mm_nesterov_step(c, v, grad, eta: float, momentum: float, stream=None):
    _check(load().mm_nesterov_step(_dev(c, c.shape, "c"), _dev(v, c.shape, "v"), _dev(grad, c.shape, "grad"), float(eta),
                                   float(momentum), c.numel(), _stream(stream)), "mm_nesterov_step")
    return c, v


def mm_basis_sparsify(h_B, n_keep: int) -> np.ndarray:
    """host helper: keep the n_keep largest |B[s][i][c]| of every (s, c) column, zero the rest (reading S26)."""
    B = np.ascontiguousarray(h_B, dtype=np.float32)
    out = np.empty_like(B)
    P, K, D = B.shape
    _check(load().mm_basis_sparsify(ctypes.c_void_p(B.ctypes.data), P, K, D, int(n_keep), ctypes.c_void_p(out.ctypes.data)), "mm_basis_sparsify")
    return out


class SparsePlan:
    """Owner of an mm_sparse_plan handle: the per-projection lists of channels with a non-zero row of the HOST matrix h_B."""

    def __init__(self, g: Geometry, h_B):
        B = np.ascontiguousarray(h_B, dtype=np.float32)
        assert B.shape[0] == g.P
        self.K, self.D = int(B.shape[1]), int(B.shape[2])
        h = ctypes.c_void_p()
        _check(load().mm_sparse_plan_create(g._h, ctypes.c_void_p(B.ctypes.data), self.K, self.D, ctypes.byref(h)), "mm_sparse_plan_create")
        self._h = h
        mx, mean = ctypes.c_int32(), ctypes.c_double()
        self.counts = np.zeros(g.P, dtype=np.int32)
        _check(load().mm_sparse_plan_info(self._h, ctypes.byref(mx), ctypes.byref(mean), ctypes.c_void_p(self.counts.ctypes.data)), "mm_sparse_plan_info")
        self.max_active, self.mean_active = mx.value, mean.value

    def __del__(self):
        if getattr(self, "_h", None) is not None and _lib is not None:
            _lib.mm_sparse_plan_destroy(self._h)
            self._h = None


def mm_forward_sparse(g: Geometry, plan: SparsePlan, B, vol, K: int, sino, stream=None):
    ldk, D = vol.shape[-1], B.shape[-1]
    _check(load().mm_forward_sparse(g._h, plan._h, _dev(B, (g.P, K, D), "B"), _dev(vol, g.vol_shape(ldk), "vol"), K, ldk, D,
                                    _dev(sino, g.proj_shape(D), "sino"), _stream(stream)), "mm_forward_sparse")
    return sino


def mm_loss_gradient_sparse(g: Geometry, plan: SparsePlan, B, vol, K: int, data, weights, grad, loss, wr_workspace, stream=None):
    import torch
    ldk, D = vol.shape[-1], B.shape[-1]
    w = ctypes.c_void_p(None) if weights is None else _dev(weights, g.proj_shape(D), "weights")
    _check(load().mm_loss_gradient_sparse(g._h, plan._h, _dev(B, (g.P, K, D), "B"), _dev(vol, g.vol_shape(ldk), "vol"), K, ldk, D,
                                          _dev(data, g.proj_shape(D), "data"), w, _dev(grad, g.vol_shape(ldk), "grad"),
                                          _dev(loss, (1,), "loss", torch.float64),
                                          _dev(wr_workspace, g.proj_shape(D), "wr_workspace"), _stream(stream)), "mm_loss_gradient_sparse")
    return grad, loss


def mm_iterate(g: Geometry, B, K: int, data, weights, c, v, losses, eta: float, momentum: float = 0.0, mu_laplacian: float = 0.0,
               mu_l2: float = 0.0, max_iter: int = 20, tol: float = 0.0, check_every: int = 1, stream=None) -> int:
    """device-resident regularised Nesterov iteration; c, v in/out, losses: CUDA float64 [max_iter]; returns n_iter."""
    import torch
    ldk, D = c.shape[-1], B.shape[-1]
    w = ctypes.c_void_p(None) if weights is None else _dev(weights, g.proj_shape(D), "weights")
    p = _IterParams(float(eta), float(momentum), float(mu_laplacian), float(mu_l2), int(max_iter), int(check_every), float(tol))
    n = ctypes.c_int32(0)
    _check(load().mm_iterate(g._h, _dev(B, (g.P, K, D), "B"), K, ldk, D, _dev(data, g.proj_shape(D), "data"), w, ctypes.byref(p),
                             _dev(c, g.vol_shape(ldk), "c"), _dev(v, g.vol_shape(ldk), "v"),
                             _dev(losses, (int(max_iter),), "losses", torch.float64), ctypes.byref(n), _stream(stream)), "mm_iterate")
    return n.value


def mm_workspace_release():
    """Return the library's cached device memory (host-call arena and stream-ordered scratch pool) to the driver."""
    _check(load().mm_workspace_release(), "mm_workspace_release")


def mm_axpy(c, grad, eta: float, stream=None):
    n = c.numel()
    _check(load().mm_axpy(_dev(c, c.shape, "c"), _dev(grad, c.shape, "grad"), float(eta), n, _stream(stream)), "mm_axpy")
    return c


def _host(a, shape, who):
    """numpy float32 C-contiguous array or CPU torch tensor -> pointer"""
    if hasattr(a, "data_ptr"):
        if a.is_cuda or not a.is_contiguous() or str(a.dtype) != "torch.float32" or tuple(a.shape) != tuple(shape):
            raise MMError(f"{who}: expected a contiguous CPU float32 tensor of shape {tuple(shape)}")
        return ctypes.c_void_p(a.data_ptr())
    if not (isinstance(a, np.ndarray) and a.dtype == np.float32 and a.flags.c_contiguous and a.shape == tuple(shape)):
        raise MMError(f"{who}: expected a C-contiguous float32 array of shape {tuple(shape)}")
    return ctypes.c_void_p(a.ctypes.data)


def mm_host_workspace_release():
    """Free the library-owned device workspace of mm_loss_gradient_host (it is kept between calls)."""
    _check(load().mm_host_workspace_release(), "mm_host_workspace_release")


def mm_loss_gradient_host(g: Geometry, h_B, h_vol, K: int, h_data, h_weights, h_grad):
    """HOST buffers in, HOST gradient out (written into h_grad); returns the loss as a Python float."""
    ldk, D = h_vol.shape[-1], h_B.shape[-1]
    loss = ctypes.c_double(0.0)
    w = ctypes.c_void_p(None) if h_weights is None else _host(h_weights, g.proj_shape(D), "h_weights")
    _check(load().mm_loss_gradient_host(g._h, _host(h_B, (g.P, K, D), "h_B"), _host(h_vol, g.vol_shape(ldk), "h_vol"),
                                        K, ldk, D, _host(h_data, g.proj_shape(D), "h_data"), w,
                                        _host(h_grad, g.vol_shape(ldk), "h_grad"),
                                        ctypes.cast(ctypes.byref(loss), ctypes.c_void_p)), "mm_loss_gradient_host")
    return loss.value


def mm_launch_count() -> int:
    return int(load().mm_launch_count())


def mm_set_phase_event(event=None):
    """event: a torch.cuda.Event(enable_timing=True) that has been recorded once (so its handle exists), or None."""
    h = None if event is None else int(event.cuda_event)
    _check(load().mm_set_phase_event(ctypes.c_void_p(h)), "mm_set_phase_event")
