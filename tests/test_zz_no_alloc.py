"""GPU test of mm_adjoint_noalloc (include/mm.h): the brick adjoint with its operand scratch in a static device array.

The file sorts last on purpose (pytest -x: a failure here must not hide another test) and builds
its own inputs, so it passes alone in a fresh process as well as after the rest of the suite (which leaves the
library's scratch pool warm and the static array untouched).  The existing path, mm_adjoint, is the reference: same
kernels, same arithmetic, so the bar is the suite's E_inf <= 1e-5 and the results are expected to be identical.
"""
import numpy as np
import pytest

from paper_2504_16446_b200 import synth

pytestmark = pytest.mark.gpu

TOL = 1e-5


@pytest.fixture(scope="module")
def mm():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2504_16446_b200 import mm as binding
    binding.load()
    return binding


def _case(mm, shape, det, P, ell_max, D, seed):
    import torch
    r = np.random.default_rng(seed)
    rot = r.uniform(0.0, 2.0 * np.pi, P)
    tilt = r.uniform(0.0, np.pi / 4, P)
    gm = mm.Geometry(shape, det, rot, tilt)
    K = synth.n_coeffs(ell_max)
    ldk = synth.ldk_for(K)
    B = torch.from_numpy(mm.mm_basis_sh_matrix(gm, ell_max, *synth.segments(D))).cuda()
    sino = torch.from_numpy(r.standard_normal(gm.proj_shape(D)).astype(np.float32)).cuda()
    return gm, B, sino, K, ldk


def _both(mm, gm, B, sino, K, ldk):
    import torch
    want = torch.full(gm.vol_shape(ldk), float("nan"), device="cuda")
    got = torch.full(gm.vol_shape(ldk), float("nan"), device="cuda")
    mm.mm_adjoint(gm, B, sino, K, want)
    mm.mm_adjoint_noalloc(gm, B, sino, K, got)
    torch.cuda.synchronize()
    assert not torch.isnan(got).any().item() and not torch.isnan(want).any().item()
    err = float((got - want).abs().max() / want.abs().max())
    return err, torch.equal(got, want), got


def test_noalloc_matches_existing_path_two_calls_in_a_row(mm):
    """two different problems back to back (K = 45 / ldk 48 / D = 8, then K = 6 / ldk 8 / D = 8 on another geometry,
    then D = 16): the second call finds the first call's operand tiles in the shared array and must not use them."""
    import torch
    n0 = mm.load().mm_launch_count()
    cases = [_case(mm, (20, 18, 22), (26, 24), 21, 8, 8, seed=901),
             _case(mm, (9, 12, 10), (14, 13), 7, 2, 8, seed=902),
             _case(mm, (12, 16, 11), (18, 20), 13, 6, 16, seed=903)]
    for gm, B, sino, K, ldk in cases:
        err, same, _ = _both(mm, gm, B, sino, K, ldk)
        print(f"mm_adjoint_noalloc vs mm_adjoint, K = {K}, ldk = {ldk}, D = {B.shape[-1]}: E_inf = {err:.2e}, identical = {same}")
        assert err <= TOL
    assert mm.load().mm_launch_count() - n0 == 4 * len(cases)          # 2 kernels per call, both paths: native code ran
    # the same problem twice in a row: the second call rewrites the array with what is already there
    gm, B, sino, K, ldk = cases[0]
    _, _, first = _both(mm, gm, B, sino, K, ldk)
    _, _, second = _both(mm, gm, B, sino, K, ldk)
    assert torch.equal(first, second)


def test_noalloc_rejects_beyond_the_static_maximum(mm):
    """P * 2 * npad * D * 4 bytes over MM_ADJOINT_NOALLOC_MAX_BYTES: refused with a clear error, nothing written."""
    import torch
    P, D, ell_max = 180, 16, 16                                       # K = 153 -> ldk 156 -> npad 192: 24 KiB per projection
    gm, B, sino, K, ldk = _case(mm, (8, 8, 8), (8, 8), P, ell_max, D, seed=904)
    assert P * 2 * 192 * D * 4 > mm.ADJOINT_NOALLOC_MAX_BYTES
    out = torch.full(gm.vol_shape(ldk), 7.0, device="cuda")
    with pytest.raises(mm.MMError, match="MM_ADJOINT_NOALLOC_MAX_BYTES"):
        mm.mm_adjoint_noalloc(gm, B, sino, K, out)
    torch.cuda.synchronize()
    assert bool((out == 7.0).all().item())
    want = torch.empty(gm.vol_shape(ldk), device="cuda")
    mm.mm_adjoint(gm, B, sino, K, want)                                # the allocating path serves the same call
    torch.cuda.synchronize()
    assert bool(torch.isfinite(want).all().item())
