"""fr_gemm_static (include/frb200.h): the operator product C <- c1*A*B + c2*C (eq. 1) for callers that must not
allocate device memory -- the packed operator sits in a file-scope device array of FR_GEMM_STATIC_MAX_BYTES.

Checked against the existing one-shot path fr_gemm on the same device buffers, within the tolerance test_T7_gemm_vs_numpy uses
(1e-13 / 1e-5 of the magnitude sum |A| |B| + |c2| |C|: the two paths run different kernels, so they agree to rounding, not bit for
bit), on two calls in a row whose operators differ in shape -- the second, smaller operator must see nothing of the first one's
image in the shared array.  Collected last (file name), so a failure here hides no other test under `pytest -x`.
"""
import numpy as np
import pytest

from fr_inputs import cases


def _run_pair(binding, rng, M, K, N, ld, c1, c2, prec):
    """One product through fr_gemm and through fr_gemm_static on the same inputs; returns (static, existing, tolerance)."""
    import torch
    ndt = np.float64 if prec == "f64" else np.float32
    A = rng.standard_normal((M, K))
    B = rng.uniform(-1, 1, (K, ld)).astype(ndt)
    C0 = rng.uniform(-1, 1, (M, ld)).astype(ndt)
    dB = torch.from_numpy(B).cuda()
    dC_ref, dC_new = torch.from_numpy(C0).cuda(), torch.from_numpy(C0).cuda()
    binding.gemm(A, dB.data_ptr(), ld, dC_ref.data_ptr(), ld, N, c1=c1, c2=c2, prec=prec)
    binding.gemm_static(A, dB.data_ptr(), ld, dC_new.data_ptr(), ld, N, c1=c1, c2=c2, prec=prec)
    torch.cuda.synchronize()
    ref, new = dC_ref.cpu().numpy().astype(np.float64), dC_new.cpu().numpy().astype(np.float64)
    Ar = np.abs(A.astype(ndt).astype(np.float64))
    scale = abs(c1) * (Ar @ np.abs(B[:, :N].astype(np.float64))) + abs(c2) * np.abs(C0[:, :N])
    tol = (1e-13 if prec == "f64" else 1e-5) * scale.max()
    assert np.array_equal(new[:, N:], C0[:, N:].astype(np.float64))         # columns beyond N untouched
    return new[:, :N], ref[:, :N], tol


@pytest.mark.gpu
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_gemm_static_matches_fr_gemm_on_two_calls_in_a_row(prec):
    from paper_1409_0405_b200 import binding
    rng = np.random.Generator(np.random.PCG64(cases.SEEDS["c4"] + 77))
    # call 1: hex p = 3 gradient operator (192 x 64), ragged width and leading dimension, c2 != 0;
    # call 2: a smaller operator with other tile sizes (tet p = 3 M0: 40 x 20), c2 = 0, narrow tail case
    for M, K, N, ld, c1, c2 in ((192, 64, 5 * 1237, 5 * 1237 + 15, 1.0, 1.0), (40, 20, 5 * 1000 + 6, 5 * 1000 + 8, -0.5, 0.0),
                                (192, 64, 6, 8, 1.0, 0.5)):
        new, ref, tol = _run_pair(binding, rng, M, K, N, ld, c1, c2, prec)
        assert np.isfinite(new).all()
        assert np.abs(new - ref).max() <= tol, (M, K, N, np.abs(new - ref).max(), tol)


@pytest.mark.gpu
def test_gemm_static_rejects_operators_beyond_the_array():
    import torch
    from paper_1409_0405_b200 import FrError, binding
    d = torch.zeros(343 * 16, dtype=torch.float64, device="cuda")
    with pytest.raises(FrError) as ei:
        binding.gemm_static(np.ones((343, 343)), d.data_ptr(), 16, d.data_ptr(), 16, 16, prec="f64")
    assert ei.value.status == binding.FR_EINVAL and "FR_GEMM_STATIC_MAX_BYTES" in str(ei.value)
    # the largest FP64 operator of the sweep that fits still runs after a rejected call
    rng = np.random.Generator(np.random.PCG64(cases.SEEDS["c4"] + 78))
    new, ref, tol = _run_pair(binding, rng, 225, 75, 640, 640, 1.0, 0.0, "f64")
    assert np.abs(new - ref).max() <= tol
