"""GPU parity for the colour decorrelation in front of RAHT (section 4): RGB -> YUV + per-channel
KLT through the C ABI against the fp64 oracle.  The transform given a basis is compared element by element; the fit is
compared on what is unique (means, covariance spectrum) and checked for validity (orthonormal, decorrelating), because
an eigenbasis is unique only up to sign and, for equal eigenvalues, rotation."""
import numpy as np
import pytest
import torch

from oracle import gsnfs_oracle as orc
from paper_2606_05650_b200 import synth

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


@pytest.fixture(scope="module")
def B():
    from paper_2606_05650_b200 import binding
    binding.lib()
    return binding


def correlated_frame(n, K, seed):
    rng = np.random.default_rng(seed)
    C = 11 + 3 * K
    a = rng.normal(0, 1, (n, C))
    a[:, 8:11] = rng.normal(0, 0.5, (n, 3))
    if K:
        _, ac = orc.sh_layout(C)
        shared = rng.normal(0, 1, (n, K)) * np.geomspace(0.08, 0.004, K)      # a component common to R, G, B: YUV pays
        for c in range(3):
            R = np.linalg.qr(rng.normal(0, 1, (K, K)))[0]
            a[:, ac[c]] = shared @ R.T * (0.8 + 0.2 * c) + rng.normal(0, 0.003, (n, K)) + rng.normal(0, 0.01, K)
    return np.ascontiguousarray(a, dtype=np.float32)


def unpack_klt(klt, K):
    st = 2 * K + K * K
    mu = np.stack([klt[c * st:c * st + K] for c in range(3)])
    lam = np.stack([klt[c * st + K:c * st + 2 * K] for c in range(3)])
    E = np.stack([klt[c * st + 2 * K:(c + 1) * st].reshape(K, K) for c in range(3)])
    return mu.astype(np.float64), lam.astype(np.float64), E.astype(np.float64)


@pytest.mark.parametrize("n,K", [(50_000, 15), (20_001, 8), (777, 3), (300_000, 15)])
def test_fit_and_transform(B, n, K):
    C = 11 + 3 * K
    a = correlated_frame(n, K, n % 97)
    ctx = B.Context(max_points=n, max_channels=C, max_depth=8)
    try:
        d_a = torch.from_numpy(a).to(DEV)
        d_klt = torch.zeros(B.gsnfs_klt_floats(C), dtype=torch.float32, device=DEV)
        B.gsnfs_klt_fit(ctx, d_a, n, None, C, d_klt)
        torch.cuda.synchronize()
        mu, lam, E = unpack_klt(d_klt.cpu().numpy(), K)
        yuv = orc.rgb_to_yuv(a)
        rmu, rlam, rE, rS = orc.klt_fit(yuv)
        scale = np.sqrt(rlam[:, :1])
        assert np.all(np.abs(mu - rmu) <= 1e-6 * scale + 1e-7)
        assert np.all(np.abs(lam - rlam) <= 2e-5 * rlam[:, :1] + 1e-12)                     # the spectrum is unique
        for c in range(3):
            assert np.allclose(E[c].T @ E[c], np.eye(K), atol=5e-6)                          # a valid basis ...
            D = E[c].T @ rS[c] @ E[c]
            assert np.all(np.abs(D - np.diag(np.diag(D))) <= 3e-5 * rlam[c, 0])              # ... that diagonalises the covariance
            for j in range(K):                                                               # well separated axes agree
                gap = min(abs(rlam[c, j] - rlam[c, i]) for i in range(K) if i != j) if K > 1 else 1.0
                if gap > 0.05 * rlam[c, 0]:
                    assert np.abs(E[c][:, j] - rE[c][:, j]).max() < 2e-3, (c, j)
        # the transform with the GPU's basis, element by element against the oracle with the same basis
        d_out = torch.empty_like(d_a)
        B.gsnfs_color_forward(ctx, d_a, n, None, C, d_klt, d_out)
        torch.cuda.synchronize()
        ref = orc.klt_forward(yuv, mu, E)
        got = d_out.cpu().numpy().astype(np.float64)
        tol = 2e-6 * np.abs(a).max(axis=0).max() * 4 + 1e-7
        assert np.abs(got - ref).max() <= tol
        assert np.array_equal(got[:, :8], a[:, :8].astype(np.float64))                      # geometry channels untouched
        d_back = torch.empty_like(d_a)
        B.gsnfs_color_inverse(ctx, d_out, n, None, C, d_klt, d_back)
        torch.cuda.synchronize()
        assert (d_back - d_a).abs().max().item() <= 4 * tol
        ref_back = orc.yuv_to_rgb(orc.klt_inverse(ref, mu, E))
        assert np.abs(d_back.cpu().numpy() - ref_back).max() <= 4 * tol
        # in place, and YUV only (d_klt == NULL)
        d_in_place = d_a.clone()
        B.gsnfs_color_forward(ctx, d_in_place, n, None, C, d_klt, d_in_place)
        d_yuv = torch.empty_like(d_a)
        B.gsnfs_color_forward(ctx, d_a, n, None, C, None, d_yuv)
        torch.cuda.synchronize()
        assert torch.equal(d_in_place, d_out)
        assert np.abs(d_yuv.cpu().numpy() - yuv).max() <= tol
        # fit twice: deterministic
        d_klt2 = torch.zeros_like(d_klt)
        B.gsnfs_klt_fit(ctx, d_a, n, None, C, d_klt2)
        torch.cuda.synchronize()
        assert torch.equal(d_klt, d_klt2)
    finally:
        ctx.close()


def test_energy_compaction_and_pipeline(B):
    """KLT concentrates the AC energy in the first coefficients ("concentrates signal energy on the first
    few coefficients") and the decorrelated frame goes through the codec path like any other 56-channel frame."""
    n, K, C = 60_000, 15, 56
    a = correlated_frame(n, K, 5)
    fr0 = synth.make_frame(2, n_override=n)
    ctx = B.Context(max_points=n, max_channels=C, max_depth=fr0.depth)
    try:
        d_a = torch.from_numpy(a).to(DEV)
        d_klt = torch.zeros(B.gsnfs_klt_floats(C), dtype=torch.float32, device=DEV)
        d_out = torch.empty_like(d_a)
        B.gsnfs_klt_fit(ctx, d_a, n, None, C, d_klt)
        B.gsnfs_color_forward(ctx, d_a, n, None, C, d_klt, d_out)
        torch.cuda.synchronize()
        y = d_out.cpu().numpy()
        _, ac = orc.sh_layout(C)
        for c in range(3):
            var_in = a[:, ac[c]].var(axis=0)
            var_out = y[:, ac[c]].var(axis=0)
            assert var_out[:3].sum() / var_out.sum() > var_in[:3].sum() / var_in.sum()
            assert np.all(np.diff(var_out) <= 1e-6 * var_out[0])
        fr = synth.Frame("klt", fr0.xyz, y, synth.qstep_from_range(y, 256), fr0.depth, 256, fr0.bbox_min, fr0.bbox_max)
        from test_gpu_parity import full_pipeline_check
        full_pipeline_check(B, ctx, fr)
    finally:
        ctx.close()
    for bad in (57, 10, 11 + 3 * 16):
        assert B.gsnfs_klt_floats(bad) == 0


def test_device_yuv_constants_against_the_bt601_definition(B):
    """The nine device constants pinned to [R15]'s definition (U = 0.492 (B - Y), V = 0.877 (R - Y) from the luma weights),
    not to the oracle's table: unit primaries through gsnfs_color_forward (YUV only), on the DC triple and on every AC
    triple, read back entry by entry to the five printed digits (+ one fp32 rounding)."""
    w = np.array([0.299, 0.587, 0.114])
    D = np.stack([w, 0.436 / (1 - w[2]) * (np.array([0, 0, 1.0]) - w), 0.615 / (1 - w[0]) * (np.array([1.0, 0, 0]) - w)])
    C, K = 56, 15
    ctx = B.Context(max_points=64, max_channels=C, max_depth=4)
    try:
        trips = [[8, 9, 10]] + [[11 + j, 11 + K + j, 11 + 2 * K + j] for j in range(K)]
        a = np.zeros((3 * len(trips), C), np.float32)
        for t, trip in enumerate(trips):
            for prim in range(3):
                a[3 * t + prim, trip[prim]] = 1.0
        a[:, :8] = 0.25                                                  # geometry channels must pass through
        d_a = torch.from_numpy(a).to(DEV)
        d_y = torch.empty_like(d_a)
        B.gsnfs_color_forward(ctx, d_a, a.shape[0], None, C, None, d_y)
        torch.cuda.synchronize()
        y = d_y.cpu().numpy().astype(np.float64)
        for t, trip in enumerate(trips):
            for prim in range(3):
                assert np.abs(y[3 * t + prim, trip] - D[:, prim]).max() < 1e-5 + 6e-8, (t, prim)
                other = np.setdiff1d(np.arange(8, C), trip)
                assert np.all(y[3 * t + prim, other] == 0.0)
        assert np.all(y[:, :8] == 0.25)
    finally:
        ctx.close()
