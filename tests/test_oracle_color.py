"""Pins for the oracle's colour decorrelation (section 4: RGB -> YUV on every SH function, one KLT per YUV
channel on the SH AC coefficients).  No GPU."""
import numpy as np
import pytest

from oracle import gsnfs_oracle as orc


def _frame(n=4000, K=15, seed=0, correlated=True):
    rng = np.random.default_rng(seed)
    C = 11 + 3 * K
    a = rng.normal(0, 1, (n, C))
    if correlated and K:
        _, ac = orc.sh_layout(C)
        for c in range(3):                                # correlated AC coefficients with distinct variances
            R = np.linalg.qr(rng.normal(0, 1, (K, K)))[0]
            s = np.geomspace(1.0, 0.02, K)
            a[:, ac[c]] = (rng.normal(0, 1, (n, K)) * s) @ R.T + rng.normal(0, 0.3, K)
    return a


def test_yuv_matrix_and_roundtrip():
    M = orc.YUV_FROM_RGB
    assert abs(M[0].sum() - 1.0) < 1e-12 and abs(M[1].sum()) < 2e-5 and abs(M[2].sum()) < 2e-5     # BT.601 as printed to 5 digits
    a = _frame(50, 15, 1)
    dc, ac = orc.sh_layout(56)
    grey = a.copy()
    for j in range(15):
        grey[:, ac[1][j]] = grey[:, ac[0][j]]; grey[:, ac[2][j]] = grey[:, ac[0][j]]
    grey[:, dc[1]] = grey[:, dc[0]]; grey[:, dc[2]] = grey[:, dc[0]]
    y = orc.rgb_to_yuv(grey)
    assert np.allclose(y[:, dc[0]], grey[:, dc[0]]) and np.abs(y[:, dc[1]]).max() < 1e-4 and np.abs(y[:, dc[2]]).max() < 1e-4
    assert np.allclose(y[:, ac[0]], grey[:, ac[0]]) and np.abs(y[:, ac[1]]).max() < 1e-4
    assert np.array_equal(y[:, :8], grey[:, :8])                     # scale, rotation, opacity untouched
    # one SH function by hand: (R, G, B) = (1, 0, 0) -> first column of the matrix
    e = np.zeros((1, 56)); e[0, dc[0]] = 1.0
    assert np.allclose(orc.rgb_to_yuv(e)[0, dc], M[:, 0])
    assert np.allclose(orc.yuv_to_rgb(orc.rgb_to_yuv(a)), a, atol=1e-12)
    with pytest.raises(ValueError):
        orc.sh_layout(57)


def bt601_yuv_from_definition():
    """[R15] by its definition, not by its printed table: luma weights (W_R, W_G, W_B) = (0.299, 0.587, 0.114); U and V are
    the colour differences B - Y and R - Y scaled to the peak excursions U_max = 0.436 and V_max = 0.615:
    U = U_max (B - Y) / (1 - W_B) = 0.492 (B - Y),  V = V_max (R - Y) / (1 - W_R) = 0.877 (R - Y)."""
    w = np.array([0.299, 0.587, 0.114])
    ku, kv = 0.436 / (1.0 - w[2]), 0.615 / (1.0 - w[0])
    assert round(ku, 3) == 0.492 and round(kv, 3) == 0.877
    b_minus_y = np.array([0.0, 0.0, 1.0]) - w
    r_minus_y = np.array([1.0, 0.0, 0.0]) - w
    return np.stack([w, ku * b_minus_y, kv * r_minus_y])


def test_yuv_matrix_is_bt601_entry_by_entry():
    """Every one of the nine constants against the definition, to the five decimals they are printed with (cut off, not rounded): a swapped pair of
    chroma coefficients, a wrong sign or a wrong U / V scale moves an entry by >= 1e-2."""
    D = bt601_yuv_from_definition()
    M = orc.YUV_FROM_RGB
    assert M.shape == (3, 3)
    assert np.array_equal(M[0], D[0])                                  # the luma weights are exact
    assert np.abs(M[1:] - D[1:]).max() < 1e-5                         # chroma rows: the table prints 5 decimals, cut off (-0.1471377 -> -0.14713)
    assert np.all(np.sign(M) == np.sign(D))
    # and through the transform itself, one unit primary at a time, on the DC triple and on an AC triple
    dc, ac = orc.sh_layout(56)
    for k, trip in enumerate((dc, [ac[0][4], ac[1][4], ac[2][4]])):
        for prim in range(3):
            e = np.zeros((1, 56)); e[0, trip[prim]] = 1.0
            assert np.abs(orc.rgb_to_yuv(e)[0, trip] - D[:, prim]).max() < 1e-5, (k, prim)


@pytest.mark.parametrize("K", [15, 8, 3])
def test_klt_is_pca(K):
    a = orc.rgb_to_yuv(_frame(6000, K, K))
    mu, lam, E, S = orc.klt_fit(a)
    _, ac = orc.sh_layout(a.shape[1])
    y = orc.klt_forward(a, mu, E)
    for c in range(3):
        assert np.allclose(E[c].T @ E[c], np.eye(K), atol=1e-12)                    # orthonormal
        assert np.all(np.diff(lam[c]) <= 1e-15)                                      # sorted, descending
        X = a[:, ac[c]]
        # independent library routine: right singular vectors of the centred data = principal axes
        U, sv, Vt = np.linalg.svd(X - X.mean(0), full_matrices=False)
        assert np.allclose(sv ** 2 / X.shape[0], lam[c], rtol=1e-9)
        for j in range(K):
            assert min(np.abs(Vt[j] - E[c][:, j]).max(), np.abs(Vt[j] + E[c][:, j]).max()) < 1e-7
            assert E[c][np.argmax(np.abs(E[c][:, j])), j] > 0                        # sign convention
        Yc = y[:, ac[c]]
        cov = Yc.T @ Yc / X.shape[0]
        assert np.allclose(cov, np.diag(lam[c]), atol=1e-10)                         # decorrelated, zero mean
        assert abs(np.abs(Yc.mean(0)).max()) < 1e-12
        assert np.isclose((Yc ** 2).sum(), ((X - mu[c]) ** 2).sum())                 # energy preserved
    assert np.allclose(orc.klt_inverse(y, mu, E), a, atol=1e-12)
    assert np.array_equal(y[:, :11], a[:, :11])                                      # only the AC coefficients move


def test_klt_recovers_a_known_covariance():
    rng = np.random.default_rng(4)
    K, n = 15, 200_000
    R = np.linalg.qr(rng.normal(0, 1, (K, K)))[0]
    s = np.linspace(2.0, 0.2, K)
    a = np.zeros((n, 56))
    _, ac = orc.sh_layout(56)
    a[:, ac[1]] = (rng.normal(0, 1, (n, K)) * s) @ R.T
    mu, lam, E, S = orc.klt_fit(a)
    assert np.allclose(lam[1], s ** 2, rtol=0.03)
    for j in range(K):
        assert abs(abs(E[1][:, j] @ R[:, j]) - 1.0) < 0.02
    assert np.allclose(lam[0], 0) and np.allclose(lam[2], 0)
