"""Pins for the oracle's RAHT and quantiser (no GPU).  References are built independently of the
oracle's level-synchronous schedule: Eq. (1) closed form, an explicit orthonormal basis from
Morton-prefix ranges, a dense separable Haar pyramid on 3-D arrays, and invariants."""
import numpy as np
import pytest

from oracle import gsnfs_oracle as orc
from paper_2606_05650_b200 import synth


def _random_voxels(rng, J, nv):
    keys = np.unique(rng.integers(0, 8 ** J, nv * 2, dtype=np.uint64))[:nv]
    return np.sort(keys)


# --------------------------------------------------------------- Eq. (1)
def test_two_voxel_closed_form():
    rng = np.random.default_rng(0)
    for (m0, m1) in [(0, 1), (0, 2), (5, 6), (0, 63), (8, 17)]:
        M = np.array([m0, m1], dtype=np.uint64)
        for w in ([1, 1], [3, 1], [2, 7]):
            A = rng.normal(0, 1, (2, 3))
            Y = orc.raht_forward(A, M, w, 2)
            wl, wr = float(w[0]), float(w[1])
            xl, xr = np.sqrt(wl) * A[0], np.sqrt(wr) * A[1]          # [R2]
            lo = (np.sqrt(wl) * xl + np.sqrt(wr) * xr) / np.sqrt(wl + wr)
            hi = (-np.sqrt(wr) * xl + np.sqrt(wl) * xr) / np.sqrt(wl + wr)
            assert np.allclose(Y[0], lo, atol=1e-14) and np.allclose(Y[1], hi, atol=1e-14)
            assert np.allclose(orc.raht_inverse(Y, M, w, 2), A, atol=1e-13)


def test_unit_weight_pair_is_haar():
    M = np.array([6, 7], dtype=np.uint64)
    Y = orc.raht_forward(np.array([[1.0], [3.0]]), M, [1, 1], 1)
    assert np.allclose(Y[:, 0], [4 / np.sqrt(2), 2 / np.sqrt(2)])


# --------------------------------------------------------------- explicit orthonormal matrix
def _msb(x):
    return int(x).bit_length() - 1


def _explicit_basis(M, w):
    """Row i of Q acts on x = sqrt(w) * a.  Built from Morton-prefix ranges only (SURVEY 8(c)
    closed form): for i > 0 with h = msb(M[i-1]^M[i]) the right node S1 = {j : M[j]>>h == M[i]>>h},
    the left node S0 = {j : M[j]>>(h+1) == M[i]>>(h+1) and bit h of M[j] == 0}."""
    M = [int(m) for m in M]
    nv = len(M)
    w = np.asarray(w, dtype=np.float64)
    Q = np.zeros((nv, nv))
    Q[0] = np.sqrt(w) / np.sqrt(w.sum())
    levels = [0]
    for i in range(1, nv):
        h = _msb(M[i - 1] ^ M[i])
        S1 = [j for j in range(nv) if (M[j] >> h) == (M[i] >> h)]
        S0 = [j for j in range(nv) if (M[j] >> (h + 1)) == (M[i] >> (h + 1)) and not (M[j] >> h) & 1]
        assert S1[0] == i and S0[-1] == i - 1
        W0, W1 = w[S0].sum(), w[S1].sum()
        Q[i, S0] = -np.sqrt(W1 / ((W0 + W1) * W0)) * np.sqrt(w[S0])
        Q[i, S1] = +np.sqrt(W0 / ((W0 + W1) * W1)) * np.sqrt(w[S1])
        levels.append(h + 1)
    return Q, levels


@pytest.mark.parametrize("J,nv,seed,weighted", [(2, 11, 0, False), (3, 16, 1, False), (4, 16, 2, True),
                                                (5, 13, 3, True), (7, 16, 4, False)])
def test_explicit_orthonormal_matrix(J, nv, seed, weighted):
    rng = np.random.default_rng(seed)
    M = _random_voxels(rng, J, nv)
    nv = len(M)
    w = rng.integers(1, 6, nv) if weighted else np.ones(nv, np.int64)
    A = rng.normal(0, 1, (nv, 4))
    Q, _ = _explicit_basis(M, w)
    assert np.allclose(Q @ Q.T, np.eye(nv), atol=1e-12)
    Y = orc.raht_forward(A, M, w, J)
    assert np.allclose(Y, Q @ (np.sqrt(w)[:, None] * A), atol=1e-12)
    assert np.allclose(orc.raht_inverse(Y, M, w, J), A, atol=1e-12)


def test_fig4_voxel_set_counts():
    # soft pin [R13]: 11 threads at the lowest level, 7 at the next
    M = np.array([24, 25, 26, 27, 28, 29, 30, 31, 33, 35, 36], dtype=np.uint64)
    sched = orc.raht_prelude(M, np.ones(11, np.int64), 2)
    assert [len(I) for (I, W, F) in sched][:2] == [11, 7]


def test_level_formula_and_butterfly_count():
    rng = np.random.default_rng(5)
    J = 6
    M = _random_voxels(rng, J, 400)
    nv = len(M)
    sched = orc.raht_prelude(M, np.ones(nv, np.int64), J)
    level_of = {}
    for l, (I, W, F) in enumerate(sched, start=1):
        for k in np.flatnonzero(F):
            level_of[int(I[k + 1])] = l
    assert len(level_of) == nv - 1                                      # exactly Nv - 1 butterflies
    for i in range(1, nv):
        assert level_of[i] == 1 + _msb(int(M[i - 1]) ^ int(M[i]))
    # run-length weights W_l (Alg. A.4 l.8) sum to Nv at every level
    for (I, W, F) in sched:
        assert int(W.sum()) == nv


# --------------------------------------------------------------- invariants
def test_dc_parseval_constant_linearity():
    rng = np.random.default_rng(6)
    J = 8
    M = _random_voxels(rng, J, 1000)
    nv = len(M)
    for w in (np.ones(nv, np.int64), rng.integers(1, 9, nv)):
        A = rng.normal(-4, 0.5, (nv, 3))
        Y = orc.raht_forward(A, M, w, J)
        assert np.allclose(Y[0], (w[:, None] * A).sum(0) / np.sqrt(w.sum()), rtol=1e-12)
        assert np.allclose((Y ** 2).sum(0), (w[:, None] * A ** 2).sum(0), rtol=1e-12)
        Yc = orc.raht_forward(np.full((nv, 1), 2.5), M, w, J)
        assert np.allclose(Yc[1:], 0.0, atol=1e-11) and np.isclose(Yc[0, 0], 2.5 * np.sqrt(w.sum()))
        B = rng.normal(0, 1, (nv, 3))
        assert np.allclose(orc.raht_forward(2 * A - 3 * B, M, w, J),
                           2 * Y - 3 * orc.raht_forward(B, M, w, J), atol=1e-10)
        # channel independence
        assert np.allclose(orc.raht_forward(A[:, 1:2], M, w, J), Y[:, 1:2], atol=0)
        assert np.allclose(orc.raht_inverse(Y, M, w, J), A, atol=1e-12)


def test_duplicates_expanded_equivalence():
    """[R2] a voxel of weight w with mean a == w coincident unit-weight points of value a, spread
    over distinct children one octree level deeper."""
    rng = np.random.default_rng(7)
    J = 4
    M = _random_voxels(rng, J, 40)
    nv = len(M)
    w = rng.integers(1, 5, nv)
    A = rng.normal(0, 1, (nv, 2))
    Y = orc.raht_forward(A, M, w, J)
    M2, A2, first = [], [], []
    for i in range(nv):
        first.append(len(M2))
        for c in range(int(w[i])):
            M2.append((int(M[i]) << 3) + c)
            A2.append(A[i])
    Y2 = orc.raht_forward(np.array(A2), np.array(M2, dtype=np.uint64), np.ones(len(M2), np.int64), J + 1)
    assert np.allclose(Y2[first], Y, atol=1e-12)
    others = np.setdiff1d(np.arange(len(M2)), first)
    assert np.allclose(Y2[others], 0.0, atol=1e-12)          # internal high-pass of a constant voxel


def _dense_haar_pyramid(cube):
    """Textbook orthonormal Haar on a dense (2^J)^3 array indexed [z, y, x]: at every octree level
    transform along x, then y, then z, always on the current low-pass sub-array only (the RAHT
    tree, PAPER.md:L198, L219 fn. 4).  Returns {(x, y, z) of the right sibling's first voxel: coef}
    plus the DC."""
    J = int(np.log2(cube.shape[0]))
    low = cube.astype(np.float64)
    out = {}
    step = 1                                   # first-voxel coordinates of a node = index * step
    s = np.sqrt(2.0)
    for _ in range(J):
        # x
        L, H = (low[:, :, 0::2] + low[:, :, 1::2]) / s, (low[:, :, 1::2] - low[:, :, 0::2]) / s
        for z in range(H.shape[0]):
            for y in range(H.shape[1]):
                for x in range(H.shape[2]):
                    out[((2 * x + 1) * step, y * step, z * step)] = H[z, y, x]
        low = L
        # y
        L, H = (low[:, 0::2, :] + low[:, 1::2, :]) / s, (low[:, 1::2, :] - low[:, 0::2, :]) / s
        for z in range(H.shape[0]):
            for y in range(H.shape[1]):
                for x in range(H.shape[2]):
                    out[(2 * x * step, (2 * y + 1) * step, z * step)] = H[z, y, x]
        low = L
        # z
        L, H = (low[0::2, :, :] + low[1::2, :, :]) / s, (low[1::2, :, :] - low[0::2, :, :]) / s
        for z in range(H.shape[0]):
            for y in range(H.shape[1]):
                for x in range(H.shape[2]):
                    out[(2 * x * step, 2 * y * step, (2 * z + 1) * step)] = H[z, y, x]
        low = L
        step *= 2
    return out, float(low[0, 0, 0])


@pytest.mark.parametrize("J", [1, 2])
def test_full_cube_is_separable_haar(J):
    rng = np.random.default_rng(8)
    side = 1 << J
    cube = rng.normal(0, 1, (side, side, side))                 # [z, y, x]
    keys = np.arange(8 ** J, dtype=np.uint64)
    coords = orc.morton_decode(keys, J)
    A = np.array([[cube[int(z), int(y), int(x)]] for (x, y, z) in coords.tolist()])
    Y = orc.raht_forward(A, keys, np.ones(len(keys), np.int64), J)
    ref, dc = _dense_haar_pyramid(cube)
    assert np.isclose(Y[0, 0], dc, atol=1e-12)
    assert len(ref) == 8 ** J - 1
    for (x, y, z), c in ref.items():
        k = int(orc.morton_encode(np.array([[x, y, z]], dtype=np.uint64), J)[0])
        assert np.isclose(Y[k, 0], c, atol=1e-12), (x, y, z)


def test_perfect_reconstruction_synthetic_frame():
    fr = synth.make_dense_frame(n=3000, depth=5, channels=7, seed=11)
    enc = orc.encode_frame(fr.xyz, fr.attr, fr.bbox_min, fr.bbox_max, fr.depth, None)
    assert enc["weights"].max() > 1
    back = orc.raht_inverse(enc["coeff"], enc["voxel_keys"], enc["weights"], fr.depth)
    assert np.allclose(back, enc["merged"], atol=1e-12)
    w = enc["weights"].astype(np.float64)
    assert np.allclose((enc["coeff"] ** 2).sum(0), (w[:, None] * enc["merged"] ** 2).sum(0), rtol=1e-12)


# --------------------------------------------------------------- quantiser (parity unpinned, R10)
@pytest.mark.parametrize("f", [0.0, 1.0 / 3.0, 0.5])
def test_quantiser_self_consistency(f):
    rng = np.random.default_rng(9)
    Y = rng.normal(0, 3, (5000, 4))
    step = np.array([0.01, 0.1, 0.5, 2.0], dtype=np.float32)
    q = orc.quantize(Y, step, f)
    s64 = step.astype(np.float64)[None, :]
    assert np.array_equal(q, -orc.quantize(-Y, step, f))                 # sign symmetry
    assert np.all(q[np.abs(Y) < (1 - f) * s64 * (1 - 1e-12)] == 0)       # dead zone
    Yh = orc.dequantize(q, step, 0.0)
    assert np.all(np.abs(Yh - Y) <= max(1 - f, f) * s64 * (1 + 1e-9) + 1e-15)
    assert np.all(np.sign(Yh) * np.sign(Y) >= 0)
    # hand-computed values at f = 1/3 for step 0.5: |y|/0.5 + 1/3 floored
    if abs(f - 1.0 / 3.0) < 1e-9:
        yy = np.array([[0.0, 0.3, 0.34, -0.34, 0.84, -1.7]]).T
        got = orc.quantize(yy, np.array([0.5], np.float32), f)[:, 0].tolist()
        assert got == [0, 0, 1, -1, 2, -3]
    assert orc.quantize(np.array([[1e30]]), np.array([1.0], np.float32), f)[0, 0] == 2**31 - 1


def test_dequantize_hand_values_and_bias_gating():
    """[R10] y^ = sign(q) (|q| + delta [q != 0]) D.  Hand-computed: D = 0.5, delta = 0.25: q = +-3 -> +-1.625,
    q = +-1 -> +-0.625, q = 0 -> 0 whatever delta; delta = 0: q = +-3 -> +-1.5.  A wrong sign of delta, a missing
    (q != 0) gate or a bias applied after the multiplication each fail one of these."""
    step = np.array([0.5], np.float32)
    q = np.array([[0], [3], [-3], [1], [-1]])
    assert orc.dequantize(q, step, 0.25)[:, 0].tolist() == [0.0, 1.625, -1.625, 0.625, -0.625]
    assert orc.dequantize(q, step, 0.0)[:, 0].tolist() == [0.0, 1.5, -1.5, 0.5, -0.5]
    assert orc.dequantize(q, step)[:, 0].tolist() == [0.0, 1.5, -1.5, 0.5, -0.5]            # default delta = 0
    # per-channel steps, and the bias moves every non-zero magnitude by exactly delta * D towards larger |y|
    rng = np.random.default_rng(3)
    qq = rng.integers(-50, 51, (200, 3))
    st = np.array([0.25, 1.0, 3.0], np.float32)
    d0, d1 = orc.dequantize(qq, st, 0.0), orc.dequantize(qq, st, 0.375)
    assert np.array_equal(d1 - d0, np.sign(qq) * 0.375 * st.astype(np.float64)[None, :])
    assert np.array_equal(d0, qq * st.astype(np.float64)[None, :])
    # round trip: quantise at f, reconstruct at delta = 1/2 - f lands mid-way in the decision interval of |q| >= 1
    f = 0.25
    y = np.array([[0.7], [1.2], [-2.6]])
    qy = orc.quantize(y, np.array([1.0], np.float32), f)
    assert qy[:, 0].tolist() == [0, 1, -2]
    assert orc.dequantize(qy, np.array([1.0], np.float32), 0.5 - f)[:, 0].tolist() == [0.0, 1.25, -2.25]


def test_quantize_reciprocal_arithmetic():
    """gsnfs.h states the arithmetic of the integer decision: floor(|y| * (1/D) + f), every operation rounded once in
    fp64.  Check against exact rational arithmetic away from the decision boundaries, and that it is the reciprocal
    form (not the division) at a value where the two differ."""
    from fractions import Fraction
    rng = np.random.default_rng(12)
    step = np.array([0.1, 1.0 / 3.0, 7.0], np.float32)
    Y = rng.normal(0, 20, (4000, 3))
    q = orc.quantize(Y, step, 1.0 / 3.0)
    for (r, c) in rng.integers(0, [4000, 3], (300, 2)).tolist():
        t = abs(Fraction(float(Y[r, c]))) / Fraction(float(step[c])) + Fraction(1.0 / 3.0)
        if abs(t - round(t)) > Fraction(1, 10**9):                       # away from a boundary both forms agree with exact
            assert abs(int(q[r, c])) == int(t // 1) and np.sign(q[r, c]) == np.sign(Y[r, c]) * (int(t // 1) > 0)
    # points where floor(|y| / D + f) and floor(|y| * (1/D) + f) differ (D = fp32(0.003): y = k D with |y| / D = k exactly
    # but |y| * (1/D) one ulp below k for many k): the oracle must follow the reciprocal form
    D = np.float64(np.float32(0.003))
    inv = 1.0 / D
    k = np.arange(1, 200000, dtype=np.float64)
    y = k * D
    a, b = np.floor(y / D), np.floor(y * inv)
    diff = np.flatnonzero(a != b)
    assert diff.size > 1000
    yy = y[diff[:200], None]
    got = orc.quantize(yy, np.array([0.003], np.float32), 0.0)[:, 0]
    assert np.array_equal(got, b[diff[:200]].astype(np.int64)) and not np.array_equal(got, a[diff[:200]].astype(np.int64))


@pytest.mark.parametrize("J,nv,seed,weighted", [(3, 40, 1, False), (4, 300, 2, True), (7, 1500, 3, True), (2, 9, 4, True)])
def test_closed_form_coefficients_equal_level_synchronous(J, nv, seed, weighted):
    """raht_coefficient_closed_form (Morton-prefix ranges, no level loop) == raht_forward (Alg. A.4 + A.6) on every row."""
    rng = np.random.default_rng(seed)
    M = _random_voxels(rng, J, nv)
    w = rng.integers(1, 9, len(M)) if weighted else np.ones(len(M), np.int64)
    A = rng.normal(0, 1, (len(M), 3))
    Y = orc.raht_forward(A, M, w, J)
    Z = orc.raht_coefficient_closed_form(A, M, w, np.arange(len(M)))
    assert np.allclose(Y, Z, atol=1e-11)
