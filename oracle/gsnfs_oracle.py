"""ORACLE -- test infrastructure, NOT part of the product.

A plain, slow, fp64 CPU restatement of what GS-NFS's per-frame codec hot path computes
(arxiv/paper_2606_05650, text in /root/reference/PAPER.md; cited below as PAPER.md:L<line>).
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import
this file.  It shares no code, tables or helpers with the CUDA path and imports nothing from it.

Every function follows the paper's own statement of the step, in the paper's order and notation,
vectorised with numpy only where the paper itself says "for ... do in parallel".  Readings of the
places where the paper is silent or garbled are the ones listed in DESIGN.md ("Readings") and are
tagged here as [O1]..[O12], [R1]..[R13].

Pins (tests/test_oracle_*.py, all `-m "not gpu"`):
  voxelize / morton        worked values PAPER.md:L136-146 (tests/golden/morton_examples.txt),
                           round trips, boundary points
  sort_by_key              python sorted() on (key, index) tuples
  octree_* / occupancy     brute-force per-level python sets; recursive level-order traversal of a
                           pointer octree; Fig. 2/3 stream (tests/golden/fig2_stream.txt);
                           full cube; single point; popcount invariants; decode(encode(P))
  merge_attributes         python-loop mean; single-Gaussian voxels copied exactly
  raht_coefficient_closed_form   the level-synchronous raht_forward on random sparse voxel sets (every row)
  raht_*                   Eq. (1) two-voxel closed form; explicit orthonormal matrix built from the
                           Morton-prefix ranges; DC = sum(w a)/sqrt(W); Parseval; constant signal;
                           dense separable 3-D Haar on a full cube (PAPER.md:L219 fn. 4);
                           duplicates-expanded equivalence [R2]; perfect reconstruction; linearity
  rgb_to_yuv / klt_*       rows of the matrix (luma weights sum to 1, chroma rows to 0), grey -> zero chroma,
                           inverse o forward = identity; KLT against an SVD of the centred data (library PCA),
                           known synthetic covariance, orthonormality, diagonal output covariance, energy
  quantize / dequantize    PARITY UNPINNED by the paper [R10]: it gives only the name "dead-zone
                           quantization" and omits de-quantisation (L259).  Pinned
                           only to self-consistency properties (dead zone, error bound, symmetry) and
                           hand-computed values (quantize at f = 1/3; dequantize with delta = 0 and 0.25).
"""
from __future__ import annotations

import numpy as np

U64 = np.uint64


# =============================================================================================
# Position coder, encoder side (section 2.1-2.2, Algorithm A.1)
# =============================================================================================
def voxelize(xyz, bbox_min, bbox_max, J):
    """Quantise positions to J bits per axis inside the bounding cuboid.

    [O1] per axis v = floor((p - lo) * 2^J / (hi - lo)), clamped to [0, 2^J - 1] (p = hi falls in
    the last voxel).  [O2] arithmetic, normative because the stream must be bit exact:
    t = fp64(p) - fp64(lo) (one rounding); s = 2^J / (fp64(hi) - fp64(lo)); u = t * s (one
    rounding, no FMA); v = floor(u).
    Returns an (N, 3) uint64 array of integer voxel coordinates (x, y, z).
    """
    p = np.asarray(xyz, dtype=np.float32).astype(np.float64).reshape(-1, 3)
    lo = np.asarray(bbox_min, dtype=np.float32).astype(np.float64)
    hi = np.asarray(bbox_max, dtype=np.float32).astype(np.float64)
    s = np.ldexp(1.0, J) / (hi - lo)
    t = p - lo
    u = t * s
    vmax = float((1 << J) - 1)
    v = np.floor(u)
    v = np.where(u < 0.0, 0.0, np.minimum(v, vmax))
    return v.astype(U64)


def morton_encode(v, J):
    """Bit-interleave (x, y, z) -> z_{J-1} y_{J-1} x_{J-1} ... z_0 y_0 x_0; 64-bit
    code, unused most-significant bits zero (L152).  [O3] bit 3b = x_b, 3b+1 = y_b, 3b+2 = z_b."""
    v = np.asarray(v, dtype=U64).reshape(-1, 3)
    key = np.zeros(v.shape[0], dtype=U64)
    one = U64(1)
    for b in range(J):
        sb = U64(b)
        key |= ((v[:, 0] >> sb) & one) << U64(3 * b)
        key |= ((v[:, 1] >> sb) & one) << U64(3 * b + 1)
        key |= ((v[:, 2] >> sb) & one) << U64(3 * b + 2)
    return key


def morton_decode(keys, J):
    """Reverse the interleaving (Alg. A.2 l.14-18 ReconstructPoints).
    [O11] shift J_v - J is taken as 0."""
    keys = np.asarray(keys, dtype=U64)
    v = np.zeros((keys.shape[0], 3), dtype=U64)
    one = U64(1)
    for b in range(J):
        sb = U64(b)
        v[:, 0] |= ((keys >> U64(3 * b)) & one) << sb
        v[:, 1] |= ((keys >> U64(3 * b + 1)) & one) << sb
        v[:, 2] |= ((keys >> U64(3 * b + 2)) & one) << sb
    return v


def sort_by_key(keys):
    """"an array sorted by the Morton code that contains a pointer to the Gaussian" (
    RadixSort in Alg. A.1 l.4).  [O8] stable: equal codes keep ascending original index.
    Returns perm with keys[perm] non-decreasing."""
    return np.argsort(np.asarray(keys, dtype=U64), kind="stable").astype(np.int64)


def unique_segments(sorted_keys):
    """Clusters of equal codes in the sorted array (Unique in Alg. A.1 l.4).
    Returns (voxel_keys[Nv], voxel_start[Nv+1], weight[Nv]) with weight = run length."""
    k = np.asarray(sorted_keys, dtype=U64)
    n = k.shape[0]
    if n == 0:
        return k.copy(), np.zeros(1, np.int64), np.zeros(0, np.int64)
    head = np.ones(n, dtype=bool)
    head[1:] = k[1:] != k[:-1]
    start = np.flatnonzero(head).astype(np.int64)
    voxel_start = np.concatenate([start, [n]]).astype(np.int64)
    return k[start].copy(), voxel_start, np.diff(voxel_start)


def merge_attributes(attr, perm, voxel_start):
    """Average the attributes of the Gaussians in one voxel.  [O9] plain
    arithmetic mean of every channel in fp64, summed in perm order, no renormalisation.
    Output Nv x C in Morton order."""
    a = np.asarray(attr).astype(np.float64)
    nv = len(voxel_start) - 1
    out = np.empty((nv, a.shape[1]), dtype=np.float64)
    cnt = np.diff(voxel_start)
    single = cnt == 1
    out[single] = a[perm[voxel_start[:-1][single]]]
    for v in np.flatnonzero(~single):
        acc = np.zeros(a.shape[1], dtype=np.float64)
        for g in range(voxel_start[v], voxel_start[v + 1]):
            acc = acc + a[perm[g]]
        out[v] = acc / float(cnt[v])
    return out


def octree_levels(voxel_keys, J):
    """Bottom-up construction L_d = Unique({c >> 3 : c in L_{d+1}}), d = J-1 .. 0
    (Alg. A.1 l.5-7).  Returns [L_0, ..., L_J]."""
    levels = [None] * (J + 1)
    levels[J] = np.asarray(voxel_keys, dtype=U64)
    for d in range(J - 1, -1, -1):
        levels[d] = np.unique(levels[d + 1] >> U64(3))
    return levels


def occ_kernel(L_d, L_d1):
    """OccKernel of Alg. A.1 l.15-25, one "thread" per parent:
    c_b = p << 3; binary-search L_{d+1} for the first code >= c_b; scan at most 8 entries while the
    code is <= c_b + 7 [O7: with an end-of-list guard]; set bit (code - c_b) [O4]."""
    L_d = np.asarray(L_d, dtype=U64)
    L_d1 = np.asarray(L_d1, dtype=U64)
    cb = L_d << U64(3)
    pos = np.searchsorted(L_d1, cb, side="left")
    occ = np.zeros(L_d.shape[0], dtype=np.uint8)
    n1 = L_d1.shape[0]
    for k in range(8):
        idx = pos + k
        inb = idx < n1
        code = L_d1[np.minimum(idx, max(n1 - 1, 0))] if n1 else np.zeros_like(cb)
        ok = inb & (code <= cb + U64(7)) & (code >= cb)
        bit = np.where(ok, code - cb, U64(0)).astype(np.uint8)
        occ |= np.where(ok, np.uint8(1) << bit, np.uint8(0)).astype(np.uint8)
    return occ


def octree_encode(voxel_keys, J):
    """Alg. A.1 steps 2-4.  [O5] bytes of level 0 first, each level contiguous, parents in
    ascending Morton order, leaves emit nothing.  [O6] the header is returned as a separate array
    level_sizes = (|L_0|, ..., |L_J|), not serialised.  Empty input: no bytes, sizes all 0."""
    vk = np.asarray(voxel_keys, dtype=U64)
    if vk.shape[0] == 0:
        return np.zeros(0, np.uint8), np.zeros(J + 1, np.int64)
    levels = octree_levels(vk, J)
    level_sizes = np.array([len(L) for L in levels], dtype=np.int64)
    parts = [occ_kernel(levels[d], levels[d + 1]) for d in range(J)]
    return np.concatenate(parts) if parts else np.zeros(0, np.uint8), level_sizes


def position_encode(xyz, bbox_min, bbox_max, J):
    """Whole encoder-side position path: voxelise -> Morton -> stable sort -> unique -> octree.
    Returns a dict with every array the C ABI's gsnfs_octree_encode emits."""
    v = voxelize(xyz, bbox_min, bbox_max, J)
    keys = morton_encode(v, J)
    perm = sort_by_key(keys)
    vk, vstart, w = unique_segments(keys[perm])
    occ, level_sizes = octree_encode(vk, J)
    return {"keys": keys, "perm": perm, "voxel_keys": vk, "voxel_start": vstart, "weights": w,
            "occ": occ, "level_sizes": level_sizes}


# =============================================================================================
# Position coder, decoder side (section 2.3, Algorithms A.2 and A.3)
# =============================================================================================
_POPCOUNT8 = np.array([bin(i).count("1") for i in range(256)], dtype=np.int64)


def expand_children(L_d, occ_d, off):
    """Alg. A.3: for each parent, for i = 0..7 ascending, if bit i is set write (parent << 3) + i at
    the running offset that starts at the parent's exclusive-scan value."""
    total = int(off[-1] + _POPCOUNT8[occ_d[-1]]) if len(occ_d) else 0
    out = np.zeros(total, dtype=U64)
    base = np.asarray(L_d, dtype=U64) << U64(3)
    w = off.copy()
    for i in range(8):
        sel = (occ_d >> np.uint8(i)) & np.uint8(1) == 1
        out[w[sel]] = base[sel] + U64(i)
        w = w + sel.astype(np.int64)
    return out


def octree_decode(occ, level_sizes, J):
    """Alg. A.2: L_0 = [0]; per level read |L_d| bytes, popcount, exclusive
    scan, expand.  Returns (leaf Morton codes L_J, integer coordinates N_v x 3, ok) where ok is
    False for a corrupt stream [O12]: a zero byte, or sum(popcount) != level_sizes[d+1]."""
    occ = np.asarray(occ, dtype=np.uint8)
    level_sizes = np.asarray(level_sizes, dtype=np.int64)
    if level_sizes[0] == 0:
        return np.zeros(0, U64), np.zeros((0, 3), U64), True
    ok = level_sizes[0] == 1
    L = np.zeros(1, dtype=U64)
    ptr = 0
    for d in range(J):
        m = L.shape[0]
        occ_d = occ[ptr:ptr + m]
        ptr += m
        if occ_d.shape[0] != m or np.any(occ_d == 0):
            return np.zeros(0, U64), np.zeros((0, 3), U64), False
        cnt = _POPCOUNT8[occ_d]
        off = np.concatenate([[0], np.cumsum(cnt)[:-1]]).astype(np.int64)
        L = expand_children(L, occ_d, off)
        if L.shape[0] != level_sizes[d + 1]:
            ok = False
    return L, morton_decode(L, J), bool(ok)


# =============================================================================================
# Attribute coder: RAHT (section 3, Appendix D, Algorithms A.4-A.6, Eq. 1)
# =============================================================================================
def raht_prelude(M, leaf_w, J):
    """Alg. A.4 (non-parallel prelude): for l = 1 .. 3J build the active index
    list I_l, weights W_l and left-sibling flags F_l = ((M_k xor M_{k+1}) and (2^{3J} - 2^l)) == 0.
    [R1] leaf weights generalise the paper's unit weights: W_l[k] = P[I_l[k+1] or Nv] - P[I_l[k]]
    with P the prefix sums of the leaf weights (equals A.4 l.8's run length when all are 1).
    [R3] l runs to 3J inclusive; [A.5 l.16] stop once a single entry is left."""
    M = np.asarray(M, dtype=U64)
    nv = M.shape[0]
    P = np.concatenate([[0], np.cumsum(np.asarray(leaf_w, dtype=np.int64))]).astype(np.int64)
    I = np.arange(nv, dtype=np.int64)
    sched = []
    full = (1 << (3 * J))
    for l in range(1, 3 * J + 1):
        if I.shape[0] <= 1:
            break
        Ml = M[I]
        nxt = np.concatenate([I[1:], [nv]])
        W = P[nxt] - P[I]
        mask = U64(full - (1 << l))
        D = Ml[:-1] ^ Ml[1:]
        F = np.concatenate([(D & mask) == U64(0), [False]])
        sched.append((I, W, F))
        Pshift = np.concatenate([[False], F[:-1]])          # A.5 l.13: marks right siblings
        I = I[~Pshift]                                      # A.5 l.15: keep left siblings + singletons
    return sched


def raht_forward(A, M, leaf_w, J):
    """Alg. A.6 forward with Eq. (1) (L213) and a, b of L621.
    [R2] the transformed signal is x_i = sqrt(w_i) * a_i (identity for the paper's unit weights).
    [R6] low-pass stays at the left index i0, high-pass goes to the right index i1.
    Returns Y (Nv x C, fp64) in place over the Morton-sorted rows: row 0 = DC."""
    A = np.asarray(A, dtype=np.float64)
    w = np.asarray(leaf_w, dtype=np.float64)
    Y = A * np.sqrt(w)[:, None]
    for (I, W, F) in raht_prelude(M, leaf_w, J):
        k = np.flatnonzero(F)
        if k.shape[0] == 0:
            continue
        i0, i1 = I[k], I[k + 1]
        w0, w1 = W[k].astype(np.float64), W[k + 1].astype(np.float64)
        a = np.sqrt(w0 / (w0 + w1))[:, None]
        b = np.sqrt(w1 / (w0 + w1))[:, None]
        y0, y1 = Y[i0], Y[i1]
        Y[i0] = a * y0 + b * y1
        Y[i1] = -b * y0 + a * y1
    return Y


def raht_inverse(Y, M, leaf_w, J):
    """Alg. A.6 inverse: the same schedule top-down with the transposed
    rotation, then [R2] un-scale by 1/sqrt(w_i)."""
    Y = np.array(Y, dtype=np.float64, copy=True)
    w = np.asarray(leaf_w, dtype=np.float64)
    for (I, W, F) in reversed(raht_prelude(M, leaf_w, J)):
        k = np.flatnonzero(F)
        if k.shape[0] == 0:
            continue
        i0, i1 = I[k], I[k + 1]
        w0, w1 = W[k].astype(np.float64), W[k + 1].astype(np.float64)
        a = np.sqrt(w0 / (w0 + w1))[:, None]
        b = np.sqrt(w1 / (w0 + w1))[:, None]
        y0, y1 = Y[i0], Y[i1]
        Y[i0] = a * y0 - b * y1
        Y[i1] = b * y0 + a * y1
    return Y / np.sqrt(w)[:, None]


def raht_coefficient_closed_form(A, M, leaf_w, rows, return_scale=False):
    """Second, independent definition of single RAHT coefficients (no level loop, no active lists): the
    closed form that follows from Eq. (1) and the run-length weights / sibling test of
    Alg. A.4 l.8-10 (L741-747) by induction over the levels.  For row i > 0 let h = msb(M[i-1] xor M[i]);
    voxel i becomes a right sibling at level h + 1, the right node is S1 = {j : M[j] >> h == M[i] >> h} =
    [i, r), the left node S0 = {j : M[j] >> (h+1) == M[i] >> (h+1), bit h of M[j] = 0} = [l, i).  A node's
    low-pass value is T_S / sqrt(W_S) with W_S = sum of leaf weights and T_S = sum of w_j a_j ([R2]:
    sqrt(w_j) x_j), hence
        Y[i] = sqrt(W0/(W0+W1)) T_S1/sqrt(W1) - sqrt(W1/(W0+W1)) T_S0/sqrt(W0),   Y[0] = T_all/sqrt(W_all).
    Used to check sampled coefficients at sizes where the level-synchronous oracle is too slow.
    Returns an array len(rows) x C (fp64); with return_scale also |T_S1|/sqrt(W1) + |T_S0|/sqrt(W0), the magnitude
    of the two low-pass values the coefficient is the difference of (what a rounding error is relative to)."""
    A = np.asarray(A)
    M = np.asarray(M, dtype=U64)
    w = np.asarray(leaf_w, dtype=np.float64)
    out = np.empty((len(rows), A.shape[1]), dtype=np.float64)
    scale = np.empty_like(out)
    for n, i in enumerate(rows):
        i = int(i)
        if i == 0:
            out[n] = (w[:, None] * A.astype(np.float64)).sum(0) / np.sqrt(w.sum())
            scale[n] = np.abs(out[n])
            continue
        h = int(M[i] ^ M[i - 1]).bit_length() - 1
        l = int(np.searchsorted(M, (M[i] >> U64(h + 1)) << U64(h + 1), side="left"))
        r = int(np.searchsorted(M, ((M[i] >> U64(h)) + U64(1)) << U64(h), side="left"))
        W0, W1 = w[l:i].sum(), w[i:r].sum()
        T0 = (w[l:i, None] * A[l:i].astype(np.float64)).sum(0)
        T1 = (w[i:r, None] * A[i:r].astype(np.float64)).sum(0)
        out[n] = np.sqrt(W0 / (W0 + W1)) * T1 / np.sqrt(W1) - np.sqrt(W1 / (W0 + W1)) * T0 / np.sqrt(W0)
        scale[n] = np.abs(T1) / np.sqrt(W1) + np.abs(T0) / np.sqrt(W0)
    return (out, scale) if return_scale else out


# ---------------------------------------------------------------------------------------------
# Dead-zone quantiser (de-quantisation omitted by the paper, L259).
# PARITY UNPINNED [R10]: q = sign(y) floor(|y|/D + f), y^ = sign(q) (|q| + delta [q != 0]) D,
# defaults f = 1/3, delta = 0.  [R9] the DC coefficient is quantised like the rest.
# ---------------------------------------------------------------------------------------------
DZ_ROUND_DEFAULT = float(np.float32(1.0 / 3.0))   # the ABI carries f as fp32
RECON_BIAS_DEFAULT = 0.0
_I32_MAX = np.float64(2**31 - 1)


def quantize(Y, qstep, dz_round=DZ_ROUND_DEFAULT):
    """q = sign(y) floor(|y| (1/D) + f) [R10].  The integer decision is taken in the arithmetic gsnfs.h states
    (the kernel's, since the paper fixes none): 1/D rounded once to fp64, the product rounded once, the sum
    rounded once (no fused multiply-add), then floor."""
    Y = np.asarray(Y, dtype=np.float64)
    step = np.asarray(qstep, dtype=np.float32).astype(np.float64)[None, :]
    inv = np.float64(1.0) / step
    mag = np.floor(np.abs(Y) * inv + np.float64(dz_round))
    mag = np.minimum(mag, _I32_MAX)                        # saturate to int32
    return (np.sign(Y) * mag).astype(np.int64)


def dequantize(q, qstep, recon_bias=RECON_BIAS_DEFAULT):
    q = np.asarray(q, dtype=np.int64)
    step = np.asarray(qstep, dtype=np.float32).astype(np.float64)[None, :]
    mag = np.abs(q).astype(np.float64) + np.float64(recon_bias) * (q != 0)
    return np.sign(q) * mag * step


# =============================================================================================
# Colour decorrelation before RAHT (section 4; Table A.8): RGB -> YUV on every
# SH function, then one Karhunen-Loeve transform per YUV channel over the SH AC coefficients.
# [R15] the paper names neither the YUV matrix nor the channel layout: BT.601 analogue YUV; channel layout of
# SURVEY 8(d) (scale 3, rotation 4, opacity 1, SH DC 3, SH AC 3 x K colour-major: AC(c, j) = 11 + K c + j).
# [R16] KLT = eigenvectors of the covariance about the mean (the textbook definition [34]), columns sorted by
# descending eigenvalue, each eigenvector signed so that its largest-magnitude component is positive;
# y = (x - mu) E, x = y E^T + mu; mu, E are side information of the frame.
# =============================================================================================
YUV_FROM_RGB = np.array([[0.299, 0.587, 0.114],
                         [-0.14713, -0.28886, 0.436],
                         [0.615, -0.51499, -0.10001]], dtype=np.float64)
SH_DC_OFFSET = 8


def sh_layout(channels):
    """(dc[3], ac[3][K]) channel indices; K = (channels - 11) / 3 SH AC coefficients per colour."""
    if channels < 11 or (channels - 11) % 3:
        raise ValueError("channels must be 11 + 3K")
    K = (channels - 11) // 3
    dc = [SH_DC_OFFSET + c for c in range(3)]
    ac = [[11 + K * c + j for j in range(K)] for c in range(3)]
    return dc, ac


def _apply_3x3(attr, M):
    a = np.array(attr, dtype=np.float64, copy=True)
    dc, ac = sh_layout(a.shape[1])
    triples = [dc] + [[ac[0][j], ac[1][j], ac[2][j]] for j in range(len(ac[0]))]
    for t in triples:                       # every SH function: (R, G, B) -> M (R, G, B)^T
        a[:, t] = a[:, t] @ M.T
    return a


def rgb_to_yuv(attr):
    return _apply_3x3(attr, YUV_FROM_RGB)


def yuv_to_rgb(attr):
    return _apply_3x3(attr, np.linalg.inv(YUV_FROM_RGB))


def klt_fit(attr_yuv):
    """Three KLTs, one per YUV channel, over the SH AC coefficients.  Returns mu[3, K], lam[3, K]
    (descending), E[3, K, K] (columns = eigenvectors) and the covariance matrices S[3, K, K]."""
    a = np.asarray(attr_yuv, dtype=np.float64)
    _, ac = sh_layout(a.shape[1])
    K = len(ac[0])
    mu, lam, E, S = np.zeros((3, K)), np.zeros((3, K)), np.zeros((3, K, K)), np.zeros((3, K, K))
    for c in range(3):
        X = a[:, ac[c]]
        mu[c] = X.mean(axis=0)
        Xc = X - mu[c]
        S[c] = Xc.T @ Xc / X.shape[0]
        w, V = np.linalg.eigh(S[c])
        order = np.argsort(-w, kind="stable")
        w, V = w[order], V[:, order]
        for j in range(K):
            if V[np.argmax(np.abs(V[:, j])), j] < 0:
                V[:, j] = -V[:, j]
        lam[c], E[c] = w, V
    return mu, lam, E, S


def klt_forward(attr_yuv, mu, E):
    a = np.array(attr_yuv, dtype=np.float64, copy=True)
    _, ac = sh_layout(a.shape[1])
    for c in range(3):
        a[:, ac[c]] = (a[:, ac[c]] - mu[c]) @ E[c]
    return a


def klt_inverse(attr_klt, mu, E):
    a = np.array(attr_klt, dtype=np.float64, copy=True)
    _, ac = sh_layout(a.shape[1])
    for c in range(3):
        a[:, ac[c]] = a[:, ac[c]] @ E[c].T + mu[c]
    return a


# =============================================================================================
# Whole-frame helpers (the order of PAPER.md:L51-59 restricted to the hot path)
# =============================================================================================
def encode_frame(xyz, attr, bbox_min, bbox_max, J, qstep, dz_round=DZ_ROUND_DEFAULT,
                 unit_weights=False):
    pos = position_encode(xyz, bbox_min, bbox_max, J)
    merged = merge_attributes(attr, pos["perm"], pos["voxel_start"])
    w = np.ones_like(pos["weights"]) if unit_weights else pos["weights"]
    Y = raht_forward(merged, pos["voxel_keys"], w, J)
    out = dict(pos)
    out.update({"merged": merged, "coeff": Y, "raht_weights": w,
                "qcoeff": quantize(Y, qstep, dz_round) if qstep is not None else None})
    return out


def decode_frame(occ, level_sizes, J, qcoeff, qstep, leaf_w, recon_bias=RECON_BIAS_DEFAULT):
    keys, coords, ok = octree_decode(occ, level_sizes, J)
    Yh = dequantize(qcoeff, qstep, recon_bias)
    attr = raht_inverse(Yh, keys, leaf_w, J)
    return {"voxel_keys": keys, "voxel_xyz": coords, "ok": ok, "attr": attr}
