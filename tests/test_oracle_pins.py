"""Pins for the CPU oracle (oracle/dkd_oracle.c) against things OTHER than itself:
brute-force python loops, torch library routines, closed forms, invariants, planted cases.
Each pin is chosen so a plausible mistake (dropped term, wrong sign/index, transposed operand,
wrong tie rule) fails it.  Citations: /root/reference/PAPER.md lines + BASELINE.json north_star.
"""
import math
import os

import numpy as np
import pytest
import torch
import torch.nn.functional as F

import oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def rng(seed):
    return np.random.default_rng(seed)


def quantised_map(H, W, seed, levels=12):
    """Random map on a coarse grid of values, so exact ties between neighbours are common."""
    g = rng(seed)
    return (g.integers(0, levels, size=(H, W)) / float(levels)).astype(np.float32)


# ------------------------------------------------------------------------------------------
# O1: NMS + border + threshold  (north_star step (1))
# ------------------------------------------------------------------------------------------
def brute_mask(S, r, thresh):
    H, W = S.shape
    m = np.zeros((H, W), np.uint8)
    for y in range(H):
        for x in range(W):
            if x < r or x >= W - r or y < r or y >= H - r:
                continue
            c = S[y, x]
            if not (c > np.float32(thresh)):
                continue
            win = S[y - r:y + r + 1, x - r:x + r + 1]
            if c >= win.max():
                m[y, x] = 1
    return m


@pytest.mark.parametrize("r", [1, 2, 4])
@pytest.mark.parametrize("shape", [(9, 11), (12, 10), (17, 23)])
def test_o1_bruteforce_tiny(r, shape):
    for seed in range(4):
        S = quantised_map(*shape, seed=100 * r + seed)
        assert np.array_equal(oracle.nms_mask(S, r, 0.3), brute_mask(S, r, 0.3))


@pytest.mark.parametrize("r", [1, 2, 3, 4])
def test_o1_equals_maxpool_library(r):
    # independent routine: mask = (S == max_pool2d(S, 2r+1, stride 1, pad r)) & (S > thresh) & interior
    for seed in range(3):
        S = quantised_map(61, 83, seed=seed, levels=40)
        S += (rng(seed + 7).random(S.shape) < 0.5).astype(np.float32) * np.float32(1 / 80)
        t = torch.from_numpy(S)[None, None]
        mp = F.max_pool2d(t, 2 * r + 1, 1, r)[0, 0].numpy()
        m = (S == mp) & (S > np.float32(0.25))
        inner = np.zeros_like(m)
        inner[r:S.shape[0] - r, r:S.shape[1] - r] = True
        assert np.array_equal(oracle.nms_mask(S, r, 0.25), (m & inner).astype(np.uint8))


def test_o1_planted_cases():
    r = 2
    S = np.zeros((15, 17), np.float32)
    S[7, 8] = 0.9                                      # isolated delta -> exactly one candidate
    m = oracle.nms_mask(S, r, 0.2)
    assert m.sum() == 1 and m[7, 8] == 1
    S[7, 9] = 0.9                                      # two equal adjacent pixels -> BOTH kept (G1)
    m = oracle.nms_mask(S, r, 0.2)
    assert m.sum() == 2 and m[7, 8] == 1 and m[7, 9] == 1
    S[7, 9] = np.nextafter(np.float32(0.9), np.float32(1))  # one ulp larger -> suppresses the other
    m = oracle.nms_mask(S, r, 0.2)
    assert m.sum() == 1 and m[7, 9] == 1
    C = np.full((11, 13), 0.5, np.float32)             # constant map above thresh: all interior px
    assert oracle.nms_mask(C, r, 0.2).sum() == (11 - 2 * r) * (13 - 2 * r)
    assert oracle.nms_mask(C, r, 0.5).sum() == 0        # S == thresh -> none (strict >, G4)
    assert oracle.nms_mask(C, r, np.nextafter(np.float32(0.5), np.float32(0))).sum() == 63
    for x, kept in [(r - 1, 0), (r, 1), (17 - r - 1, 1), (17 - r, 0)]:   # border exclusion (G3)
        S = np.zeros((15, 17), np.float32)
        S[7, x] = 0.8
        assert oracle.nms_mask(S, r, 0.2).sum() == kept
    for y, kept in [(r - 1, 0), (r, 1), (15 - r - 1, 1), (15 - r, 0)]:
        S = np.zeros((15, 17), np.float32)
        S[y, 8] = 0.8
        assert oracle.nms_mask(S, r, 0.2).sum() == kept
    # window is (2r+1)^2, not a cross or (2r)^2: a larger pixel at the window corner suppresses,
    # one just outside does not
    S = np.zeros((15, 17), np.float32)
    S[7, 8] = 0.8
    S[7 + r, 8 + r] = 0.85
    assert oracle.nms_mask(S, r, 0.2)[7, 8] == 0
    S[7 + r, 8 + r] = 0.0
    S[7 + r + 1, 8] = 0.85
    assert oracle.nms_mask(S, r, 0.2)[7, 8] == 1
    # degenerate sizes (G18): no interior -> no candidates
    assert oracle.nms_mask(np.ones((4, 9), np.float32), 2, 0.2).sum() == 0
    assert oracle.nms_mask(np.ones((5, 5), np.float32), 2, 0.2).sum() == 1


# ------------------------------------------------------------------------------------------
# O2: top-k + ordering (north_star step (2); "sorting", 210 "top-N retention")
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("top_k", [1, 5, 37, 500])
def test_o2_against_python_sorted_and_rank_count(top_k):
    S = quantised_map(40, 50, seed=3, levels=9)        # many equal scores -> index tie-break matters
    mask = oracle.nms_mask(S, 1, 0.2)
    K, idx, sc = oracle.topk(S, mask, top_k)
    cands = [(float(S.flat[p]), int(p)) for p in np.flatnonzero(mask.ravel())]
    ref = sorted(cands, key=lambda t: (-t[0], t[1]))    # library sort on the composite key
    assert K == min(top_k, len(cands))                  # G5
    assert [int(i) for i in idx[:K]] == [p for _, p in ref[:K]]
    assert np.array_equal(sc[:K], np.array([s for s, _ in ref[:K]], np.float32))
    assert np.all(idx[K:] == -1) and np.all(sc[K:] == 0)          # O5 padding
    # brute-force rank by counting: rank(i) = #{j : key_j better than key_i}
    for pos in range(K):
        s_i, p_i = float(sc[pos]), int(idx[pos])
        better = sum(1 for s, p in cands if (s > s_i) or (s == s_i and p < p_i))
        assert better == pos
    # invariants
    assert np.all(np.diff(sc[:K]) <= 0)
    eq = np.diff(sc[:K]) == 0
    assert np.all(np.diff(idx[:K])[eq] > 0)
    assert len(cands) > 37                               # the k < C branch is exercised


def test_o2_score_multiset_matches_torch_topk():
    S = rng(5).random((64, 64)).astype(np.float32)
    mask = oracle.nms_mask(S, 2, 0.5)
    K, idx, sc = oracle.topk(S, mask, 20)
    vals = torch.from_numpy(S.ravel()[mask.ravel() == 1])
    assert K == 20
    assert np.array_equal(sc[:K], torch.topk(vals, 20).values.numpy())
    assert np.array_equal(S.ravel()[idx[:K]], sc[:K])   # G7: reported score is the raw S at the peak


# ------------------------------------------------------------------------------------------
# O3: soft-argmax refinement (north_star step (3))
# ------------------------------------------------------------------------------------------
def window_map(r, centre, neighbours, fill=-1000.0, H=15, W=17, cy=7, cx=8):
    S = np.full((H, W), fill, np.float32)
    S[cy, cx] = centre
    for (i, j), v in neighbours.items():
        S[cy + j, cx + i] = v
    return S, cy * W + cx


def test_o3_closed_form_golden():
    rows = [l.split() for l in open(os.path.join(GOLD, "two_pixel_window.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) >= 5
    for i, j, delta, T, edx, edy in rows:
        i, j = int(i), int(j)
        c = np.float32(1.0)
        nb = np.float32(c - np.float32(float(delta)))
        S, idx = window_map(2, c, {(i, j): nb})
        off, kpt = oracle.refine(S, 2, float(T), np.array([idx], np.int32))
        # the fp32 inputs are what they are: closed form evaluated on the actual fp32 delta and T
        q = (float(c) - float(nb)) / float(np.float32(float(T)))
        a = i if i != 0 else j
        want = a / (1.0 + math.exp(q))
        got = off[0, 0] if i != 0 else off[0, 1]
        assert abs(got - want) < 1e-14
        assert abs(got - (float(edx) if i != 0 else float(edy))) < 2e-6    # golden (decimal delta)
        assert (off[0, 1] if i != 0 else off[0, 0]) == 0.0
        assert kpt[0, 0] == 8 + off[0, 0] and kpt[0, 1] == 7 + off[0, 1]   # (x,y) order (G10)


@pytest.mark.parametrize("r", [1, 2, 4])
def test_o3_symmetric_peak_is_exactly_zero(r):
    g = rng(r)
    H = W = 4 * r + 3
    cy = cx = 2 * r + 1
    yy, xx = np.mgrid[0:H, 0:W]
    rad2 = (yy - cy) ** 2 + (xx - cx) ** 2
    lut = g.random(rad2.max() + 1)
    S = (0.9 - 0.5 * lut[rad2] * (rad2 > 0)).astype(np.float32)   # any function of |d|^2: symmetric
    off, kpt = oracle.refine(S, r, 0.1, np.array([cy * W + cx], np.int32))
    assert off[0, 0] == 0.0 and off[0, 1] == 0.0
    assert kpt[0, 0] == cx and kpt[0, 1] == cy
    # constant window -> 0
    off, _ = oracle.refine(np.full((H, W), 0.3, np.float32), r, 0.1, np.array([cy * W + cx], np.int32))
    assert off[0, 0] == 0.0 and off[0, 1] == 0.0


@pytest.mark.parametrize("r", [1, 2, 4])
def test_o3_matches_independent_softmax_expectation_and_invariants(r):
    g = rng(10 + r)
    H, W = 33, 41
    for T in (0.1, 0.03, 1.0):
        S = g.random((H, W)).astype(np.float32)
        ys = g.integers(r, H - r, 50)
        xs = g.integers(r, W - r, 50)
        for y, x in zip(ys, xs):                        # make each centre the window max (O1 property)
            S[y, x] = S[y - r:y + r + 1, x - r:x + r + 1].max() + np.float32(0.01)
        idx = (ys * W + xs).astype(np.int32)
        off, kpt = oracle.refine(S, r, T, idx)
        Td = float(np.float32(T))
        ii = np.arange(-r, r + 1, dtype=np.float64)
        for t, (y, x) in enumerate(zip(ys, xs)):
            win = S[y - r:y + r + 1, x - r:x + r + 1].astype(np.float64)
            p = torch.softmax(torch.from_numpy(win.ravel() / Td), 0).numpy().reshape(win.shape)
            dx = (p * ii[None, :]).sum()                # expectation of i (columns)
            dy = (p * ii[:, None]).sum()                # expectation of j (rows)
            assert abs(off[t, 0] - dx) < 1e-12 and abs(off[t, 1] - dy) < 1e-12
            assert abs(off[t, 0]) <= r and abs(off[t, 1]) <= r
        # mirror: flipping the map left-right flips the sign of dx, dy unchanged (up to the
        # summation order inside Z and the row/column sums: a few ulp)
        Sm = np.ascontiguousarray(S[:, ::-1])
        idxm = (ys * W + (W - 1 - xs)).astype(np.int32)
        offm, _ = oracle.refine(Sm, r, T, idxm)
        assert np.allclose(offm[:, 0], -off[:, 0], rtol=0, atol=1e-15) and np.allclose(offm[:, 1], off[:, 1], rtol=0, atol=1e-15)
        Sv = np.ascontiguousarray(S[::-1, :])
        idxv = ((H - 1 - ys) * W + xs).astype(np.int32)
        offv, _ = oracle.refine(Sv, r, T, idxv)
        assert np.allclose(offv[:, 1], -off[:, 1], rtol=0, atol=1e-15) and np.allclose(offv[:, 0], off[:, 0], rtol=0, atol=1e-15)


def test_o3_temperature_limits():
    g = rng(77)
    r = 2
    S = (0.5 * g.random((9, 9))).astype(np.float32)
    S[4, 4] = 0.9
    idx = np.array([4 * 9 + 4], np.int32)
    off_hot, _ = oracle.refine(S, r, 1e6, idx)          # T -> inf: uniform weights -> centroid = 0
    assert np.all(np.abs(off_hot) < 1e-6)
    off_cold, _ = oracle.refine(S, r, 1e-3, idx)        # T -> 0: unique max dominates -> 0
    assert np.all(np.abs(off_cold) < 1e-100)
    assert np.all(oracle.refine(S, r, 0.1, idx)[0] != 0.0)


# ------------------------------------------------------------------------------------------
# O4: bilinear gather + L2 norm (north_star step (4))
# ------------------------------------------------------------------------------------------
def test_o4_affine_golden():
    rows = [l.split() for l in open(os.path.join(GOLD, "affine_bilinear.txt")) if l.strip() and l[0] != "#"]
    Hd, Wd = 9, 8
    v, u = np.mgrid[0:Hd, 0:Wd].astype(np.float64)
    Fm = np.stack([1 + 2 * u + 3 * v, 4 - u + 0.5 * v], -1).astype(np.float32)
    for s, px, py, d0, d1 in rows:
        out = oracle.gather(Fm, int(s), np.array([[float(px), float(py)]]))
        d = np.array([float(d0), float(d1)])
        assert np.allclose(out[0], d / np.linalg.norm(d), rtol=0, atol=1e-15)


@pytest.mark.parametrize("dtype", [np.float32, np.float16])
@pytest.mark.parametrize("stride", [1, 2, 8])
def test_o4_matches_grid_sample_library(dtype, stride):
    # library special case: grid_sample(bilinear, border, align_corners=False) with
    # grid = 2(px+0.5)/W - 1 samples at u = (px+0.5)/s - 0.5 with border clamping (G13)
    g = rng(stride)
    Hd, Wd, D = 13, 17, 8
    H, W = Hd * stride, Wd * stride
    Fm = g.standard_normal((Hd, Wd, D)).astype(dtype)
    n = 300
    kp = np.stack([g.uniform(-0.5, W - 0.5, n), g.uniform(-0.5, H - 0.5, n)], -1)
    kp[:4] = [[0, 0], [W - 1, H - 1], [0.25, H - 1], [W - 1, 0.75]]      # clamp cases
    out = oracle.gather(Fm, stride, kp)
    t = torch.from_numpy(Fm.astype(np.float64)).permute(2, 0, 1)[None]
    grid = torch.from_numpy(np.stack([2 * (kp[:, 0] + 0.5) / W - 1, 2 * (kp[:, 1] + 0.5) / H - 1], -1))
    samp = F.grid_sample(t, grid[None, None], mode="bilinear", padding_mode="border", align_corners=False)
    samp = samp[0, :, 0, :].T.numpy()
    want = samp / np.maximum(np.linalg.norm(samp, axis=1, keepdims=True), 1e-12)
    assert np.allclose(out, want, rtol=0, atol=1e-12)
    assert np.allclose(np.linalg.norm(out, axis=1), 1.0, atol=1e-12)      # unit norm (Eq. 1)


def test_o4_special_cases():
    g = rng(4)
    a = g.standard_normal(16)
    Fm = np.broadcast_to(a.astype(np.float32), (6, 7, 16)).copy()           # constant map -> a/|a| anywhere
    kp = np.stack([g.uniform(0, 6, 20), g.uniform(0, 5, 20)], -1)
    out = oracle.gather(Fm, 1, kp)
    a32 = a.astype(np.float32).astype(np.float64)
    assert np.allclose(out, a32 / np.linalg.norm(a32), atol=1e-15)
    Fm = g.standard_normal((6, 7, 16)).astype(np.float32)                   # zero offset at s=1 -> that pixel
    out = oracle.gather(Fm, 1, np.array([[3.0, 2.0]]))
    f = Fm[2, 3].astype(np.float64)
    assert np.allclose(out[0], f / np.linalg.norm(f), atol=1e-15)
    # x/y not transposed: pure x offset interpolates along the W axis
    out = oracle.gather(Fm, 1, np.array([[3.5, 2.0]]))
    f = 0.5 * (Fm[2, 3].astype(np.float64) + Fm[2, 4].astype(np.float64))
    assert np.allclose(out[0], f / np.linalg.norm(f), atol=1e-15)
    Z = np.zeros((4, 4, 8), np.float16)                                     # zero map -> zeros (G14)
    assert np.all(oracle.gather(Z, 1, np.array([[1.5, 1.5]])) == 0)
    # f16 maps are decoded exactly (incl. subnormals)
    hv = np.array([6.1e-5, 5.96e-8, -2.5, 65504.0, 1e-3, 0.333, -7e-6, 3.0], np.float16)
    Fh = np.broadcast_to(hv, (3, 3, 8)).copy()
    out = oracle.gather(Fh, 1, np.array([[1.0, 1.0]]))
    h64 = hv.astype(np.float64)
    assert np.allclose(out[0], h64 / np.linalg.norm(h64), rtol=1e-15, atol=0)
    # padding rows
    out = oracle.gather(Fm, 1, np.array([[1.0, 1.0], [2.0, 2.0]]), valid=np.array([5, -1], np.int32))
    assert np.all(out[1] == 0) and abs(np.linalg.norm(out[0]) - 1) < 1e-12


# ------------------------------------------------------------------------------------------
# Whole path: batch independence, translation, padding, count (north_star)
# ------------------------------------------------------------------------------------------
def blob_map(B, H, W, seed, nblobs=40):
    g = rng(seed)
    S = 0.1 * g.random((B, H, W))
    yy, xx = np.mgrid[0:H, 0:W]
    for b in range(B):
        for _ in range(nblobs):
            cx, cy = g.uniform(0, W), g.uniform(0, H)
            A, sg = g.uniform(0.3, 1.0), g.uniform(0.8, 2.0)
            S[b] += A * np.exp(-((xx - cx) ** 2 + (yy - cy) ** 2) / (2 * sg * sg))
    return np.clip(S, 0, 1).astype(np.float32)


def test_whole_path_invariants_and_batch_independence():
    B, H, W, D, k, r = 2, 48, 64, 16, 64, 2
    S = blob_map(B, H, W, seed=1)
    Fm = rng(2).standard_normal((B, H, W, D)).astype(np.float16)
    R = oracle.extract(S, Fm, 1, r, 0.2, k, 0.1)
    for b in range(B):
        Rb = oracle.extract(S[b:b + 1], Fm[b:b + 1], 1, r, 0.2, k, 0.1)       # G19
        for name in ("kpts", "offsets", "scores", "desc", "index"):
            assert np.array_equal(getattr(R, name)[b], getattr(Rb, name)[0]), name
        assert R.count[b] == Rb.count[0]
        K = int(R.count[b])
        C = int(oracle.nms_mask(S[b], r, 0.2).sum())
        assert K == min(k, C) and 0 < K < k                                    # count = min(top_k, candidates)
        assert np.all(np.abs(R.offsets[b]) <= r)
        assert np.allclose(np.linalg.norm(R.desc[b, :K], axis=1), 1.0, atol=1e-12)
        assert np.all(R.index[b, K:] == -1) and np.all(R.scores[b, K:] == 0)   # O5 / PAPER.md:139
        assert np.all(R.kpts[b, K:] == 0) and np.all(R.desc[b, K:] == 0) and np.all(R.offsets[b, K:] == 0)
        ys, xs = R.index[b, :K] // W, R.index[b, :K] % W
        assert np.array_equal(R.kpts[b, :K, 0], xs + R.offsets[b, :K, 0])
        assert np.array_equal(R.kpts[b, :K, 1], ys + R.offsets[b, :K, 1])
    # keypoints-only (LK pathway)
    R0 = oracle.extract(S, None, 1, r, 0.2, k, 0.1)
    assert R0.desc is None and np.array_equal(R0.kpts, R.kpts) and np.array_equal(R0.index, R.index)
    # top_k smaller than the candidate count
    R8 = oracle.extract(S, Fm, 1, r, 0.2, 8, 0.1)
    assert np.all(R8.count == 8) and np.array_equal(R8.index, R.index[:, :8])
    assert np.array_equal(R8.desc, R.desc[:, :8])


def test_whole_path_translation():
    H, W, r, k = 40, 48, 2, 32
    S = blob_map(1, H, W, seed=9, nblobs=25)[0]
    S[:r + 1] = 0; S[-r - 1:] = 0; S[:, :r + 1] = 0; S[:, -r - 1:] = 0      # keep peaks off the border
    a, b2, H2, W2 = 5, 7, 64, 80
    Sbig = np.zeros((H2, W2), np.float32)
    Sbig[b2:b2 + H, a:a + W] = S
    R1 = oracle.extract(S[None], None, 1, r, 0.2, k, 0.1)
    R2 = oracle.extract(Sbig[None], None, 1, r, 0.2, k, 0.1)
    K = int(R1.count[0])
    assert K == int(R2.count[0]) and K > 5
    # (score desc, idx asc) order can permute among equal scores after a shift only if the
    # relative index order changes; compare as sets keyed by position
    p1 = {(int(i % W) + a, int(i // W) + b2): (float(s), tuple(o)) for i, s, o in
          zip(R1.index[0, :K], R1.scores[0, :K], R1.offsets[0, :K])}
    p2 = {(int(i % W2), int(i // W2)): (float(s), tuple(o)) for i, s, o in
          zip(R2.index[0, :K], R2.scores[0, :K], R2.offsets[0, :K])}
    assert p1 == p2


def test_extract_rejects_bad_arguments():
    S = np.zeros((1, 8, 8), np.float32)
    with pytest.raises(ValueError):
        oracle.extract(S, None, 1, 0, 0.2, 4, 0.1)
    with pytest.raises(ValueError):
        oracle.extract(S, None, 1, 2, 0.2, 4, 0.0)
    with pytest.raises(ValueError):
        oracle.extract(S, None, 1, 2, 0.2, 0, 0.1)
