"""Pins for the DKD-variant oracle (oracle/dkd_variants.c, V1..V5) against things
other than itself: an independent torch restatement with library max-pooling, torch grid_sample, python filters
of the (already pinned) base oracle, planted cases.  Each pin is chosen so that a plausible mistake (mask
applied before the window maximum, product formed after it, recovery without the suppression mask, x/y swapped in
the interpolation) fails it.  Citations: /root/reference/PAPER.md:120 (original PyTorch NMS), 89-95 (heat x
reliability), 326 (validity mask), 101 (scores)."""
import numpy as np
import pytest
import torch
import torch.nn.functional as F

import oracle
import synth


def quantised_map(H, W, seed, levels=12):
    g = np.random.default_rng(seed)
    return (g.integers(0, levels, size=(H, W)) / float(levels)).astype(np.float32)


# ---- V1: iterated suppress-and-recover NMS ---------------------------------------------------------------
def torch_iterated_nms(S, r, iters):
    """The published iterative max-pool NMS restated with the library routine (max_pool2d pads with -inf, i.e.
    the window is clipped at the image edge)."""
    t = torch.from_numpy(S)[None, None].double()
    mp = lambda x: F.max_pool2d(x, 2 * r + 1, 1, r)
    M = t == mp(t)
    for _ in range(iters):
        supp = mp(M.double()) > 0
        Sp = torch.where(supp, torch.zeros_like(t), t)
        M = M | ((Sp == mp(Sp)) & ~supp)
    return M[0, 0].numpy()


@pytest.mark.parametrize("r", [1, 2, 3])
@pytest.mark.parametrize("iters", [0, 1, 2, 3])
def test_v1_equals_torch_restatement(r, iters):
    for seed in range(3):
        S = quantised_map(37, 45, seed=10 * r + seed, levels=30)
        S += (np.random.default_rng(seed).random(S.shape) < 0.4).astype(np.float32) * np.float32(1 / 64)
        M = torch_iterated_nms(S, r, iters)
        inner = np.zeros_like(M)
        inner[r:S.shape[0] - r, r:S.shape[1] - r] = True
        want = (M & inner & (S > np.float32(0.3))).astype(np.uint8)
        assert np.array_equal(oracle.nms_mask_iter(S, r, 0.3, iters), want)


def test_v1_zero_iterations_is_the_single_pass():
    for seed in range(4):
        S = synth.score_maps(1, 60, 80, 50 + seed, 0.1, 80)[0].numpy()
        for r in (1, 2, 4):
            assert np.array_equal(oracle.nms_mask_iter(S, r, 0.2, 0), oracle.nms_mask(S, r, 0.2))


def test_v1_planted_recovery_chain():
    # A > B > C on one row, r = 2: B is within A's window, C within B's but not A's.  Single pass: only A
    # (C is suppressed by B).  One recovery round: B lies in the suppression zone of A and is zeroed, so C
    # becomes the maximum of its window and is recovered; B never is (it sits inside the suppression mask).
    r = 2
    S = np.zeros((11, 21), np.float32)
    S[5, 6], S[5, 8], S[5, 10] = 0.9, 0.8, 0.7
    m0 = oracle.nms_mask_iter(S, r, 0.2, 0)
    assert m0.sum() == 1 and m0[5, 6] == 1
    m1 = oracle.nms_mask_iter(S, r, 0.2, 1)
    assert m1.sum() == 2 and m1[5, 6] == 1 and m1[5, 10] == 1 and m1[5, 8] == 0
    # a longer chain A > B > C > D > E (spacing 2): one round recovers C only (D is suppressed by C in S'),
    # the second round recovers E
    S[5, 12], S[5, 14] = 0.6, 0.5
    assert [int(x) for x in np.flatnonzero(oracle.nms_mask_iter(S, r, 0.2, 1)[5])] == [6, 10]
    assert [int(x) for x in np.flatnonzero(oracle.nms_mask_iter(S, r, 0.2, 2)[5])] == [6, 10, 14]


# ---- V2: score interpolated at the refined point ---------------------------------------------------------
def test_v2_matches_grid_sample_and_python():
    g = np.random.default_rng(3)
    S = g.random((23, 31)).astype(np.float32)
    H, W = S.shape
    pts = np.stack([g.uniform(0, W - 1, 200), g.uniform(0, H - 1, 200)], 1)
    pts[:4] = [[0, 0], [W - 1, H - 1], [W - 1, 0.5], [3.25, H - 1]]          # edges: second corner clamped
    got = np.array([oracle.bilinear_score(S, x, y) for x, y in pts])
    # library routine: align_corners=True maps pixel centre i to -1 + 2 i / (n - 1)
    grid = torch.from_numpy(np.stack([2 * pts[:, 0] / (W - 1) - 1, 2 * pts[:, 1] / (H - 1) - 1], 1))[None, None]
    want = F.grid_sample(torch.from_numpy(S).double()[None, None], grid, mode="bilinear", padding_mode="border",
                         align_corners=True)[0, 0, 0].numpy()
    assert np.abs(got - want).max() < 1e-12
    # python by hand, x and y not interchangeable: an x-only ramp
    R = np.tile(np.arange(W, dtype=np.float32), (H, 1))
    assert abs(oracle.bilinear_score(R, 4.25, 9.75) - 4.25) < 1e-12
    assert abs(oracle.bilinear_score(R.T.copy(), 4.25, 9.75) - 9.75) < 1e-12


def test_v2_whole_path_symmetric_peak_keeps_raw_score_and_others_interpolate():
    S = np.zeros((1, 21, 25), np.float32)
    S[0, 10, 12] = 0.8
    S[0, 10, 11] = S[0, 10, 13] = S[0, 9, 12] = S[0, 11, 12] = 0.3       # symmetric -> offset exactly 0
    S[0, 4, 5] = 0.9
    S[0, 4, 6] = 0.6                                                      # asymmetric -> dx > 0
    raw = oracle.extract_var(S, None, 1, 2, 0.2, 4, 0.1, score_mode=0)
    bil = oracle.extract_var(S, None, 1, 2, 0.2, 4, 0.1, score_mode=1)
    assert np.array_equal(raw.index, bil.index) and np.array_equal(raw.kpts, bil.kpts)   # selection unaffected
    i_sym = list(raw.index[0]).index(10 * 25 + 12)
    assert bil.scores[0, i_sym] == raw.scores[0, i_sym] == np.float32(0.8)
    i_asym = list(raw.index[0]).index(4 * 25 + 5)
    dx, dy = raw.offsets[0, i_asym]
    assert dx > 0 and dy == 0
    want = (1 - dx) * float(np.float32(0.9)) + dx * float(np.float32(0.6))
    assert abs(bil.scores[0, i_asym] - want) < 1e-12 and bil.scores[0, i_asym] < raw.scores[0, i_asym]


# ---- V3: threshold-only mode (total count beside the capped count) --------------------------------------
def test_v3_total_and_capped_count():
    S = synth.score_maps(2, 64, 96, 7, 0.1, 90).numpy()
    for cap in (8, 4096):
        R = oracle.extract_var(S, None, 1, 2, 0.2, cap, 0.1)
        for b in range(2):
            C = int(oracle.nms_mask(S[b], 2, 0.2).sum())
            assert R.total[b] == C and R.count[b] == min(C, cap)
    base = oracle.extract(S, None, 1, 2, 0.2, 64, 0.1)
    var = oracle.extract_var(S, None, 1, 2, 0.2, 64, 0.1)
    assert np.array_equal(base.index, var.index) and np.array_equal(base.kpts, var.kpts)
    assert np.array_equal(base.scores.astype(np.float64), var.scores)


# ---- V4: heat x reliability ------------------------------------------------------------------------------
def test_v4_equals_base_path_on_the_fp32_product_map():
    heat = synth.score_maps(2, 48, 72, 11, 0.1, 60).numpy()
    rel = np.random.default_rng(5).random(heat.shape).astype(np.float32)
    desc = synth.desc_maps(2, 48, 72, 16, 4, torch.float32).numpy()
    prod = heat * rel                                                     # numpy float32 multiply: one rounding
    assert prod.dtype == np.float32
    got = oracle.extract_var(heat, desc, 1, 2, 0.05, 40, 0.1, reliability=rel)
    want = oracle.extract(prod, desc, 1, 2, 0.05, 40, 0.1)
    assert np.array_equal(got.index, want.index) and np.array_equal(got.count, want.count)
    assert np.array_equal(got.scores, want.scores.astype(np.float64))
    assert np.array_equal(got.kpts, want.kpts) and np.array_equal(got.desc, want.desc)
    # the product is formed BEFORE the window maximum: NMS on the heat alone gives another answer
    heat_only = oracle.extract(heat, None, 1, 2, 0.05, 40, 0.1)
    assert not np.array_equal(heat_only.index, got.index)


def test_v4_planted():
    heat = np.zeros((1, 15, 17), np.float32)
    heat[0, 7, 8] = 0.9
    heat[0, 7, 9] = 0.5
    ones = np.ones_like(heat)
    assert oracle.extract_var(heat, None, 1, 2, 0.2, 4, 0.1, reliability=ones).index[0, 0] == 7 * 17 + 8
    rel = ones.copy()
    rel[0, 7, 8] = 0.0                                                    # unreliable peak: gone, its neighbour wins
    R = oracle.extract_var(heat, None, 1, 2, 0.2, 4, 0.1, reliability=rel)
    assert R.count[0] == 1 and R.index[0, 0] == 7 * 17 + 9 and R.scores[0, 0] == np.float32(0.5)
    rel[0, 7, 9] = 0.3                                                    # 0.5 * 0.3 = 0.15 < thresh
    assert oracle.extract_var(heat, None, 1, 2, 0.2, 4, 0.1, reliability=rel).count[0] == 0


# ---- V5: validity mask -----------------------------------------------------------------------------------
def test_v5_is_a_filter_on_candidate_centres_only():
    S = synth.score_maps(2, 56, 88, 21, 0.1, 120).numpy()
    g = np.random.default_rng(9)
    vm = (g.random(S.shape) < 0.6).astype(np.uint8)
    top_k = 30
    got = oracle.extract_var(S, None, 1, 2, 0.2, top_k, 0.1, valid_mask=vm)
    for b in range(2):
        m = oracle.nms_mask(S[b], 2, 0.2)                                 # base candidates (pinned elsewhere)
        cands = [(float(S[b].flat[p]), int(p)) for p in np.flatnonzero(m.ravel()) if vm[b].flat[p]]
        ref = sorted(cands, key=lambda t: (-t[0], t[1]))[:top_k]
        assert got.count[b] == len(ref) and got.total[b] == len(cands)
        assert [int(i) for i in got.index[b, :len(ref)]] == [p for _, p in ref]
    ones = np.ones_like(vm)
    base = oracle.extract(S, None, 1, 2, 0.2, top_k, 0.1)
    allv = oracle.extract_var(S, None, 1, 2, 0.2, top_k, 0.1, valid_mask=ones)
    assert np.array_equal(base.index, allv.index)
    assert oracle.extract_var(S, None, 1, 2, 0.2, top_k, 0.1, valid_mask=0 * ones).count.sum() == 0


def test_v5_masked_neighbour_still_suppresses():
    S = np.zeros((1, 15, 17), np.float32)
    S[0, 7, 8] = 0.9
    S[0, 7, 9] = 0.5
    vm = np.ones(S.shape, np.uint8)
    vm[0, 7, 8] = 0                                                       # the stronger pixel is outside the valid area
    R = oracle.extract_var(S, None, 1, 2, 0.2, 4, 0.1, valid_mask=vm)
    assert R.count[0] == 0                                                # ... and still suppresses its neighbour


def test_variants_compose():
    heat = synth.score_maps(1, 40, 60, 31, 0.1, 50).numpy()
    rel = np.random.default_rng(1).random(heat.shape).astype(np.float32)
    vm = (np.random.default_rng(2).random(heat.shape) < 0.7).astype(np.uint8)
    R = oracle.extract_var(heat, None, 1, 2, 0.05, 20, 0.1, reliability=rel, valid_mask=vm, nms_iters=2, score_mode=1)
    prod = heat * rel
    m = oracle.nms_mask_iter(prod[0], 2, 0.05, 2) & vm[0]
    assert R.total[0] == m.sum()
    K = int(R.count[0])
    assert K == min(20, m.sum()) and all(m.flat[i] for i in R.index[0, :K])
    for i in range(K):
        assert abs(R.scores[0, i] - oracle.bilinear_score(prod[0], *R.kpts[0, i])) < 1e-12
