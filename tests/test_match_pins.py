"""Pins for the matching / retrieval / stereo-validation / covariance oracle (oracle/match_oracle.c; SURVEY.md
8(f) f3, f4; M1..M8, S1..S4, C1..C4) against things other than itself: brute-force python loops,
torch library routines on float64, planted sets, closed forms worked by hand (tests/golden/chol2x2.txt).
Citations: /root/reference/PAPER.md:157 (cosine NN + Lowe ratio), 151-153 Eq. 4, 348 (skip 50, tau 0.60),
145 (stereo gates), 586-603 Eq. 9-11 (covariance weighting)."""
import math
import os

import numpy as np
import pytest
import torch

import oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def unit_rows(n, D, seed, dtype=np.float32):
    g = np.random.default_rng(seed)
    x = g.standard_normal((n, D))
    x /= np.linalg.norm(x, axis=1, keepdims=True)
    return x.astype(dtype)


# ---- (1) cosine nearest neighbour + Lowe ratio + mutual check -------------------------------------------
def brute_match(A, B, na, nb, ratio, mutual):
    A = A.astype(np.float64)
    B = B.astype(np.float64)
    out = []
    for i in range(A.shape[0]):
        if i >= na or nb == 0:
            out.append((-1, 0.0, 0.0))
            continue
        sims = [sum(A[i, c] * B[j, c] for c in range(A.shape[1])) for j in range(nb)]
        j1 = max(range(nb), key=lambda j: (sims[j], -j))                  # ties -> smallest j
        s1 = sims[j1]
        rest = [sims[j] for j in range(nb) if j != j1]
        s2 = max(rest) if rest else -1.0
        keep = max(0.0, 2 - 2 * s1) < ratio * ratio * max(0.0, 2 - 2 * s2) if ratio < 1e9 else True
        if keep and mutual:
            col = [sum(A[ii, c] * B[j1, c] for c in range(A.shape[1])) for ii in range(na)]
            keep = max(range(na), key=lambda ii: (col[ii], -ii)) == i
        out.append((j1 if keep else -1, s1, s2))
    return out


@pytest.mark.parametrize("dtype", [np.float32, np.float16])
@pytest.mark.parametrize("mutual", [False, True])
def test_m_bruteforce_tiny(dtype, mutual):
    for seed in range(3):
        A = unit_rows(9, 8, seed, dtype)
        B = unit_rows(7, 8, 100 + seed, dtype)
        B[2] = A[4]                                                       # a planted duplicate
        for na, nb in ((9, 7), (6, 5), (9, 1), (0, 7)):
            idx, s1, s2 = oracle.match_nn(A, B, na, nb, ratio=0.9, mutual=mutual)
            ref = brute_match(A, B, na, nb, 0.9, mutual)
            assert [int(i) for i in idx] == [r[0] for r in ref]
            assert np.allclose(s1, [r[1] for r in ref], atol=1e-14) and np.allclose(s2, [r[2] for r in ref], atol=1e-14)


def test_m_against_torch_topk_on_float64_matmul():
    A = unit_rows(200, 64, 1, np.float16)
    B = unit_rows(300, 64, 2, np.float16)
    noisy = A[:150].astype(np.float64) + 0.15 * unit_rows(150, 64, 3)                          # true matches + noise,
    B[:150] = (noisy / np.linalg.norm(noisy, axis=1, keepdims=True)).astype(np.float16)        # l2-normalised (Eq. 1)
    idx, s1, s2, S = oracle.match_nn(A, B, ratio=1e9, want_sim=True)
    St = torch.from_numpy(A.astype(np.float64)) @ torch.from_numpy(B.astype(np.float64)).T
    assert np.abs(S - St.numpy()).max() < 1e-13
    top = torch.topk(St, 2, dim=1)
    assert np.array_equal(idx, top.indices[:, 0].numpy().astype(np.int32))   # (no exact ties in this data)
    assert np.allclose(s1, top.values[:, 0].numpy(), atol=1e-13) and np.allclose(s2, top.values[:, 1].numpy(), atol=1e-13)
    # ratio test == the test on Euclidean distances computed independently
    for rho in (0.6, 0.8, 0.95):
        got, _, _ = oracle.match_nn(A, B, ratio=rho)
        d = torch.cdist(torch.from_numpy(A.astype(np.float64)), torch.from_numpy(B.astype(np.float64)))
        dd = torch.topk(d, 2, dim=1, largest=False)
        keep = (dd.values[:, 0] < rho * dd.values[:, 1]).numpy()
        # cdist uses the descriptors as stored (f16-rounded: unit norm to ~1e-3 only): compare where the margin is clear
        clear = np.abs(dd.values[:, 0].numpy() - rho * dd.values[:, 1].numpy()) > 5e-3
        assert np.array_equal((got >= 0)[clear], keep[clear])
        assert (got[:150] >= 0).mean() > 0.9 or rho < 0.7


def test_m_planted_duplicates_orthogonal_ties_padding():
    D = 16
    E = np.eye(D, dtype=np.float32)
    # exact duplicates: sim 1, distance 0 -> always passes the ratio test
    idx, s1, s2 = oracle.match_nn(E[:5], E[[3, 0, 4, 1, 2]], ratio=0.8)
    assert [int(i) for i in idx] == [1, 3, 4, 0, 2] and np.all(s1 == 1.0) and np.all(s2 == 0.0)
    # orthogonal sets: every sim 0 -> nearest = smallest j (tie rule), d1 == d2 -> ratio test rejects
    idx, s1, s2 = oracle.match_nn(E[:4], E[8:12], ratio=0.8)
    assert np.all(idx == -1) and np.all(s1 == 0) and np.all(s2 == 0)
    idx, _, _ = oracle.match_nn(E[:4], E[8:12], ratio=1e9)
    assert np.all(idx == 0)
    # exact tie between two columns: the smaller index wins, and the ratio test rejects (d1 == d2)
    B = np.stack([E[1], E[0], E[0]])
    idx, s1, s2 = oracle.match_nn(E[:1], B, ratio=1e9)
    assert idx[0] == 1 and s1[0] == 1.0 and s2[0] == 1.0
    assert oracle.match_nn(E[:1], B, ratio=0.99)[0][0] == -1
    # mutual check: rows 0 and 1 both prefer column 0; only the better one keeps it
    A = np.stack([E[0], (0.8 * E[0] + 0.6 * E[1]).astype(np.float32)])
    B = np.stack([E[0], E[5]])
    assert [int(i) for i in oracle.match_nn(A, B, ratio=1e9)[0]] == [0, 0]
    assert [int(i) for i in oracle.match_nn(A, B, ratio=1e9, mutual=True)[0]] == [0, -1]
    # zero padding: rows >= na report -1 / 0 / 0 and columns >= nb are never matched
    A = np.zeros((6, D), np.float32)
    A[:3] = E[:3]
    B = np.zeros((5, D), np.float32)
    B[:2] = E[[2, 7]]
    idx, s1, s2 = oracle.match_nn(A, B, na=3, nb=2, ratio=1e9)
    assert [int(i) for i in idx] == [0, 0, 0, -1, -1, -1] and np.all(s1[3:] == 0) and np.all(s2[3:] == 0)
    assert s1[2] == 1.0
    # the Lowe test on hand numbers: s1 = 0.9, s2 = 0.5 -> d1^2 = 0.2, d2^2 = 1.0: kept iff rho^2 > 0.2
    a = E[0]
    B = np.stack([(0.9 * E[0] + math.sqrt(1 - 0.81) * E[1]), (0.5 * E[0] + math.sqrt(0.75) * E[2])]).astype(np.float64)
    A64 = a[None].astype(np.float32)
    B32 = B.astype(np.float32)
    assert oracle.match_nn(A64, B32, ratio=0.46)[0][0] == 0              # 0.46^2 = 0.2116 > 0.2
    assert oracle.match_nn(A64, B32, ratio=0.44)[0][0] == -1             # 0.44^2 = 0.1936 < 0.2


# ---- (2) retrieval scan ----------------------------------------------------------------------------------
def test_r_bruteforce_and_topk():
    D, n = 96, 400
    db = unit_rows(n, D, 5, np.float16)
    q = unit_rows(1, D, 6, np.float16)[0]
    for k in (10, 50, 120, 360, 399):                                     # planted revisits, one inside the recent window
        db[k] = (0.8 * q.astype(np.float64) + 0.6 * unit_rows(1, D, k)[0] * 0.5).astype(np.float16)
    sim, cand, K = oracle.retrieval_scan(db, q, n_exclude=50, tau=0.60, max_cand=8)
    ref = [sum(float(q[e]) * float(db[k, e]) for e in range(D)) for k in range(n)]
    assert np.allclose(sim, ref, atol=1e-13)
    elig = [(s, k) for k, s in enumerate(ref) if k < n - 50 and s > 0.60]
    elig.sort(key=lambda t: (-t[0], t[1]))
    assert K == min(8, len(elig)) and [int(c) for c in cand[:K]] == [k for _, k in elig[:K]]
    assert np.all(cand[K:] == -1)
    assert 360 not in cand and 399 not in cand and 10 in cand            # the recent window is excluded
    # library routine on float64
    st = torch.from_numpy(db.astype(np.float64)) @ torch.from_numpy(q.astype(np.float64))
    assert np.abs(st.numpy() - sim).max() < 1e-13
    # truncation, strict gate, empty database, window larger than the database
    _, c2, K2 = oracle.retrieval_scan(db, q, 50, 0.60, 2)
    assert K2 == 2 and [int(c) for c in c2] == [k for _, k in elig[:2]]
    top = max(s for s, _ in elig)
    assert oracle.retrieval_scan(db, q, 50, top, 8)[2] == 0              # sim == tau is NOT a candidate
    assert oracle.retrieval_scan(db[:0], q, 50, 0.6, 4)[2] == 0
    assert oracle.retrieval_scan(db[:30], q, 50, -1.0, 4)[2] == 0
    # ties -> the older keyframe (smaller k) first
    db2 = np.stack([q, q, q]).astype(np.float16)
    assert [int(c) for c in oracle.retrieval_scan(db2, q, 0, 0.5, 3)[1]] == [0, 1, 2]


# ---- (3) stereo validation ---------------------------------------------------------------------------------
def test_s_planted_points_round_trip_and_gates():
    fx, fy, cx, cy, bl = 458.0, 457.0, 367.0, 248.0, 0.11
    g = np.random.default_rng(0)
    P = np.stack([g.uniform(-2, 2, 50), g.uniform(-1, 1, 50), g.uniform(0.5, 20, 50)], 1)   # 3-D points, left frame
    pl = np.stack([fx * P[:, 0] / P[:, 2] + cx, fy * P[:, 1] / P[:, 2] + cy], 1)
    pr = np.stack([fx * (P[:, 0] - bl) / P[:, 2] + cx, fy * P[:, 1] / P[:, 2] + cy], 1)
    valid, xyz, disp, err = oracle.stereo_validate(pl, pr, fx, fy, cx, cy, bl, 0.5, 0.3, 30.0)
    assert np.allclose(xyz, P, atol=1e-9) and np.allclose(disp, fx * bl / P[:, 2]) and np.all(err < 1e-9)
    assert np.array_equal(valid, (disp > 0.5).astype(np.uint8))
    # vertical disagreement dv: the least-squares point sits half way, so each view is off by dv / 2
    pr2 = pr.copy()
    pr2[:, 1] += 2.0
    v2, xyz2, _, err2 = oracle.stereo_validate(pl, pr2, fx, fy, cx, cy, bl, 0.0, 0.3, 30.0)
    assert np.allclose(err2, 1.0) and np.all(v2 == 1)
    pr2[:, 1] += 1.2                                                      # dv = 3.2 -> 1.6 px > 1.5
    assert oracle.stereo_validate(pl, pr2, fx, fy, cx, cy, bl, 0.0, 0.3, 30.0)[0].sum() == 0
    # gates one at a time
    one_l, one_r = np.array([[400.0, 250.0]]), np.array([[390.0, 250.0]])   # d = 10 -> z = 458 * 0.11 / 10 = 5.038
    z = fx * bl / 10.0
    assert oracle.stereo_validate(one_l, one_r, fx, fy, cx, cy, bl, 1.0, 0.3, 30.0)[0][0] == 1
    assert oracle.stereo_validate(one_l, one_r, fx, fy, cx, cy, bl, 10.0, 0.3, 30.0)[0][0] == 0    # d <= d_min: negligible
    assert oracle.stereo_validate(one_l, one_r, fx, fy, cx, cy, bl, 1.0, 0.3, z)[0][0] == 0        # z < z_max strict
    assert oracle.stereo_validate(one_l, one_r, fx, fy, cx, cy, bl, 1.0, z, 30.0)[0][0] == 0
    assert oracle.stereo_validate(one_r, one_l, fx, fy, cx, cy, bl, -100.0, 0.3, 30.0)[0][0] == 0  # negative depth
    xyz1 = oracle.stereo_validate(one_l, one_r, fx, fy, cx, cy, bl, 1.0, 0.3, 30.0)[1][0]
    assert np.allclose(xyz1, [(400 - cx) * z / fx, (250 - cy) * z / fy, z])


# ---- (4) covariance-weighted square-root information -------------------------------------------------------
def test_c_golden_cholesky_by_hand():
    rows = [l.split() for l in open(os.path.join(GOLD, "chol2x2.txt")) if l.strip() and not l.startswith("#")]
    for r in rows:
        l11, l21, l22, scale, flo, fx, fy, lam, lmin, s0 = map(float, r[:10])
        want = np.array(list(map(float, r[10:14]))).reshape(2, 2)
        om, ok = oracle.cov_sqrt_info(np.array([[l11, l21, l22]]), scale, flo, fx, fy, lam, lmin, s0)
        assert ok[0] == int(float(r[14])), r
        assert np.allclose(om[0], want, rtol=1e-12, atol=1e-12), (om[0], want)


def test_c_properties_and_fallback():
    g = np.random.default_rng(4)
    Lf = np.stack([g.uniform(0.2, 3, 100), g.uniform(-2, 2, 100), g.uniform(0.2, 3, 100)], 1)
    scale, flo, fx, fy, lam, lmin, s0 = 1.25, 0.01, 460.0, 455.0, 0.3, 0.05, 1.5 / 460.0
    om, ok = oracle.cov_sqrt_info(Lf, scale, flo, fx, fy, lam, lmin, s0)
    assert ok.all()
    for i in range(100):
        L = np.array([[Lf[i, 0], 0], [Lf[i, 1], Lf[i, 2]]])
        Spx = scale ** 2 * (L @ L.T) + flo * np.eye(2)
        J = np.diag([1 / fx, 1 / fy])
        Sn = J @ Spx @ J.T
        info = lam * np.linalg.inv(Sn)                                    # Eq. 11
        assert np.allclose(om[i].T @ om[i], info, rtol=1e-9)              # Omega^T Omega = Sigma_eff^-1 (Eq. 10)
        assert om[i][1, 0] == 0 and om[i][0, 0] > 0 and om[i][1, 1] > 0   # upper triangular
        assert np.allclose(om[i], np.linalg.cholesky(info).T, rtol=1e-9)  # library Cholesky
        r = g.standard_normal(2)
        assert math.isclose(float(np.sum((om[i] @ r) ** 2)), float(r @ info @ r), rel_tol=1e-9)
    # lower clamp on the gain
    a, _ = oracle.cov_sqrt_info(Lf[:3], scale, flo, fx, fy, 0.001, 0.05, s0)
    b, _ = oracle.cov_sqrt_info(Lf[:3], scale, flo, fx, fy, 0.05, 0.05, s0)
    assert np.array_equal(a, b)
    # isotropic covariance sigma^2 I with lambda = 1 recovers 1/sigma_n on the diagonal
    om1, _ = oracle.cov_sqrt_info(np.array([[2.0, 0.0, 2.0]]), 1.0, 0.0, 400.0, 400.0, 1.0, 0.0, 1.0)
    assert np.allclose(om1[0], np.eye(2) * 400.0 / 2.0)
    # failures -> isotropic fallback sigma0^-1 I, flag 0
    bad = np.array([[0.0, 1.0, 0.0], [1.0, 1.0, 0.0], [np.nan, 0.0, 1.0], [np.inf, 0.0, 1.0]])
    omb, okb = oracle.cov_sqrt_info(bad, 1.0, 0.0, fx, fy, 0.5, 0.05, 0.25)
    assert not okb.any() and np.allclose(omb, np.eye(2)[None] * 4.0)
    # ... and the optional floor rescues a singular prediction
    omf, okf = oracle.cov_sqrt_info(bad[:2], 1.0, 0.5, fx, fy, 0.5, 0.05, 0.25)
    assert okf.all()
