"""GPU parity of the descriptor consumers against oracle/match_oracle.c on the same seeded
inputs: dkd_match (tcgen05 similarity + fused top-2 + Lowe ratio + mutual check), dkd_retrieval_scan, dkd_stereo_validate,
dkd_cov_sqrt_info.

Tolerances (derived in DESIGN.md "Matching"):
  * similarities of dkd_match: fp16 x fp16 products are exact in fp32; the tensor core accumulates D <= 256 of them in
    fp32 -> |err| <= D * 2^-23 * sum|a_i b_i| <= 3.1e-5 for unit vectors; TOL_SIM = 1e-4 against the fp64 oracle;
  * an ARGMAX decided in fp32 can differ from the fp64 one only between columns whose fp64 similarities are within
    2 * TOL_SIM of the maximum: the GPU index must be one of those columns, and must equal the oracle's when there is
    only one; ratio / mutual decisions are compared where the fp64 margin exceeds the propagated tolerance;
  * retrieval similarities: fp32 accumulation of 12288 products in a fixed tree -> TOL_SCAN = 2e-5;
  * stereo / covariance: fp32 arithmetic against fp64, relative 2e-5.
"""
import numpy as np
import pytest
import torch

import oracle
import synth

pytestmark = pytest.mark.gpu
TOL_SIM = 1e-4
TOL_SCAN = 2e-5


@pytest.fixture(scope="module")
def ctx():
    import paper_2607_01757_b200 as dkd
    c = dkd.DKD(max_batch=2, max_h=64, max_w=128, max_top_k=64, max_dim=0)
    yield c
    c.close()


def check_pair(A, B, na, nb, ratio, mutual, nn_idx, nn_sim, dec_idx, rows=None):
    """A [Na,D], B [Nb,D] f16 numpy; nn_*: GPU result with the ratio test off and no mutual check; dec_idx: GPU result with
    (ratio, mutual).  `rows`: subset of A rows to check (default all)."""
    Na = A.shape[0]
    rows = np.arange(Na) if rows is None else np.asarray(rows)
    live = rows[rows < na]
    idx_o, s1_o, s2_o, S = oracle.match_nn(A[live], B, len(live), nb, ratio=1e9, want_sim=True)
    amb = 0
    for t, i in enumerate(live):
        near = np.flatnonzero(S[t] >= S[t].max() - 2 * TOL_SIM)
        assert nn_idx[i] in near, (i, nn_idx[i], near)
        if len(near) == 1:
            assert nn_idx[i] == idx_o[t]
        assert abs(nn_sim[i, 0] - s1_o[t]) <= TOL_SIM and abs(nn_sim[i, 1] - s2_o[t]) <= TOL_SIM, (i, nn_sim[i], s1_o[t], s2_o[t])
        # decisions: compare where the fp64 margins are clear
        d1, d2 = max(0.0, 2 - 2 * s1_o[t]), max(0.0, 2 - 2 * s2_o[t])
        margin = ratio * ratio * d2 - d1
        clear = abs(margin) > 2 * TOL_SIM * (1 + ratio * ratio) * 2 and len(near) == 1
        keep = margin > 0
        if mutual and keep and clear:
            col = (A[:na].astype(np.float64) @ B[idx_o[t]].astype(np.float64))
            cnear = np.flatnonzero(col >= col.max() - 2 * TOL_SIM)
            if len(cnear) == 1:
                keep = cnear[0] == i
            else:
                clear = False
        if clear:
            assert (dec_idx[i] == idx_o[t]) if keep else (dec_idx[i] == -1), (i, dec_idx[i], idx_o[t], keep, margin)
        else:
            amb += 1
    dead = rows[rows >= na]
    assert np.all(nn_idx[dead] == -1) and np.all(dec_idx[dead] == -1) and np.all(nn_sim[dead] == 0)   # padding rows
    return amb, len(live)


@pytest.mark.parametrize("D", [64, 128, 256])
@pytest.mark.parametrize("shape", [(300, 260), (128, 128), (513, 1100), (97, 40)])
@pytest.mark.parametrize("mutual", [False, True])
def test_match_small_and_ragged(ctx, D, shape, mutual):
    Na, Nb = shape
    ca, cb = [Na - 17, Na], [Nb, max(Nb - 33, 1)]
    A, B, cta, ctb = synth.match_sets(2, Na, Nb, D, seed=D + Na + int(mutual), count_a=ca, count_b=cb)
    Ad, Bd, cad, cbd = A.cuda(), B.cuda(), cta.cuda(), ctb.cuda()
    nn, nsim = ctx.match(Ad, Bd, cad, cbd, ratio=1e9, mutual=False)
    dec, _ = ctx.match(Ad, Bd, cad, cbd, ratio=0.8, mutual=mutual)
    torch.cuda.synchronize()
    amb = tot = 0
    for p in range(2):
        a, n = check_pair(A[p].numpy(), B[p].numpy(), ca[p], cb[p], 0.8, mutual, nn[p].cpu().numpy(), nsim[p].cpu().numpy(),
                          dec[p].cpu().numpy())
        amb, tot = amb + a, tot + n
    assert amb <= 0.03 * tot + 2                                  # the comparison is not vacuous
    assert (dec >= 0).sum() > 0.3 * min(Na, Nb)                   # the planted matches are found


@pytest.mark.parametrize("D", [64, 192, 256])
@pytest.mark.parametrize("mutual", [False, True])
def test_match_wide_tiles_ragged(ctx, D, mutual):
    """Sizes at which the kernel takes its 256-column tiles (row blocks x pairs x 256-wide tiles fill the machine) with
    set sizes that are multiples of neither 128 nor 256 and ragged counts; ~160 rows per pair (tile edges + a random sample)
    checked against the oracle over every column."""
    Na, Nb = 1300, 2100
    ca, cb = [Na - 17, Na], [Nb, Nb - 333]
    A, B, cta, ctb = synth.match_sets(2, Na, Nb, D, seed=D + int(mutual), count_a=ca, count_b=cb)
    Ad, Bd, cad, cbd = A.cuda(), B.cuda(), cta.cuda(), ctb.cuda()
    nn, nsim = ctx.match(Ad, Bd, cad, cbd, ratio=1e9, mutual=False)
    dec, _ = ctx.match(Ad, Bd, cad, cbd, ratio=0.8, mutual=mutual)
    torch.cuda.synchronize()
    amb = tot = 0
    g = np.random.default_rng(D)
    for p in range(2):
        rows = np.unique(np.concatenate([g.choice(ca[p], 150, replace=False), [0, 127, 128, 255, 256, 1279, 1280, ca[p] - 1, Na - 1]]))
        a, n = check_pair(A[p].numpy(), B[p].numpy(), ca[p], cb[p], 0.8, mutual, nn[p].cpu().numpy(), nsim[p].cpu().numpy(),
                          dec[p].cpu().numpy(), rows=rows)
        amb, tot = amb + a, tot + n
    assert amb <= 0.03 * tot + 2
    assert (dec >= 0).sum() > 0.3 * min(Na, Nb)


def test_match_planted_exact_cases(ctx):
    D = 64
    E = torch.eye(D, dtype=torch.float16)
    A = torch.zeros((1, 128, D), dtype=torch.float16)
    B = torch.zeros((1, 128, D), dtype=torch.float16)
    A[0, :5] = E[:5]
    B[0, :5] = E[[3, 0, 4, 1, 2]]
    B[0, 5] = E[0]                                                # exact duplicate column of B[1]: tie -> smallest j, ratio rejects
    m, s = ctx.match(A.cuda(), B.cuda(), torch.tensor([5], dtype=torch.int32).cuda(), torch.tensor([6], dtype=torch.int32).cuda(),
                     ratio=1e9)
    torch.cuda.synchronize()
    assert m[0, :5].tolist() == [1, 3, 4, 0, 2] and torch.all(m[0, 5:] == -1)
    assert s[0, 0].tolist() == [1.0, 1.0] and s[0, 1].tolist() == [1.0, 0.0]
    m2, _ = ctx.match(A.cuda(), B.cuda(), torch.tensor([5], dtype=torch.int32).cuda(), torch.tensor([6], dtype=torch.int32).cuda(),
                      ratio=0.8)
    torch.cuda.synchronize()
    assert m2[0, :5].tolist() == [-1, 3, 4, 0, 2]                 # d1 == d2 for the duplicated column
    ref = oracle.match_nn(A[0].numpy(), B[0].numpy(), 5, 6, ratio=0.8)[0]
    assert m2[0].cpu().numpy().tolist() == ref.tolist()
    # a single valid column: s2 = -1 (M2); no valid column / row: -1
    m3, s3 = ctx.match(A.cuda(), B.cuda(), torch.tensor([5], dtype=torch.int32).cuda(), torch.tensor([1], dtype=torch.int32).cuda(),
                       ratio=1e9)
    torch.cuda.synchronize()
    assert m3[0, :5].tolist() == [0] * 5 and s3[0, 3].tolist() == [1.0, -1.0]
    m4, _ = ctx.match(A.cuda(), B.cuda(), torch.tensor([5], dtype=torch.int32).cuda(), torch.tensor([0], dtype=torch.int32).cuda())
    m5, _ = ctx.match(A.cuda(), B.cuda(), torch.tensor([0], dtype=torch.int32).cuda(), torch.tensor([6], dtype=torch.int32).cuda())
    torch.cuda.synchronize()
    assert torch.all(m4 == -1) and torch.all(m5 == -1)


def test_match_full_size_sampled(ctx):
    """N_max = 4096, D = 256, P = 2 (temporal + stereo pair) in the launch configuration bench.py times; the
    oracle evaluates, per pair, one random row of EVERY 32-row TMEM lane quadrant of every 128-row block (128 rows: every
    row block, every epilogue warp) plus the block and count edges, against every column."""
    A, B, ca, cb = synth.match_sets(2, 4096, 4096, 256, seed=77, count_a=[4096, 3900], count_b=[4000, 4096])
    nn, nsim = ctx.match(A.cuda(), B.cuda(), ca.cuda(), cb.cuda(), ratio=1e9)
    dec, _ = ctx.match(A.cuda(), B.cuda(), ca.cuda(), cb.cuda(), ratio=0.8)
    torch.cuda.synchronize()
    g = np.random.default_rng(0)
    for p in range(2):
        strat = 32 * np.arange(128) + g.integers(0, 32, 128)
        rows = np.unique(np.concatenate([strat, [0, 127, 128, 3899, 3900, 4095]]))
        amb, tot = check_pair(A[p].numpy(), B[p].numpy(), int(ca[p]), int(cb[p]), 0.8, False, nn[p].cpu().numpy(),
                              nsim[p].cpu().numpy(), dec[p].cpu().numpy(), rows=rows)
        assert amb <= 6 and tot >= 120
    assert (dec >= 0).sum() > 0.5 * 4096 * 2 * 0.7 * 0.8
    nn_ok = nn[0, :4096]
    assert int(nn_ok.min()) >= 0 and int(nn_ok.max()) < 4000      # never a padding column


def test_match_error_codes(ctx):
    import paper_2607_01757_b200 as dkd
    a16 = torch.zeros((1, 128, 64), dtype=torch.float16, device="cuda")
    with pytest.raises(dkd.DKDError) as e:
        ctx.match(a16.float(), a16.float())
    assert e.value.code == -2                                     # fp32 sets: the tensor-core path is fp16
    with pytest.raises(dkd.DKDError) as e:
        ctx.match(a16[..., :48].contiguous(), a16[..., :48].contiguous())
    assert e.value.code == -2                                     # D not a multiple of 64
    with pytest.raises(dkd.DKDError) as e:
        ctx.match(a16, a16, ratio=0.0)
    assert e.value.code == -1


def test_first_match_and_scan_calls_inside_a_capture():
    """A context created with max_match_n / max_scan_rows owns its scratch from the start: the FIRST dkd_match and the
    first dkd_retrieval_scan of its life are made while the stream is being captured (no allocation may happen there),
    the graph is replayed, and the results equal those of an ordinary context."""
    import paper_2607_01757_b200 as dkd
    A, B, ca, cb = synth.match_sets(2, 700, 900, 128, seed=5, count_a=[650, 700], count_b=[900, 801])
    Ad, Bd, cad, cbd = A.cuda(), B.cuda(), ca.cuda(), cb.cuda()
    db, q = synth.keyframe_db(3000, 1024, seed=4, revisits=[10, 1500], dtype=torch.float16)
    dbd, qd = db.cuda(), q.cuda()
    c = dkd.DKD(2, 64, 128, 64, 0, max_match_n=900, max_match_pairs=2, max_scan_rows=3000, max_radius=2)
    ref = dkd.DKD(2, 64, 128, 64, 0)
    try:
        ws0 = c.workspace_bytes
        assert ws0 > ref.workspace_bytes
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            m, s = c.match(Ad, Bd, cad, cbd, ratio=0.8, mutual=True)
            sim, cand, csim, cnt = c.retrieval_scan(dbd, qd, n_exclude=50, tau=0.6, max_cand=4, want_sim=False)
        g.replay()
        torch.cuda.synchronize()
        assert c.workspace_bytes == ws0                         # nothing grew
        m_r, s_r = ref.match(Ad, Bd, cad, cbd, ratio=0.8, mutual=True)
        _, cand_r, csim_r, cnt_r = ref.retrieval_scan(dbd, qd, n_exclude=50, tau=0.6, max_cand=4, want_sim=False)
        torch.cuda.synchronize()
        assert torch.equal(m, m_r) and torch.equal(s, s_r) and int((m >= 0).sum()) > 300
        assert torch.equal(cand, cand_r) and torch.equal(csim, csim_r) and int(cnt[0]) == int(cnt_r[0]) == 2
        # max_radius is a capacity of the context
        sc = torch.zeros((1, 32, 128), device="cuda")
        with pytest.raises(dkd.DKDError) as e:
            c.extract(sc, None, 1, 3, 0.2, 8, 0.1)
        assert e.value.code == -3
        c.extract(sc, None, 1, 2, 0.2, 8, 0.1)
    finally:
        c.close()
        ref.close()
    with pytest.raises(dkd.DKDError):
        dkd.DKD(2, 64, 128, 64, 0, max_radius=5)


# ---- retrieval scan -----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,D,dtype", [(700, 12288, torch.float16), (333, 4096, torch.float32), (1, 12288, torch.float16),
                                       (51, 384, torch.float16), (4000, 12288, torch.float16),
                                       (20000, 12288, torch.float16),     # the size bench.py times: three passes per warp
                                       (30011, 512, torch.float32)])      # four passes, ragged last step
def test_retrieval_scan(ctx, n, D, dtype):
    rev = [k for k in (3, n // 3, n // 2, n - 60, n - 20, n - 1) if 0 <= k < n]
    db, q = synth.keyframe_db(n, D, seed=n + D, revisits=rev, dtype=dtype)
    sim, cand, csim, cnt = ctx.retrieval_scan(db.cuda(), q.cuda(), n_exclude=50, tau=0.60, max_cand=4)
    torch.cuda.synchronize()
    sim_o, cand_o, K = oracle.retrieval_scan(db.numpy(), q.numpy(), 50, 0.60, 4)
    assert np.abs(sim.cpu().numpy() - sim_o).max() <= TOL_SCAN
    assert int(cnt[0]) == K                                       # planted similarities are far from tau and from each other
    assert cand.cpu().numpy().tolist() == cand_o.tolist()
    cs = csim.cpu().numpy()
    assert np.all(np.abs(cs[:K] - sim_o[cand_o[:K]]) <= TOL_SCAN) and np.all(cs[K:] == 0)
    assert all(k < n - 50 for k in cand_o[:K])                    # the 50 most recent keyframes are never candidates


def test_retrieval_scan_many_candidates_and_gate(ctx):
    n, D = 3000, 1024
    db, q = synth.keyframe_db(n, D, seed=9, revisits=[], dtype=torch.float16)
    sim, cand, csim, cnt = ctx.retrieval_scan(db.cuda(), q.cuda(), n_exclude=100, tau=-1.0, max_cand=512)   # every eligible row passes
    torch.cuda.synchronize()
    sim_o, cand_o, K = oracle.retrieval_scan(db.numpy(), q.numpy(), 100, -1.0, 512)
    assert int(cnt[0]) == K == 512
    got = cand.cpu().numpy()
    cs = csim.cpu().numpy()
    assert np.all(np.diff(cs) <= 0) and np.all(got < n - 100)     # ranked, window respected
    assert np.abs(cs - sim_o[got]).max() <= TOL_SCAN
    assert np.abs(np.sort(sim_o[got])[::-1] - sim_o[cand_o]).max() <= 2 * TOL_SCAN    # the same top-512 up to near-ties
    # nothing passes a gate above every similarity; the all-rows output is still complete
    _, c2, _, k2 = ctx.retrieval_scan(db.cuda(), q.cuda(), n_exclude=0, tau=0.99, max_cand=8)
    torch.cuda.synchronize()
    assert int(k2[0]) == 0 and torch.all(c2 == -1)


# ---- stereo validation / covariance -------------------------------------------------------------------------------
def test_stereo_validate(ctx):
    fx, fy, cx, cy, bl = 458.0, 457.0, 367.0, 248.0, 0.11
    g = np.random.default_rng(1)
    n = 5000
    P = np.stack([g.uniform(-3, 3, n), g.uniform(-2, 2, n), g.uniform(0.2, 40, n)], 1)
    pl = np.stack([fx * P[:, 0] / P[:, 2] + cx, fy * P[:, 1] / P[:, 2] + cy], 1).astype(np.float32)
    pr = np.stack([fx * (P[:, 0] - bl) / P[:, 2] + cx, fy * P[:, 1] / P[:, 2] + cy + g.normal(0, 1.2, n)], 1).astype(np.float32)
    perm = g.permutation(n).astype(np.int32)
    match = perm.copy()
    match[g.random(n) < 0.2] = -1
    pr_shuffled = np.empty_like(pr)
    pr_shuffled[perm] = pr                                         # right keypoint of left i sits at perm[i]
    args = dict(fx=fx, fy=fy, cx=cx, cy=cy, baseline=bl, d_min=1.0, z_min=0.3, z_max=30.0, max_reproj=1.5)
    valid, xyz, disp, err = ctx.stereo_validate(torch.from_numpy(pl).cuda(), torch.from_numpy(pr_shuffled).cuda(),
                                                torch.from_numpy(match).cuda(), **args)
    torch.cuda.synchronize()
    has = match >= 0
    v_o, xyz_o, d_o, e_o = oracle.stereo_validate(pl[has].astype(np.float64), pr_shuffled[match[has]].astype(np.float64), fx, fy, cx, cy, bl,
                                                  1.0, 0.3, 30.0, 1.5)
    v, x, d, e = valid.cpu().numpy(), xyz.cpu().numpy(), disp.cpu().numpy(), err.cpu().numpy()
    assert np.all(v[~has] == 0) and np.all(x[~has] == 0)
    tri = d_o > 1.0
    assert np.allclose(d[has], d_o, atol=1e-4) and np.allclose(e[has][tri], e_o[tri], atol=1e-5)
    assert np.allclose(x[has][tri], xyz_o[tri], rtol=2e-5, atol=1e-5)
    z = xyz_o[:, 2]
    clear = (np.abs(d_o - 1.0) > 1e-3) & (np.abs(z - 0.3) > 1e-3) & (np.abs(z - 30.0) > 1e-2) & (np.abs(e_o - 1.5) > 1e-4)
    assert np.array_equal(v[has][clear], v_o[clear]) and clear.mean() > 0.95 and 0.2 < v_o.mean() < 0.9
    # match == NULL: pairs i <-> i
    v2, x2, _, _ = ctx.stereo_validate(torch.from_numpy(pl).cuda(), torch.from_numpy(pr).cuda(), None, **args)
    torch.cuda.synchronize()
    v2_o = oracle.stereo_validate(pl.astype(np.float64), pr.astype(np.float64), fx, fy, cx, cy, bl, 1.0, 0.3, 30.0, 1.5)[0]
    v2_o, xyz2_o, d2_o, e2_o = oracle.stereo_validate(pl.astype(np.float64), pr.astype(np.float64), fx, fy, cx, cy, bl, 1.0, 0.3, 30.0, 1.5)
    z2 = xyz2_o[:, 2]
    clear2 = (np.abs(d2_o - 1.0) > 1e-3) & (np.abs(z2 - 0.3) > 1e-3) & (np.abs(z2 - 30.0) > 1e-2) & (np.abs(e2_o - 1.5) > 1e-4)
    assert np.array_equal(v2.cpu().numpy()[clear2], v2_o[clear2]) and clear2.mean() > 0.95      # exact away from the gates


def test_cov_sqrt_info(ctx):
    g = np.random.default_rng(2)
    n = 4000
    Lf = np.stack([g.uniform(0.2, 3, n), g.uniform(-2, 2, n), g.uniform(0.2, 3, n)], 1).astype(np.float32)
    Lf[:4] = [[0, 1, 0], [1, 1, 0], [np.nan, 0, 1], [np.inf, 0, 1]]          # failures -> isotropic fallback
    par = dict(scale=1.25, floor_px=0.0, fx=460.0, fy=455.0, lam=0.3, lam_min=0.05, sigma0=1.5 / 460.0)
    om, ok = ctx.cov_sqrt_info(torch.from_numpy(Lf).cuda(), **par)
    torch.cuda.synchronize()
    om_o, ok_o = oracle.cov_sqrt_info(Lf.astype(np.float64), par["scale"], par["floor_px"], par["fx"], par["fy"], par["lam"],
                                      par["lam_min"], par["sigma0"])
    assert np.array_equal(ok.cpu().numpy(), ok_o) and not ok_o[:4].any() and ok_o[4:].all()
    o = om.cpu().numpy().astype(np.float64)
    assert np.allclose(o, om_o, rtol=3e-5, atol=1e-3)             # entries are O(100..1000): relative bound
    assert np.all(o[:, 1, 0] == 0)
    assert np.allclose(o[:4], np.eye(2)[None] * (460.0 / 1.5), rtol=1e-6)
    # with the optional floor the singular predictions factor too; lambda below the clamp equals the clamp
    par2 = dict(par, floor_px=0.5)
    _, ok2 = ctx.cov_sqrt_info(torch.from_numpy(Lf[:2]).cuda(), **par2)
    a, _ = ctx.cov_sqrt_info(torch.from_numpy(Lf[4:9]).cuda(), **dict(par, lam=0.001))
    b, _ = ctx.cov_sqrt_info(torch.from_numpy(Lf[4:9]).cuda(), **dict(par, lam=0.05))
    torch.cuda.synchronize()
    assert ok2.all() and torch.equal(a, b)
