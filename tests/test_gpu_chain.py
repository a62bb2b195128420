"""The front-end chain on the device, stage feeding stage ("Both sets stay resident on the GPU ... the
temporal pair and the stereo pair ... resolve in one batch-2 ... launch"; PAPER.md:139 zero-padded sets + counts handed
downstream; PAPER.md:145 stereo matches validated by calibrated geometry):

    dkd_extract (B = 4: L(t-1), L(t), R(t), R(t-1))
      -> dkd_match, P = 2, on VIEWS of the extract outputs (out_desc[0:2] vs out_desc[1:3], out_count likewise: no copy,
         no host read of the counts): pair 0 = temporal L(t-1)/L(t), pair 1 = stereo L(t)/R(t)
      -> dkd_stereo_validate(out_kpts[L(t)], out_kpts[R(t)], out_match[pair 1])

against the composed oracle oracle.extract -> oracle.match_nn -> oracle.stereo_validate, each oracle stage fed with the
ORACLE's upstream result.  Two levels:
  1. interface fit, exact: the oracle matcher run on the product's own extract outputs (downloaded) must agree with the
     product's matcher at the matcher's tolerance TOL_SIM — layout, padding rows, device-side counts, keypoint order;
  2. the chain: between the stages the oracle's descriptors are stored in the boundary's dtype (f16, like out_desc).  The
     product's f16 descriptors can differ from those by one f16 rounding step per element (the fp32 value before the
     store is within ~1e-6 of the fp64 one), |delta_i| <= 2^-10 |d_i|, hence a similarity differs by at most
     2 * 2^-10 * sum|a_i||b_i| <= 2^-9 (Cauchy-Schwarz, unit vectors) on top of TOL_SIM:  TOL_CHAIN = 2^-9 + 1e-4.
     Argmax / ratio / mutual decisions are compared where the fp64 margins exceed that (the ambiguous-argmax rule of
     tests/test_gpu_match.py), and the stereo results on the rows whose match is unambiguous.
"""
import numpy as np
import pytest
import torch

import oracle
import synth
from _parity import compare

pytestmark = pytest.mark.gpu
TOL_SIM = 1e-4
TOL_CHAIN = 2.0 ** -9 + TOL_SIM
H, W, D, R, THRESH, T = 480, 752, 128, 2, 0.2, 0.1               # c2's shapes and parameters
CAM = dict(fx=458.0, fy=457.0, cx=367.0, cy=248.0, baseline=0.11, d_min=1.0, z_min=0.3, z_max=30.0, max_reproj=1.5)


def check_match(A, B, na, nb, ratio, mutual, nn_idx, nn_sim, dec_idx, tol):
    """Oracle matcher on (A, B) against the product's results.  Returns (oracle decision [na] (-1: none), clear [na])."""
    idx_o, s1_o, s2_o, S = oracle.match_nn(A[:na], B, na, nb, ratio=1e9, want_sim=True)
    want = np.full(na, -1, np.int64)
    clear = np.zeros(na, bool)
    for i in range(na):
        near = np.flatnonzero(S[i] >= S[i].max() - 2 * tol)
        assert nn_idx[i] in near, (i, nn_idx[i], near)
        if len(near) == 1:
            assert nn_idx[i] == idx_o[i]
        assert abs(nn_sim[i, 0] - s1_o[i]) <= tol and abs(nn_sim[i, 1] - s2_o[i]) <= tol, (i, nn_sim[i], s1_o[i], s2_o[i])
        d1, d2 = max(0.0, 2 - 2 * s1_o[i]), max(0.0, 2 - 2 * s2_o[i])
        margin = ratio * ratio * d2 - d1
        ok = abs(margin) > 2 * tol * (1 + ratio * ratio) * 2 and len(near) == 1
        keep = margin > 0
        if mutual and keep and ok:
            col = A[:na].astype(np.float64) @ B[idx_o[i]].astype(np.float64)
            cnear = np.flatnonzero(col >= col.max() - 2 * tol)
            if len(cnear) == 1:
                keep = cnear[0] == i
            else:
                ok = False
        if ok:
            want[i] = idx_o[i] if keep else -1
            assert dec_idx[i] == want[i], (i, dec_idx[i], idx_o[i], keep, margin)
        clear[i] = ok
    assert np.all(nn_idx[na:] == -1) and np.all(dec_idx[na:] == -1) and np.all(nn_sim[na:] == 0)   # padding rows
    return want, clear


def run_chain(ctx, score_d, desc_d, cap, out=None):
    res = ctx.extract(score_d, desc_d, 1, R, THRESH, cap, T, out=out)
    da, db, ca, cb = res.desc[0:2], res.desc[1:3], res.count[0:2], res.count[1:3]      # views: nothing is copied
    assert da.data_ptr() == res.desc.data_ptr() and db.data_ptr() == res.desc[1].data_ptr()
    nn, nsim = ctx.match(da, db, ca, cb, ratio=1e9, mutual=False)
    dec, _ = ctx.match(da, db, ca, cb, ratio=0.8, mutual=True)
    stereo = ctx.stereo_validate(res.kpts[1], res.kpts[2], dec[1], **CAM)
    return res, nn, nsim, dec, stereo


@pytest.mark.parametrize("cap,disparity", [(256, 20), (1024, 7)])
def test_extract_match_stereo_chain_against_the_composed_oracle(cap, disparity):
    import paper_2607_01757_b200 as dkd
    score, desc = synth.stereo_sequence(H, W, D, seed=100 + cap, disparity=disparity, device="cuda")
    ctx = dkd.DKD(4, H, W, cap, D)
    try:
        res, nn, nsim, dec, (valid, xyz, disp, err) = run_chain(ctx, score.cuda(), desc, cap)
        torch.cuda.synchronize()
        # stage 1 against the oracle
        ref = oracle.extract(score.numpy(), desc.cpu().numpy(), 1, R, THRESH, cap, T)
        compare(res, ref, torch.float16)
        cnt = ref.count
        assert cnt.min() > 0.5 * cap
        g_desc = res.desc.cpu().numpy()
        o_desc = ref.desc.astype(np.float16)                       # the boundary's storage dtype between the stages
        nn_h, nsim_h, dec_h = nn.cpu().numpy(), nsim.cpu().numpy(), dec.cpu().numpy()
        n_clear = n_live = 0
        for p in range(2):
            ia, ib = p, p + 1
            # level 1: the oracle matcher on the product's own sets — exact interface fit
            check_match(g_desc[ia], g_desc[ib], cnt[ia], cnt[ib], 0.8, True, nn_h[p], nsim_h[p], dec_h[p], TOL_SIM)
            # level 2: the oracle's sets
            want, clear = check_match(o_desc[ia], o_desc[ib], cnt[ia], cnt[ib], 0.8, True, nn_h[p], nsim_h[p], dec_h[p], TOL_CHAIN)
            n_clear, n_live = n_clear + int(clear.sum()), n_live + int(cnt[ia])
            if p == 1:
                stereo_want, stereo_clear = want, clear
        assert n_clear >= 0.75 * n_live                            # the comparison is not vacuous
        assert (dec_h[0] >= 0).sum() > 0.5 * cnt[:2].min() and (dec_h[1] >= 0).sum() > 0.5 * cnt[1:3].min()   # the views do match
        # stage 3 against the oracle fed with the oracle's keypoints and the oracle chain's matches
        rows = np.flatnonzero(stereo_clear & (stereo_want >= 0))
        assert len(rows) > 0.4 * cnt[1]
        pl, pr = ref.kpts[1][rows], ref.kpts[2][stereo_want[rows]]
        v_o, xyz_o, d_o, e_o = oracle.stereo_validate(pl, pr, *[CAM[k] for k in ("fx", "fy", "cx", "cy", "baseline", "d_min", "z_min",
                                                                                 "z_max", "max_reproj")])
        v, x, d, e = valid.cpu().numpy(), xyz.cpu().numpy(), disp.cpu().numpy(), err.cpu().numpy()
        assert np.allclose(d[rows], d_o, atol=1e-4) and np.allclose(e[rows], e_o, atol=2e-5)
        assert np.allclose(x[rows], xyz_o, rtol=2e-5, atol=1e-4)
        z = xyz_o[:, 2]
        away = (np.abs(d_o - 1.0) > 1e-3) & (np.abs(z - 0.3) > 1e-3) & (np.abs(z - 30.0) > 1e-2) & (np.abs(e_o - 1.5) > 1e-4)
        assert np.array_equal(v[rows][away], v_o[away]) and away.mean() > 0.95
        assert np.abs(d_o - disparity).max() < 1e-3 and v_o.mean() > 0.95       # the planted geometry comes back
        no_match = np.flatnonzero(dec_h[1] < 0)
        assert np.all(v[no_match] == 0) and np.all(x[no_match] == 0)
    finally:
        ctx.close()


def test_chain_replays_from_one_caller_graph():
    """After one eager pass (the matcher's scratch is sized by then) the whole chain is captured into ONE graph of the
    caller's and replayed on new inputs written into the same buffers: results identical to the eager chain."""
    import paper_2607_01757_b200 as dkd
    cap = 256
    s0, d0 = synth.stereo_sequence(H, W, D, seed=7, disparity=12, device="cuda")
    s1, d1 = synth.stereo_sequence(H, W, D, seed=8, disparity=16, device="cuda")
    ctx = dkd.DKD(4, H, W, cap, D)
    try:
        score_d, desc_d = s0.cuda(), d0.clone()
        out = ctx.alloc_outputs(4, cap, desc_d, D)
        run_chain(ctx, score_d, desc_d, cap, out=out)              # eager warm-up
        torch.cuda.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):
            _, nn_g, nsim_g, dec_g, st_g = run_chain(ctx, score_d, desc_d, cap, out=out)
        for s, d in ((s1, d1), (s0, d0)):
            score_d.copy_(s)
            desc_d.copy_(d)
            graph.replay()
            torch.cuda.synchronize()
            got = [t.clone() for t in (out.kpts, out.desc, out.count, nn_g, nsim_g, dec_g, *st_g)]
            out2 = ctx.alloc_outputs(4, cap, desc_d, D)
            _, nn_e, nsim_e, dec_e, st_e = run_chain(ctx, score_d, desc_d, cap, out=out2)
            torch.cuda.synchronize()
            for a, b in zip(got, (out2.kpts, out2.desc, out2.count, nn_e, nsim_e, dec_e, *st_e)):
                assert torch.equal(a, b)
            assert int((dec_e >= 0).sum()) > cap // 2
    finally:
        ctx.close()
