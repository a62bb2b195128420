"""GPU parity of the DKD variants (dkd_extract_var) against oracle.extract_var on the same
seeded inputs.  Integer results (indices, order, counts, totals) bit-exact; raw scores bit-exact (the fp32
product heat x reliability is one correctly rounded multiply on both sides); interpolated scores within 2e-6
(three fp32 fma roundings on values <= 1, each <= 6e-8, against the fp64 oracle); offsets / descriptors within
the north_star tolerances of tests/_parity.py."""
import numpy as np
import pytest
import torch

import oracle
import synth
from _parity import TOL_DESC, TOL_OFFSET, half_ulp_f32

pytestmark = pytest.mark.gpu
TOL_BILINEAR_SCORE = 2e-6


@pytest.fixture(scope="module")
def ctx():
    import paper_2607_01757_b200 as dkd
    c = dkd.DKD(max_batch=4, max_h=1100, max_w=1930, max_top_k=8192, max_dim=256)
    yield c
    c.close()


def compare_var(res, ref, desc_dtype=None, bilinear=False):
    torch.cuda.synchronize()
    assert np.array_equal(res.count.cpu().numpy(), ref.count), (res.count, ref.count)
    if res.total is not None:
        assert np.array_equal(res.total.cpu().numpy(), ref.total), (res.total, ref.total)
    assert np.array_equal(res.index.cpu().numpy(), ref.index), "index / order mismatch"
    sc = res.scores.cpu().numpy()
    if bilinear:
        assert np.abs(sc.astype(np.float64) - ref.scores).max() <= TOL_BILINEAR_SCORE
    else:
        assert np.array_equal(sc.astype(np.float64), ref.scores), "scores not bit-exact"
    off = res.offsets.cpu().numpy().astype(np.float64)
    assert np.abs(off - ref.offsets).max() <= TOL_OFFSET
    kp = res.kpts.cpu().numpy().astype(np.float64)
    assert np.all(np.abs(kp - ref.kpts) <= TOL_OFFSET + half_ulp_f32(ref.kpts))
    if ref.desc is not None:
        d = res.desc.cpu().numpy().astype(np.float64)
        assert np.abs(d - ref.desc).max() <= TOL_DESC[desc_dtype]


def inputs(B, H, W, seed, nblobs, D=0, dtype=torch.float16, stride=1, base=0.1):
    score = synth.score_maps(B, H, W, seed, base, nblobs)
    desc = synth.desc_maps(B, H // stride, W // stride, D, seed, dtype, "cuda") if D else None
    g = torch.Generator().manual_seed(seed)
    rel = torch.rand((B, H, W), generator=g)
    vm = (torch.rand((B, H, W), generator=g) < 0.7).to(torch.uint8)
    return score, desc, rel, vm


@pytest.mark.parametrize("r", [1, 2, 3, 4])
@pytest.mark.parametrize("HW", [(75, 300), (67, 301), (203, 252)])          # TMA loader, plain loader (W % 4 != 0), several units
def test_heat_times_reliability(ctx, r, HW):
    H, W = HW
    score, desc, rel, _ = inputs(3, H, W, seed=7 * r + H, nblobs=250, D=64)
    res = ctx.extract(score.cuda(), desc, 1, r, 0.05, 128, 0.1, reliability=rel.cuda(), want_total=True)
    ref = oracle.extract_var(score.numpy(), desc.cpu().numpy(), 1, r, 0.05, 128, 0.1, reliability=rel.numpy())
    compare_var(res, ref, torch.float16)
    assert ref.count.min() > 20
    # the product is formed BEFORE the window maximum: the heat map alone selects other pixels
    alone = ctx.extract(score.cuda(), None, 1, r, 0.05, 128, 0.1)
    torch.cuda.synchronize()
    assert not torch.equal(alone.index, res.index)


@pytest.mark.parametrize("r", [1, 2, 4])
@pytest.mark.parametrize("W", [256, 301])
def test_validity_mask(ctx, r, W):
    score, desc, _, vm = inputs(2, 120, W, seed=r + W, nblobs=300, D=32, dtype=torch.float32)
    res = ctx.extract(score.cuda(), desc, 1, r, 0.2, 200, 0.1, valid_mask=vm.cuda(), want_total=True)
    ref = oracle.extract_var(score.numpy(), desc.cpu().numpy(), 1, r, 0.2, 200, 0.1, valid_mask=vm.numpy())
    compare_var(res, ref, torch.float32)
    unmasked = oracle.extract_var(score.numpy(), None, 1, r, 0.2, 200, 0.1)
    assert np.all(ref.total < unmasked.total)                                 # the mask removes candidates
    idx = res.index.cpu().numpy()
    for b in range(2):                                                        # every reported keypoint is on a valid pixel
        k = idx[b][idx[b] >= 0]
        assert np.all(vm[b].numpy().ravel()[k] != 0)
    none = ctx.extract(score.cuda(), None, 1, r, 0.2, 200, 0.1, valid_mask=torch.zeros_like(vm).cuda(), want_total=True)
    torch.cuda.synchronize()
    assert int(none.count.sum()) == 0 and int(none.total.sum()) == 0


@pytest.mark.parametrize("unit", [0, 1, 4, 8])
def test_validity_mask_with_more_candidates_than_the_sort_capacity(ctx, unit):
    """A plateau map (tens of thousands of tied candidates) under a validity mask: the staged dense filter of k_select
    overflows its 8192-key capacity, the first pass is repeated with the per-lane filter, the radix narrowing reads the
    mask too — for one-tile and multi-tile NMS units (1, 2, 4, 8 lanes per candidate segment in the gather).  Also the
    case where the UNMASKED candidates fit although the staged ones do not."""
    from paper_2607_01757_b200.binding import OPT_NMS_UNIT
    g = torch.Generator().manual_seed(11 + unit)
    s = (torch.randint(0, 4, (2, 300, 400), generator=g).float() / 4.0)
    s = torch.nn.functional.max_pool2d(s[None], 3, 1, 1)[0]                    # plateaus -> lots of tied maxima
    dense = (torch.rand((2, 300, 400), generator=g) < 0.7).to(torch.uint8)    # > 8192 unmasked candidates
    sparse = (torch.rand((2, 300, 400), generator=g) < 0.05).to(torch.uint8)  # staged > 8192, unmasked < 8192
    try:
        ctx.set_option(OPT_NMS_UNIT, unit)
        for vm, top_k in ((dense, 500), (dense, 8192), (sparse, 3000)):
            res = ctx.extract(s.cuda(), None, 1, 1, 0.2, top_k, 0.1, valid_mask=vm.cuda(), want_total=True)
            ref = oracle.extract_var(s.numpy(), None, 1, 1, 0.2, top_k, 0.1, valid_mask=vm.numpy())
            compare_var(res, ref)
        staged = int(oracle.nms_mask(s[0].numpy(), 1, 0.2).sum())
        assert staged > 8192 and ref.total.max() < 8192
    finally:
        ctx.set_option(OPT_NMS_UNIT, 0)


@pytest.mark.parametrize("r", [1, 2, 3, 4])
def test_score_at_refined_point(ctx, r):
    score, desc, _, _ = inputs(2, 96, 200, seed=30 + r, nblobs=200, D=0)
    res = ctx.extract(score.cuda(), None, 1, r, 0.2, 128, 0.1, score_mode=1)
    ref = oracle.extract_var(score.numpy(), None, 1, r, 0.2, 128, 0.1, score_mode=1)
    compare_var(res, ref, bilinear=True)
    raw = ctx.extract(score.cuda(), None, 1, r, 0.2, 128, 0.1)
    torch.cuda.synchronize()
    assert torch.equal(raw.index, res.index) and torch.equal(raw.kpts, res.kpts)     # selection is unaffected
    assert not torch.equal(raw.scores, res.scores)
    assert torch.all(res.scores <= raw.scores + 1e-6)                                # the peak is the window maximum


def test_threshold_only_mode_reports_the_total(ctx):
    score, _, _, _ = inputs(2, 150, 400, seed=5, nblobs=600)
    for cap in (16, 8192):                                                    # capacity below / above the candidate count
        res = ctx.extract(score.cuda(), None, 1, 2, 0.2, cap, 0.1, want_total=True)
        ref = oracle.extract_var(score.numpy(), None, 1, 2, 0.2, cap, 0.1)
        compare_var(res, ref)
        tot, cnt = res.total.cpu().numpy(), res.count.cpu().numpy()
        assert np.array_equal(cnt, np.minimum(tot, cap))
    assert np.all(tot > 16) and np.all(tot < 8192)
    # more candidates than the in-kernel sort capacity: the total still counts every candidate
    s = torch.full((1, 128, 256), 0.7)
    res = ctx.extract(s.cuda(), None, 1, 2, 0.2, 100, 0.1, want_total=True)
    torch.cuda.synchronize()
    assert int(res.total[0]) == 124 * 252 and int(res.count[0]) == 100


def test_variants_compose_and_graph_updates_keep_them(ctx):
    score, desc, rel, vm = inputs(2, 110, 260, seed=9, nblobs=300, D=128)
    sd, rd, md = score.cuda(), rel.cuda(), vm.cuda()
    ref = oracle.extract_var(score.numpy(), desc.cpu().numpy(), 1, 2, 0.05, 256, 0.1, reliability=rel.numpy(),
                             valid_mask=vm.numpy(), score_mode=1)
    for rep in range(3):                                                      # fresh outputs: cached graph, updated nodes
        res = ctx.extract(sd, desc, 1, 2, 0.05, 256, 0.1, reliability=rd, valid_mask=md, score_mode=1, want_total=True)
        compare_var(res, ref, torch.float16, bilinear=True)
    # same call without the variants still gives the base result (separate graph)
    base = ctx.extract(sd, desc, 1, 2, 0.05, 256, 0.1)
    bref = oracle.extract(score.numpy(), desc.cpu().numpy(), 1, 2, 0.05, 256, 0.1)
    torch.cuda.synchronize()
    assert np.array_equal(base.index.cpu().numpy(), bref.index)


def test_xfeat_like_config_with_reliability_full_size():
    """c4's shapes (720x1280, stride-8 64-d map, k = 4096) with a reliability map: the XFeat-style workload."""
    import paper_2607_01757_b200 as dkd
    cfg = synth.CONFIGS["c4"]
    c = dkd.DKD(cfg.B, cfg.H, cfg.W, cfg.top_k, cfg.D)
    try:
        score, desc = synth.make_inputs(cfg, device="cuda")
        rel = torch.rand(score.shape, generator=torch.Generator().manual_seed(4)) * 0.5 + 0.5
        res = c.extract(score.cuda(), desc, cfg.stride, cfg.r, cfg.thresh, cfg.top_k, cfg.T, reliability=rel.cuda(),
                        want_total=True)
        ref = oracle.extract_var(score.numpy(), desc.cpu().numpy(), cfg.stride, cfg.r, cfg.thresh, cfg.top_k, cfg.T,
                                 reliability=rel.numpy())
        compare_var(res, ref, torch.float16)
        assert ref.count.min() > 1000
    finally:
        c.close()


@pytest.mark.parametrize("r,iters", [(1, 1), (2, 1), (2, 2), (3, 2), (4, 2), (2, 3), (1, 5)])
@pytest.mark.parametrize("HW", [(75, 300), (130, 97), (203, 252)])
def test_iterated_suppress_and_recover_nms(ctx, r, iters, HW):
    H, W = HW
    score, desc, rel, vm = inputs(2, H, W, seed=11 * r + iters + H, nblobs=400, D=64)
    res = ctx.extract(score.cuda(), desc, 1, r, 0.15, 256, 0.1, nms_iters=iters, want_total=True)
    ref = oracle.extract_var(score.numpy(), desc.cpu().numpy(), 1, r, 0.15, 256, 0.1, nms_iters=iters)
    compare_var(res, ref, torch.float16)
    single = oracle.extract_var(score.numpy(), None, 1, r, 0.15, 256, 0.1)
    assert np.all(ref.total > single.total)                                   # recovery adds candidates


def test_iterated_nms_composes_with_the_other_variants_and_plateaus(ctx):
    score, desc, rel, vm = inputs(2, 140, 260, seed=3, nblobs=300, D=32, dtype=torch.float32)
    res = ctx.extract(score.cuda(), desc, 1, 2, 0.05, 300, 0.1, nms_iters=2, reliability=rel.cuda(), valid_mask=vm.cuda(),
                      score_mode=1, want_total=True)
    ref = oracle.extract_var(score.numpy(), desc.cpu().numpy(), 1, 2, 0.05, 300, 0.1, nms_iters=2, reliability=rel.numpy(),
                             valid_mask=vm.numpy(), score_mode=1)
    compare_var(res, ref, torch.float32, bilinear=True)
    # plateaus and exact ties (quantised map), image smaller than one tile, border pixels
    g = torch.Generator().manual_seed(8)
    q = (torch.randint(0, 6, (1, 40, 50), generator=g).float() / 6.0)
    res = ctx.extract(q.cuda(), None, 1, 2, 0.1, 2048, 0.1, nms_iters=2, want_total=True)
    ref = oracle.extract_var(q.numpy(), None, 1, 2, 0.1, 2048, 0.1, nms_iters=2)
    compare_var(res, ref)
    assert ref.total[0] > 50


def test_iterated_nms_full_size_c2():
    import paper_2607_01757_b200 as dkd
    cfg = synth.CONFIGS["c2"]
    c = dkd.DKD(cfg.B, cfg.H, cfg.W, cfg.top_k, cfg.D)
    try:
        score, desc = synth.make_inputs(cfg, device="cuda")
        res = c.extract(score.cuda(), desc, cfg.stride, cfg.r, cfg.thresh, cfg.top_k, cfg.T, nms_iters=2, want_total=True)
        ref = oracle.extract_var(score.numpy(), desc.cpu().numpy(), cfg.stride, cfg.r, cfg.thresh, cfg.top_k, cfg.T, nms_iters=2)
        compare_var(res, ref, torch.float16)
    finally:
        c.close()


def test_iterated_nms_limits(ctx):
    import paper_2607_01757_b200 as dkd
    s = torch.zeros((1, 32, 128), device="cuda")
    with pytest.raises(dkd.DKDError) as e:
        ctx.extract(s, None, 1, 4, 0.2, 8, 0.1, nms_iters=5)                  # (2*5+1)*4 = 44 > 40
    assert e.value.code == -2
    with pytest.raises(dkd.DKDError) as e:
        ctx.extract(s, None, 1, 2, 0.2, 8, 0.1, nms_iters=-1)
    assert e.value.code == -1


def test_iterated_nms_finest_tiling_at_the_context_maximum():
    """r = 3, nms_iters = 6: halo 39, 24 x 24 tiles — more tiles (1080) than the context has single-pass NMS units, at the
    very shape the context was created for: the per-tile counts must fit the workspace (they are sized for this tiling)."""
    import paper_2607_01757_b200 as dkd
    B, H, W = 2, 480, 640
    c = dkd.DKD(B, H, W, 512, 0)
    try:
        score = synth.score_maps(B, H, W, 5, 0.1, 600)
        res = c.extract(score.cuda(), None, 1, 3, 0.15, 512, 0.1, nms_iters=6, want_total=True)
        ref = oracle.extract_var(score.numpy(), None, 1, 3, 0.15, 512, 0.1, nms_iters=6)
        compare_var(res, ref)
        assert ref.count.min() > 50
        again = c.extract(score.cuda(), None, 1, 2, 0.15, 512, 0.1)           # the workspace after it is intact
        compare_var(again, oracle.extract_var(score.numpy(), None, 1, 2, 0.15, 512, 0.1))
    finally:
        c.close()


@pytest.mark.parametrize("unit", [0, 8])
def test_reliability_at_1080p_in_the_batch64_launch_shape(ctx, unit):
    """The heat x reliability NMS kernel at 1920 x 1080 with 8-tile units (the shape it is launched in at batch 64:
    one CTA per SM, both TMA rings), on B = 4 frames the oracle finishes in seconds."""
    from paper_2607_01757_b200.binding import OPT_NMS_UNIT
    cfg = synth.CONFIGS["c5"]
    B = 4
    score = synth.score_maps(B, cfg.H, cfg.W, 31, 0.1, 4000)
    desc = synth.desc_maps(B, cfg.H, cfg.W, 128, 31, torch.float16, "cuda")
    rel = torch.rand(score.shape, generator=torch.Generator().manual_seed(6)) * 0.5 + 0.5
    try:
        ctx.set_option(OPT_NMS_UNIT, unit)
        res = ctx.extract(score.cuda(), desc, 1, cfg.r, cfg.thresh, cfg.top_k, cfg.T, reliability=rel.cuda(), want_total=True)
        torch.cuda.synchronize()
    finally:
        ctx.set_option(OPT_NMS_UNIT, 0)
    ref = oracle.extract_var(score.numpy(), desc.cpu().numpy(), 1, cfg.r, cfg.thresh, cfg.top_k, cfg.T, reliability=rel.numpy())
    compare_var(res, ref, torch.float16)
    assert ref.count.min() > 500
