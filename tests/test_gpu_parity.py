"""GPU parity: the CUDA path (through the C-ABI) vs the CPU oracle, element by element, on the same
seeded inputs.  Sizes span several 128x32 tiles with ragged tails; configs c1-c5 run at full size
(c5 in the launch configuration bench.py times; its oracle runs on every image for steps 1-3 and on
sampled images for step 4).  north_star tolerances live in tests/_parity.py."""
import numpy as np
import pytest
import torch

import oracle
import synth
from _parity import compare, run_both

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    import paper_2607_01757_b200 as dkd
    c = dkd.DKD(max_batch=4, max_h=1100, max_w=1930, max_top_k=8192, max_dim=1024)
    yield c
    c.close()


def small_inputs(B, H, W, seed, nblobs, D, dtype, stride, base=0.1):
    score = synth.score_maps(B, H, W, seed, base, nblobs)
    desc = None
    if D:
        desc = synth.desc_maps(B, max(H // stride, 1), max(W // stride, 1), D, seed, dtype, "cuda")
    return score, desc


# ---- multi-tile small cases, ragged tails, every radius, both loaders ---------------------------
@pytest.mark.parametrize("r", [1, 2, 3, 4])
@pytest.mark.parametrize("HW", [(75, 300), (67, 301), (33, 129), (200, 136)])
def test_small_multitile(ctx, r, HW):
    H, W = HW
    score, desc = small_inputs(3, H, W, seed=10 * r + H, nblobs=150, D=64, dtype=torch.float16, stride=1)
    res, ref = run_both(ctx, score, desc, 1, r, 0.2, 96, 0.1)
    st = compare(res, ref, torch.float16)
    assert ref.count.min() > 10
    assert st["max_offset_err"] <= 1e-5


@pytest.mark.parametrize("r", [1, 2, 3, 4])
@pytest.mark.parametrize("unit", [2, 3, 8])
def test_nms_units_of_several_strip_tiles(ctx, r, unit):
    # a warp walks down `unit` strip-tiles carrying the last 2r rows in registers (the default picks
    # units > 1 only for large batches): tall image, ragged last unit, every radius
    from paper_2607_01757_b200.binding import OPT_NMS_UNIT
    score, _ = small_inputs(2, 203, 250, seed=100 + 10 * r + unit, nblobs=500, D=0, dtype=None, stride=1)
    try:
        ctx.set_option(OPT_NMS_UNIT, unit)
        res, ref = run_both(ctx, score, None, 1, r, 0.15, 512, 0.1)
        compare(res, ref)
    finally:
        ctx.set_option(OPT_NMS_UNIT, 0)
    assert ref.count.min() > 100


@pytest.mark.parametrize("dtype,D", [(torch.float32, 4), (torch.float32, 64), (torch.float32, 512),
                                      (torch.float16, 8), (torch.float16, 128), (torch.float16, 256),
                                      (torch.float16, 1024), (torch.float16, 72)])
@pytest.mark.parametrize("stride", [1, 2, 8])
def test_descriptor_shapes_and_strides(ctx, dtype, D, stride):
    score, desc = small_inputs(2, 96, 160, seed=D + stride, nblobs=120, D=D, dtype=dtype, stride=stride)
    res, ref = run_both(ctx, score, desc, stride, 2, 0.2, 128, 0.1)
    compare(res, ref, dtype)


def test_stride_clamp_and_nonmultiple_map(ctx):
    # descriptor map smaller than H/s: positions clamp to the map (G13); r = 4 near the border
    score = synth.score_maps(2, 80, 120, 5, 0.01, 200)
    desc = synth.desc_maps(2, 9, 14, 64, 5, torch.float16, "cuda")
    res, ref = run_both(ctx, score, desc, 8, 4, 0.005, 256, 0.1)
    compare(res, ref, torch.float16)
    u = (ref.kpts[..., 0] + 0.5) / 8 - 0.5
    assert (u < 0).any() and (u > 13).any()                    # both clamps exercised


@pytest.mark.parametrize("T", [0.03, 0.1, 1.0])
def test_temperature(ctx, T):
    score, desc = small_inputs(1, 64, 128, seed=3, nblobs=60, D=0, dtype=None, stride=1)
    res, ref = run_both(ctx, score, None, 1, 2, 0.2, 64, T)
    compare(res, ref)


# ---- seeded random sweep over shapes and parameters ---------------------------------------------
@pytest.mark.parametrize("case", range(48))
def test_random_shapes_and_parameters(ctx, case):
    """Random small problems (ragged widths incl. W % 4 != 0 -> plain loader, images smaller than a
    strip-tile, every radius / stride / descriptor type, top_k above and below the candidate count,
    forced NMS unit lengths) against the oracle."""
    from paper_2607_01757_b200.binding import OPT_NMS_UNIT
    g = np.random.default_rng(1000 + case)
    B = int(g.integers(1, 4))
    H = int(g.integers(3, 140))
    W = int(g.integers(3, 400))
    if case % 3 == 0:
        W = 4 * max(W // 4, 1)                                    # TMA path
    r = int(g.integers(1, 5))
    stride = int(g.choice([1, 1, 2, 4, 8]))
    dtype, D = [(torch.float16, 64), (torch.float16, 8), (torch.float32, 32), (torch.float16, 264), (None, 0)][case % 5]
    top_k = int(g.choice([1, 7, 64, 300, 2048]))
    thresh = float(g.choice([0.0, 0.05, 0.2, 0.6]))
    T = float(g.choice([0.05, 0.1, 0.5]))
    score = synth.score_maps(B, H, W, 5000 + case, 0.1, int(g.integers(0, 200)))
    desc = None
    if D:
        desc = synth.desc_maps(B, max(H // stride, 1), max(W // stride, 1), D, case, dtype, "cuda")
    try:
        ctx.set_option(OPT_NMS_UNIT, int(g.integers(0, 9)))
        res, ref = run_both(ctx, score, desc, stride, r, thresh, top_k, T)
        compare(res, ref, dtype)
    finally:
        ctx.set_option(OPT_NMS_UNIT, 0)


# ---- full-size configs c1-c4 ---------------------------------------------------------------------
@pytest.mark.parametrize("name", ["c1", "c2", "c3", "c4"])
def test_config_full_size(name):
    import paper_2607_01757_b200 as dkd
    cfg = synth.CONFIGS[name]
    c = dkd.DKD(cfg.B, cfg.H, cfg.W, cfg.top_k, cfg.D)
    try:
        score, desc = synth.make_inputs(cfg, device="cuda")
        res, ref = run_both(c, score, desc, cfg.stride, cfg.r, cfg.thresh, cfg.top_k, cfg.T)
        st = compare(res, ref, synth.torch_dtype(cfg.desc_dtype))
        print(name, "counts", ref.count, st)
        assert (ref.scores == 1.0).sum() > 10                   # exact-1.0 ties head every ranking (G1)
        if name in ("c2", "c4"):
            assert np.all(ref.count < cfg.top_k)                # K_b < k branch
        else:
            assert np.all(ref.count == cfg.top_k)
    finally:
        c.close()


def lazy_desc_reference(cfg, b, idx, kpts):
    """Oracle descriptors of image b's kept keypoints WITHOUT the descriptor map: the four corner rows of every keypoint
    are evaluated from the counter-based generator (synth.desc_elements), stacked into a [2K, 2, D] map (keypoint i owns
    rows 2i, 2i+1), and sampled by the oracle's own gather at the keypoint's position relative to its cell.  Bilinear
    interpolation is local, so this is the oracle's O4 on the full map (the c5 map is 34 GB)."""
    K = int((idx >= 0).sum())
    px, py = kpts[:K, 0], kpts[:K, 1]
    x0 = np.clip(np.floor(px).astype(np.int64), 0, cfg.Wd - 2)
    y0 = np.clip(np.floor(py).astype(np.int64), 0, cfg.Hd - 2)
    cells = ((y0[:, None, None] + np.arange(2)[None, :, None]) * cfg.Wd + x0[:, None, None] + np.arange(2)[None, None, :])
    e = torch.from_numpy(cells[..., None] * cfg.D + np.arange(cfg.D))          # [K, 2, 2, D] element offsets
    F = synth.desc_elements(cfg.seed, b, e.reshape(-1), torch.float16).reshape(2 * K, 2, cfg.D).numpy()
    local = np.stack([px - x0, py - y0 + 2 * np.arange(K)], 1)
    return oracle.gather(F, 1, local)


def test_config_c5_full_size_all_images():
    """B=64 1080p in the launch configuration bench.py times.  Steps 1-3 are checked on EVERY image (oracle without
    descriptors), and so is step 4: the oracle's corner rows come lazily from the generator, for all 64 images."""
    import paper_2607_01757_b200 as dkd
    cfg = synth.CONFIGS["c5"]
    free, _ = torch.cuda.mem_get_info()
    need = cfg.B * cfg.Hd * cfg.Wd * cfg.D * 2 + 4 * cfg.B * cfg.H * cfg.W * 4
    if free < need + (4 << 30):
        pytest.fail(f"c5 needs {need >> 30} GiB of device memory, {free >> 30} GiB free")
    c = dkd.DKD(cfg.B, cfg.H, cfg.W, cfg.top_k, cfg.D)
    try:
        score = synth.score_maps(cfg.B, cfg.H, cfg.W, cfg.seed, cfg.base, cfg.nblobs)
        desc = synth.desc_maps(cfg.B, cfg.Hd, cfg.Wd, cfg.D, cfg.seed, torch.float16, "cuda")
        res = c.extract(score.cuda(), desc, cfg.stride, cfg.r, cfg.thresh, cfg.top_k, cfg.T)
        torch.cuda.synchronize()
        ref = oracle.extract(score.numpy(), None, 1, cfg.r, cfg.thresh, cfg.top_k, cfg.T)
        res_nodesc = type(res)(res.kpts, res.scores, None, res.count, res.index, res.offsets)
        st = compare(res_nodesc, ref)
        assert np.all(ref.count == cfg.top_k)
        got = res.desc.cpu().numpy().astype(np.float64)
        worst = 0.0
        for b in range(cfg.B):                                     # step 4 on all 64 images
            want = lazy_desc_reference(cfg, b, ref.index[b], ref.kpts[b])
            worst = max(worst, float(np.abs(got[b, :want.shape[0]] - want).max()))
        assert worst <= 2e-3, worst
        # the lazy reference is the oracle on the real map: one image end to end through oracle.extract
        refb = oracle.extract(score[37:38].numpy(), desc[37:38].cpu().numpy(), 1, cfg.r, cfg.thresh, cfg.top_k, cfg.T)
        compare(res, refb, torch.float16, images=[37])
        assert np.abs(refb.desc[0] - lazy_desc_reference(cfg, 37, ref.index[37], ref.kpts[37])).max() < 1e-12
        # device-side generator == host evaluation on sampled elements
        e = torch.randint(0, cfg.Hd * cfg.Wd * cfg.D, (100000,))
        assert torch.equal(desc[11].view(-1)[e.cuda()].cpu(), synth.desc_elements(cfg.seed, 11, e, torch.float16))
    finally:
        c.close()


def test_random_sweep_and_worst_cases_under_the_debug_build():
    """compute-sanitizer is closed on this GPU pool, so memory safety is checked by the library itself: libdkd_debug.so
    is the same source with -DDKD_DEBUG, i.e. a device-side assert on every candidate-segment / shared-memory index and
    on the mbarrier ring arithmetic.  The random sweep, the worst-case (every pixel a candidate), the radix-select and the
    multi-unit tests run under it in a child process; a failed assert is a CUDA error and fails them."""
    import os
    import subprocess
    import sys
    from paper_2607_01757_b200 import build
    if os.environ.get("DKD_LIBRARY") == "libdkd_debug.so":
        pytest.skip("already running under the debug build")          # (the child process must not start another one)
    build.build(debug=True)
    env = dict(os.environ, DKD_LIBRARY="libdkd_debug.so")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    sel = "random_shapes or worst_case or many_candidates or units_of_several or small_multitile or ties_at_clamp or back_to_back"
    r = subprocess.run([sys.executable, "-m", "pytest", "tests/test_gpu_parity.py", "tests/test_gpu_variants.py",
                        "tests/test_gpu_match.py", "-q", "-x", "-m", "gpu", "-k",
                        "(" + sel + " or reliability or validity or retrieval or match_small or wide_tiles) and not debug_build"],
                       cwd=root, env=env, capture_output=True, text=True, timeout=1500)
    assert r.returncode == 0, r.stdout[-3000:] + r.stderr[-2000:]
    assert "DKD_DEBUG" in subprocess.run([sys.executable, "-c", "import paper_2607_01757_b200 as d, ctypes; L = d.load_library(); "
                                          "L.dkd_version.restype = ctypes.c_char_p; print(L.dkd_version().decode())"],
                                         cwd=root, env=env, capture_output=True, text=True).stdout


# ---- larger shapes than the configs: 4K frames, the plain loader at scale, the largest cap -------------
@pytest.mark.parametrize("case", ["4k_r4_k8192_d256_s8", "plain_1081x1923", "tall_narrow", "d1024_f16"])
def test_large_and_odd_shapes(case):
    import paper_2607_01757_b200 as dkd
    B, H, W, r, thresh, k, T, D, dtype, stride, base, blobs = {
        "4k_r4_k8192_d256_s8": (2, 2160, 3840, 4, 0.05, 8192, 0.1, 256, torch.float16, 8, 0.05, 20000),
        "plain_1081x1923": (2, 1081, 1923, 2, 0.2, 2048, 0.1, 64, torch.float32, 1, 0.1, 4000),
        "tall_narrow": (3, 4000, 132, 3, 0.2, 1024, 0.05, 128, torch.float16, 2, 0.1, 3000),
        "d1024_f16": (1, 300, 500, 2, 0.2, 512, 0.1, 1024, torch.float16, 4, 0.1, 800),
    }[case]
    c = dkd.DKD(B, H, W, k, D)
    try:
        score = synth.score_maps(B, H, W, 99, base, blobs)
        desc = synth.desc_maps(B, H // stride, W // stride, D, 99, dtype, "cuda")
        res, ref = run_both(c, score, desc, stride, r, thresh, k, T)
        st = compare(res, ref, dtype)
        assert ref.count.min() > 500 and st["max_offset_err"] <= 1e-5
    finally:
        c.close()


# ---- degenerate and adversarial inputs -----------------------------------------------------------
def test_no_candidates_and_tiny_images(ctx):
    score = torch.full((2, 40, 140), 0.1)
    desc = synth.desc_maps(2, 40, 140, 32, 1, torch.float16, "cuda")
    res, ref = run_both(ctx, score, desc, 1, 2, 0.2, 16, 0.1)
    compare(res, ref, torch.float16)
    assert int(res.count.sum()) == 0 and float(res.kpts.abs().sum()) == 0 and int((res.index != -1).sum()) == 0
    for H, W in [(4, 9), (5, 5), (1, 1), (9, 4)]:               # H or W < 2r+1 -> no interior (G18)
        s = torch.ones((1, H, W))
        res, ref = run_both(ctx, s, None, 1, 2, 0.2, 8, 0.1)
        compare(res, ref)


def test_threshold_is_strict_and_border_excluded(ctx):
    s = torch.zeros((1, 40, 140))
    s[0, 10, 20] = 0.5                   # == thresh -> dropped
    s[0, 20, 30] = float(np.nextafter(np.float32(0.5), np.float32(1)))
    s[0, 1, 50] = 0.9                    # inside the r-border -> dropped
    s[0, 2, 60] = 0.9                    # first kept row
    s[0, 37, 137] = 0.8                  # last kept row / column
    s[0, 38, 100] = 0.9
    res, ref = run_both(ctx, s, None, 1, 2, 0.5, 8, 0.1)
    compare(res, ref)
    assert int(res.count[0]) == 3


def test_constant_map_worst_case_radix_select(ctx):
    # every interior pixel is a candidate (n = 124*252 = 31248 > 8192): MSB radix select must walk
    # into the index bits; result = the first top_k interior pixels in raster order
    s = torch.full((2, 128, 256), 0.7)
    s[1] = 0.3
    for top_k in (1, 100, 8192):
        res, ref = run_both(ctx, s, None, 1, 2, 0.2, top_k, 0.1)
        compare(res, ref)
        assert int(res.count[0]) == top_k
        assert int(res.index[0, 0]) == 2 * 256 + 2


def test_many_candidates_mixed_scores_radix_select(ctx):
    # > 8192 candidates with few distinct scores and a big tie class straddling the k-th place
    g = torch.Generator().manual_seed(5)
    s = (torch.randint(0, 4, (1, 300, 400), generator=g).float() / 4.0)
    s = torch.nn.functional.max_pool2d(s[None], 3, 1, 1)[0]     # plateaus -> lots of tied maxima
    for top_k in (500, 4096, 8192):
        res, ref = run_both(ctx, s, None, 1, 1, 0.2, top_k, 0.1)
        compare(res, ref)
    n = int(oracle.nms_mask(s[0].numpy(), 1, 0.2).sum())
    assert n > 8192


def test_ties_at_clamp_value_adjacent(ctx):
    s = synth.score_maps(1, 96, 200, 8, 0.1, 900)               # dense blobs -> many exact 1.0, some adjacent
    res, ref = run_both(ctx, s, None, 1, 2, 0.2, 512, 0.1)
    compare(res, ref)
    assert (ref.scores == 1.0).sum() > 20


def test_negative_threshold_and_signed_zero(ctx):
    s = torch.zeros((1, 40, 140))
    s[0, 10, 10] = -0.0
    s[0, 20, 20] = -0.25
    s[0, 30, 30] = 0.25
    res, ref = run_both(ctx, s - 0.0, None, 1, 2, -0.5, 4096, 0.1)
    compare(res, ref)


# ---- API surface -----------------------------------------------------------------------------------
def test_loader_graph_and_literal_variants_agree(ctx):
    from paper_2607_01757_b200.binding import OPT_USE_GRAPH, OPT_USE_TMA, OPT_USE_PDL
    score, desc = small_inputs(2, 100, 260, seed=21, nblobs=200, D=128, dtype=torch.float16, stride=1)
    sd = score.cuda()
    base = ctx.extract(sd, desc, 1, 2, 0.2, 256, 0.1)
    torch.cuda.synchronize()
    try:
        for graph in (0, 1):
            for tma in (0, 1):
                for pdl in (0, 1):
                    ctx.set_option(OPT_USE_GRAPH, graph)
                    ctx.set_option(OPT_USE_TMA, tma)
                    ctx.set_option(OPT_USE_PDL, pdl)
                    for rep in range(3):                          # later calls replay the cached graph
                        r2 = ctx.extract(sd, desc, 1, 2, 0.2, 256, 0.1)
                        torch.cuda.synchronize()
                        for n in ("kpts", "scores", "desc", "count", "index", "offsets"):
                            assert torch.equal(getattr(base, n), getattr(r2, n)), (graph, tma, pdl, n)
    finally:
        ctx.set_option(OPT_USE_GRAPH, 1)
        ctx.set_option(OPT_USE_TMA, 1)
        ctx.set_option(OPT_USE_PDL, 1)
    lit = ctx.alloc_outputs(2, 256, desc, 128, want_index=False, want_offsets=False)
    ctx.extract_literal(sd, desc, 1, 2, 0.2, 256, 0.1, lit)
    torch.cuda.synchronize()
    for n in ("kpts", "scores", "desc", "count"):
        assert torch.equal(getattr(base, n), getattr(lit, n)), n


def test_back_to_back_stream_launches_overlap_safely(ctx):
    """Plain launches with programmatic dependent launch: the NMS kernel of call i+1 is launched while the refine /
    gather kernel of call i still runs (both use the context's candidate workspace).  200 calls alternating between
    two different inputs, never synchronised in between, must give exactly the results of isolated calls; a producer
    kernel of the caller enqueued right before a call (it writes the score map) must be seen completely."""
    from paper_2607_01757_b200.binding import OPT_USE_GRAPH
    ins = [small_inputs(2, 120, 380, seed=40 + j, nblobs=300 + 100 * j, D=128, dtype=torch.float16, stride=1) for j in range(2)]
    sds = [i[0].cuda() for i in ins]
    want = []
    for j in range(2):
        want.append(ctx.extract(sds[j], ins[j][1], 1, 2, 0.2, 256, 0.1))
        torch.cuda.synchronize()
    try:
        ctx.set_option(OPT_USE_GRAPH, 0)
        outs = [ctx.alloc_outputs(2, 256, ins[0][1], 128) for _ in range(200)]
        for i in range(200):
            ctx.extract(sds[i % 2], ins[i % 2][1], 1, 2, 0.2, 256, 0.1, out=outs[i])
        torch.cuda.synchronize()
        for i in range(200):
            for n in ("kpts", "scores", "desc", "count", "index", "offsets"):
                assert torch.equal(getattr(want[i % 2], n), getattr(outs[i], n)), (i, n)
        # the score map is produced by a kernel of the caller right before the call
        buf = torch.zeros_like(sds[0])
        for i in range(20):
            buf.copy_(sds[i % 2] * 1.0)                          # (an elementwise kernel on the same stream)
            ctx.extract(buf, ins[i % 2][1], 1, 2, 0.2, 256, 0.1, out=outs[i])
        torch.cuda.synchronize()
        for i in range(20):
            for n in ("kpts", "scores", "desc", "count", "index", "offsets"):
                assert torch.equal(getattr(want[i % 2], n), getattr(outs[i], n)), ("producer", i, n)
    finally:
        ctx.set_option(OPT_USE_GRAPH, 1)


def test_batch_equals_single_images_and_keypoints_only(ctx):
    score, desc = small_inputs(3, 90, 200, seed=2, nblobs=100, D=64, dtype=torch.float32, stride=1)
    sd = score.cuda()
    full = ctx.extract(sd, desc, 1, 2, 0.2, 64, 0.1)
    nod = ctx.extract(sd, None, 1, 2, 0.2, 64, 0.1)             # LK pathway
    torch.cuda.synchronize()
    assert nod.desc is None and torch.equal(nod.kpts, full.kpts) and torch.equal(nod.index, full.index)
    for b in range(3):
        one = ctx.extract(sd[b:b + 1].contiguous(), desc[b:b + 1].contiguous(), 1, 2, 0.2, 64, 0.1)
        torch.cuda.synchronize()
        for n in ("kpts", "scores", "desc", "count", "index", "offsets"):
            assert torch.equal(getattr(full, n)[b], getattr(one, n)[0]), n


def test_host_path_matches_device_path(ctx):
    score, desc = small_inputs(2, 90, 200, seed=4, nblobs=100, D=128, dtype=torch.float16, stride=1)
    dev = ctx.extract(score.cuda(), desc, 1, 2, 0.2, 128, 0.1)
    torch.cuda.synchronize()
    # pinned buffers: descriptor rows sampled in place over PCIe (the gather touches 128*4 of 18000 rows),
    # outputs stored straight into the host tensors; pageable buffers: staged copies; resident: uploaded once
    sp, dp = score.pin_memory(), desc.cpu().pin_memory()
    pageable_out = ctx.alloc_outputs(2, 128, desc, 128, device="cpu", pin=False)
    for s_in, d_in, out, resident in ((sp, dp, None, False), (sp, dp, None, True), (sp, dp, None, True),
                                      (score, desc.cpu(), pageable_out, False), (sp, dp, pageable_out, False),
                                      (score, desc.cpu(), None, False)):
        host = ctx.extract_host(s_in, d_in, 1, 2, 0.2, 128, 0.1, out=out, desc_resident=resident)
        for n in ("kpts", "scores", "desc", "count", "index", "offsets"):
            assert not getattr(host, n).is_cuda
            assert torch.equal(getattr(dev, n).cpu(), getattr(host, n)), n
        for n in ("kpts", "scores", "desc", "count", "index", "offsets"):
            getattr(host, n).zero_()


def test_capture_safe_inside_a_user_graph(ctx):
    score, desc = small_inputs(2, 64, 256, seed=6, nblobs=80, D=64, dtype=torch.float16, stride=1)
    sd = score.cuda()
    want = ctx.extract(sd, desc, 1, 2, 0.2, 64, 0.1)
    out = ctx.alloc_outputs(2, 64, desc, 64)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):                                     # the caller captures: no sync / alloc inside
        ctx.extract(sd, desc, 1, 2, 0.2, 64, 0.1, out=out)
    for t in (out.kpts, out.scores, out.desc, out.count, out.index, out.offsets):
        t.zero_()
    g.replay()
    torch.cuda.synchronize()
    for n in ("kpts", "scores", "desc", "count", "index", "offsets"):
        assert torch.equal(getattr(want, n), getattr(out, n)), n


def test_graph_cache_is_keyed_on_shapes_not_pointers():
    """1000 calls that rotate through fresh output buffers and several input maps (and change thresh / T) stay
    correct, and the library never captures or instantiates a second graph for the shape: the kernel nodes of the
    cached graph are re-pointed in place."""
    import paper_2607_01757_b200 as dkd
    c = dkd.DKD(2, 96, 256, 128, 64)
    try:
        inputs = []
        for seed in range(4):
            score, desc = small_inputs(2, 96, 256, seed=40 + seed, nblobs=150, D=64, dtype=torch.float16, stride=1)
            inputs.append((score, score.cuda(), desc))
        params = [(0.2, 0.1), (0.3, 0.1), (0.2, 0.25)]
        refs = {}
        for i, (score, _, desc) in enumerate(inputs):
            for j, (th, T) in enumerate(params):
                refs[(i, j)] = oracle.extract(score.numpy(), desc.cpu().numpy(), 1, 2, th, 128, T)
        outs = []
        for it in range(1000):
            i, j = it % 4, (it // 4) % 3
            res = c.extract(inputs[i][1], inputs[i][2], 1, 2, params[j][0], 128, params[j][1])   # fresh outputs every call
            outs.append((i, j, res))
            if len(outs) == 50:                                   # check in batches (keeps 50 output sets alive at once)
                for (ii, jj, rr) in outs:
                    compare(rr, refs[(ii, jj)], torch.float16)
                outs = []
        st = c.graph_stats()
        assert st["instantiated"] == 1, st                        # one shape -> one graph, ever
        assert st["updated"] >= 990 and st["stream"] == 0, st
        # a different shape (other top_k) is a second graph; the first one is still valid afterwards
        c.extract(inputs[0][1], inputs[0][2], 1, 2, 0.2, 64, 0.1)
        res = c.extract(inputs[1][1], inputs[1][2], 1, 2, 0.2, 128, 0.1)
        compare(res, refs[(1, 0)], torch.float16)
        assert c.graph_stats()["instantiated"] == 2
    finally:
        c.close()


def test_unaligned_outputs_are_rejected_not_faulted(ctx):
    import paper_2607_01757_b200 as dkd
    s = torch.zeros((1, 32, 128), device="cuda")
    out = ctx.alloc_outputs(1, 8, None, 0)
    flat = torch.zeros(1 * 8 * 2 + 1, device="cuda")
    out.kpts = flat[1:].view(1, 8, 2)                             # 4-byte aligned only: the kernel stores float2
    with pytest.raises(dkd.DKDError) as e:
        ctx.extract(s, None, 1, 2, 0.2, 8, 0.1, out=out)
    assert e.value.code == -2
    out = ctx.alloc_outputs(1, 8, None, 0)
    out.scores = torch.zeros((1, 9), device="cuda")               # wrong shape: caught by the binding
    with pytest.raises(dkd.DKDError):
        ctx.extract(s, None, 1, 2, 0.2, 8, 0.1, out=out)
    torch.cuda.synchronize()                                      # the context is still usable
    ctx.extract(s, None, 1, 2, 0.2, 8, 0.1)
    torch.cuda.synchronize()


def test_host_path_validates_before_any_copy(ctx):
    import paper_2607_01757_b200 as dkd
    s = torch.zeros((1, 32, 128)).pin_memory()
    for bad in (dict(r=0), dict(T=0.0), dict(r=7), dict(top_k=0)):
        kw = dict(r=2, T=0.1, top_k=8)
        kw.update(bad)
        with pytest.raises(dkd.DKDError):
            ctx.extract_host(s, None, 1, kw["r"], 0.2, kw["top_k"], kw["T"])


def test_deterministic_across_runs(ctx):
    score, desc = small_inputs(2, 150, 400, seed=12, nblobs=500, D=64, dtype=torch.float16, stride=1)
    sd = score.cuda()
    a = ctx.extract(sd, desc, 1, 2, 0.2, 512, 0.1)
    torch.cuda.synchronize()
    for _ in range(5):
        b = ctx.extract(sd, desc, 1, 2, 0.2, 512, 0.1)
        torch.cuda.synchronize()
        for n in ("kpts", "scores", "desc", "count", "index", "offsets"):
            assert torch.equal(getattr(a, n), getattr(b, n)), n


def test_error_codes(ctx):
    import paper_2607_01757_b200 as dkd
    s = torch.zeros((1, 32, 128), device="cuda")
    d = torch.zeros((1, 32, 128, 64), device="cuda", dtype=torch.float16)
    def code(fn):
        with pytest.raises(dkd.DKDError) as e:
            fn()
        return e.value.code
    assert code(lambda: ctx.extract(s, None, 1, 0, 0.2, 8, 0.1)) == -1          # r < 1
    assert code(lambda: ctx.extract(s, None, 1, 2, 0.2, 8, 0.0)) == -1          # T <= 0
    assert code(lambda: ctx.extract(s, None, 1, 2, 0.2, 8, float("inf"))) == -1
    assert code(lambda: ctx.extract(s, None, 1, 2, 0.2, 0, 0.1)) == -1          # top_k < 1
    assert code(lambda: ctx.extract(s, None, 1, 5, 0.2, 8, 0.1)) == -2          # r > DKD_MAX_RADIUS
    assert code(lambda: ctx.extract(s, d[..., :4].contiguous(), 1, 2, 0.2, 8, 0.1)) == -2   # 8-byte rows
    assert code(lambda: ctx.extract(s, None, 1, 2, 0.2, 9000, 0.1)) == -3       # top_k > max
    big = torch.zeros((5, 32, 128), device="cuda")
    assert code(lambda: ctx.extract(big, None, 1, 2, 0.2, 8, 0.1)) == -3        # B > max_batch
    assert code(lambda: dkd.DKD(1, 8, 8, 9000)) == -2                           # max_top_k > DKD_MAX_TOP_K
    assert ctx.workspace_bytes > 0 and ctx.launches_per_extract() == 3
