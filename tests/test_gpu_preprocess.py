"""GPU parity of the fused input pre-processing kernel (dkd_preprocess) and of the keypoint
un-shift (DKD_OPT_ORIGIN_X/Y) against the CPU oracle.  Tolerances: f32 output
<= 5e-6 absolute (three fp32 roundings of the luminance, one fma, rounded constants), f16 output <= 2.5e-3
(half an f16 ulp at |out| <= 4); padding exactly pad_value; the exact-copy case bit-exact."""
import numpy as np
import pytest
import torch

import oracle
import synth
from _parity import compare

pytestmark = pytest.mark.gpu

MEAN, INV_STD = (0.485, 0.456, 0.406), (1 / 0.229, 1 / 0.224, 1 / 0.225)


@pytest.fixture(scope="module")
def ctx():
    import paper_2607_01757_b200 as dkd
    c = dkd.DKD(max_batch=2, max_h=512, max_w=800, max_top_k=1024, max_dim=128)
    yield c
    c.close()


def images(B, H, W, C, seed):
    return torch.from_numpy(np.random.default_rng(seed).integers(0, 256, (B, H, W, C), dtype=np.uint8))


@pytest.mark.parametrize("cin,cout", [(1, 1), (1, 3), (3, 1), (3, 3)])
@pytest.mark.parametrize("dtype", [torch.float32, torch.float16])
@pytest.mark.parametrize("HW,grid", [((480, 752), 32), ((480, 752), 8), ((37, 50), 32), ((61, 43), 5), ((64, 64), 32)])
def test_preprocess_matches_oracle(ctx, cin, cout, dtype, HW, grid):
    H, W = HW
    img = images(2, H, W, cin, seed=H * 7 + W + cin + cout)
    bgr = (H + cout) % 2 == 1
    out = ctx.preprocess(img.cuda(), cout, grid, bgr=bgr, mean=MEAN, inv_std=INV_STD, pad_value=-0.5, out_dtype=dtype)
    torch.cuda.synchronize()
    ref = oracle.preprocess(img.numpy(), cout, grid, bgr=bgr, mean=MEAN, inv_std=INV_STD, pad_value=-0.5)
    assert tuple(out.shape) == ref.shape
    err = np.abs(out.cpu().double().numpy() - ref).max()
    assert err <= (5e-6 if dtype == torch.float32 else 2.5e-3), err
    Hp, Wp, oy, ox = ctx.padded_size(H, W, grid)
    mask = torch.ones((Hp, Wp), dtype=torch.bool)
    mask[oy:oy + H, ox:ox + W] = False
    assert torch.all(out.cpu()[:, :, mask] == -0.5)


@pytest.mark.parametrize("cin,cout,dtype", [(1, 3, torch.float16), (3, 1, torch.float32)])
def test_preprocess_1080p_bench_shape(cin, cout, dtype):
    """1080 x 1920 -> 1088 x 1920 (grid 32): the shape bench.py times — the interior fast path with word loads plus the
    padded rows — mono -> 3 channels f16 (the bench leg) and colour -> luminance f32."""
    import paper_2607_01757_b200 as dkd
    c = dkd.DKD(max_batch=2, max_h=1088, max_w=1920, max_top_k=64, max_dim=0)
    try:
        img = images(2, 1080, 1920, cin, seed=cin + 40)
        out = c.preprocess(img.cuda(), cout, 32, bgr=False, mean=MEAN, inv_std=INV_STD, pad_value=-0.5, out_dtype=dtype)
        torch.cuda.synchronize()
        ref = oracle.preprocess(img.numpy(), cout, 32, bgr=False, mean=MEAN, inv_std=INV_STD, pad_value=-0.5)
        assert tuple(out.shape) == ref.shape == (2, cout, 1088, 1920)
        err = np.abs(out.cpu().double().numpy() - ref).max()
        assert err <= (5e-6 if dtype == torch.float32 else 2.5e-3), err
        Hp, Wp, oy, ox = c.padded_size(1080, 1920, 32)
        mask = torch.ones((Hp, Wp), dtype=torch.bool)
        mask[oy:oy + 1080, ox:ox + 1920] = False
        assert torch.all(out.cpu()[:, :, mask] == -0.5)
    finally:
        c.close()


def test_exact_copy_is_bit_exact(ctx):
    img = images(2, 100, 136, 1, seed=1)
    out = ctx.preprocess(img.cuda(), 1, 8, scale=1.0)
    torch.cuda.synchronize()
    ref = oracle.preprocess(img.numpy(), 1, 8, scale=1.0)
    assert np.array_equal(out.cpu().double().numpy(), ref)


def test_preprocess_error_codes(ctx):
    import paper_2607_01757_b200 as dkd
    img = images(1, 16, 16, 1, seed=2).cuda()
    with pytest.raises(dkd.DKDError):
        ctx.preprocess(img, 2, 8)
    with pytest.raises(dkd.DKDError):
        ctx.preprocess(img, 1, 0)
    with pytest.raises(dkd.DKDError):
        ctx.preprocess(img.cpu(), 1, 8)


def test_keypoints_are_shifted_back_to_native_coordinates(ctx):
    """A score map computed on the padded frame: with the letterbox offset set, the extracted keypoints equal the
    oracle's keypoints minus (ox, oy); indices, scores, descriptors are unchanged."""
    from paper_2607_01757_b200.binding import OPT_ORIGIN_X, OPT_ORIGIN_Y
    H, W, grid = 100, 150, 32
    Hp, Wp, oy, ox = ctx.padded_size(H, W, grid)
    score = synth.score_maps(2, Hp, Wp, 77, 0.1, 150)
    desc = synth.desc_maps(2, Hp, Wp, 64, 77, torch.float16, "cuda")
    try:
        ctx.set_option(OPT_ORIGIN_X, ox)
        ctx.set_option(OPT_ORIGIN_Y, oy)
        res = ctx.extract(score.cuda(), desc, 1, 2, 0.2, 128, 0.1)
        torch.cuda.synchronize()
    finally:
        ctx.set_option(OPT_ORIGIN_X, 0)
        ctx.set_option(OPT_ORIGIN_Y, 0)
    ref = oracle.extract(score.numpy(), desc.cpu().numpy(), 1, 2, 0.2, 128, 0.1)
    valid = np.arange(128)[None, :] < ref.count[:, None]
    ref.kpts[valid] -= np.array([ox, oy], np.float64)
    compare(res, ref, torch.float16)
    assert ox > 0 and oy > 0
