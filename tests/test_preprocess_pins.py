"""Pins of the pre-processing oracle (oracle.preprocess) against what
the definition fixes: a hand-worked fixture, closed forms, invariants, and an independent torch routine."""
import os

import numpy as np
import pytest
import torch

import oracle

HERE = os.path.dirname(os.path.abspath(__file__))


def test_golden_tiny_luma_letterbox():
    exp = np.loadtxt(os.path.join(HERE, "golden", "preprocess_tiny.txt"))
    img = np.array([[[255, 0, 0], [0, 255, 0], [0, 0, 255]],
                    [[255, 255, 255], [0, 0, 0], [10, 20, 30]]], np.uint8)[None]
    out = oracle.preprocess(img, 1, 4, mean=(0.5,) * 3, inv_std=(2.0,) * 3, pad_value=-1.0)
    assert out.shape == (1, 1, 4, 4)
    assert np.abs(out[0, 0] - exp).max() < 1e-12
    # the same image stored B,G,R gives the same luminance
    out_bgr = oracle.preprocess(img[..., ::-1], 1, 4, bgr=True, mean=(0.5,) * 3, inv_std=(2.0,) * 3, pad_value=-1.0)
    assert np.array_equal(out, out_bgr)


@pytest.mark.parametrize("H,W,grid", [(480, 752, 8), (480, 752, 32), (7, 5, 8), (32, 64, 32), (33, 65, 32), (600, 960, 32)])
def test_padded_size_and_centred_offset(H, W, grid):
    Hp, Wp, oy, ox = oracle.padded_size(H, W, grid)
    assert Hp % grid == 0 and Wp % grid == 0 and 0 <= Hp - H < grid and 0 <= Wp - W < grid      # P1
    assert oy == (Hp - H) // 2 and ox == (Wp - W) // 2                                           # P2
    g = np.random.default_rng(H * W)
    img = g.integers(0, 256, (2, H, W, 1), dtype=np.uint8)
    out = oracle.preprocess(img, 1, grid, scale=1.0, pad_value=-7.0)
    assert out.shape == (2, 1, Hp, Wp)
    inner = out[:, :, oy:oy + H, ox:ox + W]
    assert np.array_equal(inner[:, 0], img[..., 0].astype(np.float64))                           # exact copy
    mask = np.ones((Hp, Wp), bool)
    mask[oy:oy + H, ox:ox + W] = False
    assert np.all(out[:, :, mask] == -7.0)                                                       # P3
    assert mask.sum() == Hp * Wp - H * W


def test_mono_replication_and_per_channel_normalisation():
    g = np.random.default_rng(3)
    img = g.integers(0, 256, (1, 9, 11, 1), dtype=np.uint8)
    mean, inv_std = (0.485, 0.456, 0.406), (1 / 0.229, 1 / 0.224, 1 / 0.225)
    out = oracle.preprocess(img, 3, 8, mean=mean, inv_std=inv_std)
    Hp, Wp, oy, ox = oracle.padded_size(9, 11, 8)
    v = img[0, :, :, 0].astype(np.float64) / 255.0
    for c in range(3):                                                                           # P5, P6
        assert np.abs(out[0, c, oy:oy + 9, ox:ox + 11] - (v - mean[c]) * inv_std[c]).max() < 1e-15
    same = oracle.preprocess(img, 3, 8)
    assert np.array_equal(same[0, 0], same[0, 1]) and np.array_equal(same[0, 0], same[0, 2])


def test_luma_closed_forms_and_channel_order():
    def one(px, **kw):
        return oracle.preprocess(np.array(px, np.uint8).reshape(1, 1, 1, 3), 1, 1, scale=1.0, **kw)[0, 0, 0, 0]
    assert abs(one([255, 0, 0]) - 0.299 * 255) < 1e-12 and abs(one([0, 255, 0]) - 0.587 * 255) < 1e-12
    assert abs(one([0, 0, 255]) - 0.114 * 255) < 1e-12
    assert abs(one([200, 200, 200]) - 200.0) < 1e-10                                             # weights sum to 1
    assert abs(one([0, 0, 255], bgr=True) - 0.299 * 255) < 1e-12
    rgb = oracle.preprocess(np.array([[[[1, 2, 3]]]], np.uint8), 3, 1, scale=1.0)
    bgr = oracle.preprocess(np.array([[[[3, 2, 1]]]], np.uint8), 3, 1, scale=1.0, bgr=True)
    assert rgb[0, :, 0, 0].tolist() == [1.0, 2.0, 3.0] and np.array_equal(rgb, bgr)              # planes R,G,B


@pytest.mark.parametrize("cin,cout,grid", [(1, 1, 8), (1, 3, 32), (3, 1, 8), (3, 3, 32)])
def test_matches_independent_torch_routine(cin, cout, grid):
    """Library special case: the same pipeline from torch tensor ops in float64 (pad, permute, matmul)."""
    g = np.random.default_rng(cin * 10 + cout)
    B, H, W = 2, 37, 50
    img = g.integers(0, 256, (B, H, W, cin), dtype=np.uint8)
    mean, inv_std = (0.1, 0.2, 0.3), (1.5, 2.5, 0.5)
    out = oracle.preprocess(img, cout, grid, mean=mean, inv_std=inv_std, pad_value=0.25)
    t = torch.from_numpy(img).to(torch.float64).permute(0, 3, 1, 2)                              # NCHW
    if cin == 1 and cout == 3:
        t = t.expand(-1, 3, -1, -1)
    elif cin == 3 and cout == 1:
        t = (t * torch.tensor([0.299, 0.587, 0.114], dtype=torch.float64).view(1, 3, 1, 1)).sum(1, keepdim=True)
    m = torch.tensor(mean[:cout], dtype=torch.float64).view(1, cout, 1, 1)
    s = torch.tensor(inv_std[:cout], dtype=torch.float64).view(1, cout, 1, 1)
    t = (t / 255.0 - m) * s
    Hp, Wp, oy, ox = oracle.padded_size(H, W, grid)
    t = torch.nn.functional.pad(t, (ox, Wp - W - ox, oy, Hp - H - oy), value=0.25)
    assert np.abs(out - t.numpy()).max() < 1e-12


def test_keypoint_unshift_round_trip():
    """P2: a bright pixel at native (x,y) sits at (x+ox, y+oy) in the padded map; subtracting the offset
    from a keypoint found there gives the native position back."""
    H, W, grid = 21, 45, 32
    Hp, Wp, oy, ox = oracle.padded_size(H, W, grid)
    img = np.zeros((1, H, W, 1), np.uint8)
    img[0, 13, 30, 0] = 255
    out = oracle.preprocess(img, 1, grid)
    yp, xp = np.unravel_index(np.argmax(out[0, 0]), (Hp, Wp))
    assert (xp - ox, yp - oy) == (30, 13)


def test_rejects_bad_arguments():
    with pytest.raises(ValueError):
        oracle.preprocess(np.zeros((1, 4, 4, 2), np.uint8), 1, 8)
    with pytest.raises(ValueError):
        oracle.preprocess(np.zeros((1, 4, 4, 1), np.uint8), 2, 8)
