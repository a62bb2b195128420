"""Seeded input generator (synth/): determinism, recipe properties, CPU/any-device equality of the
descriptor hash.  Inputs stand in for the paper's datasets — DESIGN.md."""
import numpy as np
import torch

import synth


def test_score_maps_deterministic_and_in_range():
    a = synth.score_maps(2, 60, 94, seed=7, base=0.1, nblobs=40)
    b = synth.score_maps(2, 60, 94, seed=7, base=0.1, nblobs=40)
    c = synth.score_maps(2, 60, 94, seed=8, base=0.1, nblobs=40)
    assert a.dtype == torch.float32 and a.shape == (2, 60, 94)
    assert torch.equal(a, b) and not torch.equal(a, c)
    assert not torch.equal(a[0], a[1])
    assert float(a.min()) >= 0.0 and float(a.max()) <= 1.0
    noise = synth.score_maps(1, 60, 94, seed=7, base=0.1, nblobs=0)
    assert float(noise.max()) < 0.1 and float(noise.min()) >= 0.0
    assert abs(float(noise.mean()) - 0.05) < 0.005
    assert torch.all(a[0] >= noise[0])                      # blobs only add
    # clamp produces exact 1.0 ties with enough blobs (G1)
    dense = synth.score_maps(1, 60, 94, seed=3, base=0.1, nblobs=400)
    assert int((dense == 1.0).sum()) > 0


def test_desc_hash_matches_independent_numpy_and_is_standard_normal():
    B, Hd, Wd, D, seed = 2, 5, 7, 16, 11
    d = synth.desc_maps(B, Hd, Wd, D, seed, torch.float16, "cpu", chunk_elems=97)
    # independent numpy uint64 evaluation of the same recipe
    M = np.uint64(0xFFFFFFFFFFFFFFFF)
    with np.errstate(over="ignore"):
        for b in range(B):
            e = np.arange(Hd * Wd * D, dtype=np.uint64)
            x = e ^ np.uint64((seed ^ (3 << 56) ^ (b << 40)) & int(M))
            z = x + np.uint64(0x9E3779B97F4A7C15)
            z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
            z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
            z = z ^ (z >> np.uint64(31))
            want = synth.qtab(torch.float16).numpy()[(z >> np.uint64(48)).astype(np.int64)]
            assert np.array_equal(d[b].numpy().ravel(), want)
    big = synth.desc_maps(1, 64, 64, 64, 5, torch.float32)
    assert abs(float(big.mean())) < 0.01 and abs(float(big.std()) - 1.0) < 0.01
    # single elements can be evaluated alone (lazy evaluation for config 5)
    e = torch.tensor([0, 17, 4095, 64 * 64 * 64 - 1])
    assert torch.equal(synth.desc_elements(5, 0, e, torch.float32), big.view(-1)[e])


def test_configs_match_baseline_json():
    import json, os
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    cfgs = json.load(open(os.path.join(root, "BASELINE.json")))["configs"]
    assert len(cfgs) == 5
    c = synth.CONFIGS
    assert (c["c1"].B, c["c1"].H, c["c1"].W, c["c1"].top_k, c["c1"].D, c["c1"].desc_dtype) == (1, 480, 752, 256, 64, "f32")
    assert "top_k=1024" in cfgs[1] and c["c2"].top_k == 1024 and c["c2"].nblobs == 800
    assert "r=4" in cfgs[2] and c["c3"].r == 4 and c["c3"].stride == 8 and c["c3"].D == 256 and (c["c3"].Hd, c["c3"].Wd) == (60, 94)
    assert "720x1280" in cfgs[3] and (c["c4"].H, c["c4"].W, c["c4"].Hd, c["c4"].Wd) == (720, 1280, 90, 160)
    assert "B=64" in cfgs[4] and (c["c5"].B, c["c5"].H, c["c5"].W, c["c5"].top_k) == (64, 1080, 1920, 2048)
