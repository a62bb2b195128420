"""Shared helper for the GPU parity tests: runs the CUDA path (through the C-ABI binding) and the
CPU oracle on the same inputs and compares element by element.

Tolerances (BASELINE.json north_star):
  * integer positions, order, counts, scores: bit-exact;
  * sub-pixel offsets (dx,dy): <= 1e-5 px absolute;
  * stored fp32 coordinates: <= 1e-5 + half an fp32 ulp of the oracle's value (G11);
  * descriptors: <= 2e-3 absolute for f16 maps, <= 1e-5 for f32 maps;
  * padding slots: exactly zero / index -1.
"""
import numpy as np
import torch

import oracle

TOL_OFFSET = 1e-5
TOL_DESC = {torch.float16: 2e-3, torch.float32: 1e-5}


def half_ulp_f32(x64: np.ndarray) -> np.ndarray:
    x32 = np.abs(x64).astype(np.float32)
    return 0.5 * (np.nextafter(x32, np.float32(np.inf)) - x32).astype(np.float64)


def compare(res, ref, desc_dtype=None, images=None):
    """res: DKDResult (cuda tensors); ref: oracle.OracleResult.  `images`: the batch indices of
    `res` that `ref` covers (default: all)."""
    torch.cuda.synchronize()
    sel = slice(None) if images is None else list(images)
    count = res.count.cpu().numpy()[sel]
    assert np.array_equal(count, ref.count), f"count {count} vs {ref.count}"
    if res.index is not None:
        assert np.array_equal(res.index.cpu().numpy()[sel], ref.index), "index / order mismatch"
    sc = res.scores.cpu().numpy()[sel]
    assert np.array_equal(sc.view(np.uint32), ref.scores.view(np.uint32)), "scores not bit-exact"
    if res.offsets is not None:
        off = res.offsets.cpu().numpy()[sel].astype(np.float64)
        err = np.abs(off - ref.offsets).max() if off.size else 0.0
        assert err <= TOL_OFFSET, f"offset error {err}"
    kp = res.kpts.cpu().numpy()[sel].astype(np.float64)
    bound = TOL_OFFSET + half_ulp_f32(ref.kpts)
    assert np.all(np.abs(kp - ref.kpts) <= bound), f"kpt error {np.abs(kp - ref.kpts).max()}"
    stats = {"max_offset_err": float(np.abs(res.offsets.cpu().numpy()[sel] - ref.offsets).max())
             if res.offsets is not None and ref.offsets.size else 0.0}
    if ref.desc is not None:
        d = res.desc.cpu().numpy()[sel].astype(np.float64)
        tol = TOL_DESC[desc_dtype]
        err = np.abs(d - ref.desc).max() if d.size else 0.0
        assert err <= tol, f"descriptor error {err} > {tol}"
        stats["max_desc_err"] = float(err)
        k = ref.index.shape[1]
        pad = np.arange(k)[None, :] >= ref.count[:, None]
        assert np.all(d[pad] == 0.0), "descriptor padding not zero"
        nrm = np.linalg.norm(d[~pad], axis=-1)
        if nrm.size:
            assert np.abs(nrm - 1.0).max() <= (2e-3 if desc_dtype == torch.float16 else 1e-5)
    return stats


def run_both(ctx, score_cpu, desc_dev, stride, r, thresh, top_k, T, **kw):
    score_dev = score_cpu.cuda()
    res = ctx.extract(score_dev, desc_dev, stride, r, thresh, top_k, T, **kw)
    ref = oracle.extract(score_cpu.numpy(), None if desc_dev is None else desc_dev.cpu().numpy(),
                         stride, r, thresh, top_k, T)
    return res, ref
