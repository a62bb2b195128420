"""CPU oracle for the DKD + descriptor-sampling hot path — TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  The product
(``paper_2607_01757_b200``) never does, and this package never imports the product.

The arithmetic lives in ``dkd_oracle.c`` (the hot path), ``dkd_variants.c`` (the DKD variants, SURVEY.md
8(f) f2) and ``match_oracle.c`` (descriptor matching, retrieval scan, stereo validation, covariance weighting:
f3, f4) — plain C99, fp64, naive loops; see their headers for the passages of /root/reference/PAPER.md and the
DESIGN.md readings they follow.  This file only compiles them with gcc and marshals numpy arrays through ctypes.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRCS = [os.path.join(_HERE, f) for f in ("dkd_oracle.c", "dkd_variants.c", "match_oracle.c")]
_LIB = os.path.join(_HERE, "libdkd_oracle.so")

F32, F16 = 0, 1
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp (no -ffast-math) -> oracle/libdkd_oracle.so."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(f) for f in _SRCS):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-fopenmp", "-shared", "-fPIC",
                               *_SRCS, "-o", tmp, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        vp, i, f = ctypes.c_void_p, ctypes.c_int, ctypes.c_float
        L.dkd_oracle_num_threads.restype = i
        L.dkd_oracle_nms.restype = ctypes.c_long
        L.dkd_oracle_nms.argtypes = [vp, i, i, i, f, vp]
        L.dkd_oracle_topk.restype = i
        L.dkd_oracle_topk.argtypes = [vp, vp, i, i, i, vp, vp]
        L.dkd_oracle_refine.restype = None
        L.dkd_oracle_refine.argtypes = [vp, i, i, i, f, i, vp, vp, vp]
        L.dkd_oracle_gather.restype = None
        L.dkd_oracle_gather.argtypes = [vp, i, i, i, i, i, i, vp, vp, vp]
        L.dkd_oracle_preprocess.restype = i
        L.dkd_oracle_preprocess.argtypes = [vp, i, i, i, i, i, i, i, ctypes.c_double, vp, vp, ctypes.c_double, vp]
        L.dkd_oracle_extract.restype = i
        L.dkd_oracle_extract.argtypes = [vp, i, i, i, vp, i, i, i, i, i, i, f, i, f,
                                         vp, vp, vp, vp, vp, vp]
        d = ctypes.c_double
        L.dkd_oracle_nms_iter.restype = ctypes.c_long
        L.dkd_oracle_nms_iter.argtypes = [vp, i, i, i, f, i, vp]
        L.dkd_oracle_bilinear_score.restype = d
        L.dkd_oracle_bilinear_score.argtypes = [vp, i, i, d, d]
        L.dkd_oracle_extract_var.restype = i
        L.dkd_oracle_extract_var.argtypes = [vp, vp, vp, i, i, i, vp, i, i, i, i, i, i, f, i, f, i, i,
                                             vp, vp, vp, vp, vp, vp, vp]
        L.match_oracle_nn.restype = i
        L.match_oracle_nn.argtypes = [vp, vp, i, i, i, i, i, i, d, i, vp, vp, vp, vp]
        L.retrieval_oracle_scan.restype = i
        L.retrieval_oracle_scan.argtypes = [vp, vp, i, i, i, i, d, i, vp, vp]
        L.stereo_oracle_validate.restype = i
        L.stereo_oracle_validate.argtypes = [vp, vp, i, d, d, d, d, d, d, d, d, d, vp, vp, vp, vp]
        L.cov_oracle_sqrt_info.restype = i
        L.cov_oracle_sqrt_info.argtypes = [vp, i, d, d, d, d, d, d, d, vp, vp]
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().dkd_oracle_num_threads())


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _c(a, dtype):
    a = np.ascontiguousarray(a, dtype=dtype)
    return a


def _desc_arg(desc):
    if desc is None:
        return None, F32
    if desc.dtype == np.float16:
        return np.ascontiguousarray(desc), F16
    if desc.dtype == np.float32:
        return np.ascontiguousarray(desc), F32
    raise TypeError("descriptor map must be float16 or float32")


# ---- step functions (one image) -------------------------------------------------------------
def nms_mask(S, r, thresh):
    """O1 -> uint8 mask [H,W]."""
    S = _c(S, np.float32)
    H, W = S.shape
    mask = np.zeros((H, W), np.uint8)
    n = lib().dkd_oracle_nms(_p(S), H, W, int(r), float(thresh), _p(mask))
    assert n == int(mask.sum())
    return mask


def topk(S, mask, top_k):
    """O2 -> (K, idx[top_k] int32 (-1 padded), score[top_k] f32 (0 padded))."""
    S = _c(S, np.float32)
    mask = _c(mask, np.uint8)
    H, W = S.shape
    idx = np.empty(top_k, np.int32)
    sc = np.empty(top_k, np.float32)
    K = lib().dkd_oracle_topk(_p(S), _p(mask), H, W, int(top_k), _p(idx), _p(sc))
    return int(K), idx, sc


def refine(S, r, T, idx):
    """O3 -> (off[n,2] f64 (dx,dy), kpt[n,2] f64 (x,y))."""
    S = _c(S, np.float32)
    idx = _c(idx, np.int32)
    H, W = S.shape
    n = idx.shape[0]
    off = np.empty((n, 2), np.float64)
    kpt = np.empty((n, 2), np.float64)
    lib().dkd_oracle_refine(_p(S), H, W, int(r), float(T), n, _p(idx), _p(off), _p(kpt))
    return off, kpt


def gather(F, stride, kpt, valid=None):
    """O4 -> out[n,D] f64.  F [Hd,Wd,D] f16|f32; kpt [n,2] f64 in score-map pixels."""
    F, dt = _desc_arg(F)
    Hd, Wd, D = F.shape
    kpt = _c(kpt, np.float64)
    n = kpt.shape[0]
    v = None if valid is None else _c(valid, np.int32)
    out = np.empty((n, D), np.float64)
    lib().dkd_oracle_gather(_p(F), dt, Hd, Wd, D, int(stride), n, _p(kpt), _p(v), _p(out))
    return out


# ---- whole path -----------------------------------------------------------------------------
@dataclass
class OracleResult:
    kpts: np.ndarray     # [B,k,2] f64 (x,y)
    offsets: np.ndarray  # [B,k,2] f64 (dx,dy)
    scores: np.ndarray   # [B,k]   f32
    desc: np.ndarray     # [B,k,D] f64 or None
    count: np.ndarray    # [B]     i32
    index: np.ndarray    # [B,k]   i32, -1 padding


def extract(score, desc, stride, r, thresh, top_k, T) -> OracleResult:
    """O1..O5 over a batch.  score [B,H,W] f32; desc [B,Hd,Wd,D] f16|f32 or None."""
    score = _c(score, np.float32)
    B, H, W = score.shape
    desc, dt = _desc_arg(desc)
    if desc is not None:
        assert desc.shape[0] == B
        _, Hd, Wd, D = desc.shape
    else:
        Hd = Wd = D = 0
    k = int(top_k)
    kp = np.empty((B, k, 2), np.float64)
    off = np.empty((B, k, 2), np.float64)
    sc = np.empty((B, k), np.float32)
    de = np.empty((B, k, D), np.float64) if desc is not None else None
    cnt = np.empty(B, np.int32)
    idx = np.empty((B, k), np.int32)
    rc = lib().dkd_oracle_extract(_p(score), B, H, W, _p(desc), dt, Hd, Wd, D, int(stride),
                                  int(r), float(thresh), k, float(T),
                                  _p(kp), _p(off), _p(sc), _p(de), _p(cnt), _p(idx))
    if rc != 0:
        raise ValueError("dkd_oracle_extract: invalid argument")
    return OracleResult(kp, off, sc, de, cnt, idx)


# ---- fused input pre-processing ---------------------------
def padded_size(H: int, W: int, grid: int):
    """(Hp, Wp, oy, ox): padded size on the resolution grid and the centred letterbox offset (P1, P2)."""
    Hp, Wp = (H + grid - 1) // grid * grid, (W + grid - 1) // grid * grid
    return Hp, Wp, (Hp - H) // 2, (Wp - W) // 2


def preprocess(src, out_channels, grid, bgr=False, scale=1.0 / 255.0, mean=(0.0, 0.0, 0.0),
               inv_std=(1.0, 1.0, 1.0), pad_value=0.0) -> np.ndarray:
    """src [B,H,W,Cin] u8 -> [B,Cout,Hp,Wp] f64 (letterbox, colour conversion, normalisation, NCHW)."""
    src = _c(src, np.uint8)
    B, H, W, Cin = src.shape
    Hp, Wp, _, _ = padded_size(H, W, grid)
    m = _c(np.asarray(mean, np.float64), np.float64)
    s = _c(np.asarray(inv_std, np.float64), np.float64)
    out = np.empty((B, int(out_channels), Hp, Wp), np.float64)
    rc = lib().dkd_oracle_preprocess(_p(src), B, H, W, Cin, int(out_channels), int(grid), int(bool(bgr)),
                                     float(scale), _p(m), _p(s), float(pad_value), _p(out))
    if rc != 0:
        raise ValueError("dkd_oracle_preprocess: invalid argument")
    return out



# ---- DKD variants (dkd_variants.c) ------------------------------------------------
def nms_mask_iter(S, r, thresh, iters):
    """V1 -> uint8 mask [H,W] of the iterated suppress-and-recover NMS (iters = 0: the single pass)."""
    S = _c(S, np.float32)
    H, W = S.shape
    mask = np.zeros((H, W), np.uint8)
    n = lib().dkd_oracle_nms_iter(_p(S), H, W, int(r), float(thresh), int(iters), _p(mask))
    assert n == int(mask.sum())
    return mask


def bilinear_score(S, px, py):
    """V2 -> S interpolated bilinearly at (px, py) (fp64)."""
    S = _c(S, np.float32)
    H, W = S.shape
    return float(lib().dkd_oracle_bilinear_score(_p(S), H, W, float(px), float(py)))


@dataclass
class OracleVarResult(OracleResult):
    total: np.ndarray = None   # [B] i32: candidates before the cap (V3)


def extract_var(score, desc, stride, r, thresh, top_k, T, reliability=None, valid_mask=None, nms_iters=0,
                score_mode=0) -> OracleVarResult:
    """The whole path with the variants V1..V5.  `scores` is float64 (exactly the fp32 score in raw mode)."""
    score = _c(score, np.float32)
    B, H, W = score.shape
    rel = None if reliability is None else _c(reliability, np.float32)
    vm = None if valid_mask is None else _c(valid_mask, np.uint8)
    assert rel is None or rel.shape == score.shape
    assert vm is None or vm.shape == score.shape
    desc, dt = _desc_arg(desc)
    if desc is not None:
        _, Hd, Wd, D = desc.shape
    else:
        Hd = Wd = D = 0
    k = int(top_k)
    kp = np.empty((B, k, 2), np.float64)
    off = np.empty((B, k, 2), np.float64)
    sc = np.empty((B, k), np.float64)
    de = np.empty((B, k, D), np.float64) if desc is not None else None
    cnt = np.empty(B, np.int32)
    idx = np.empty((B, k), np.int32)
    tot = np.empty(B, np.int32)
    rc = lib().dkd_oracle_extract_var(_p(score), _p(rel), _p(vm), B, H, W, _p(desc), dt, Hd, Wd, D, int(stride),
                                      int(r), float(thresh), k, float(T), int(nms_iters), int(score_mode),
                                      _p(kp), _p(off), _p(sc), _p(de), _p(cnt), _p(idx), _p(tot))
    if rc != 0:
        raise ValueError("dkd_oracle_extract_var: invalid argument")
    return OracleVarResult(kp, off, sc, de, cnt, idx, tot)


# ---- descriptor matching / retrieval / stereo validation / covariance (f3, f4; match_oracle.c) -----------
def _mdt(a):
    if a.dtype == np.float16:
        return F16
    if a.dtype == np.float32:
        return F32
    raise TypeError("descriptors must be float16 or float32")


def match_nn(A, Bm, na=None, nb=None, ratio=0.8, mutual=False, want_sim=False):
    """M1..M5.  A [Na,D], Bm [Nb,D] (f16|f32, same dtype) -> (idx [Na] i32, s1 [Na] f64, s2 [Na] f64[, S [na,nb]])."""
    A = np.ascontiguousarray(A)
    Bm = np.ascontiguousarray(Bm)
    assert A.dtype == Bm.dtype and A.shape[1] == Bm.shape[1]
    Na, D = A.shape
    Nb = Bm.shape[0]
    na = Na if na is None else int(na)
    nb = Nb if nb is None else int(nb)
    idx = np.empty(Na, np.int32)
    s1 = np.empty(Na, np.float64)
    s2 = np.empty(Na, np.float64)
    S = np.empty((na, nb), np.float64) if want_sim else None
    rc = lib().match_oracle_nn(_p(A), _p(Bm), _mdt(A), Na, Nb, D, na, nb, float(ratio), int(bool(mutual)),
                               _p(idx), _p(s1), _p(s2), _p(S))
    if rc < 0:
        raise ValueError("match_oracle_nn: invalid argument")
    return (idx, s1, s2, S) if want_sim else (idx, s1, s2)


def retrieval_scan(db, q, n_exclude=50, tau=0.60, max_cand=16):
    """M6..M8.  db [n,D], q [D] (f16|f32) -> (sim [n] f64, cand [max_cand] i32 (-1 padded), count)."""
    db = np.ascontiguousarray(db)
    q = np.ascontiguousarray(q)
    assert db.dtype == q.dtype and db.shape[1] == q.shape[0]
    n, D = db.shape
    sim = np.empty(n, np.float64)
    cand = np.empty(max_cand, np.int32)
    K = lib().retrieval_oracle_scan(_p(db), _p(q), _mdt(db), n, D, int(n_exclude), float(tau), int(max_cand),
                                    _p(sim), _p(cand))
    if K < 0:
        raise ValueError("retrieval_oracle_scan: invalid argument")
    return sim, cand, int(K)


def stereo_validate(pl, pr, fx, fy, cx, cy, baseline, d_min, z_min, z_max, max_reproj=1.5):
    """S1..S4 -> (valid [n] u8, xyz [n,3], disparity [n], reproj_err [n])."""
    pl = _c(pl, np.float64)
    pr = _c(pr, np.float64)
    n = pl.shape[0]
    xyz = np.empty((n, 3), np.float64)
    disp = np.empty(n, np.float64)
    err = np.empty(n, np.float64)
    valid = np.empty(n, np.uint8)
    lib().stereo_oracle_validate(_p(pl), _p(pr), n, float(fx), float(fy), float(cx), float(cy), float(baseline),
                                 float(d_min), float(z_min), float(z_max), float(max_reproj),
                                 _p(xyz), _p(disp), _p(err), _p(valid))
    return valid, xyz, disp, err


def cov_sqrt_info(Lf, scale, floor_px, fx, fy, lam, lam_min, sigma0):
    """C1..C4.  Lf [n,3] = (l11, l21, l22) -> (omega [n,2,2] f64, ok [n] u8)."""
    Lf = _c(Lf, np.float64)
    n = Lf.shape[0]
    om = np.empty((n, 2, 2), np.float64)
    ok = np.empty(n, np.uint8)
    lib().cov_oracle_sqrt_info(_p(Lf), n, float(scale), float(floor_px), float(fx), float(fy), float(lam),
                               float(lam_min), float(sigma0), _p(om), _p(ok))
    return om, ok
