"""CPU oracle for the DKD + descriptor-sampling hot path — TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  The product
(``paper_2607_01757_b200``) never does, and this package never imports the product.

The arithmetic lives in ``dkd_oracle.c`` (plain C99, fp64, naive loops; see its header for the
passages of /root/reference/PAPER.md and the DESIGN.md readings it follows).  This file only
compiles it with gcc and marshals numpy arrays through ctypes.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dkd_oracle.c")
_LIB = os.path.join(_HERE, "libdkd_oracle.so")

F32, F16 = 0, 1
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp (no -ffast-math) -> oracle/libdkd_oracle.so."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-fopenmp", "-shared", "-fPIC",
                               _SRC, "-o", tmp, "-lm"])
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

