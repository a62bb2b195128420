"""Seeded synthetic inputs for the DKD hot path (serves both the oracle and the CUDA path).

Holds none of the method's arithmetic — only the input recipe of DESIGN.md "Input recipe"
(BASELINE.json configs 1-5).  These inputs stand in for the paper's
EuRoC / NTU-VIRAL / Botanic Garden / SubT-MRS frames and pretrained-network outputs
(Table III, 171), which are not available: only their shapes
(752x480, D in {64,128,256}, 1/8-resolution coarse maps, stereo = batch 2) are taken.

* score maps: host C generator (``score_gen.c``), deterministic, rounded once to fp32;
* descriptor maps "N(0,1)": ``QTAB[splitmix64(seed ^ 3<<56 ^ b<<40 ^ e) >> 48]`` with QTAB the
  65536-entry normal quantile table — integer hash + table lookup, so the torch implementation
  gives identical bits on CPU and on CUDA, and any element can be evaluated alone
  (``desc_elements``) without materialising the map (config 5's map is 34 GB).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, replace

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "score_gen.c")
_LIB = os.path.join(_HERE, "libscore_gen.so")
_lib = None


@dataclass(frozen=True)
class Config:
    name: str
    B: int
    H: int
    W: int
    base: float        # noise amplitude: U[0, base)
    nblobs: int        # Gaussian blobs per image
    r: int
    thresh: float
    top_k: int
    T: float
    D: int
    desc_dtype: str    # "f16" | "f32"
    stride: int
    seed: int

    @property
    def Hd(self):
        return self.H // self.stride

    @property
    def Wd(self):
        return self.W // self.stride

    def scaled(self, **kw) -> "Config":
        return replace(self, **kw)


# BASELINE.json `configs` 0..4 == c1..c5
CONFIGS = {
    "c1": Config("c1", 1, 480, 752, 0.1, 600, 2, 0.2, 256, 0.1, 64, "f32", 1, 1),
    "c2": Config("c2", 2, 480, 752, 0.1, 800, 2, 0.2, 1024, 0.1, 128, "f16", 1, 2),
    "c3": Config("c3", 2, 480, 752, 0.01, 1000, 4, 0.005, 1024, 0.1, 256, "f16", 8, 3),
    "c4": Config("c4", 2, 720, 1280, 0.05, 3000, 2, 0.05, 4096, 0.1, 64, "f16", 8, 4),
    "c5": Config("c5", 64, 1080, 1920, 0.1, 4000, 2, 0.2, 2048, 0.1, 128, "f16", 1, 5),
}


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-fopenmp", "-shared", "-fPIC",
                               _SRC, "-o", tmp, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _get_lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        L.synth_score_maps.restype = ctypes.c_int
        L.synth_score_maps.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                       ctypes.c_uint64, ctypes.c_double, ctypes.c_int]
        _lib = L
    return _lib


def score_maps(B, H, W, seed, base, nblobs, pin_memory=False) -> torch.Tensor:
    """[B,H,W] fp32 CPU tensor (optionally pinned)."""
    out = torch.empty((B, H, W), dtype=torch.float32, pin_memory=pin_memory)
    rc = _get_lib().synth_score_maps(ctypes.c_void_p(out.data_ptr()), B, H, W,
                                     ctypes.c_uint64(seed), float(base), int(nblobs))
    if rc != 0:
        raise MemoryError("synth_score_maps")
    return out


# ---- descriptor maps ------------------------------------------------------------------------
_QTAB64 = None


def qtab(dtype: torch.dtype) -> torch.Tensor:
    """Normal quantile table Phi^-1((i+0.5)/65536), i in [0,65536), rounded once to `dtype`."""
    global _QTAB64
    if _QTAB64 is None:
        from scipy.special import ndtri
        _QTAB64 = torch.from_numpy(ndtri((np.arange(65536, dtype=np.float64) + 0.5) / 65536.0))
    return _QTAB64.to(dtype)


def _s64(v: int) -> int:
    v &= (1 << 64) - 1
    return v - (1 << 64) if v >= (1 << 63) else v


def _lsr(z: torch.Tensor, n: int) -> torch.Tensor:
    return (z >> n) & ((1 << (64 - n)) - 1)


def _splitmix64(x: torch.Tensor) -> torch.Tensor:
    z = x + _s64(0x9E3779B97F4A7C15)
    z = (z ^ _lsr(z, 30)) * _s64(0xBF58476D1CE4E5B9)
    z = (z ^ _lsr(z, 27)) * _s64(0x94D049BB133111EB)
    return z ^ _lsr(z, 31)


def desc_elements(seed: int, b: int, e: torch.Tensor, dtype: torch.dtype) -> torch.Tensor:
    """Values of image b's descriptor map at flat element offsets e (int64 tensor, any device)."""
    key = _s64(seed ^ (3 << 56) ^ (b << 40))
    h = _splitmix64(e ^ key)
    return qtab(dtype).to(e.device)[_lsr(h, 48)]


def desc_maps(B, Hd, Wd, D, seed, dtype=torch.float16, device="cpu", out=None,
              chunk_elems=1 << 26) -> torch.Tensor:
    """[B,Hd,Wd,D] channel-last descriptor map, filled chunk by chunk on `device`."""
    n = Hd * Wd * D
    if out is None:
        out = torch.empty((B, Hd, Wd, D), dtype=dtype, device=device)
    flat = out.view(B, n)
    for b in range(B):
        for s in range(0, n, chunk_elems):
            e = torch.arange(s, min(n, s + chunk_elems), dtype=torch.int64, device=out.device)
            flat[b, s:s + e.numel()] = desc_elements(seed, b, e, dtype)
    return out


def torch_dtype(name: str) -> torch.dtype:
    return {"f16": torch.float16, "f32": torch.float32}[name]


def make_inputs(cfg: Config, device="cpu", with_desc=True, pin_memory=False):
    """(score [B,H,W] f32 on CPU, desc [B,Hd,Wd,D] on `device` or None) for a Config."""
    score = score_maps(cfg.B, cfg.H, cfg.W, cfg.seed, cfg.base, cfg.nblobs, pin_memory=pin_memory)
    desc = None
    if with_desc:
        desc = desc_maps(cfg.B, cfg.Hd, cfg.Wd, cfg.D, cfg.seed, torch_dtype(cfg.desc_dtype), device)
    return score, desc


# ---- a stereo sequence for the composed chain extract -> match -> stereo validation ------
def stereo_sequence(H, W, D, seed, disparity, motion=(5, -3), base=0.1, nblobs=900, dtype=torch.float16, device="cpu",
                    margin=32):
    """Four views of ONE synthetic world, as crops of a larger score map and descriptor map (stride 1), in the batch
    order [L(t-1), L(t), R(t), R(t-1)]: the right camera sees every world point `disparity` pixels further left
    (x_R = x_L - disparity: a fronto-parallel scene at depth fx * baseline / disparity), and between t-1 and t the image
    content moves by motion = (dx, dy) pixels.  Integer shifts, so corresponding keypoints have identical windows and
    identical bilinear samples: descriptors of true correspondences agree to rounding; points near the crop borders
    have no partner.  Returns (score [4,H,W] f32 CPU, desc [4,H,W,D] `dtype` on `device`).  Stands in for consecutive
    stereo frames of the paper's datasets (EuRoC-like 752 x 480), which are not available."""
    dx, dy = int(motion[0]), int(motion[1])
    d = int(disparity)
    assert max(abs(dx), abs(dy)) <= margin and 0 <= d <= margin
    Hb, Wb = H + 2 * margin, W + 2 * margin
    world_s = score_maps(1, Hb, Wb, seed, base, nblobs)[0]
    world_d = desc_maps(1, Hb, Wb, D, seed, dtype, device)[0]
    # top-left corner of each view in the world: a point at world column c appears at c - x0 in the view
    corners = [(margin - dy, margin - dx), (margin, margin), (margin, margin + d), (margin - dy, margin - dx + d)]
    score = torch.stack([world_s[y0:y0 + H, x0:x0 + W] for y0, x0 in corners]).contiguous()
    desc = torch.stack([world_d[y0:y0 + H, x0:x0 + W] for y0, x0 in corners]).contiguous()
    return score, desc


# ---- inputs for the consumers of the descriptor output ---------------------------------
def _unit_rows(g: torch.Generator, n: int, D: int) -> torch.Tensor:
    x = torch.randn((n, D), generator=g, dtype=torch.float64)
    return x / x.norm(dim=1, keepdim=True)


def match_sets(P, Na, Nb, D, seed, overlap=0.7, noise=0.35, count_a=None, count_b=None):
    """Two zero-padded, l2-normalised fp16 descriptor sets per pair, like two views of one scene: a fraction
    `overlap` of A's rows reappears in B at a random position with additive noise (true matches, cosine about
    1 / sqrt(1 + noise^2)), the rest of B are unrelated descriptors.  Returns (A [P,Na,D] f16, B [P,Nb,D] f16,
    count_a [P] i32, count_b [P] i32); rows past the counts are zero.  Stands in for the
    ALIKED / SuperPoint / XFeat descriptors of two frames, which are not available."""
    g = torch.Generator().manual_seed(int(seed))
    A = torch.zeros((P, Na, D), dtype=torch.float16)
    B = torch.zeros((P, Nb, D), dtype=torch.float16)
    ca = torch.empty(P, dtype=torch.int32)
    cb = torch.empty(P, dtype=torch.int32)
    for p in range(P):
        na = Na if count_a is None else int(count_a[p])
        nb = Nb if count_b is None else int(count_b[p])
        a = _unit_rows(g, na, D)
        b = _unit_rows(g, nb, D)
        m = min(int(overlap * na), nb)
        src = torch.randperm(na, generator=g)[:m]
        dst = torch.randperm(nb, generator=g)[:m]
        nz = a[src] + noise * _unit_rows(g, m, D)
        b[dst] = nz / nz.norm(dim=1, keepdim=True)
        A[p, :na] = a.to(torch.float16)
        B[p, :nb] = b.to(torch.float16)
        ca[p], cb[p] = na, nb
    return A, B, ca, cb


def keyframe_db(n, D, seed, revisits=(), revisit_sim=0.8, dtype=torch.float16):
    """A keyframe database of n l2-normalised global descriptors (rows in insertion order) and a query: unrelated
    unit vectors, except that the rows listed in `revisits` are earlier views of the query's place (cosine about
    `revisit_sim`, each a little lower than the one before so that the ranking is unambiguous).  Stands in for the
    AnyLoc DINOv2-VLAD descriptors, g in R^{32*384}, which need trained weights."""
    g = torch.Generator().manual_seed(int(seed))
    q = _unit_rows(g, 1, D)[0]
    db = torch.empty((n, D), dtype=dtype)
    for s in range(0, n, 4096):
        db[s:s + 4096] = _unit_rows(g, min(4096, n - s), D).to(dtype)
    for i, k in enumerate(revisits):
        s = revisit_sim - 0.004 * i
        o = _unit_rows(g, 1, D)[0]
        o = o - (o @ q) * q
        o = o / o.norm()
        db[k] = (s * q + (1 - s * s) ** 0.5 * o).to(dtype)
    return db, q.to(dtype)
