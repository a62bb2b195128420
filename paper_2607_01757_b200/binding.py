"""ctypes binding of include/dkd.h — same names, argument marshalling only."""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass
from typing import Optional

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
F32, F16 = 0, 1
OPT_USE_GRAPH, OPT_USE_TMA, OPT_PROFILE, OPT_USE_PDL, OPT_NMS_UNIT, OPT_ORIGIN_X, OPT_ORIGIN_Y, OPT_SEL_PREFETCH = 0, 1, 2, 3, 4, 5, 6, 7
MAX_RADIUS, MAX_TOP_K, MAX_ROW_BYTES = 4, 8192, 2048

SCORE_RAW, SCORE_BILINEAR = 0, 1

EXPORTED_SYMBOLS = (
    "dkd_create", "dkd_destroy", "dkd_last_error", "dkd_workspace_bytes", "dkd_set_option",
    "dkd_extract", "dkd_extract_ex", "dkd_extract_var", "dkd_extract_host", "dkd_launches_per_extract", "dkd_version",
    "dkd_profile_read", "dkd_kernel_name", "dkd_pre_padded_size", "dkd_preprocess", "dkd_graph_stats",
    "dkd_match", "dkd_match_static", "dkd_retrieval_scan", "dkd_stereo_validate", "dkd_cov_sqrt_info",
)


class DKDError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"dkd error {code}: {msg}")
        self.code = code


class _CreateParams(ctypes.Structure):
    _fields_ = [("device", ctypes.c_int), ("max_batch", ctypes.c_int), ("max_h", ctypes.c_int),
                ("max_w", ctypes.c_int), ("max_top_k", ctypes.c_int), ("max_dim", ctypes.c_int),
                ("max_radius", ctypes.c_int), ("max_match_n", ctypes.c_int), ("max_match_pairs", ctypes.c_int),
                ("max_scan_rows", ctypes.c_int)]


class _PreParams(ctypes.Structure):
    _fields_ = [("in_channels", ctypes.c_int), ("out_channels", ctypes.c_int), ("grid", ctypes.c_int),
                ("bgr", ctypes.c_int), ("out_dtype", ctypes.c_int), ("scale", ctypes.c_float),
                ("mean", ctypes.c_float * 3), ("inv_std", ctypes.c_float * 3), ("pad_value", ctypes.c_float)]


class _VariantParams(ctypes.Structure):
    _fields_ = [("reliability", ctypes.c_void_p), ("valid_mask", ctypes.c_void_p), ("nms_iters", ctypes.c_int),
                ("score_mode", ctypes.c_int), ("out_total", ctypes.c_void_p)]


class _StereoParams(ctypes.Structure):
    _fields_ = [(n, ctypes.c_float) for n in ("fx", "fy", "cx", "cy", "baseline", "d_min", "z_min", "z_max", "max_reproj")]


class _CovParams(ctypes.Structure):
    _fields_ = [(n, ctypes.c_float) for n in ("scale", "floor_px", "fx", "fy", "lam", "lambda_min", "sigma0")]


def lib_path() -> str:
    """The in-tree library.  DKD_LIBRARY selects another build of it by file name (libdkd_debug.so: the
    -DDKD_DEBUG build with device-side bounds checks)."""
    return os.path.join(_HERE, os.environ.get("DKD_LIBRARY", "libdkd.so"))


_lib = None


def load_library():
    """Loads libdkd.so (in-tree).  Fails loudly if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    path = lib_path()
    if not os.path.exists(path):
        raise DKDError(-4, f"{path} not built — run `python -m paper_2607_01757_b200.build` "
                           "(or __graft_entry__.build()); there is no CPU fallback")
    L = ctypes.CDLL(path)
    vp, i, f = ctypes.c_void_p, ctypes.c_int, ctypes.c_float
    L.dkd_create.restype = i
    L.dkd_create.argtypes = [ctypes.POINTER(_CreateParams), ctypes.POINTER(vp)]
    L.dkd_destroy.restype = i
    L.dkd_destroy.argtypes = [vp]
    L.dkd_last_error.restype = ctypes.c_char_p
    L.dkd_last_error.argtypes = [vp]
    L.dkd_workspace_bytes.restype = ctypes.c_size_t
    L.dkd_workspace_bytes.argtypes = [vp]
    L.dkd_set_option.restype = i
    L.dkd_set_option.argtypes = [vp, i, i]
    L.dkd_launches_per_extract.restype = i
    L.dkd_launches_per_extract.argtypes = [vp, i]
    L.dkd_version.restype = ctypes.c_char_p
    L.dkd_profile_read.restype = i
    L.dkd_profile_read.argtypes = [vp, ctypes.POINTER(ctypes.c_float), i]
    L.dkd_kernel_name.restype = ctypes.c_char_p
    L.dkd_kernel_name.argtypes = [i]
    ip = ctypes.POINTER(ctypes.c_int)
    L.dkd_pre_padded_size.restype = i
    L.dkd_pre_padded_size.argtypes = [i, i, i, ip, ip, ip, ip]
    L.dkd_preprocess.restype = i
    L.dkd_preprocess.argtypes = [vp, vp, i, i, i, ctypes.POINTER(_PreParams), vp, vp]
    common = [vp, vp, i, i, i, vp, i, i, i, i, i, i, f, i, f, vp, vp, vp, vp]
    L.dkd_extract.restype = i
    L.dkd_extract.argtypes = common + [vp]
    L.dkd_extract_ex.restype = i
    L.dkd_extract_ex.argtypes = common + [vp, vp, vp]
    L.dkd_extract_var.restype = i
    L.dkd_extract_var.argtypes = common + [vp, vp, ctypes.POINTER(_VariantParams), vp]
    L.dkd_match.restype = i
    L.dkd_match.argtypes = [vp, vp, vp, i, vp, vp, i, i, i, i, f, i, vp, vp, vp]
    L.dkd_match_static.restype = i
    L.dkd_match_static.argtypes = [vp, vp, i, vp, vp, i, i, i, i, f, i, vp, vp, vp, ctypes.c_char_p, i]
    L.dkd_retrieval_scan.restype = i
    L.dkd_retrieval_scan.argtypes = [vp, vp, i, i, i, vp, i, f, i, vp, vp, vp, vp, vp]
    L.dkd_stereo_validate.restype = i
    L.dkd_stereo_validate.argtypes = [vp, vp, vp, vp, i, ctypes.POINTER(_StereoParams), vp, vp, vp, vp, vp]
    L.dkd_cov_sqrt_info.restype = i
    L.dkd_cov_sqrt_info.argtypes = [vp, vp, i, ctypes.POINTER(_CovParams), vp, vp, vp]
    u64p = ctypes.POINTER(ctypes.c_uint64)
    L.dkd_graph_stats.restype = i
    L.dkd_graph_stats.argtypes = [vp, u64p, u64p, u64p, u64p]
    L.dkd_extract_host.restype = i
    L.dkd_extract_host.argtypes = common + [vp, vp, i, vp]
    _lib = L
    return L


@dataclass
class DKDResult:
    kpts: torch.Tensor                 # [B,k,2] f32 (x,y)
    scores: torch.Tensor               # [B,k]   f32
    desc: Optional[torch.Tensor]       # [B,k,D] f16|f32
    count: torch.Tensor                # [B]     i32
    index: Optional[torch.Tensor]      # [B,k]   i32 (-1 padding)
    offsets: Optional[torch.Tensor]    # [B,k,2] f32 (dx,dy)
    total: Optional[torch.Tensor] = None   # [B] i32: candidates before the cap (variants only)


def _dt(t: Optional[torch.Tensor]) -> int:
    if t is None or t.dtype == torch.float32:
        return F32
    if t.dtype == torch.float16:
        return F16
    raise DKDError(-2, "descriptor map must be float16 or float32")


def _ptr(t: Optional[torch.Tensor]):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


MATCH_STATIC_MAX_RECS = 65536


def match_static(desc_a: torch.Tensor, desc_b: torch.Tensor, out_match: torch.Tensor,
                 out_sim: Optional[torch.Tensor] = None, count_a: Optional[torch.Tensor] = None,
                 count_b: Optional[torch.Tensor] = None, ratio: float = 0.8, mutual: bool = False, stream=None) -> None:
    """dkd_match_static: the matcher for callers that may not allocate device memory (no context; the scratch is a
    1 MiB array built into the library, shared by all calls on a device — keep them on one stream).  Nothing is
    allocated here either: the caller passes the outputs.  desc_a [P,Na,D], desc_b [P,Nb,D] f16 cuda contiguous;
    out_match [P,Na] i32, out_sim [P,Na,2] f32 or None; counts [P] i32 cuda or None.  Runs on desc_a's device, on
    torch's current stream of that device unless `stream` is given.  Raises DKDError (code -3: the problem needs
    more than MATCH_STATIC_MAX_RECS partial records)."""
    L = load_library()
    for t in (desc_a, desc_b):
        if not (t.is_cuda and t.is_contiguous() and t.dim() == 3):
            raise DKDError(-1, "descriptor sets must be contiguous CUDA [P,N,D] tensors")
    P, Na, D = desc_a.shape
    Nb = desc_b.shape[1]
    if desc_b.shape[0] != P or desc_b.shape[2] != D or desc_a.dtype != desc_b.dtype or desc_b.device != desc_a.device:
        raise DKDError(-1, "desc_a / desc_b disagree in P, D, dtype or device")
    for c in (count_a, count_b):
        if c is not None and not (c.device == desc_a.device and c.dtype == torch.int32 and c.is_contiguous() and c.numel() == P):
            raise DKDError(-1, "counts must be contiguous CUDA int32 [P] tensors")
    if not (out_match.device == desc_a.device and out_match.dtype == torch.int32 and out_match.is_contiguous()
            and tuple(out_match.shape) == (P, Na)):
        raise DKDError(-1, "out_match must be a contiguous CUDA int32 [P,Na] tensor")
    if out_sim is not None and not (out_sim.device == desc_a.device and out_sim.dtype == torch.float32
                                    and out_sim.is_contiguous() and tuple(out_sim.shape) == (P, Na, 2)):
        raise DKDError(-1, "out_sim must be a contiguous CUDA float32 [P,Na,2] tensor")
    err = ctypes.create_string_buffer(256)
    with torch.cuda.device(desc_a.device):                       # the entry point runs on the current device
        st = torch.cuda.current_stream(desc_a.device) if stream is None else stream
        rc = L.dkd_match_static(_ptr(desc_a), _ptr(count_a), Na, _ptr(desc_b), _ptr(count_b), Nb, D, _dt(desc_a), P,
                                float(ratio), int(bool(mutual)), _ptr(out_match), _ptr(out_sim),
                                ctypes.c_void_p(st.cuda_stream), err, len(err))
    if rc != 0:
        raise DKDError(rc, err.value.decode(errors="replace"))


class DKD:
    """One context = one device workspace.  `extract` mirrors dkd_extract_ex, `extract_host`
    mirrors dkd_extract_host."""

    def __init__(self, max_batch: int, max_h: int, max_w: int, max_top_k: int, max_dim: int = 0,
                 device: int = 0, max_radius: int = 0, max_match_n: int = 0, max_match_pairs: int = 0,
                 max_scan_rows: int = 0):
        """dkd_create.  The maxima after `device` may stay 0 (dkd.h): max_match_n / max_match_pairs / max_scan_rows size the
        scratch of match / retrieval_scan at create, so that those calls never allocate (capture-safe from the first)."""
        self._h = None
        L = load_library()
        if not torch.cuda.is_available():
            raise DKDError(-4, "no CUDA device: libdkd has no CPU fallback")
        self._L = L
        self.device = torch.device("cuda", device)
        p = _CreateParams(device, max_batch, max_h, max_w, max_top_k, max_dim, max_radius, max_match_n, max_match_pairs,
                          max_scan_rows)
        h = ctypes.c_void_p()
        rc = L.dkd_create(ctypes.byref(p), ctypes.byref(h))
        if rc != 0:
            raise DKDError(rc, L.dkd_last_error(None).decode())
        self._h = h

    def close(self):
        if self._h is not None:
            self._L.dkd_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc: int):
        if rc != 0:
            raise DKDError(rc, self._L.dkd_last_error(self._h).decode())

    def set_option(self, option: int, value: int):
        self._check(self._L.dkd_set_option(self._h, option, value))

    @property
    def workspace_bytes(self) -> int:
        return int(self._L.dkd_workspace_bytes(self._h))

    def launches_per_extract(self, with_desc: bool = True) -> int:
        return int(self._L.dkd_launches_per_extract(self._h, int(with_desc)))

    def profile_read(self) -> dict:
        """dkd_profile_read: {kernel name: ms} of the last call made with OPT_PROFILE set (waits for it)."""
        buf = (ctypes.c_float * 8)()
        n = self._L.dkd_profile_read(self._h, buf, 8)
        if n < 0:
            self._check(n)
        return {self._L.dkd_kernel_name(j).decode(): float(buf[j]) for j in range(n)}

    def graph_stats(self) -> dict:
        """dkd_graph_stats: {instantiated, updated, replayed, stream} call counts since the context was created."""
        v = [ctypes.c_uint64() for _ in range(4)]
        self._check(self._L.dkd_graph_stats(self._h, *[ctypes.byref(x) for x in v]))
        return dict(zip(("instantiated", "updated", "replayed", "stream"), (int(x.value) for x in v)))

    # -- consumers of the descriptor output (dkd_match / dkd_retrieval_scan / dkd_stereo_validate / dkd_cov_sqrt_info) --
    def _stream(self, stream):
        st = torch.cuda.current_stream(self.device) if stream is None else stream
        return ctypes.c_void_p(st.cuda_stream)

    def match(self, desc_a: torch.Tensor, desc_b: torch.Tensor, count_a: Optional[torch.Tensor] = None,
              count_b: Optional[torch.Tensor] = None, ratio: float = 0.8, mutual: bool = False, want_sim: bool = True,
              stream=None):
        """dkd_match.  desc_a [P,Na,D], desc_b [P,Nb,D] f16 cuda contiguous; counts [P] i32 cuda or None.
        Returns (match [P,Na] i32, sim [P,Na,2] f32 or None)."""
        for t in (desc_a, desc_b):
            if not (t.is_cuda and t.is_contiguous() and t.dim() == 3):
                raise DKDError(-1, "descriptor sets must be contiguous CUDA [P,N,D] tensors")
        P, Na, D = desc_a.shape
        if desc_b.shape[0] != P or desc_b.shape[2] != D or desc_a.dtype != desc_b.dtype:
            raise DKDError(-1, "desc_a / desc_b disagree in P, D or dtype")
        for c in (count_a, count_b):
            if c is not None and not (c.is_cuda and c.dtype == torch.int32 and c.is_contiguous() and c.numel() == P):
                raise DKDError(-1, "counts must be contiguous CUDA int32 [P] tensors")
        Nb = desc_b.shape[1]
        out = torch.empty((P, Na), dtype=torch.int32, device=desc_a.device)
        sim = torch.empty((P, Na, 2), dtype=torch.float32, device=desc_a.device) if want_sim else None
        self._check(self._L.dkd_match(self._h, _ptr(desc_a), _ptr(count_a), Na, _ptr(desc_b), _ptr(count_b), Nb, D,
                                      _dt(desc_a), P, float(ratio), int(bool(mutual)), _ptr(out), _ptr(sim),
                                      self._stream(stream)))
        return out, sim

    def retrieval_scan(self, db: torch.Tensor, query: torch.Tensor, n_exclude: int = 50, tau: float = 0.60,
                       max_cand: int = 16, want_sim: bool = True, stream=None):
        """dkd_retrieval_scan.  db [n,D], query [D] f16|f32 cuda contiguous.
        Returns (sim [n] f32 or None, cand [max_cand] i32, cand_sim [max_cand] f32, count [1] i32)."""
        if not (db.is_cuda and db.is_contiguous() and db.dim() == 2 and query.is_cuda and query.is_contiguous()
                and query.dim() == 1 and query.shape[0] == db.shape[1] and query.dtype == db.dtype):
            raise DKDError(-1, "db must be a contiguous CUDA [n,D] tensor and query a matching [D] tensor")
        n, D = db.shape
        sim = torch.empty((n,), dtype=torch.float32, device=db.device) if want_sim else None
        cand = torch.empty((max_cand,), dtype=torch.int32, device=db.device)
        csim = torch.empty((max_cand,), dtype=torch.float32, device=db.device)
        cnt = torch.empty((1,), dtype=torch.int32, device=db.device)
        self._check(self._L.dkd_retrieval_scan(self._h, _ptr(db), _dt(db), n, D, _ptr(query), int(n_exclude), float(tau),
                                               int(max_cand), _ptr(sim), _ptr(cand), _ptr(csim), _ptr(cnt),
                                               self._stream(stream)))
        return sim, cand, csim, cnt

    def stereo_validate(self, kpts_l: torch.Tensor, kpts_r: torch.Tensor, match: Optional[torch.Tensor], fx, fy, cx, cy,
                        baseline, d_min, z_min, z_max, max_reproj=1.5, stream=None):
        """dkd_stereo_validate.  kpts_l [n,2], kpts_r [m,2] f32 cuda; match [n] i32 cuda or None.
        Returns (valid [n] u8, xyz [n,3], disparity [n], reproj_err [n])."""
        for t in (kpts_l, kpts_r):
            if not (t.is_cuda and t.is_contiguous() and t.dtype == torch.float32 and t.dim() == 2 and t.shape[1] == 2):
                raise DKDError(-1, "keypoints must be contiguous CUDA float32 [n,2] tensors")
        if match is not None and not (match.is_cuda and match.dtype == torch.int32 and match.is_contiguous()
                                      and match.numel() == kpts_l.shape[0]):
            raise DKDError(-1, "match must be a contiguous CUDA int32 [n] tensor")
        n = kpts_l.shape[0]
        dev = kpts_l.device
        xyz = torch.empty((n, 3), dtype=torch.float32, device=dev)
        disp = torch.empty((n,), dtype=torch.float32, device=dev)
        err = torch.empty((n,), dtype=torch.float32, device=dev)
        valid = torch.empty((n,), dtype=torch.uint8, device=dev)
        p = _StereoParams(fx, fy, cx, cy, baseline, d_min, z_min, z_max, max_reproj)
        self._check(self._L.dkd_stereo_validate(self._h, _ptr(kpts_l), _ptr(kpts_r), _ptr(match), n, ctypes.byref(p),
                                                _ptr(xyz), _ptr(disp), _ptr(err), _ptr(valid), self._stream(stream)))
        return valid, xyz, disp, err

    def cov_sqrt_info(self, L: torch.Tensor, scale, floor_px, fx, fy, lam, lam_min, sigma0, stream=None):
        """dkd_cov_sqrt_info.  L [n,3] f32 cuda (l11, l21, l22).  Returns (omega [n,2,2] f32, ok [n] u8)."""
        if not (L.is_cuda and L.is_contiguous() and L.dtype == torch.float32 and L.dim() == 2 and L.shape[1] == 3):
            raise DKDError(-1, "L must be a contiguous CUDA float32 [n,3] tensor")
        n = L.shape[0]
        om = torch.empty((n, 2, 2), dtype=torch.float32, device=L.device)
        ok = torch.empty((n,), dtype=torch.uint8, device=L.device)
        p = _CovParams(scale, floor_px, fx, fy, lam, lam_min, sigma0)
        self._check(self._L.dkd_cov_sqrt_info(self._h, _ptr(L), n, ctypes.byref(p), _ptr(om), _ptr(ok),
                                              self._stream(stream)))
        return om, ok

    # -- fused input pre-processing (dkd_pre_padded_size / dkd_preprocess) ---------------------
    @staticmethod
    def padded_size(H: int, W: int, grid: int):
        """(Hp, Wp, oy, ox) of dkd_pre_padded_size."""
        v = [ctypes.c_int() for _ in range(4)]
        rc = load_library().dkd_pre_padded_size(H, W, grid, *[ctypes.byref(x) for x in v])
        if rc != 0:
            raise DKDError(rc, "dkd_pre_padded_size: H, W, grid must be >= 1")
        return tuple(x.value for x in v)

    def preprocess(self, src: torch.Tensor, out_channels: int, grid: int, bgr=False, scale=1.0 / 255.0,
                   mean=(0.0, 0.0, 0.0), inv_std=(1.0, 1.0, 1.0), pad_value=0.0, out_dtype=torch.float32,
                   out: Optional[torch.Tensor] = None, stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
        """src [B,H,W,Cin] u8 cuda contiguous -> [B,out_channels,Hp,Wp] f32|f16 (dkd_preprocess)."""
        if not (src.is_cuda and src.is_contiguous() and src.dtype == torch.uint8 and src.dim() == 4):
            raise DKDError(-1, "src must be a contiguous CUDA uint8 [B,H,W,C] tensor")
        B, H, W, Cin = src.shape
        Hp, Wp, _, _ = self.padded_size(H, W, grid)
        if out is None:
            out = torch.empty((B, out_channels, Hp, Wp), dtype=out_dtype, device=src.device)
        p = _PreParams(Cin, int(out_channels), int(grid), int(bool(bgr)), _dt(out), float(scale),
                       (ctypes.c_float * 3)(*mean), (ctypes.c_float * 3)(*inv_std), float(pad_value))
        st = torch.cuda.current_stream(self.device) if stream is None else stream
        self._check(self._L.dkd_preprocess(self._h, _ptr(src), B, H, W, ctypes.byref(p), _ptr(out),
                                           ctypes.c_void_p(st.cuda_stream)))
        return out

    # -- device buffers ---------------------------------------------------------------------
    def alloc_outputs(self, B: int, top_k: int, desc: Optional[torch.Tensor], D: int = 0,
                      want_index=True, want_offsets=True, device=None, pin=False) -> DKDResult:
        dev = self.device if device is None else device
        kw = dict(device=dev, pin_memory=pin) if pin else dict(device=dev)
        return DKDResult(
            kpts=torch.empty((B, top_k, 2), dtype=torch.float32, **kw),
            scores=torch.empty((B, top_k), dtype=torch.float32, **kw),
            desc=None if desc is None else torch.empty((B, top_k, D), dtype=desc.dtype, **kw),
            count=torch.empty((B,), dtype=torch.int32, **kw),
            index=torch.empty((B, top_k), dtype=torch.int32, **kw) if want_index else None,
            offsets=torch.empty((B, top_k, 2), dtype=torch.float32, **kw) if want_offsets else None,
        )

    def _check_out(self, out: DKDResult, B: int, top_k: int, desc, D: int, cuda: bool):
        """A caller-supplied output set must have exactly the shapes / dtypes / placement the C call writes."""
        want = [("kpts", (B, top_k, 2), torch.float32, True), ("scores", (B, top_k), torch.float32, True),
                ("count", (B,), torch.int32, True), ("index", (B, top_k), torch.int32, False),
                ("offsets", (B, top_k, 2), torch.float32, False), ("total", (B,), torch.int32, False)]
        if desc is not None:
            want.append(("desc", (B, top_k, D), desc.dtype, True))
        elif out.desc is not None:
            raise DKDError(-1, "out.desc given without a descriptor map")
        for name, shape, dtype, required in want:
            t = getattr(out, name)
            if t is None:
                if required:
                    raise DKDError(-1, f"out.{name} is missing")
                continue
            if tuple(t.shape) != shape or t.dtype != dtype or not t.is_contiguous() or t.is_cuda != cuda:
                raise DKDError(-1, f"out.{name} must be a contiguous {'CUDA' if cuda else 'CPU'} {dtype} tensor of shape {shape}")
            if cuda and t.device != self.device:
                raise DKDError(-1, f"out.{name} is on {t.device}, the context is on {self.device}")

    def extract(self, score: torch.Tensor, desc: Optional[torch.Tensor], stride: int, r: int,
                thresh: float, top_k: int, T: float, out: Optional[DKDResult] = None,
                stream: Optional[torch.cuda.Stream] = None, want_index=True, want_offsets=True,
                reliability: Optional[torch.Tensor] = None, valid_mask: Optional[torch.Tensor] = None,
                nms_iters: int = 0, score_mode: int = SCORE_RAW, want_total: bool = False) -> DKDResult:
        """score [B,H,W] f32 cuda contiguous; desc [B,Hd,Wd,D] f16|f32 cuda contiguous or None.
        Asynchronous on `stream` (default: the current torch stream).  The keyword arguments after
        `want_offsets` are the variants of dkd_extract_var (dkd.h)."""
        if not (score.is_cuda and score.is_contiguous() and score.dtype == torch.float32 and score.dim() == 3):
            raise DKDError(-1, "score must be a contiguous CUDA float32 [B,H,W] tensor")
        B, H, W = score.shape
        Hd = Wd = D = 0
        if desc is not None:
            if not (desc.is_cuda and desc.is_contiguous() and desc.dim() == 4 and desc.shape[0] == B):
                raise DKDError(-1, "desc must be a contiguous CUDA [B,Hd,Wd,D] tensor")
            _, Hd, Wd, D = desc.shape
        if reliability is not None and not (reliability.is_cuda and reliability.is_contiguous() and
                                            reliability.dtype == torch.float32 and reliability.shape == score.shape):
            raise DKDError(-1, "reliability must be a contiguous CUDA float32 tensor shaped like score")
        if valid_mask is not None and not (valid_mask.is_cuda and valid_mask.is_contiguous() and
                                           valid_mask.dtype == torch.uint8 and valid_mask.shape == score.shape):
            raise DKDError(-1, "valid_mask must be a contiguous CUDA uint8 tensor shaped like score")
        if out is None:
            out = self.alloc_outputs(B, top_k, desc, D, want_index, want_offsets)
        else:
            self._check_out(out, B, top_k, desc, D, cuda=True)
        if want_total and out.total is None:
            out.total = torch.empty((B,), dtype=torch.int32, device=score.device)
        st = torch.cuda.current_stream(self.device) if stream is None else stream
        v = _VariantParams(_ptr(reliability), _ptr(valid_mask), int(nms_iters), int(score_mode), _ptr(out.total))
        rc = self._L.dkd_extract_var(self._h, _ptr(score), B, H, W, _ptr(desc), _dt(desc), Hd, Wd, D,
                                     int(stride), int(r), float(thresh), int(top_k), float(T),
                                     _ptr(out.kpts), _ptr(out.scores), _ptr(out.desc), _ptr(out.count),
                                     _ptr(out.index), _ptr(out.offsets), ctypes.byref(v),
                                     ctypes.c_void_p(st.cuda_stream))
        self._check(rc)
        return out

    def bind(self, score, desc, stride, r, thresh, top_k, T, out: DKDResult, stream=None):
        """Pre-marshals one dkd_extract_ex call (fixed buffers) and returns a zero-argument callable that
        enqueues it — keeps Python's per-call marshalling out of a timed launch loop."""
        B, H, W = score.shape
        Hd = Wd = D = 0
        if desc is not None:
            _, Hd, Wd, D = desc.shape
        st = torch.cuda.current_stream(self.device) if stream is None else stream
        ci, cf = ctypes.c_int, ctypes.c_float
        args = (self._h, _ptr(score), ci(B), ci(H), ci(W), _ptr(desc), ci(_dt(desc)), ci(Hd), ci(Wd), ci(D),
                ci(int(stride)), ci(int(r)), cf(float(thresh)), ci(int(top_k)), cf(float(T)),
                _ptr(out.kpts), _ptr(out.scores), _ptr(out.desc), _ptr(out.count),
                _ptr(out.index), _ptr(out.offsets), ctypes.c_void_p(st.cuda_stream))
        fn, check = self._L.dkd_extract_ex, self._check
        keep = (score, desc, out)                                 # the call holds raw pointers

        def call(_keep=keep):
            rc = fn(*args)
            if rc:
                check(rc)
        return call

    def extract_literal(self, score, desc, stride, r, thresh, top_k, T, out: DKDResult, stream=None):
        """dkd_extract (the literal north_star signature: no index / offset outputs)."""
        B, H, W = score.shape
        Hd = Wd = D = 0
        if desc is not None:
            _, Hd, Wd, D = desc.shape
        st = torch.cuda.current_stream(self.device) if stream is None else stream
        rc = self._L.dkd_extract(self._h, _ptr(score), B, H, W, _ptr(desc), _dt(desc), Hd, Wd, D,
                                 int(stride), int(r), float(thresh), int(top_k), float(T),
                                 _ptr(out.kpts), _ptr(out.scores), _ptr(out.desc), _ptr(out.count),
                                 ctypes.c_void_p(st.cuda_stream))
        self._check(rc)
        return out

    def extract_host(self, score: torch.Tensor, desc: Optional[torch.Tensor], stride: int, r: int,
                     thresh: float, top_k: int, T: float, out: Optional[DKDResult] = None,
                     desc_resident: bool = False, stream: Optional[torch.cuda.Stream] = None) -> DKDResult:
        """HOST tensors in, HOST tensors out (copies inside the call, synchronous on return).
        desc_resident: False/0, True/1 (re-use the uploaded map; do not modify it meanwhile) or 2 (upload again
        and keep resident) — see dkd.h."""
        if score.is_cuda or not score.is_contiguous() or score.dtype != torch.float32 or score.dim() != 3:
            raise DKDError(-1, "score must be a contiguous CPU float32 [B,H,W] tensor")
        B, H, W = score.shape
        Hd = Wd = D = 0
        if desc is not None:
            if desc.is_cuda or not desc.is_contiguous() or desc.dim() != 4 or desc.shape[0] != B:
                raise DKDError(-1, "desc must be a contiguous CPU [B,Hd,Wd,D] tensor")
            _, Hd, Wd, D = desc.shape
        if out is None:
            out = self.alloc_outputs(B, top_k, desc, D, device="cpu", pin=True)
        else:
            self._check_out(out, B, top_k, desc, D, cuda=False)
        st = torch.cuda.current_stream(self.device) if stream is None else stream
        rc = self._L.dkd_extract_host(self._h, _ptr(score), B, H, W, _ptr(desc), _dt(desc), Hd, Wd, D,
                                      int(stride), int(r), float(thresh), int(top_k), float(T),
                                      _ptr(out.kpts), _ptr(out.scores), _ptr(out.desc), _ptr(out.count),
                                      _ptr(out.index), _ptr(out.offsets), int(desc_resident),
                                      ctypes.c_void_p(st.cuda_stream))
        self._check(rc)
        return out
