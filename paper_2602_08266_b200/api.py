"""Thin Python binding of libnbv (include/nbv.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of csrc/.  PyTorch supplies device memory (tensors whose
data_ptr() is passed through) and the current CUDA stream; nothing is computed here.  There is no CPU
fallback: without the built library and a CUDA device every call raises.

Names mirror the C ABI: NBV.load_gaussians -> nbv_load_gaussians, NBV.accumulate_training ->
nbv_accumulate_training, NBV.score_candidates -> nbv_score_candidates, ...
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

from .synth import CAMERA_DTYPE

_PKG = Path(__file__).resolve().parent
LIB_PATH = _PKG / "libnbv.so"

P = 14
NBLK = 105
CH_RGB, CH_DEPTH, CH_RGBD, CH_MASK = 7, 8, 15, 16

STATUS = {
    0: "NBV_OK", -1: "NBV_ERR_INVALID_ARG", -2: "NBV_ERR_BAD_DATA", -3: "NBV_ERR_NOT_LOADED",
    -4: "NBV_ERR_EMPTY_CANDIDATES", -5: "NBV_ERR_UNKNOWN_TARGET", -6: "NBV_ERR_OOM", -7: "NBV_ERR_CUDA",
    -8: "NBV_ERR_CAPACITY",
}

# every symbol include/nbv.h declares (tests check that the library exports all of them)
EXPORTS = [
    "nbv_default_config", "nbv_create", "nbv_destroy", "nbv_last_error", "nbv_load_gaussians", "nbv_reset_training",
    "nbv_accumulate_training", "nbv_score_candidates", "nbv_score_candidates_host", "nbv_last_view_stats",
    "nbv_projected", "nbv_tile_lists", "nbv_render", "nbv_view_hessian", "nbv_training_hessian", "nbv_confidence",
    "nbv_gaussian_gains", "nbv_set_stage_timing", "nbv_stage_times", "nbv_kernel_launches", "nbv_set_concurrency",
    "nbv_tile_walk", "nbv_score_candidates_fused", "nbv_select_greedy", "nbv_block_size", "nbv_render_mask", "nbv_measure_ffma_peak",
    "nbv_chain", "nbv_load_sh", "nbv_exp_spec_pairs", "nbv_exclusive_scan_noalloc", "nbv_noalloc_last_error", "nbv_batch_views",
]

STAGES = ["project", "depth_sort", "bin", "coarse_sort", "forward", "backward", "expand_gain"]


class NBVError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__("%s (%d): %s" % (STATUS.get(code, "?"), code, msg))
        self.code = code
        self.status = STATUS.get(code, "?")


class Config(C.Structure):
    """nbv_config"""
    _fields_ = [
        ("near_plane", C.c_float), ("blur", C.c_float), ("alpha_min", C.c_float), ("alpha_max", C.c_float),
        ("t_stop", C.c_float), ("bg", C.c_float * 3), ("channel_mask", C.c_int32), ("channel_weight", C.c_float * 4),
        ("opacity_coord", C.c_int32), ("alpha_obj", C.c_float), ("alpha_opa", C.c_float), ("p_floor", C.c_float),
        ("sigma_floor", C.c_float), ("prior_precision", C.c_float * 14), ("mask_bg_channel", C.c_int32),
        ("prior_precision_obj", C.c_float), ("weight_mode", C.c_int32), ("criterion", C.c_int32),
    ]


class ViewStats(C.Structure):
    """nbv_view_stats"""
    _fields_ = [("n_visible", C.c_int64), ("n_keys", C.c_int64), ("n_entries", C.c_int64), ("n_pairs", C.c_int64),
                ("n_touched", C.c_int64), ("n_coarse", C.c_int64)]

    def as_dict(self):
        return {k: int(getattr(self, k)) for k, _ in self._fields_}


_lib = None


def load_library(path: Path | None = None):
    """dlopen libnbv.so (built in-tree by paper_2602_08266_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = Path(path) if path else LIB_PATH
    if not p.exists():
        raise FileNotFoundError("%s not built: run `python -m paper_2602_08266_b200.build` (nvcc, sm_100a)" % p)
    lib = C.CDLL(str(p))
    lib.nbv_last_error.restype = C.c_char_p
    lib.nbv_last_error.argtypes = [C.c_void_p]
    lib.nbv_destroy.restype = None
    lib.nbv_destroy.argtypes = [C.c_void_p]
    lib.nbv_default_config.restype = None
    lib.nbv_kernel_launches.restype = C.c_int64
    lib.nbv_noalloc_last_error.restype = C.c_char_p
    lib.nbv_noalloc_last_error.argtypes = []
    lib.nbv_block_size.restype = C.c_int64
    lib.nbv_block_size.argtypes = [C.c_void_p]
    if path is None:
        _lib = lib
    return lib


def default_config(**overrides) -> Config:
    cfg = Config()
    load_library().nbv_default_config(C.byref(cfg))
    for k, v in overrides.items():
        if k in ("bg", "channel_weight", "prior_precision"):
            arr = getattr(cfg, k)
            vals = list(v) if np.ndim(v) else [v] * len(arr)
            for i, x in enumerate(vals):
                arr[i] = float(x)
        else:
            setattr(cfg, k, v)
    return cfg


def _cams(cams) -> np.ndarray:
    a = np.ascontiguousarray(np.asarray(cams, dtype=CAMERA_DTYPE).reshape(-1))
    return a


def _stream():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else None


class NBV:
    """One libnbv context (one GPU)."""

    def __init__(self, cfg: Config | None = None, **overrides):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("libnbv needs a CUDA device (sm_100a); there is no CPU fallback")
        self._torch = torch
        self.lib = load_library()
        self.cfg = cfg if cfg is not None else default_config(**overrides)
        self._h = C.c_void_p()
        rc = self.lib.nbv_create(C.byref(self._h), C.byref(self.cfg))
        if rc != 0:
            raise NBVError(rc, "nbv_create failed")
        self.N = 0
        self.K = 0
        self.device = torch.device("cuda", torch.cuda.current_device())

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            self.lib.nbv_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc: int):
        if rc != 0:
            msg = self.lib.nbv_last_error(self._h)
            raise NBVError(rc, msg.decode() if msg else "")

    def _dev(self, a, dtype=None):
        torch = self._torch
        if isinstance(a, torch.Tensor):
            t = a.to(device=self.device, dtype=dtype or torch.float32)
        else:
            t = torch.as_tensor(np.ascontiguousarray(a), device=self.device).to(dtype or torch.float32)
        return t.contiguous()

    # ---- hot path -----------------------------------------------------------------------------
    def load_gaussians(self, mean, logscale, quat, opacity, rgb, obj_logits):
        """nbv_load_gaussians.  Arguments: torch CUDA tensors (used in place) or numpy arrays (copied to the GPU)."""
        m, ls, q = self._dev(mean), self._dev(logscale), self._dev(quat)
        o, c, lg = self._dev(opacity), self._dev(rgb), self._dev(obj_logits)
        N = int(m.shape[0])
        if N == 0 or lg.ndim != 2:
            raise NBVError(-1, "empty Gaussian set or malformed object logits")
        K = int(lg.shape[1])
        self._check(self.lib.nbv_load_gaussians(self._h, N, K, _ptr(m), _ptr(ls), _ptr(q), _ptr(o), _ptr(c), _ptr(lg), _stream()))
        self.N, self.K = N, K

    def load_scene(self, scene):
        self.load_gaussians(scene.mean, scene.logscale, scene.quat, scene.opacity, scene.rgb, scene.obj_logits)

    def load_sh(self, sh45):
        """nbv_load_sh: (N, 45) float32 SH coefficients of degree 1..3 (coefficient-major); blocks become 59 x 59"""
        torch = self._torch
        a = np.ascontiguousarray(sh45, dtype=np.float32)
        if a.size != self.N * 45:
            raise ValueError("load_sh expects N x 45 coefficients for the %d Gaussians loaded, got %d values" % (self.N, a.size))
        t = torch.as_tensor(a.reshape(-1), device=self.device).contiguous()
        self._check(self.lib.nbv_load_sh(self._h, _ptr(t), _stream()))

    def reset_training(self):
        self._check(self.lib.nbv_reset_training(self._h, _stream()))

    def accumulate_training(self, cams):
        cams = _cams(cams)
        self._check(self.lib.nbv_accumulate_training(self._h, C.c_void_p(cams.ctypes.data), int(cams.shape[0]), _stream()))

    def score_candidates(self, cams, target_obj: int = -1, scores=None, best=None):
        """nbv_score_candidates: returns (scores, best) as CUDA tensors (no host synchronisation)."""
        torch = self._torch
        cams = _cams(cams)
        n = int(cams.shape[0])
        if scores is None:
            scores = torch.empty(max(n, 1), dtype=torch.float32, device=self.device)
        if best is None:
            best = torch.empty(1, dtype=torch.int32, device=self.device)
        self._check(self.lib.nbv_score_candidates(self._h, C.c_void_p(cams.ctypes.data), n, int(target_obj), _ptr(scores), _ptr(best), _stream()))
        return scores[:n], best

    def score_candidates_host(self, cams, target_obj: int = -1):
        """nbv_score_candidates_host: HOST outputs (numpy scores, int best); synchronises."""
        cams = _cams(cams)
        n = int(cams.shape[0])
        scores = np.zeros(max(n, 1), dtype=np.float32)
        best = C.c_int32(-1)
        self._check(self.lib.nbv_score_candidates_host(self._h, C.c_void_p(cams.ctypes.data), n, int(target_obj),
                                                       C.c_void_p(scores.ctypes.data), C.byref(best), _stream()))
        return scores[:n], int(best.value)

    def select_greedy(self, cams, rounds: int, target_obj: int = -1, want_scores: bool = True):
        """nbv_select_greedy: returns (order: numpy int32 (rounds,), scores: CUDA tensor (rounds, n) or None).
        H_T contains the selected views afterwards."""
        torch = self._torch
        cams = _cams(cams)
        n = int(cams.shape[0])
        order = np.full(max(int(rounds), 1), -1, dtype=np.int32)
        scores = torch.empty((max(int(rounds), 1), max(n, 1)), dtype=torch.float32, device=self.device) if want_scores else None
        self._check(self.lib.nbv_select_greedy(self._h, C.c_void_p(cams.ctypes.data), n, int(rounds), int(target_obj),
                                               C.c_void_p(order.ctypes.data), _ptr(scores), _stream()))
        return order[:rounds], (scores[:rounds, :n] if want_scores else None)

    def batch_views(self, width: int, height: int) -> int:
        """nbv_batch_views: views per batch a call with images of this size would use"""
        return int(self.lib.nbv_batch_views(self._h, int(width), int(height)))

    def set_concurrency(self, views_in_flight: int):
        self._check(self.lib.nbv_set_concurrency(self._h, int(views_in_flight)))

    def last_view_stats(self) -> dict:
        st = ViewStats()
        self._check(self.lib.nbv_last_view_stats(self._h, C.byref(st), _stream()))
        return st.as_dict()

    # ---- measurement ----------------------------------------------------------------------------
    def set_stage_timing(self, enable: bool = True):
        self._check(self.lib.nbv_set_stage_timing(self._h, int(bool(enable)), _stream()))

    def stage_times(self) -> tuple[dict, int]:
        """({stage: milliseconds summed over the timed views}, number of views)"""
        ms = (C.c_double * len(STAGES))()
        views = C.c_int64(0)
        self._check(self.lib.nbv_stage_times(self._h, ms, C.byref(views), _stream()))
        return {k: float(ms[i]) for i, k in enumerate(STAGES)}, int(views.value)

    def kernel_launches(self) -> int:
        return int(self.lib.nbv_kernel_launches())

    # ---- parity / debug exports ------------------------------------------------------------------
    def projected(self, cam):
        torch = self._torch
        cam = _cams(cam)
        vis = torch.empty(self.N, dtype=torch.int32, device=self.device)
        rec = torch.empty((self.N, 9), dtype=torch.float32, device=self.device)
        rect = torch.empty((self.N, 4), dtype=torch.int32, device=self.device)
        self._check(self.lib.nbv_projected(self._h, C.c_void_p(cam.ctypes.data), _ptr(vis), _ptr(rec), _ptr(rect), _stream()))
        return vis, rec, rect

    def tile_lists(self, cam):
        torch = self._torch
        cam = _cams(cam)
        W, H = int(cam["width"][0]), int(cam["height"][0])
        nt = ((W + 15) // 16) * ((H + 15) // 16)
        offsets = torch.empty(nt + 1, dtype=torch.int64, device=self.device)
        total = C.c_int64(0)
        rc = self.lib.nbv_tile_lists(self._h, C.c_void_p(cam.ctypes.data), _ptr(offsets), None, C.c_int64(0), C.byref(total), _stream())
        if rc not in (0, -8):
            self._check(rc)
        ids = torch.empty(max(int(total.value), 1), dtype=torch.int32, device=self.device)
        self._check(self.lib.nbv_tile_lists(self._h, C.c_void_p(cam.ctypes.data), _ptr(offsets), _ptr(ids), C.c_int64(ids.numel()),
                                            C.byref(total), _stream()))
        return offsets, ids[: int(total.value)]

    def tile_walk(self, cam):
        """nbv_tile_walk: (walked per tile, last per pixel)"""
        torch = self._torch
        cam = _cams(cam)
        W, H = int(cam["width"][0]), int(cam["height"][0])
        nt = ((W + 15) // 16) * ((H + 15) // 16)
        walked = torch.empty(nt, dtype=torch.int32, device=self.device)
        last = torch.empty((H, W), dtype=torch.int32, device=self.device)
        self._check(self.lib.nbv_tile_walk(self._h, C.c_void_p(cam.ctypes.data), _ptr(walked), _ptr(last), _stream()))
        return walked, last

    def render(self, cam):
        torch = self._torch
        cam = _cams(cam)
        W, H = int(cam["width"][0]), int(cam["height"][0])
        rgb = torch.empty((H, W, 3), dtype=torch.float32, device=self.device)
        depth = torch.empty((H, W), dtype=torch.float32, device=self.device)
        T = torch.empty((H, W), dtype=torch.float32, device=self.device)
        nc = torch.empty((H, W), dtype=torch.int32, device=self.device)
        self._check(self.lib.nbv_render(self._h, C.c_void_p(cam.ctypes.data), _ptr(rgb), _ptr(depth), _ptr(T), _ptr(nc), _stream()))
        return dict(rgb=rgb, depth=depth, T=T, ncontrib=nc)

    def block_size(self) -> int:
        """nbv_block_size: floats per packed block (105, or L (L + 1) / 2 with L = 11 + K in a mask context)"""
        return int(self.lib.nbv_block_size(self._h))

    def render_mask(self, cam):
        """nbv_render_mask: (H, W, K) blended object vector (mask contexts)"""
        torch = self._torch
        cam = _cams(cam)
        W, H = int(cam["width"][0]), int(cam["height"][0])
        mask = torch.empty((H, W, self.K), dtype=torch.float32, device=self.device)
        self._check(self.lib.nbv_render_mask(self._h, C.c_void_p(cam.ctypes.data), _ptr(mask), _stream()))
        return mask

    def view_hessian(self, cam):
        torch = self._torch
        cam = _cams(cam)
        blocks = torch.empty((self.N, self.block_size()), dtype=torch.float32, device=self.device)
        self._check(self.lib.nbv_view_hessian(self._h, C.c_void_p(cam.ctypes.data), _ptr(blocks), _stream()))
        return blocks

    def training_hessian(self):
        torch = self._torch
        blocks = torch.empty((self.N, self.block_size()), dtype=torch.float32, device=self.device)
        self._check(self.lib.nbv_training_hessian(self._h, _ptr(blocks), _stream()))
        return blocks

    def chain(self, cam):
        """nbv_chain: (N, 53) = d(mx,my,a,b,c)/d(mu,logscale,quat) (5 x 10, row-major) then dz/dmu (3), per Gaussian"""
        torch = self._torch
        cam = _cams(cam)
        out = torch.empty((self.N, 53), dtype=torch.float32, device=self.device)
        self._check(self.lib.nbv_chain(self._h, C.c_void_p(cam.ctypes.data), _ptr(out), _stream()))
        return out

    def confidence(self, target_obj: int = -1):
        torch = self._torch
        conf = torch.empty(self.N, dtype=torch.float32, device=self.device)
        self._check(self.lib.nbv_confidence(self._h, int(target_obj), _ptr(conf), _stream()))
        return conf

    def gaussian_gains(self, cam, target_obj: int = -1):
        torch = self._torch
        cam = _cams(cam)
        gains = torch.empty(self.N, dtype=torch.float32, device=self.device)
        self._check(self.lib.nbv_gaussian_gains(self._h, C.c_void_p(cam.ctypes.data), int(target_obj), _ptr(gains), _stream()))
        return gains


def exp_spec_pairs(x):
    """nbv_exp_spec_pairs: the raster kernels' packed exp_spec on a CUDA float32 tensor (returns a tensor of the same shape)."""
    import torch
    x = x.contiguous()
    y = torch.empty_like(x)
    rc = load_library().nbv_exp_spec_pairs(_ptr(x), _ptr(y), C.c_int64(x.numel()), _stream())
    if rc != 0:
        raise NBVError(rc, "nbv_exp_spec_pairs failed")
    return y


SCAN_NOALLOC_MAX = 16777216      # NBV_SCAN_NOALLOC_MAX


def exclusive_scan_noalloc(x, out=None, total=None):
    """nbv_exclusive_scan_noalloc: exclusive prefix sum of a CUDA int32 / uint32 tensor (the bits are taken as uint32) with the
    scratch in the library's static device array -- the call itself allocates nothing; the tensors are the caller's: `out`
    (same size, may be x) and `total` (1 element) are created here only when not passed in.  Returns (out, total)."""
    import torch
    x = x.contiguous()
    if out is None:
        out = torch.empty_like(x)
    if total is None:
        total = torch.empty(1, dtype=x.dtype, device=x.device)
    lib = load_library()
    rc = lib.nbv_exclusive_scan_noalloc(_ptr(x), _ptr(out), C.c_int64(x.numel()), _ptr(total), _stream())
    if rc != 0:
        raise NBVError(rc, (lib.nbv_noalloc_last_error() or b"").decode())
    return out, total


def measure_ffma_peak() -> float:
    """nbv_measure_ffma_peak: TFLOP/s of an FFMA-chain microbenchmark on the current CUDA device."""
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("libnbv needs a CUDA device (sm_100a); there is no CPU fallback")
    v = C.c_double(0.0)
    rc = load_library().nbv_measure_ffma_peak(C.byref(v), _stream())
    if rc != 0:
        raise NBVError(rc, "nbv_measure_ffma_peak failed")
    return float(v.value)


def score_candidates_fused(nbv_rgb: NBV, nbv_depth: NBV, train_cams, cams, target_obj: int = -1, beta_d: float = 10.0,
                           nbv_mask: NBV | None = None, beta_o: float = 1.0):
    """nbv_score_candidates_fused (Eq. 10-11): returns dict(fused (n,), raw (F, n), denom (F,), best (1,)) of
    CUDA tensors, F = 2 (rgb, depth) or 3 (+ mask).  The contexts hold the same map with channel masks RGB / DEPTH /
    MASK and have `train_cams` already accumulated."""
    torch = nbv_rgb._torch
    tc, cc = _cams(train_cams), _cams(cams)
    n, nt = int(cc.shape[0]), int(tc.shape[0])
    F = 3 if nbv_mask is not None else 2
    dev = nbv_rgb.device
    fused = torch.empty(max(n, 1), dtype=torch.float32, device=dev)
    raw = torch.empty((F, max(n, 1)), dtype=torch.float32, device=dev)
    denom = torch.empty(F, dtype=torch.float32, device=dev)
    best = torch.empty(1, dtype=torch.int32, device=dev)
    rc = nbv_rgb.lib.nbv_score_candidates_fused(nbv_rgb._h, nbv_depth._h, nbv_mask._h if nbv_mask is not None else None,
                                                C.c_void_p(tc.ctypes.data), nt, C.c_void_p(cc.ctypes.data), n, int(target_obj),
                                                C.c_float(beta_d), C.c_float(beta_o), _ptr(fused), _ptr(raw), _ptr(denom),
                                                _ptr(best), _stream())
    nbv_rgb._check(rc)
    return dict(fused=fused[:n], raw=raw[:, :n] if n else raw[:, :0], denom=denom, best=best)
