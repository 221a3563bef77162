"""CPU oracle, Python side.  TEST INFRASTRUCTURE -- see the header of nbv_oracle.cpp.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl
reference` legs may import this.  It imports nothing from
paper_2602_08266_b200: inputs arrive as plain numpy arrays.

C++ part (nbv_oracle.cpp, via ctypes): activation, projection, depth order, tile
lists, per-pixel compositing, analytic Jacobian rows and J^T J blocks.
numpy part (this file): confidence (Eq. 7, 8, 12), confidence-weighted
block-diagonal log-det information gain (Eq. 5, 6, 9) with numpy.linalg.slogdet
as the library primitive, and the arg-max over candidates (Eq. 5).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "nbv_oracle.cpp"
_EXT = _HERE / "nbv_oracle_ext.inc"
_LIB = _HERE / "libnbv_oracle.so"

P = 14
NB = 105

CAMERA_DTYPE = np.dtype([("width", "<i4"), ("height", "<i4"), ("fx", "<f4"), ("fy", "<f4"), ("cx", "<f4"),
                         ("cy", "<f4"), ("R", "<f4", (9,)), ("t", "<f4", (3,))])


class Config(C.Structure):
    _fields_ = [
        ("near_plane", C.c_float), ("blur", C.c_float), ("alpha_min", C.c_float), ("alpha_max", C.c_float),
        ("t_stop", C.c_float), ("power_min", C.c_float), ("bg", C.c_float * 3), ("channel_mask", C.c_int32),
        ("channel_weight", C.c_float * 4), ("opacity_coord", C.c_int32),
    ]


def default_config(channel_mask: int = 7, bg=(0.0, 0.0, 0.0), opacity_coord: int = 0,
                   channel_weight=(1.0, 1.0, 1.0, 1.0)) -> Config:
    cfg = Config()
    cfg.near_plane = 0.01
    cfg.blur = 0.3
    cfg.alpha_min = np.float32(1.0 / 255.0)
    cfg.alpha_max = 0.99
    cfg.t_stop = 1e-4
    cfg.power_min = -6.0
    cfg.bg = (C.c_float * 3)(*bg)
    cfg.channel_mask = channel_mask
    cfg.channel_weight = (C.c_float * 4)(*channel_weight)
    cfg.opacity_coord = opacity_coord
    return cfg


def build(force: bool = False) -> Path:
    """Compile the oracle shared library (g++, OpenMP, no FP contraction)."""
    if _LIB.exists() and not force and _LIB.stat().st_mtime >= max(_SRC.stat().st_mtime, _EXT.stat().st_mtime):
        return _LIB
    flags = ["-O2", "-std=c++17", "-fopenmp", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC"]
    try:
        if " fma " in open("/proc/cpuinfo").read():
            flags.append("-mfma")  # std::fmaf inlined; without it libm's (correctly rounded) fmaf is called
    except OSError:
        pass
    tmp = _LIB.with_suffix(".so.tmp%d" % os.getpid())
    subprocess.check_call(["g++", *flags, str(_SRC), "-o", str(tmp)])
    os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(str(build()))
        _lib.orc_create.restype = C.c_void_p
        _lib.orc_exp_spec.restype = C.c_float
        _lib.orc_exp_spec.argtypes = [C.c_float]
        _lib.orc_log_bound.restype = C.c_float
        _lib.orc_log_bound.argtypes = [C.c_float]
        _lib.orc_tile_lists.restype = C.c_int64
        _lib.orc_trace.restype = C.c_int64
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def _cam(cam) -> np.ndarray:
    """one camera record as a contiguous (1,) CAMERA_DTYPE array"""
    return np.ascontiguousarray(np.asarray(cam, dtype=CAMERA_DTYPE).reshape(-1)[:1])


def _wh(cam):
    return int(cam["width"][0]), int(cam["height"][0])


def exp_spec(x) -> np.ndarray:
    x = np.atleast_1d(np.asarray(x, dtype=np.float32))
    return np.array([lib().orc_exp_spec(C.c_float(float(v))) for v in x], dtype=np.float32)


def log_bound(s) -> np.ndarray:
    s = np.atleast_1d(np.asarray(s, dtype=np.float32))
    return np.array([lib().orc_log_bound(C.c_float(float(v))) for v in s], dtype=np.float32)


def num_threads() -> int:
    return int(lib().orc_num_threads())


class OracleScene:
    """Gaussian map G held by the C++ oracle."""

    def __init__(self, mean, logscale, quat, opacity, rgb, obj_logits, cfg: Config | None = None):
        f = lambda a: np.ascontiguousarray(a, dtype=np.float32)
        self.mean, self.logscale, self.quat = f(mean), f(logscale), f(quat)
        self.opacity, self.rgb, self.obj_logits = f(opacity), f(rgb), f(obj_logits)
        self.N = int(self.mean.shape[0])
        self.K = int(self.obj_logits.shape[1]) if self.obj_logits.ndim == 2 else 0
        self.cfg = cfg if cfg is not None else default_config()
        self._h = C.c_void_p(lib().orc_create(self.N, self.K, _p(self.mean), _p(self.logscale), _p(self.quat),
                                              _p(self.opacity), _p(self.rgb), C.byref(self.cfg)))

    def __del__(self):
        try:
            if self._h:
                lib().orc_destroy(self._h)
                self._h = None
        except Exception:
            pass

    @property
    def bad_data(self) -> bool:
        return bool(lib().orc_bad_data(self._h))

    def activation(self) -> np.ndarray:
        M = np.zeros((self.N, 9), dtype=np.float32)
        lib().orc_activation(self._h, _p(M))
        return M

    def project(self, cam):
        """decision-path splats: visible (N,), rec (N,9) = mx,my,qa,qb,qc,z,a,b,c ; rect (N,4) tx0,ty0,tx1,ty1"""
        cam = _cam(cam)
        vis = np.zeros(self.N, dtype=np.int32)
        rec = np.zeros((self.N, 9), dtype=np.float32)
        rect = np.zeros((self.N, 4), dtype=np.int32)
        lib().orc_project(self._h, _p(cam), _p(vis), _p(rec), _p(rect))
        return vis, rec, rect

    def depth_order(self, cam) -> np.ndarray:
        cam = _cam(cam)
        order = np.zeros(self.N, dtype=np.int32)
        n = lib().orc_depth_order(self._h, _p(cam), _p(order))
        return order[:n].copy()

    def tile_lists(self, cam):
        cam = _cam(cam)
        W, H = _wh(cam)
        tx, ty = (W + 15) // 16, (H + 15) // 16
        offsets = np.zeros(tx * ty + 1, dtype=np.int64)
        total = lib().orc_tile_lists(self._h, _p(cam), _p(offsets), None, C.c_int64(0))
        ids = np.zeros(max(int(total), 1), dtype=np.int32)
        total2 = lib().orc_tile_lists(self._h, _p(cam), _p(offsets), _p(ids), C.c_int64(ids.size))
        assert total2 == total
        return offsets, ids[:total]

    def render(self, cam, pixel_mask=None):
        """dict(rgb (H,W,3), depth, T (binary64 value path), T32 (decision path), ncontrib)"""
        cam = _cam(cam)
        W, H = _wh(cam)
        rgb = np.zeros((H, W, 3))
        depth = np.zeros((H, W))
        T = np.ones((H, W))
        T32 = np.ones((H, W), dtype=np.float32)
        nc = np.zeros((H, W), dtype=np.int32)
        pm = None if pixel_mask is None else np.ascontiguousarray(pixel_mask, dtype=np.uint8)
        lib().orc_render(self._h, _p(cam), _p(pm), _p(rgb), _p(depth), _p(T), _p(T32), _p(nc))
        return dict(rgb=rgb, depth=depth, T=T, T32=T32, ncontrib=nc)

    def trace(self, cam):
        """per-pixel contributor lists, CSR: offsets (H*W+1,), ids, clamped"""
        cam = _cam(cam)
        W, H = _wh(cam)
        offsets = np.zeros(H * W + 1, dtype=np.int64)
        total = lib().orc_trace(self._h, _p(cam), _p(offsets), None, None, C.c_int64(0))
        ids = np.zeros(max(int(total), 1), dtype=np.int32)
        cl = np.zeros(max(int(total), 1), dtype=np.uint8)
        lib().orc_trace(self._h, _p(cam), _p(offsets), _p(ids), _p(cl), C.c_int64(ids.size))
        return offsets, ids[:total], cl[:total]

    def view_hessian(self, cam, pixel_mask=None, out=None) -> np.ndarray:
        """(N,105) packed upper triangles of sum_pixels sum_channels omega J^T J; accumulates into `out`."""
        cam = _cam(cam)
        if out is None:
            out = np.zeros((self.N, NB))
        pm = None if pixel_mask is None else np.ascontiguousarray(pixel_mask, dtype=np.uint8)
        lib().orc_view_hessian(self._h, _p(cam), _p(pm), _p(out))
        return out

    def theta(self) -> np.ndarray:
        """(N,14) binary64 parameter vectors [mu | logscale | quat | opacity logit | rgb]"""
        th = np.zeros((self.N, P))
        th[:, 0:3] = self.mean
        th[:, 3:6] = self.logscale
        th[:, 6:10] = self.quat
        s = self.opacity.astype(np.float64)
        th[:, 10] = np.log(s) - np.log1p(-s)
        th[:, 11:14] = self.rgb
        return th


# ---- object-mask output (Eq. 1-2) -----------------------------
def mask_block_size(K: int) -> int:
    L = 11 + K
    return L * (L + 1) // 2


def unpack_blocks_L(packed: np.ndarray, L: int) -> np.ndarray:
    iu = np.triu_indices(L)
    packed = np.asarray(packed, dtype=np.float64)
    full = np.zeros(packed.shape[:-1] + (L, L))
    full[..., iu[0], iu[1]] = packed
    full[..., iu[1], iu[0]] = packed
    return full


def render_mask(scene: "OracleScene", cam, bg_channel: int = 0) -> np.ndarray:
    """(H,W,K) per-pixel object vector: O' = sum_i softmax(o_i) alpha_i T_i (Eq. 1) plus the residual 1 - 1^T O' on the
    background channel (Eq. 2)."""
    cam = _cam(cam)
    W, H = _wh(cam)
    prob = np.ascontiguousarray(softmax(scene.obj_logits))
    out = np.zeros((H, W, scene.K))
    lib().orc_render_mask(scene._h, _p(cam), scene.K, int(bg_channel), _p(prob), _p(out))
    return out


def view_hessian_mask(scene: "OracleScene", cam, bg_channel: int = 0, out=None) -> np.ndarray:
    """(N, L(L+1)/2), L = 11 + K: packed J^T J blocks of the mask output w.r.t. [mu, logscale, quat, opacity | logits];
    accumulates into `out`."""
    cam = _cam(cam)
    prob = np.ascontiguousarray(softmax(scene.obj_logits))
    if out is None:
        out = np.zeros((scene.N, mask_block_size(scene.K)))
    lib().orc_view_hessian_mask(scene._h, _p(cam), scene.K, int(bg_channel), _p(prob), _p(out))
    return out


def render_mask_smooth(theta11, logits, cam, cfg, offsets, ids, clamped, bg_channel: int = 0) -> np.ndarray:
    cam = _cam(cam)
    theta11 = np.ascontiguousarray(theta11, dtype=np.float64)
    logits = np.ascontiguousarray(logits, dtype=np.float64)
    W, H = _wh(cam)
    N, K = logits.shape
    out = np.zeros((H, W, K))
    lib().orc_render_mask_smooth(N, K, int(bg_channel), _p(theta11), _p(logits), _p(cam), C.byref(cfg), _p(offsets), _p(ids),
                                 _p(clamped), _p(out))
    return out


def view_hessian_mask_smooth(theta11, logits, cam, cfg, offsets, ids, clamped, bg_channel: int = 0) -> np.ndarray:
    cam = _cam(cam)
    theta11 = np.ascontiguousarray(theta11, dtype=np.float64)
    logits = np.ascontiguousarray(logits, dtype=np.float64)
    N, K = logits.shape
    out = np.zeros((N, mask_block_size(K)))
    lib().orc_view_hessian_mask_smooth(N, K, int(bg_channel), _p(theta11), _p(logits), _p(cam), C.byref(cfg), _p(offsets),
                                       _p(ids), _p(clamped), _p(out))
    return out


def gaussian_gains_L(H_T, H_c, c, prior, L: int) -> np.ndarray:
    """gaussian_gains for blocks of L x L parameters (prior: L diagonal entries of Lambda)."""
    Lam = np.diag(np.asarray(prior, dtype=np.float64))
    A, B = unpack_blocks_L(H_T, L), unpack_blocks_L(H_c, L)
    c = np.asarray(c, dtype=np.float64)[:, None, None]
    s1, l1 = np.linalg.slogdet(c * (A + B) + Lam)
    s0, l0 = np.linalg.slogdet(c * A + Lam)
    assert np.all(s1 > 0) and np.all(s0 > 0)
    return l1 - l0


def score_candidates_mask(scene: "OracleScene", train_cams, cand_cams, target=-1, alpha_obj=0.3, alpha_opa=0.3, prior=None,
                          bg_channel: int = 0):
    """IG_o(T, c) (Eq. 5, 6, 9 on the mask output's blocks).  Returns dict(H_T, scores, best)."""
    L = 11 + scene.K
    prior = np.ones(L) if prior is None else np.asarray(prior, dtype=np.float64)
    H_T = np.zeros((scene.N, mask_block_size(scene.K)))
    for cam in np.atleast_1d(train_cams):
        view_hessian_mask(scene, cam, bg_channel, out=H_T)
    conf = confidence(scene.obj_logits, scene.opacity, alpha_obj, alpha_opa, target)
    scores = np.array([gaussian_gains_L(H_T, view_hessian_mask(scene, cam, bg_channel), conf, prior, L).sum()
                       for cam in np.atleast_1d(cand_cams)])
    return dict(H_T=H_T, scores=scores, best=argmax_lowest(scores))


def render_smooth(theta, cam, cfg, offsets, ids, clamped) -> np.ndarray:
    cam = _cam(cam)
    theta = np.ascontiguousarray(theta, dtype=np.float64)
    W, H = _wh(cam)
    out = np.zeros((H, W, 4))
    lib().orc_render_smooth(theta.shape[0], _p(theta), _p(cam), C.byref(cfg), _p(offsets), _p(ids), _p(clamped), _p(out))
    return out


def view_hessian_smooth(theta, cam, cfg, offsets, ids, clamped) -> np.ndarray:
    cam = _cam(cam)
    theta = np.ascontiguousarray(theta, dtype=np.float64)
    out = np.zeros((theta.shape[0], NB))
    lib().orc_view_hessian_smooth(theta.shape[0], _p(theta), _p(cam), C.byref(cfg), _p(offsets), _p(ids), _p(clamped), _p(out))
    return out


def chain(theta14, cam, cfg):
    """binary64 projection of one Gaussian and its derivatives: (mx,my,a,b,c,z), G (5,10), dz (3,)"""
    cam = _cam(cam)
    th = np.ascontiguousarray(theta14, dtype=np.float64)
    out6 = np.zeros(6)
    G = np.zeros((5, 10))
    dz = np.zeros(3)
    lib().orc_chain(_p(cam), C.byref(cfg), _p(th), _p(out6), _p(G), _p(dz))
    return out6, G, dz


# ---------------------------------------------------------------------------
# numpy part: blocks, confidence, gain, arg-max
# ---------------------------------------------------------------------------
_IU = np.triu_indices(P)


def unpack_blocks(packed: np.ndarray) -> np.ndarray:
    """(N,105) -> (N,14,14) symmetric."""
    packed = np.asarray(packed, dtype=np.float64)
    full = np.zeros(packed.shape[:-1] + (P, P))
    full[..., _IU[0], _IU[1]] = packed
    full[..., _IU[1], _IU[0]] = packed
    return full


def pack_blocks(full: np.ndarray) -> np.ndarray:
    return np.asarray(full)[..., _IU[0], _IU[1]]


def softmax(logits: np.ndarray) -> np.ndarray:
    z = np.asarray(logits, dtype=np.float64)
    z = z - z.max(axis=1, keepdims=True)
    e = np.exp(z)
    return e / e.sum(axis=1, keepdims=True)


def confidence(obj_logits, opacity, alpha_obj=0.3, alpha_opa=0.3, target=-1, p_floor=1e-4, s_floor=1e-4) -> np.ndarray:
    """PAPER.md Eq. 7 (L229-232): c_g = max_k(p_gk)^-alpha_obj * sigma_g^-alpha_opa, p_g = softmax(o_g) (L146).
    Eq. 12 (L698-704) with a target object: p_{g,obj} replaces the max, and c_g = 0 unless argmax_k p_gk = obj.
    Floors on p and sigma: reading R-14."""
    p = softmax(obj_logits)
    s = np.maximum(np.asarray(opacity, dtype=np.float64), s_floor)
    if target < 0:
        pm = np.maximum(p.max(axis=1), p_floor)
        return pm ** (-alpha_obj) * s ** (-alpha_opa)
    am = p.argmax(axis=1)  # lowest index on ties
    pt = np.maximum(p[:, target], p_floor)
    c = pt ** (-alpha_obj) * s ** (-alpha_opa)
    return np.where(am == target, c, 0.0)


def gaussian_gains(H_T, H_c, c, prior, weight_mode: int = 0) -> np.ndarray:
    """Per-Gaussian information gain (Eq. 5, 6, 9; block-diagonal, L210).  H_T, H_c: (N,105) packed; c: (N,);
    prior: (14,) diagonal of Lambda (reading R-13).  Where the confidence acts (reading R-14):
      weight_mode 0 (R1, Eq. 9 literal "H := J^T C J"): log det(c (H_T + H_c) + Lambda) - log det(c H_T + Lambda)
      weight_mode 1 (R2, L61 "weighting each Gaussian's information gain"): c [log det(H_T + H_c + Lambda) - log det(H_T + Lambda)]
      weight_mode 2 (R3, L238 "scale each Jacobian ... during information gain computation", candidate only):
                     log det(H_T + c H_c + Lambda) - log det(H_T + Lambda)"""
    Lam = np.diag(np.asarray(prior, dtype=np.float64))
    A = unpack_blocks(H_T)
    B = unpack_blocks(H_c)
    cv = np.asarray(c, dtype=np.float64)
    c3 = cv[:, None, None]
    if weight_mode == 0:
        M1, M0, out_scale = c3 * (A + B) + Lam, c3 * A + Lam, 1.0
    elif weight_mode == 1:
        M1, M0, out_scale = A + B + Lam, A + Lam, cv
    else:
        M1, M0, out_scale = A + c3 * B + Lam, A + Lam, 1.0
    s1, l1 = np.linalg.slogdet(M1)
    s0, l0 = np.linalg.slogdet(M0)
    assert np.all(s1 > 0) and np.all(s0 > 0)
    return out_scale * (l1 - l0)


def argmax_lowest(scores) -> int:
    """PAPER.md Eq. 5: c* = argmax_c IG(T,c); ties -> lowest index (R-15)."""
    scores = np.asarray(scores)
    return int(np.flatnonzero(scores == scores.max())[0])


def score_candidates(scene: OracleScene, train_cams, cand_cams, target=-1, alpha_obj=0.3, alpha_opa=0.3,
                     prior=None, H_T=None, weight_mode: int = 0):
    """The whole hot path on the CPU.  Returns dict(H_T, scores, best, conf, gains (C,N))."""
    prior = np.ones(P) if prior is None else np.asarray(prior, dtype=np.float64)
    if H_T is None:
        H_T = np.zeros((scene.N, NB))
        for cam in np.atleast_1d(train_cams):
            scene.view_hessian(cam, out=H_T)
    conf = confidence(scene.obj_logits, scene.opacity, alpha_obj, alpha_opa, target)
    scores, gains = [], []
    for cam in np.atleast_1d(cand_cams):
        H_c = scene.view_hessian(cam)
        g = gaussian_gains(H_T, H_c, conf, prior, weight_mode)
        gains.append(g)
        scores.append(g.sum())
    scores = np.array(scores)
    return dict(H_T=H_T, scores=scores, best=argmax_lowest(scores), conf=conf, gains=np.array(gains))


# ---------------------------------------------------------------------------------------------------
# per-output normalisation and fusion (Eq. 10-11), greedy selection.
# ---------------------------------------------------------------------------------------------------
def normalized_gain(raw, training_gains):
    """PAPER.md Eq. 10 (L251-257): IG~_f(T,c) = IG_f(T,c) / ( (1/|T|) sum_{t in T} IG_f(T,t) )."""
    tg = np.asarray(training_gains, dtype=np.float64)
    return np.asarray(raw, dtype=np.float64) / (tg.sum() / tg.size)


def fused_gain(ig_rgb_n, ig_d_n, beta_d=10.0):
    """PAPER.md Eq. 11 (L261-265) without the object-mask output (NEXT-2, not built): IG~ = IG~_rgb + beta_d IG~_d;
    beta_d = 10 (L742)."""
    return np.asarray(ig_rgb_n, dtype=np.float64) + beta_d * np.asarray(ig_d_n, dtype=np.float64)


def fused_gain3(ig_rgb_n, ig_d_n, ig_o_n, beta_d=10.0, beta_o=1.0):
    """PAPER.md Eq. 11 (L261-265): IG~ = IG~_rgb + beta_d IG~_d + beta_o IG~_o; beta_d = 10, beta_o = 1 (L742)."""
    return fused_gain(ig_rgb_n, ig_d_n, beta_d) + beta_o * np.asarray(ig_o_n, dtype=np.float64)


def score_candidates_fused(scene_rgb: OracleScene, scene_d: OracleScene, train_cams, cand_cams, target=-1, beta_d=10.0,
                           alpha_obj=0.3, alpha_opa=0.3, prior=None, scene_mask: OracleScene | None = None, beta_o=1.0,
                           bg_channel: int = 0):
    """Per-output gains (L248: each output has its own Jacobian, hence its own Hessian and gain), normalised by the
    mean gain of the training views re-scored as candidates on top of the full H_T (Eq. 10), fused (Eq. 11), arg-max
    (Eq. 5).  scene_rgb / scene_d: the same map with channel masks {r,g,b} / {depth}; scene_mask (optional): the same
    map again, scored on its object-mask output.
    Returns dict(raw (F,C), denom (F,), normalized (F,C), fused (C,), best), F = 2 or 3."""
    raw, denom = [], []
    for scn in (scene_rgb, scene_d):
        H_T = np.zeros((scn.N, NB))
        for cam in np.atleast_1d(train_cams):
            scn.view_hessian(cam, out=H_T)
        r_c = score_candidates(scn, train_cams[:0], cand_cams, target, alpha_obj, alpha_opa, prior, H_T=H_T)["scores"]
        r_t = score_candidates(scn, train_cams[:0], train_cams, target, alpha_obj, alpha_opa, prior, H_T=H_T)["scores"]
        raw.append(r_c)
        denom.append(r_t.sum() / r_t.size)
    if scene_mask is not None:
        r_c = score_candidates_mask(scene_mask, train_cams, cand_cams, target, alpha_obj, alpha_opa, None, bg_channel)["scores"]
        r_t = score_candidates_mask(scene_mask, train_cams, train_cams, target, alpha_obj, alpha_opa, None, bg_channel)["scores"]
        raw.append(r_c)
        denom.append(r_t.sum() / r_t.size)
    raw, denom = np.array(raw), np.array(denom)
    norm = np.array([normalized_gain(raw[f], [denom[f]]) for f in range(len(raw))])
    fused = fused_gain(norm[0], norm[1], beta_d) if scene_mask is None else fused_gain3(norm[0], norm[1], norm[2], beta_d, beta_o)
    return dict(raw=raw, denom=denom, normalized=norm, fused=fused, best=argmax_lowest(fused))


def select_greedy(scene: OracleScene, train_cams, cand_cams, rounds, target=-1, alpha_obj=0.3, alpha_opa=0.3, prior=None):
    """Greedy multi-view selection without retraining (Eq. 5 applied repeatedly; L746 "6 rounds"):
    in every round score the not-yet-selected candidates against the current H_T, pick the arg-max (lowest index on
    ties), and add that view's Hessian to H_T (Eq. 6: the sum over the view set).
    Returns dict(order (rounds,), scores (rounds, C) with NaN at already selected candidates)."""
    prior = np.ones(P) if prior is None else np.asarray(prior, dtype=np.float64)
    cand_cams = np.atleast_1d(cand_cams)
    H_T = np.zeros((scene.N, NB))
    for cam in np.atleast_1d(train_cams):
        scene.view_hessian(cam, out=H_T)
    conf = confidence(scene.obj_logits, scene.opacity, alpha_obj, alpha_opa, target)
    H_c = [scene.view_hessian(cam) for cam in cand_cams]       # a view's block does not depend on H_T
    order, table = [], []
    for _ in range(rounds):
        row = np.full(len(cand_cams), np.nan)
        for i in range(len(cand_cams)):
            if i not in order:
                row[i] = gaussian_gains(H_T, H_c[i], conf, prior).sum()
        best = int(np.flatnonzero(row == np.nanmax(row))[0])
        order.append(best)
        table.append(row)
        H_T = H_T + H_c[best]
    return dict(order=np.array(order), scores=np.array(table))
