"""CPU oracle, view-dependent colour (SH degree 3).  TEST INFRASTRUCTURE -- same rules as nbv_oracle.py.

SURVEY.md section 8(f) NEXT-4; PAPER.md L131 (SH coefficients c in R^{3(d+1)^2}), L156 (d = 0 during NBV), L166 (degree 3
for the final reconstruction).  Reading R-18: colour_ch(dir) = rgb_ch + sum_{j=1}^{15} B_j(dir) k_{j,ch}; block of
L = 59 parameters [mu logscale quat opacity | rgb | k_1 .. k_15 (3 each)].  C++ part: oracle/nbv_oracle_ext.inc.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import nbv_oracle as orc

L = 59
LB = L * (L + 1) // 2
NK = 45


def _k(k45, N):
    k = np.ascontiguousarray(k45, dtype=np.float32).reshape(N, NK)
    return k


def basis(direction):
    """B (16,), dB/d(x,y,z) (16,3) at the normalised direction"""
    d = np.ascontiguousarray(direction, dtype=np.float64)
    B, dB = np.zeros(16), np.zeros((16, 3))
    orc.lib().orc_sh_basis(orc._p(d), orc._p(B), orc._p(dB))
    return B, dB


def colours(scene: "orc.OracleScene", cam, k45) -> np.ndarray:
    cam = orc._cam(cam)
    k = _k(k45, scene.N)
    out = np.zeros((scene.N, 3))
    orc.lib().orc_sh_colours(scene._h, orc._p(cam), orc._p(k), orc._p(out))
    return out


def render(scene: "orc.OracleScene", cam, k45):
    cam = orc._cam(cam)
    W, H = orc._wh(cam)
    k = _k(k45, scene.N)
    rgb, depth, nc = np.zeros((H, W, 3)), np.zeros((H, W)), np.zeros((H, W), dtype=np.int32)
    orc.lib().orc_render_sh(scene._h, orc._p(cam), orc._p(k), orc._p(rgb), orc._p(depth), orc._p(nc))
    return dict(rgb=rgb, depth=depth, ncontrib=nc)


def view_hessian(scene: "orc.OracleScene", cam, k45, out=None) -> np.ndarray:
    """(N, 1770) packed 59 x 59 blocks; accumulates into `out`"""
    cam = orc._cam(cam)
    k = _k(k45, scene.N)
    if out is None:
        out = np.zeros((scene.N, LB))
    orc.lib().orc_view_hessian_sh(scene._h, orc._p(cam), orc._p(k), orc._p(out))
    return out


def theta(scene: "orc.OracleScene", k45) -> np.ndarray:
    """(N, 59) binary64 parameter vectors"""
    return np.concatenate([scene.theta(), _k(k45, scene.N).astype(np.float64)], axis=1)


def render_smooth(theta59, cam, cfg, offsets, ids, clamped) -> np.ndarray:
    cam = orc._cam(cam)
    th = np.ascontiguousarray(theta59, dtype=np.float64)
    W, H = orc._wh(cam)
    out = np.zeros((H, W, 4))
    orc.lib().orc_render_sh_smooth(th.shape[0], orc._p(th), orc._p(cam), C.byref(cfg), orc._p(offsets), orc._p(ids), orc._p(clamped),
                                   orc._p(out))
    return out


def view_hessian_smooth(theta59, cam, cfg, offsets, ids, clamped) -> np.ndarray:
    cam = orc._cam(cam)
    th = np.ascontiguousarray(theta59, dtype=np.float64)
    out = np.zeros((th.shape[0], LB))
    orc.lib().orc_view_hessian_sh_smooth(th.shape[0], orc._p(th), orc._p(cam), C.byref(cfg), orc._p(offsets), orc._p(ids),
                                         orc._p(clamped), orc._p(out))
    return out


def score_candidates(scene: "orc.OracleScene", k45, train_cams, cand_cams, target=-1, alpha_obj=0.3, alpha_opa=0.3, prior=None):
    """Eq. 5, 6, 9 on the 59 x 59 blocks.  Returns dict(H_T, scores, best, gains (C, N))."""
    prior = np.ones(L) if prior is None else np.asarray(prior, dtype=np.float64)
    H_T = np.zeros((scene.N, LB))
    for cam in np.atleast_1d(train_cams):
        view_hessian(scene, cam, k45, out=H_T)
    conf = orc.confidence(scene.obj_logits, scene.opacity, alpha_obj, alpha_opa, target)
    gains = [orc.gaussian_gains_L(H_T, view_hessian(scene, cam, k45), conf, prior, L) for cam in np.atleast_1d(cand_cams)]
    scores = np.array([g.sum() for g in gains])
    return dict(H_T=H_T, scores=scores, best=orc.argmax_lowest(scores), gains=np.array(gains))
