"""CPU oracle, alternative selection criteria.  TEST INFRASTRUCTURE -- same rules as nbv_oracle.py (only tests/,
__graft_entry__.smoke() and bench.py's oracle legs may import this; nothing shared with the CUDA path).

PAPER.md L199 (section III.B.1, before Eq. 6): "Several choices exist for f such as the trace-based trace(H^-1)^-1 or the
determinant det(H) of the Hessian, but we adopt the log-determinant log(det(H))"; L739 (section IV.A.2): the T- / D-optimality
criteria of the comparison systems.  With Eq. 5, IG(T,c) = f(T u c) - f(T), the block-diagonal H of L210 and the
confidence / prior of readings R-13, R-14 (H_V := blockdiag_g(c_g H_V,g + Lambda); weight_mode 0 only):

  trace:  f(V) = 1 / trace(H_V^-1) = 1 / sum_g trace((c_g H_V,g + Lambda)^-1)         -- the sum runs over ALL Gaussians
          IG   = 1 / (S_T - D_c) - 1 / S_T,   S_T = sum_g trace((c_g H_T,g + Lambda)^-1),
                 D_c = sum_g [trace((c_g H_T,g + Lambda)^-1) - trace((c_g (H_T,g + H_c,g) + Lambda)^-1)] >= 0
          (D_c only has terms where H_c,g != 0; IG is increasing in D_c, so arg max IG = arg max D_c)
  det:    f(V) = det(H_V) = prod_g det(c_g H_V,g + Lambda);  IG = det(H_T) (exp(L_c) - 1) with L_c the log-det gain of Eq. 6.
          det(H_T) is a product of N numbers and over- or underflows binary64 for any real map, so the criterion is carried
          in the log domain: the score is L_c = log(det(H_{T u c}) / det(H_T)), which orders the candidates exactly as the
          literal IG does (reading R-17).  `det_gain_literal` evaluates the literal difference for tiny inputs (pins).

Everything is written with numpy's dense inverse / slogdet as the library primitive.
"""
from __future__ import annotations

import numpy as np

from . import nbv_oracle as orc

LOGDET, TRACE, DET = 0, 1, 2


def _weighted(H, c, prior):
    Lam = np.diag(np.asarray(prior, dtype=np.float64))
    return np.asarray(c, dtype=np.float64)[:, None, None] * orc.unpack_blocks(H) + Lam


def trace_inverse_terms(H, c, prior) -> np.ndarray:
    """(N,) trace((c_g H_g + Lambda)^-1)"""
    return np.trace(np.linalg.inv(_weighted(H, c, prior)), axis1=1, axis2=2)


def trace_reduction(H_T, H_c, c, prior) -> np.ndarray:
    """(N,) per-Gaussian D_g = trace((c H_T + L)^-1) - trace((c (H_T + H_c) + L)^-1)  (>= 0, 0 where H_c = 0)"""
    return trace_inverse_terms(H_T, c, prior) - trace_inverse_terms(np.asarray(H_T) + np.asarray(H_c), c, prior)


def trace_gain(H_T, H_c, c, prior) -> float:
    """IG(T,c) = f(T u c) - f(T) with f = 1 / trace(H^-1) over the whole block-diagonal H (Eq. 5)"""
    S_T = trace_inverse_terms(H_T, c, prior).sum()
    return float(1.0 / (S_T - trace_reduction(H_T, H_c, c, prior).sum()) - 1.0 / S_T)


def det_gain_literal(H_T, H_c, c, prior) -> float:
    """det(H_{T u c}) - det(H_T), literally (tiny inputs only: a product over all Gaussians)"""
    d1 = np.prod(np.linalg.det(_weighted(np.asarray(H_T) + np.asarray(H_c), c, prior)))
    d0 = np.prod(np.linalg.det(_weighted(H_T, c, prior)))
    return float(d1 - d0)


def score_candidates(scene: "orc.OracleScene", train_cams, cand_cams, criterion: int, target=-1, alpha_obj=0.3, alpha_opa=0.3,
                     prior=None, H_T=None):
    """The hot path under another criterion.  Returns dict(scores (C,), best, terms (C, N): the per-Gaussian terms whose sum
    (log-det gain, or trace reduction D_g) determines the score)."""
    prior = np.ones(orc.P) if prior is None else np.asarray(prior, dtype=np.float64)
    if H_T is None:
        H_T = np.zeros((scene.N, orc.NB))
        for cam in np.atleast_1d(train_cams):
            scene.view_hessian(cam, out=H_T)
    conf = orc.confidence(scene.obj_logits, scene.opacity, alpha_obj, alpha_opa, target)
    scores, terms = [], []
    S_T = trace_inverse_terms(H_T, conf, prior).sum() if criterion == TRACE else None
    for cam in np.atleast_1d(cand_cams):
        H_c = scene.view_hessian(cam)
        if criterion == TRACE:
            d = trace_reduction(H_T, H_c, conf, prior)
            terms.append(d)
            scores.append(1.0 / (S_T - d.sum()) - 1.0 / S_T)
        else:                       # LOGDET, and DET in the log domain (R-17)
            g = orc.gaussian_gains(H_T, H_c, conf, prior)
            terms.append(g)
            scores.append(g.sum())
    scores = np.array(scores)
    return dict(scores=scores, best=orc.argmax_lowest(scores), terms=np.array(terms), S_T=S_T)
