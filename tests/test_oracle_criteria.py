"""Pins of oracle/criteria.py (the trace-based trace(H^-1)^-1 and the determinant det(H) as alternatives to
the log-determinant; Eq. 5 IG(T,c) = f(T u c) - f(T); block-diagonal H, L210).  None of them re-types the oracle's formula:
closed forms on diagonal blocks, the dense inverse / determinant of the assembled block-diagonal matrix, invariants."""
import numpy as np
import pytest
import scipy.linalg

from oracle import criteria as crit
from oracle import nbv_oracle as orc
from paper_2602_08266_b200 import synth
from conftest import make_oracle_scene


def _rand_blocks(n, rank, seed, scale=1.0):
    rng = np.random.default_rng(seed)
    J = rng.standard_normal((n, rank, 14)) * scale
    return orc.pack_blocks(np.einsum("nri,nrj->nij", J, J))


def test_trace_gain_on_diagonal_blocks_closed_form():
    # H_T = diag(a), H_c = diag(b), Lambda = diag(l): trace((c a + l)^-1) = sum 1 / (c a_i + l_i), by hand
    a = np.arange(1.0, 15.0); b = np.linspace(0.5, 2.0, 14); lam = np.full(14, 0.25); c = 2.0
    HT = orc.pack_blocks(np.diag(a)[None]); HC = orc.pack_blocks(np.diag(b)[None])
    S0 = (1.0 / (c * a + lam)).sum(); S1 = (1.0 / (c * (a + b) + lam)).sum()
    assert crit.trace_inverse_terms(HT, [c], lam)[0] == pytest.approx(S0, rel=1e-13)
    assert crit.trace_reduction(HT, HC, [c], lam)[0] == pytest.approx(S0 - S1, rel=1e-12)
    assert crit.trace_gain(HT, HC, [c], lam) == pytest.approx(1.0 / S1 - 1.0 / S0, rel=1e-12)
    # scalar toy: one parameter observed, the rest prior only
    HT1 = np.zeros((1, 105)); HC1 = np.zeros((1, 105)); HC1[0, 0] = 3.0
    assert crit.trace_gain(HT1, HC1, [1.0], np.ones(14)) == pytest.approx(1.0 / (13 + 0.25) - 1.0 / 14, rel=1e-13)


def test_trace_and_det_against_the_dense_block_diagonal_matrix():
    """3 Gaussians: assemble the 42 x 42 matrix blockdiag(c_g H_g + Lambda) and use the dense inverse / determinant"""
    HT, HC = _rand_blocks(3, 9, 1), _rand_blocks(3, 5, 2, 0.7)
    c = np.array([0.8, 1.7, 2.5]); lam = np.linspace(0.5, 1.5, 14)
    def dense(H):
        return scipy.linalg.block_diag(*[c[g] * orc.unpack_blocks(H[g]) + np.diag(lam) for g in range(3)])
    A0, A1 = dense(HT), dense(HT + HC)
    f0, f1 = 1.0 / np.trace(np.linalg.inv(A0)), 1.0 / np.trace(np.linalg.inv(A1))
    assert crit.trace_gain(HT, HC, c, lam) == pytest.approx(f1 - f0, rel=1e-10)
    assert crit.det_gain_literal(HT, HC, c, lam) == pytest.approx(np.linalg.det(A1) - np.linalg.det(A0), rel=1e-9)
    # the log-domain score of the det criterion maps onto the literal one: IG_det = det(H_T) (exp(L) - 1)
    L = orc.gaussian_gains(HT, HC, c, lam).sum()
    assert crit.det_gain_literal(HT, HC, c, lam) == pytest.approx(np.linalg.det(A0) * np.expm1(L), rel=1e-9)


def test_trace_invariants():
    HT, HC = _rand_blocks(40, 8, 3), _rand_blocks(40, 6, 4)
    HC[::3] = 0.0                                        # Gaussians the candidate does not touch
    c = np.random.default_rng(5).uniform(0.5, 3.0, 40); lam = np.ones(14)
    d = crit.trace_reduction(HT, HC, c, lam)
    assert np.all(d[::3] == 0.0) and np.all(d[HC.any(axis=1)] > 0)        # more information never raises the covariance trace
    assert crit.trace_gain(HT, HC, c, lam) > 0
    assert crit.trace_gain(HT, 0 * HC, c, lam) == 0.0
    # c_g = 0 (Eq. 12, non-target): the block is the prior alone, the candidate adds nothing there
    c0 = c.copy(); c0[:20] = 0.0
    assert np.all(crit.trace_reduction(HT, HC, c0, lam)[:20] == 0.0)
    assert crit.trace_inverse_terms(HT, c0, lam)[:20] == pytest.approx(14.0)
    # the gain is increasing in the total trace reduction: same arg-max
    cands = [_rand_blocks(40, 6, 10 + i, 0.3 + 0.2 * i) for i in range(5)]
    gains = [crit.trace_gain(HT, h, c, lam) for h in cands]
    reds = [crit.trace_reduction(HT, h, c, lam).sum() for h in cands]
    assert np.argsort(gains).tolist() == np.argsort(reds).tolist()


def test_score_candidates_under_the_criteria_on_a_small_scene():
    wl = synth.make_workload(0, n_gaussians=300)
    scn = make_oracle_scene(wl.scene)
    base = orc.score_candidates(scn, wl.train_cams, wl.cand_cams)
    det = crit.score_candidates(scn, wl.train_cams, wl.cand_cams, crit.DET)
    assert det["scores"] == pytest.approx(base["scores"], rel=1e-13) and det["best"] == base["best"]     # R-17: log domain
    tr = crit.score_candidates(scn, wl.train_cams, wl.cand_cams, crit.TRACE)
    assert np.all(tr["scores"] > 0) and tr["terms"].shape == (4, 300)
    # literal definition on the whole map, one candidate: f(T u c) - f(T) with the inverse of every block
    conf = orc.confidence(wl.scene.obj_logits, wl.scene.opacity)
    Hc = scn.view_hessian(wl.cand_cams[2])
    inv_tr = lambda H: np.trace(np.linalg.inv(conf[:, None, None] * orc.unpack_blocks(H) + np.eye(14)), axis1=1, axis2=2).sum()
    assert tr["scores"][2] == pytest.approx(1.0 / inv_tr(base["H_T"] + Hc) - 1.0 / inv_tr(base["H_T"]), rel=1e-9)
    assert tr["best"] == int(np.argmax(tr["terms"].sum(axis=1)))
