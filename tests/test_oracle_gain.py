"""Pins for confidence (Eq. 7, 8, 12), the confidence-weighted block-diagonal log-det gain
(Eq. 5, 6, 9) and the arg-max (Eq. 5) of the oracle's numpy part."""
import json
import os

import numpy as np
import pytest

from oracle import nbv_oracle as orc
from conftest import make_oracle_scene

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "spec_examples.json")))
P, NB = 14, 105


def _rand_psd(rng, n, rank=14, scale=1.0):
    A = rng.standard_normal((n, P, rank)) * scale
    return orc.pack_blocks(np.einsum("nik,njk->nij", A, A))


# ------------------------------------------------------------------ confidence
def test_confidence_zero_exponents_give_unit_weights():
    rng = np.random.default_rng(0)
    c = orc.confidence(rng.standard_normal((50, 4)), rng.uniform(0.01, 0.99, 50), 0.0, 0.0)
    np.testing.assert_array_equal(c, 1.0)  # unweighted FisherRF recovered


def test_confidence_worked_example():
    g = GOLD["confidence_example"]
    # softmax of (0,0) = (0.5, 0.5): p_max = 0.5 ; sigma = 0.25
    c = orc.confidence(np.zeros((1, 2)), np.array([g["sigma"]]), g["alpha_obj"], g["alpha_opa"])
    assert c[0] == pytest.approx(g["value"], rel=1e-12)
    assert c[0] == pytest.approx(2 ** 0.9, rel=1e-12)


def test_confidence_object_mode():
    logits = np.array([[5.0, 0.0, 0.0], [0.0, 5.0, 0.0], [0.0, 0.0, 5.0], [1.0, 1.0, 0.0]])
    sig = np.full(4, 0.5)
    c = orc.confidence(logits, sig, 0.3, 0.3, target=1)
    assert c[0] == 0 and c[2] == 0  # Eq. 12 else-branch
    assert c[3] == 0  # tie between 0 and 1: argmax = lowest index = 0 != target
    p = np.exp(5) / (np.exp(5) + 2)
    assert c[1] == pytest.approx(p ** -0.3 * 0.5 ** -0.3, rel=1e-12)
    # target's own probability replaces the max (Eq. 12): here they coincide for Gaussian 1
    assert c[1] == pytest.approx(orc.confidence(logits, sig, 0.3, 0.3)[1], rel=1e-12)


def test_confidence_decreases_with_opacity_and_object_probability():
    sig = np.linspace(0.01, 0.99, 30)
    c = orc.confidence(np.zeros((30, 3)), sig)
    assert np.all(np.diff(c) < 0)
    lg = np.zeros((30, 3))
    lg[:, 0] = np.linspace(0.0, 6.0, 30)
    c = orc.confidence(lg, np.full(30, 0.5))
    assert np.all(np.diff(c) < 0)
    assert np.all(c > 0)  # whole-scene mode: all weights > 0


def test_confidence_floors():
    c = orc.confidence(np.zeros((1, 2)), np.array([1e-9]), 0.3, 0.3)
    assert c[0] == pytest.approx(0.5 ** -0.3 * 1e-4 ** -0.3, rel=1e-12)  # sigma floored at 1e-4


# ------------------------------------------------------------------ log-det gain
def test_gain_zero_candidate_block_is_zero():
    rng = np.random.default_rng(1)
    HT = _rand_psd(rng, 20)
    g = orc.gaussian_gains(HT, np.zeros_like(HT), np.ones(20), np.ones(P))
    np.testing.assert_allclose(g, 0.0, atol=1e-12)


def test_gain_scalar_toy_example():
    e = GOLD["scalar_gain_example"]
    HT = np.zeros((1, NB))
    Hc = np.zeros((1, NB))
    Hc[0, 0] = e["block"]  # single unit entry on the diagonal
    g = orc.gaussian_gains(HT, Hc, np.ones(1), np.full(P, e["ridge"]))
    assert g[0] == pytest.approx(e["value"], rel=1e-9)  # ln(1+1e-6) - ln(1e-6)


def test_gain_of_unobserved_gaussian_is_sum_log1p_of_scaled_eigenvalues():
    rng = np.random.default_rng(2)
    Hc = _rand_psd(rng, 10, rank=5)
    c = rng.uniform(0.5, 3.0, 10)
    lam = 0.7
    g = orc.gaussian_gains(np.zeros_like(Hc), Hc, c, np.full(P, lam))
    ev = np.linalg.eigvalsh(orc.unpack_blocks(Hc))
    want = np.log1p(np.maximum(ev, 0) * c[:, None] / lam).sum(axis=1)
    np.testing.assert_allclose(g, want, rtol=1e-9)


def test_gain_equals_dense_block_diagonal_assembly():
    rng = np.random.default_rng(3)
    n = 3
    HT, Hc = _rand_psd(rng, n, rank=9), _rand_psd(rng, n, rank=4)
    c = rng.uniform(0.5, 2.0, n)
    prior = rng.uniform(0.5, 2.0, P)
    big0 = np.zeros((n * P, n * P))
    big1 = np.zeros((n * P, n * P))
    for g in range(n):
        sl = slice(g * P, (g + 1) * P)
        big0[sl, sl] = c[g] * orc.unpack_blocks(HT[g]) + np.diag(prior)
        big1[sl, sl] = c[g] * orc.unpack_blocks(HT[g] + Hc[g]) + np.diag(prior)
    want = np.linalg.slogdet(big1)[1] - np.linalg.slogdet(big0)[1]  # Eq. 5 with Eq. 6, full matrix
    got = orc.gaussian_gains(HT, Hc, c, prior).sum()
    assert got == pytest.approx(want, abs=1e-8)


def test_gain_diag_example_and_monotonicity():
    e = GOLD["diag_logdet_example"]
    # block = diag(1,2,4,0,...): log det(B + I) - log det(I) = ln 2 + ln 3 + ln 5
    Hc = np.zeros((1, P, P))
    Hc[0, 0, 0], Hc[0, 1, 1], Hc[0, 2, 2] = e["diag"]
    g = orc.gaussian_gains(np.zeros((1, NB)), orc.pack_blocks(Hc), np.ones(1), np.ones(P))
    assert g[0] == pytest.approx(np.log(2 * 3 * 5), rel=1e-12)
    rng = np.random.default_rng(4)
    HT, Hc = _rand_psd(rng, 200, rank=6), _rand_psd(rng, 200, rank=3)
    g = orc.gaussian_gains(HT, Hc, rng.uniform(0, 2, 200), np.ones(P))
    assert np.all(g >= -1e-9)


def test_zero_confidence_gives_exactly_zero_gain():
    rng = np.random.default_rng(5)
    HT, Hc = _rand_psd(rng, 5), _rand_psd(rng, 5)
    g = orc.gaussian_gains(HT, Hc, np.zeros(5), np.ones(P))
    assert np.all(g == 0.0)  # Eq. 12: non-target Gaussians contribute exactly 0


def test_pack_unpack_roundtrip_and_order():
    F = np.arange(P * P, dtype=float).reshape(P, P)
    F = F + F.T
    pk = orc.pack_blocks(F[None])[0]
    assert pk.shape == (NB,)
    for r in range(P):
        for c in range(r, P):
            assert pk[r * P - r * (r - 1) // 2 + (c - r)] == F[r, c]
    np.testing.assert_array_equal(orc.unpack_blocks(pk[None])[0], F)


# ------------------------------------------------------------------ arg-max and the whole path
def test_argmax_lowest_index_on_ties():
    assert orc.argmax_lowest([1.0]) == 0
    assert orc.argmax_lowest([1.0, 3.0, 3.0, 2.0]) == 1
    assert orc.argmax_lowest([-1.0, -1.0]) == 0


def test_score_candidates_properties(wl0):
    scn = make_oracle_scene(wl0.scene)
    res = orc.score_candidates(scn, wl0.train_cams, wl0.cand_cams)
    assert res["scores"].shape == (4,) and np.all(res["scores"] > 0)
    assert res["best"] == int(np.argmax(res["scores"]))
    assert np.all(res["gains"] >= -1e-9)
    # a duplicate of the training view still has strictly positive gain
    dup = orc.score_candidates(scn, wl0.train_cams, wl0.train_cams[:1], H_T=res["H_T"])
    assert dup["scores"][0] > 0
    # object-centric: only Gaussians whose argmax is the target contribute (Eq. 12)
    tgt = 1
    rt = orc.score_candidates(scn, wl0.train_cams, wl0.cand_cams, target=tgt, H_T=res["H_T"])
    am = orc.softmax(wl0.scene.obj_logits).argmax(axis=1)
    assert np.all(rt["gains"][:, am != tgt] == 0)
    assert np.all(rt["scores"] < res["scores"])
    # whole-scene machinery with the non-target confidences forced to 0 gives the same scores
    c_forced = np.where(am == tgt, rt["conf"], 0.0)
    for i, cam in enumerate(wl0.cand_cams):
        g = orc.gaussian_gains(res["H_T"], scn.view_hessian(cam), c_forced, np.ones(P))
        assert g.sum() == pytest.approx(rt["scores"][i], rel=1e-9)


def test_weight_modes_closed_forms_and_limits():
    """Where the confidence acts (reading R-14): scalar closed forms on a block a e1 e1^T + candidate b e1 e1^T, lambda = 1."""
    a, b, c = 3.0, 5.0, 1.7
    H_T = np.zeros((1, orc.NB)); H_c = np.zeros((1, orc.NB))
    H_T[0, 0], H_c[0, 0] = a, b
    one = np.ones(14)
    g0 = orc.gaussian_gains(H_T, H_c, [c], one, 0)[0]
    g1 = orc.gaussian_gains(H_T, H_c, [c], one, 1)[0]
    g2 = orc.gaussian_gains(H_T, H_c, [c], one, 2)[0]
    assert g0 == pytest.approx(np.log((c * (a + b) + 1) / (c * a + 1)), rel=1e-12)     # Eq. 9 literal
    assert g1 == pytest.approx(c * np.log((a + b + 1) / (a + 1)), rel=1e-12)          # c weights the gain
    assert g2 == pytest.approx(np.log((a + c * b + 1) / (a + 1)), rel=1e-12)          # c weights the candidate only
    rng = np.random.default_rng(0)
    X = rng.standard_normal((5, 14, 20)); Y = rng.standard_normal((5, 14, 6))
    HT, HC = orc.pack_blocks(X @ X.transpose(0, 2, 1)), orc.pack_blocks(Y @ Y.transpose(0, 2, 1))
    ones = np.ones(5)
    ref = orc.gaussian_gains(HT, HC, ones, one, 0)
    for m in (1, 2):
        np.testing.assert_allclose(orc.gaussian_gains(HT, HC, ones, one, m), ref, rtol=1e-12)    # c = 1: all readings agree
    cs = rng.uniform(0.5, 3.0, 5)
    np.testing.assert_allclose(orc.gaussian_gains(HT, HC, 2 * cs, one, 1), 2 * orc.gaussian_gains(HT, HC, cs, one, 1), rtol=1e-12)
    zero = np.zeros_like(HT)
    np.testing.assert_allclose(orc.gaussian_gains(zero, HC, cs, one, 0), orc.gaussian_gains(zero, HC, cs, one, 2), rtol=1e-12)
    for m in (0, 1, 2):
        assert np.all(orc.gaussian_gains(HT, HC, np.zeros(5), one, m) == 0.0)                      # c = 0 (Eq. 12): exactly zero
    assert np.all(orc.gaussian_gains(HT, HC, 2 * cs, one, 2) > orc.gaussian_gains(HT, HC, cs, one, 2))
