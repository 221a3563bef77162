"""Pins of the oracle's per-output normalisation / fusion (Eq. 10-11) and greedy selection (Eq. 5 repeated)."""
import numpy as np
import pytest

from conftest import make_oracle_scene
from oracle import nbv_oracle as orc
from paper_2602_08266_b200 import synth


def _small_workload(n_train=3, n_cand=4):
    wl = synth.make_workload(0, n_gaussians=300)
    c = synth.CONFIGS[0]
    f = synth._intrinsics(c)
    rng = np.random.default_rng(77)
    wl.train_cams = synth.hemisphere_cameras(n_train, c["radius"], 32, 32, f / 2, f / 2, rng)
    wl.cand_cams = synth.hemisphere_cameras(n_cand, c["radius"], 32, 32, f / 2, f / 2, rng)
    return wl


def test_fusion_weight_defaults_are_the_papers():
    import inspect, json, os
    gold = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "spec_examples.json")))["fusion_weights"]
    sig = inspect.signature(orc.fused_gain3).parameters
    assert sig["beta_d"].default == gold["beta_d"] and sig["beta_o"].default == gold["beta_o"]
    assert inspect.signature(orc.score_candidates_fused).parameters["beta_d"].default == gold["beta_d"]


def test_normalized_and_fused_gain_hand_numbers():
    # Eq. 10: 3 / mean(1, 2, 3) = 1.5 ; Eq. 11 with beta_d = 10: 0.5 + 10 * 0.2 = 2.5
    assert orc.normalized_gain(3.0, [1.0, 2.0, 3.0]) == pytest.approx(1.5, abs=1e-15)
    assert orc.fused_gain(0.5, 0.2, 10.0) == pytest.approx(2.5, abs=1e-15)
    tg = np.array([0.3, 1.7, 4.0, 2.2])
    assert orc.normalized_gain(tg, tg).mean() == pytest.approx(1.0, abs=1e-15)      # "a typical training view has unit gain"


def test_training_views_as_candidates_have_unit_mean_per_output():
    wl = _small_workload()
    s_rgb, s_d = make_oracle_scene(wl.scene, 7), make_oracle_scene(wl.scene, 8)
    r = orc.score_candidates_fused(s_rgb, s_d, wl.train_cams, wl.train_cams)
    assert r["normalized"].mean(axis=1) == pytest.approx([1.0, 1.0], abs=1e-12)
    assert r["fused"].mean() == pytest.approx(11.0, abs=1e-10)                      # 1 + beta_d * 1
    assert np.all(r["raw"] > 0) and np.all(r["denom"] > 0)


def test_fusion_limits_and_ranking():
    wl = _small_workload()
    s_rgb, s_d = make_oracle_scene(wl.scene, 7), make_oracle_scene(wl.scene, 8)
    r0 = orc.score_candidates_fused(s_rgb, s_d, wl.train_cams, wl.cand_cams, beta_d=0.0)
    plain = orc.score_candidates(s_rgb, wl.train_cams, wl.cand_cams)
    assert r0["raw"][0] == pytest.approx(plain["scores"], rel=1e-12)                # the rgb output alone is the plain path
    assert r0["best"] == plain["best"]                                               # a positive rescaling keeps the arg-max
    r = orc.score_candidates_fused(s_rgb, s_d, wl.train_cams, wl.cand_cams, beta_d=10.0)
    assert r["fused"] == pytest.approx(r["raw"][0] / r["denom"][0] + 10.0 * r["raw"][1] / r["denom"][1], rel=1e-12)
    big = orc.score_candidates_fused(s_rgb, s_d, wl.train_cams, wl.cand_cams, beta_d=1e9)
    assert big["best"] == int(np.argmax(r["raw"][1]))                                # depth dominates as beta_d grows


def test_depth_only_block_lives_in_the_11x11_geometry_subblock():
    """L248: depth uses position, scale, rotation, opacity only -> colour rows are zero, and the 14x14 log-det gain
    with the prior equals the gain of the 11x11 sub-block (the colour prior cancels)."""
    wl = _small_workload()
    s_d = make_oracle_scene(wl.scene, 8)
    H_T = s_d.view_hessian(wl.train_cams[0])
    H_c = s_d.view_hessian(wl.cand_cams[0])
    full_T, full_c = orc.unpack_blocks(H_T), orc.unpack_blocks(H_c)
    assert np.all(full_T[:, 11:, :] == 0) and np.all(full_c[:, :, 11:] == 0) and np.abs(full_c).max() > 0
    conf = orc.confidence(s_d.obj_logits, s_d.opacity)
    g14 = orc.gaussian_gains(H_T, H_c, conf, np.ones(14))
    A, B = full_T[:, :11, :11], full_c[:, :11, :11]
    c = conf[:, None, None]
    g11 = np.linalg.slogdet(c * (A + B) + np.eye(11))[1] - np.linalg.slogdet(c * A + np.eye(11))[1]
    assert g14 == pytest.approx(g11, rel=1e-9, abs=1e-12)


def test_greedy_selection_rounds():
    wl = _small_workload(n_train=2, n_cand=5)
    scn = make_oracle_scene(wl.scene, 7)
    g = orc.select_greedy(scn, wl.train_cams, wl.cand_cams, rounds=3)
    order = g["order"]
    assert len(set(order.tolist())) == 3
    first = orc.score_candidates(scn, wl.train_cams, wl.cand_cams)
    assert g["scores"][0] == pytest.approx(first["scores"], rel=1e-12) and order[0] == first["best"]
    # Eq. 6: round 2 is plain scoring against the training set extended by the selected view
    ext = np.concatenate([wl.train_cams, wl.cand_cams[order[:1]]])
    second = orc.score_candidates(scn, ext, wl.cand_cams)["scores"]
    keep = np.arange(5) != order[0]
    assert g["scores"][1][keep] == pytest.approx(second[keep], rel=1e-10)
    assert np.isnan(g["scores"][1][order[0]]) and np.isnan(g["scores"][2][order[:2]]).all()
    # re-observing the selected view is worth less the second time (diminishing returns of the log-det)
    assert second[order[0]] < first["scores"][order[0]]


def test_greedy_tie_takes_the_lowest_index():
    wl = _small_workload(n_train=1, n_cand=3)
    scn = make_oracle_scene(wl.scene, 7)
    g = orc.select_greedy(scn, wl.train_cams, wl.cand_cams[[0, 0]], rounds=2)      # the same camera twice
    row = g["scores"][0]
    # the oracle sums a view's pixels band by band in a fixed order: the same camera gives the same bits, run to run
    assert row[0] == row[1]
    assert g["order"].tolist() == [0, 1]
    assert orc.argmax_lowest(np.array([1.0, 3.0, 3.0, 2.0])) == 1                  # the rule itself (R-15)
