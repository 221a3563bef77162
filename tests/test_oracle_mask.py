"""Pins of the oracle's object-mask output (Eq. 1-2)."""
import numpy as np
import pytest

from conftest import make_oracle_scene, scene_from_arrays
from oracle import nbv_oracle as orc
from paper_2602_08266_b200 import synth


def _micro(n=4, K=3, seed=3):
    sc = synth.micro_scene(n, seed, K=K)
    rng = np.random.default_rng(seed + 50)
    sc.obj_logits[:] = rng.standard_normal((n, K)).astype(np.float32)
    return sc


def test_mask_sums_to_one_and_is_nonnegative(wl0):
    scn = make_oracle_scene(wl0.scene)
    O = orc.render_mask(scn, wl0.cand_cams[1])
    assert O.shape == (64, 64, 3)
    np.testing.assert_allclose(O.sum(axis=2), 1.0, atol=1e-12)            # Eq. 2
    assert O.min() >= 0.0
    r = scn.render(wl0.cand_cams[1])
    empty = r["ncontrib"] == 0
    assert empty.any() and np.all(O[empty] == [1.0, 0.0, 0.0])             # nothing hit: pure background channel
    # O' = O - e_bg T_end ; its channel sum is the accumulated alpha 1 - T_end (softmax sums to one)
    np.testing.assert_allclose((O.sum(axis=2) - r["T"]), 1.0 - r["T"], atol=1e-12)
    O1 = orc.render_mask(scn, wl0.cand_cams[1], bg_channel=2)
    np.testing.assert_allclose(O1[..., 2] - O[..., 2], r["T"], atol=1e-12)
    np.testing.assert_allclose(O[..., 0] - O1[..., 0], r["T"], atol=1e-12)


def test_mask_equals_rgb_compositing_of_the_probabilities():
    """With K = 3 the mask is the (already pinned) colour compositing of the 'colours' softmax(o) over the background
    colour e_0: values, and the 11 x 11 geometry sub-block of the Hessian."""
    sc = _micro(5, 3)
    cam = synth.simple_camera(24, 24, 60.0, 0.5)
    p = orc.softmax(sc.obj_logits)
    as_rgb = scene_from_arrays(sc.mean, sc.logscale, sc.quat, sc.opacity, p.astype(np.float32), K=3)
    s_mask = make_oracle_scene(sc, 7)
    s_rgb = make_oracle_scene(as_rgb, 7, bg=(1.0, 0.0, 0.0))
    O = orc.render_mask(s_mask, cam)
    np.testing.assert_allclose(O, s_rgb.render(cam)["rgb"], atol=2e-7)    # colours were rounded to binary32
    Hm = orc.unpack_blocks_L(orc.view_hessian_mask(s_mask, cam), 14)
    Hr = orc.unpack_blocks(s_rgb.view_hessian(cam))
    scale = np.abs(Hr[:, :11, :11]).max()
    assert scale > 0 and np.abs(Hm[:, :11, :11] - Hr[:, :11, :11]).max() < 1e-6 * scale


@pytest.mark.parametrize("K", [2, 5])
def test_mask_blocks_match_finite_differences(K):
    sc = _micro(3, K, seed=4 + K)
    cam = synth.simple_camera(12, 12, 30.0, 0.5)
    scn = make_oracle_scene(sc)
    offsets, ids, clamped = scn.trace(cam)
    th = scn.theta()[:, :11].copy()
    lg = sc.obj_logits.astype(np.float64)
    L = 11 + K
    N = th.shape[0]
    Han = orc.unpack_blocks_L(orc.view_hessian_mask_smooth(th, lg, cam, scn.cfg, offsets, ids, clamped), L)
    step = 1e-5
    for g in range(N):
        Jg = np.zeros((12 * 12 * K, L))
        for k in range(L):
            tp, tm, lp, lm = th.copy(), th.copy(), lg.copy(), lg.copy()
            if k < 11:
                tp[g, k] += step; tm[g, k] -= step
            else:
                lp[g, k - 11] += step; lm[g, k - 11] -= step
            d = (orc.render_mask_smooth(tp, lp, cam, scn.cfg, offsets, ids, clamped)
                 - orc.render_mask_smooth(tm, lm, cam, scn.cfg, offsets, ids, clamped)) / (2 * step)
            Jg[:, k] = d.reshape(-1)
        Hfd = Jg.T @ Jg
        assert np.linalg.norm(Han[g] - Hfd) <= 1e-6 * max(np.linalg.norm(Hfd), 1e-12), g
    # normal mode (binary32 splat, binary64 values) agrees with smooth mode
    Hn = orc.unpack_blocks_L(orc.view_hessian_mask(scn, cam), L)
    assert np.abs(Hn - Han).max() <= 1e-4 * np.abs(Han).max()


def test_mask_block_invariants(wl0):
    scn = make_oracle_scene(wl0.scene)
    K, L = 3, 14
    H = orc.unpack_blocks_L(orc.view_hessian_mask(scn, wl0.cand_cams[0]), L)
    seen = np.abs(H).max(axis=(1, 2)) > 0
    assert 0 < seen.sum() < scn.N
    ev = np.linalg.eigvalsh(H[seen])
    assert ev.min() >= -1e-9 * ev.max()                                      # PSD
    ones = np.zeros(L); ones[11:] = 1.0                                       # softmax is shift invariant
    assert np.abs(H[seen] @ ones).max() <= 1e-9 * np.abs(H[seen]).max()
    q = np.zeros((scn.N, L)); q[:, 6:10] = wl0.scene.quat                     # quaternion gauge (R-10)
    assert np.abs(np.einsum("nij,nj->ni", H, q)).max() <= 1e-7 * np.abs(H).max()
    # two identical views double the block; gain against itself is positive
    H2 = orc.view_hessian_mask(scn, wl0.cand_cams[0])
    orc.view_hessian_mask(scn, wl0.cand_cams[0], out=H2)
    np.testing.assert_allclose(orc.unpack_blocks_L(H2, L), 2 * H, rtol=1e-9, atol=1e-18)
    r = orc.score_candidates_mask(scn, wl0.train_cams, wl0.cand_cams)
    assert np.all(r["scores"] > 0) and r["best"] == int(np.argmax(r["scores"]))


def test_saturated_one_hot_logits_give_a_hard_mask_and_no_logit_information():
    sc = _micro(2, 3)
    sc.obj_logits[:] = np.array([[0, 60, 0], [0, 0, 60]], dtype=np.float32)  # p = e_1, e_2 to 1e-26
    cam = synth.simple_camera(16, 16, 40.0, 0.5)
    scn = make_oracle_scene(sc)
    O = orc.render_mask(scn, cam)
    r = scn.render(cam)
    np.testing.assert_allclose(O[..., 0], r["T"], atol=1e-12)                # background = what is left over
    H = orc.unpack_blocks_L(orc.view_hessian_mask(scn, cam), 14)
    assert np.abs(H[:, 11:, :]).max() < 1e-20 and np.abs(H[:, :11, :11]).max() > 0   # dp/do = p(delta - p) = 0


def test_three_output_fusion_hand_numbers_and_unit_mean(wl0):
    assert orc.fused_gain3(0.5, 0.2, 0.3, 10.0, 1.0) == pytest.approx(2.8, abs=1e-15)     # Eq. 11
    wl = synth.make_workload(0, n_gaussians=200)
    rng = np.random.default_rng(5)
    train = synth.hemisphere_cameras(2, (0.6, 0.6), 24, 24, 20.0, 20.0, rng)
    s7, s8, sm = make_oracle_scene(wl.scene, 7), make_oracle_scene(wl.scene, 8), make_oracle_scene(wl.scene, 7)
    r = orc.score_candidates_fused(s7, s8, train, train, scene_mask=sm)
    assert r["raw"].shape == (3, 2) and r["normalized"].mean(axis=1) == pytest.approx([1.0, 1.0, 1.0], abs=1e-12)
    assert r["fused"].mean() == pytest.approx(12.0, abs=1e-10)                            # 1 + beta_d + beta_o
    two = orc.score_candidates_fused(s7, s8, train, train)
    assert r["raw"][:2] == pytest.approx(two["raw"], rel=1e-12)
