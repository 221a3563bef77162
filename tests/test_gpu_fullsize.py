"""GPU-vs-oracle parity at BASELINE.json's full sizes, through the calls and in the launch configuration bench.py times
(nbv_score_candidates with several views in flight), plus the structure the two-level binning adds.

The oracle walks every Gaussian at every pixel, so at full size it is run on ONE or TWO views per config (tens of
seconds on the box's host cores) or on a pixel sample; everything else is checked through properties that hold at
any size.  Tolerances are the ones of B: north_star (see test_gpu_parity.py).
"""
import numpy as np
import pytest

from oracle import nbv_oracle as orc
from paper_2602_08266_b200 import synth
from conftest import make_oracle_scene
from test_gpu_parity import _nbv, block_rel_err

pytestmark = pytest.mark.gpu


def _pixel_sample(W, H, n, seed, full_tiles=((0, 0),)):
    """random pixels + a few complete 16x16 tiles (so that whole-tile behaviour is covered too)"""
    rng = np.random.default_rng(seed)
    m = np.zeros((H, W), dtype=np.uint8)
    m.reshape(-1)[rng.choice(W * H, size=n, replace=False)] = 1
    for tx, ty in full_tiles:
        m[ty * 16:(ty + 1) * 16, tx * 16:(tx + 1) * 16] = 1
    return m


def _check_sampled_render(nbv, scn, cam, mask):
    ro = scn.render(cam, pixel_mask=mask)
    rg = {k: v.cpu().numpy() for k, v in nbv.render(cam).items()}
    sel = mask.astype(bool)
    np.testing.assert_array_equal(rg["ncontrib"][sel], ro["ncontrib"][sel])                       # bit-exact
    np.testing.assert_array_equal(rg["T"][sel].view(np.uint32), ro["T32"][sel].view(np.uint32))   # decision path
    np.testing.assert_allclose(rg["rgb"][sel], ro["rgb"][sel], rtol=0, atol=1e-5)
    np.testing.assert_allclose(rg["depth"][sel], ro["depth"][sel], rtol=0, atol=1e-5)
    return rg


def _check_walk_invariants(nbv, cam):
    """what S3 walked is a prefix of each tile list that reaches the last composited entry of every pixel"""
    W, H = int(cam["width"]), int(cam["height"])
    walked, last = [t.cpu().numpy() for t in nbv.tile_walk(cam)]
    tx, ty = (W + 15) // 16, (H + 15) // 16
    pad = np.zeros((ty * 16, tx * 16), dtype=last.dtype)
    pad[:H, :W] = last
    tile_max = pad.reshape(ty, 16, tx, 16).max(axis=(1, 3)).reshape(-1)
    assert np.all(tile_max <= walked)
    off, _ = nbv.tile_lists(cam)
    lens = np.diff(off.cpu().numpy())
    assert np.all(walked <= lens)          # the ellipse test only removes entries: never longer than the R-5 list
    return walked, lens


def _block_properties(Hg, quat):
    """symmetric by construction (packed); PSD; exact null vector (0,..,q_hat,..,0) of R-10"""
    F = orc.unpack_blocks(Hg)
    touched = np.abs(Hg).sum(axis=1) > 0
    Ft = F[touched]
    tr = np.einsum("nii->n", Ft)
    ev = np.linalg.eigvalsh(Ft)
    assert np.all(ev[:, 0] >= -2e-5 * tr), float((ev[:, 0] / tr).min())
    qh = quat[touched] / np.linalg.norm(quat[touched], axis=1, keepdims=True)
    v = np.zeros((Ft.shape[0], 14))
    v[:, 6:10] = qh
    nq = np.sqrt(np.maximum(np.einsum("ni,nij,nj->n", v, Ft, v), 0))
    assert np.all(nq <= 2e-3 * np.sqrt(tr) + 1e-3), float((nq / np.sqrt(tr)).max())
    return int(touched.sum())


def test_cfg0_scene_on_a_multi_supertile_image():
    """2,000 Gaussians seen at 304 x 200 (19 x 13 tiles -> 3 x 2 supertiles, ragged right and bottom): lists, images, blocks"""
    wl = synth.make_workload(0)
    cam = synth.hemisphere_cameras(1, (0.6, 0.6), 304, 200, 260.0, 260.0, np.random.default_rng(11))[0]
    scn = make_oracle_scene(wl.scene, channel_mask=15)
    nbv = _nbv(wl.scene, channel_mask=15)
    off_o, ids_o = scn.tile_lists(cam)
    off_g, ids_g = [t.cpu().numpy() for t in nbv.tile_lists(cam)]
    np.testing.assert_array_equal(off_g, off_o)
    np.testing.assert_array_equal(ids_g, ids_o)
    _check_sampled_render(nbv, scn, cam, np.ones((200, 304), dtype=np.uint8))
    walked, lens = _check_walk_invariants(nbv, cam)
    assert walked.sum() < lens.sum()
    Ho = scn.view_hessian(cam)
    Hg = nbv.view_hessian(cam).cpu().numpy().astype(np.float64)
    np.testing.assert_array_equal(np.abs(Hg).sum(axis=1) > 0, np.abs(Ho).sum(axis=1) > 0)
    assert block_rel_err(Hg, Ho).max() < 1e-3


def test_cfg1_scoring_call_matches_the_oracle():
    """config 1 (50,000 Gaussians, 640 x 480): the timed call itself, 2 training views + 3 candidates in flight together"""
    wl = synth.make_workload(1)
    scn = make_oracle_scene(wl.scene)
    nbv = _nbv(wl.scene)
    train, cand = wl.train_cams[:2], wl.cand_cams[:3]
    nbv.accumulate_training(train)
    res = orc.score_candidates(scn, train, cand)
    HT = nbv.training_hessian().cpu().numpy().astype(np.float64)
    assert block_rel_err(HT, res["H_T"]).max() < 1e-3
    scores, best = nbv.score_candidates(cand)
    np.testing.assert_allclose(scores.cpu().numpy(), res["scores"], rtol=1e-3, atol=1e-6)
    assert int(best.item()) == res["best"]
    # the number of views in flight changes nothing but the order of S4's binary32 reductions
    nbv.set_concurrency(1)
    s1, b1 = nbv.score_candidates(cand)
    np.testing.assert_allclose(s1.cpu().numpy(), scores.cpu().numpy(), rtol=1e-5)
    assert int(b1.item()) == int(best.item())
    _check_walk_invariants(nbv, cand[0])


@pytest.fixture(scope="module")
def wl2():
    return synth.make_workload(2)


def test_cfg2_sampled_pixels_and_walk(wl2):
    """config 2 (200,000 Gaussians, 1280 x 720): 3,000 random pixels + 3 whole tiles of one candidate, bit-exact counts"""
    scn = make_oracle_scene(wl2.scene, channel_mask=15)
    nbv = _nbv(wl2.scene, channel_mask=15)
    cam = wl2.cand_cams[7]
    mask = _pixel_sample(1280, 720, 3000, 2, full_tiles=((40, 22), (0, 44), (79, 0)))
    rg = _check_sampled_render(nbv, scn, cam, mask)
    st = nbv.last_view_stats()
    assert st["n_pairs"] == int(rg["ncontrib"].sum())
    walked, lens = _check_walk_invariants(nbv, cam)
    assert walked.sum() == st["n_entries"] and lens.sum() == st["n_keys"]
    assert walked.sum() < 0.05 * lens.sum()      # the dense-fog structure the lazy lists exploit


def _full_view_check(wl, target):
    """H_T of one training view, every block of one candidate, its per-Gaussian gains and the score of the scoring call"""
    scn = make_oracle_scene(wl.scene, channel_mask=wl.channel_mask)
    nbv = _nbv(wl.scene, channel_mask=wl.channel_mask)
    train, cand = wl.train_cams[:1], wl.cand_cams[3:4]
    nbv.accumulate_training(train)
    # the oracle's hot path written out (oracle.score_candidates without a second pass over the candidate)
    HTo = scn.view_hessian(train[0])
    Ho = scn.view_hessian(cand[0])
    conf = orc.confidence(wl.scene.obj_logits, wl.scene.opacity, target=target)
    go = orc.gaussian_gains(HTo, Ho, conf, np.ones(14))
    res = dict(H_T=HTo, conf=conf, gains=[go], scores=np.array([go.sum()]), best=0)
    HT = nbv.training_hessian().cpu().numpy().astype(np.float64)
    assert block_rel_err(HT, res["H_T"]).max() < 1e-3
    Hg = nbv.view_hessian(cand[0]).cpu().numpy().astype(np.float64)
    np.testing.assert_array_equal(np.abs(Hg).sum(axis=1) > 0, np.abs(Ho).sum(axis=1) > 0)
    assert block_rel_err(Hg, Ho).max() < 1e-3
    assert _block_properties(Hg, wl.scene.quat) == nbv.last_view_stats()["n_touched"]
    scores, best = nbv.score_candidates(cand, target_obj=target)
    np.testing.assert_allclose(scores.cpu().numpy(), res["scores"], rtol=1e-3, atol=1e-6)
    assert int(best.item()) == res["best"]
    # per-Gaussian terms: the tolerance of B: north_star, every Gaussian
    g = nbv.gaussian_gains(cand[0], target_obj=target).cpu().numpy()
    go = res["gains"][0]
    np.testing.assert_allclose(g, go, rtol=1e-3, atol=1e-6)
    return nbv, res, g


def test_cfg2_full_view_blocks_and_gains(wl2):
    """config 2: whole-scene gain, RGB + depth Jacobians, every one of the 200,000 blocks of one candidate"""
    _full_view_check(wl2, -1)


def test_cfg3_object_centric_full_view():
    """config 3: the gain restricted to the (small, partly occluded) target object, Eq. 12"""
    wl3 = synth.make_workload(3)
    assert wl3.target_obj >= 0
    nbv, res, g = _full_view_check(wl3, int(wl3.target_obj))
    conf = nbv.confidence(int(wl3.target_obj)).cpu().numpy()
    np.testing.assert_array_equal(conf == 0, res["conf"] == 0)
    assert np.all(g[res["conf"] == 0] == 0)          # non-target Gaussians contribute exactly 0
    assert (res["conf"] > 0).sum() < 0.2 * len(conf)


def test_cfg4_full_view_blocks_and_gains():
    """config 4 (1,000,000 Gaussians, dense small splats, RGB): H_T of one training view, every block of one candidate, its
    per-Gaussian gains and the score, against the oracle"""
    _full_view_check(synth.make_workload(4), -1)


def test_cfg4_sampled_pixels_and_block_properties():
    """config 4 (1,000,000 Gaussians, dense small splats): 1,500 random pixels + 2 tiles bit-exact; block invariants"""
    wl = synth.make_workload(4)
    scn = make_oracle_scene(wl.scene)
    nbv = _nbv(wl.scene)
    cam = wl.cand_cams[100]
    mask = _pixel_sample(1280, 720, 1500, 4, full_tiles=((33, 20), (5, 40)))
    _check_sampled_render(nbv, scn, cam, mask)
    _check_walk_invariants(nbv, cam)
    Hg = nbv.view_hessian(cam).cpu().numpy().astype(np.float64)
    assert _block_properties(Hg, wl.scene.quat) == nbv.last_view_stats()["n_touched"]
    # repeatability of the scoring call across views in flight
    cands = wl.cand_cams[:6]
    s4, b4 = nbv.score_candidates(cands)
    nbv.set_concurrency(1)
    s1, b1 = nbv.score_candidates(cands)
    # the order of S4's cross-tile red.global.add.f64 is all that varies with the number of views in flight
    np.testing.assert_allclose(s4.cpu().numpy(), s1.cpu().numpy(), rtol=1e-9)       # see test_gpu_golden.py on the bound
    assert int(b4.item()) == int(b1.item())


@pytest.mark.parametrize("W,H,f", [(1296, 1104, 1100.0), (2576, 1680, 2200.0)])
def test_large_supertile_grids(W, H, f):
    """Grids of more than 64 supertiles (1296 x 1104: 11 x 9 = 99 of 8 x 8 tiles -- the comparison path of the multi-split)
    and of more than 256 at 8 x 8 (2576 x 1680: 161 x 105 tiles -> supertiles of 16 x 16 tiles, 11 x 7): tile lists
    bit-exact, blocks and gains against the oracle."""
    wl = synth.make_workload(0)
    cam = synth.hemisphere_cameras(1, (0.6, 0.6), W, H, f, f, np.random.default_rng(13))[0]
    scn = make_oracle_scene(wl.scene)
    nbv = _nbv(wl.scene)
    off_o, ids_o = scn.tile_lists(cam)
    off_g, ids_g = [t.cpu().numpy() for t in nbv.tile_lists(cam)]
    np.testing.assert_array_equal(off_g, off_o)
    np.testing.assert_array_equal(ids_g, ids_o)
    Ho = scn.view_hessian(cam)
    Hg = nbv.view_hessian(cam).cpu().numpy().astype(np.float64)
    np.testing.assert_array_equal(np.abs(Hg).sum(axis=1) > 0, np.abs(Ho).sum(axis=1) > 0)
    assert block_rel_err(Hg, Ho).max() < 1e-3
    nbv.accumulate_training(wl.train_cams)
    ref = orc.score_candidates(scn, wl.train_cams, np.array([cam]))
    s, _ = nbv.score_candidates(np.array([cam]))
    np.testing.assert_allclose(s.cpu().numpy(), ref["scores"], rtol=1e-3)
