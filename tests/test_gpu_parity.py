"""GPU-vs-oracle parity through the C ABI (B: north_star tolerances).

  tile lists, depth order, per-pixel contributor counts, projected splats : bit-exact
  rendered colour / depth / transmittance                                  : 1e-5 abs
  Hessian blocks                                                           : 1e-3 relative (1e-6 abs floor)
  information gains                                                        : 1e-3 relative (1e-6 abs floor)
  chosen next-best-view index                                              : identical

"Relative" for a block entry (k,l) is taken against sqrt(H_kk H_ll), the Cauchy-Schwarz scale of that entry
(off-diagonal entries are sums with cancellation; their own magnitude is not a scale).
"""
import numpy as np
import pytest

from oracle import nbv_oracle as orc
from paper_2602_08266_b200 import synth
from conftest import make_oracle_scene, scene_from_arrays

pytestmark = pytest.mark.gpu

P, NB = 14, 105


def _nbv(scene, channel_mask=7, **kw):
    from paper_2602_08266_b200 import api
    n = api.NBV(channel_mask=channel_mask, **kw)
    n.load_scene(scene)
    return n


def block_rel_err(Hg, Ho):
    """max over entries of |Hg - Ho| / (sqrt(Ho_kk Ho_ll) + floor), per Gaussian"""
    Fo = orc.unpack_blocks(Ho)
    d = np.sqrt(np.maximum(np.einsum("nii->ni", Fo), 0))
    scale = orc.pack_blocks(d[:, :, None] * d[:, None, :])
    return np.abs(Hg - Ho) / (scale + 1e-6 / 1e-3)


CASES = [
    # (scene builder, camera builder, channel mask)
    ("cfg0_train", lambda: synth.make_workload(0), 7),
    ("cfg0_rgbd", lambda: synth.make_workload(0), 15),
]


def _ragged_camera():
    # 70 x 50: ragged right / bottom tiles (5 x 4 tiles, the last ones partly outside the image)
    return synth.hemisphere_cameras(1, (0.6, 0.6), 70, 50, 60.0, 60.0, np.random.default_rng(5))[0]


@pytest.fixture(scope="module")
def wl():
    return synth.make_workload(0)


@pytest.mark.parametrize("which", ["train0", "cand2", "ragged"])
def test_projection_order_and_tile_lists_bit_exact(wl, which):
    cam = {"train0": wl.train_cams[0], "cand2": wl.cand_cams[2], "ragged": _ragged_camera()}[which]
    scn = make_oracle_scene(wl.scene)
    nbv = _nbv(wl.scene)
    vis_o, rec_o, rect_o = scn.project(cam)
    vis_g, rec_g, rect_g = [t.cpu().numpy() for t in nbv.projected(cam)]
    np.testing.assert_array_equal(vis_g, vis_o)
    v = vis_o > 0
    np.testing.assert_array_equal(rec_g[v].view(np.uint32), rec_o[v].view(np.uint32))  # bit-exact floats
    np.testing.assert_array_equal(rect_g[v], rect_o[v])
    off_o, ids_o = scn.tile_lists(cam)
    off_g, ids_g = [t.cpu().numpy() for t in nbv.tile_lists(cam)]
    np.testing.assert_array_equal(off_g, off_o)
    np.testing.assert_array_equal(ids_g, ids_o)
    st = nbv.last_view_stats()
    assert st["n_visible"] == int(v.sum()) and st["n_keys"] == len(ids_o)


@pytest.mark.parametrize("which,mask", [("train0", 7), ("cand1", 15), ("ragged", 15)])
def test_render_and_contributor_counts(wl, which, mask):
    cam = {"train0": wl.train_cams[0], "cand1": wl.cand_cams[1], "ragged": _ragged_camera()}[which]
    bg = (0.2, 0.4, 0.6)
    scn = make_oracle_scene(wl.scene, channel_mask=mask, bg=bg)
    nbv = _nbv(wl.scene, channel_mask=mask, bg=bg)
    ro = scn.render(cam)
    rg = {k: v.cpu().numpy() for k, v in nbv.render(cam).items()}
    np.testing.assert_array_equal(rg["ncontrib"], ro["ncontrib"])                       # bit-exact
    np.testing.assert_array_equal(rg["T"].view(np.uint32), ro["T32"].view(np.uint32))   # decision-path transmittance
    np.testing.assert_allclose(rg["rgb"], ro["rgb"], rtol=0, atol=1e-5)
    np.testing.assert_allclose(rg["depth"], ro["depth"], rtol=0, atol=1e-5)
    assert nbv.last_view_stats()["n_pairs"] == int(ro["ncontrib"].sum())


@pytest.mark.parametrize("which,mask,coord", [("train0", 7, 0), ("cand3", 15, 0), ("ragged", 15, 1), ("cand0", 8, 0)])
def test_view_hessian_blocks(wl, which, mask, coord):
    cam = {"train0": wl.train_cams[0], "cand3": wl.cand_cams[3], "cand0": wl.cand_cams[0], "ragged": _ragged_camera()}[which]
    kw = dict(bg=(0.1, 0.2, 0.3), opacity_coord=coord, channel_weight=(1.0, 0.5, 2.0, 3.0))
    scn = make_oracle_scene(wl.scene, channel_mask=mask, **kw)
    nbv = _nbv(wl.scene, channel_mask=mask, **kw)
    Ho = scn.view_hessian(cam)
    Hg = nbv.view_hessian(cam).cpu().numpy().astype(np.float64)
    touched_o = np.abs(Ho).sum(axis=1) > 0
    touched_g = np.abs(Hg).sum(axis=1) > 0
    np.testing.assert_array_equal(touched_g, touched_o)
    err = block_rel_err(Hg, Ho)
    assert err.max() < 1e-3, (err.max(), np.unravel_index(err.argmax(), err.shape))
    assert nbv.last_view_stats()["n_touched"] == int(touched_o.sum())


def test_training_accumulation_and_gains_and_argmax(wl):
    scn = make_oracle_scene(wl.scene)
    nbv = _nbv(wl.scene)
    # two training views (the config's one + a candidate) so that H_T is a sum
    train = np.concatenate([wl.train_cams, wl.cand_cams[3:4]])
    nbv.accumulate_training(train)
    res = orc.score_candidates(scn, train, wl.cand_cams)
    HT = nbv.training_hessian().cpu().numpy().astype(np.float64)
    assert block_rel_err(HT, res["H_T"]).max() < 1e-3
    conf = nbv.confidence(-1).cpu().numpy()
    np.testing.assert_allclose(conf, res["conf"], rtol=2e-6)
    scores, best = nbv.score_candidates(wl.cand_cams)
    scores = scores.cpu().numpy()
    np.testing.assert_allclose(scores, res["scores"], rtol=1e-3, atol=1e-6)
    assert int(best.item()) == res["best"]
    hs, hb = nbv.score_candidates_host(wl.cand_cams)
    np.testing.assert_allclose(hs, scores, rtol=1e-5)
    assert hb == res["best"]
    # per-Gaussian terms of one candidate
    g = nbv.gaussian_gains(wl.cand_cams[1]).cpu().numpy()
    go = res["gains"][1]
    assert np.all(g[go == 0] == 0)          # Gaussians the view does not touch: exactly zero
    assert np.all(g[go > 1e-6] > 0)
    np.testing.assert_allclose(g, go, rtol=1e-3, atol=1e-6)


def test_object_centric_scoring(wl):
    scn = make_oracle_scene(wl.scene)
    nbv = _nbv(wl.scene)
    nbv.accumulate_training(wl.train_cams)
    for tgt in (0, 2):
        res = orc.score_candidates(scn, wl.train_cams, wl.cand_cams, target=tgt)
        conf = nbv.confidence(tgt).cpu().numpy()
        np.testing.assert_array_equal(conf == 0, res["conf"] == 0)
        np.testing.assert_allclose(conf, res["conf"], rtol=5e-6)
        scores, best = nbv.score_candidates(wl.cand_cams, target_obj=tgt)
        np.testing.assert_allclose(scores.cpu().numpy(), res["scores"], rtol=1e-3, atol=1e-6)
        assert int(best.item()) == res["best"]
        g = nbv.gaussian_gains(wl.cand_cams[0], target_obj=tgt).cpu().numpy()
        assert np.all(g[res["conf"] == 0] == 0)  # Eq. 12: non-target Gaussians contribute exactly 0


def test_scoring_without_training_views_uses_the_prior_only(wl):
    scn = make_oracle_scene(wl.scene)
    nbv = _nbv(wl.scene)
    res = orc.score_candidates(scn, wl.train_cams[:0], wl.cand_cams[:2])
    scores, best = nbv.score_candidates(wl.cand_cams[:2])
    np.testing.assert_allclose(scores.cpu().numpy(), res["scores"], rtol=1e-3, atol=1e-6)
    assert int(best.item()) == res["best"]


def test_reset_training_and_repeatability(wl):
    nbv = _nbv(wl.scene)
    nbv.accumulate_training(wl.train_cams)
    s1, b1 = nbv.score_candidates(wl.cand_cams)
    s1 = s1.cpu().numpy().copy()
    nbv.reset_training()
    assert float(nbv.training_hessian().abs().sum()) == 0.0
    nbv.accumulate_training(wl.train_cams)
    s2, b2 = nbv.score_candidates(wl.cand_cams)
    # H_T is added up view by view and a score block by block in a fixed order; only the order of S4's cross-tile
    # red.global.add.f64 varies, and a binary64 sum of widened binary32 tile sums is exact for these data
    np.testing.assert_allclose(s2.cpu().numpy(), s1, rtol=1e-9)
    assert int(b1.item()) == int(b2.item())


# ------------------------------------------------------------------ micro scenes and edge cases
def test_micro_scenes_match_the_oracle():
    for n, seed, size in ((1, 0, 12), (2, 1, 8), (5, 3, 33)):
        sc = synth.micro_scene(n, seed)
        cam = synth.simple_camera(size, size, 40.0, dist=0.5)
        scn = make_oracle_scene(sc, channel_mask=15)
        nbv = _nbv(sc, channel_mask=15)
        ro = scn.render(cam)
        rg = {k: v.cpu().numpy() for k, v in nbv.render(cam).items()}
        np.testing.assert_array_equal(rg["ncontrib"], ro["ncontrib"])
        np.testing.assert_allclose(rg["rgb"], ro["rgb"], atol=1e-5, rtol=0)
        Ho = scn.view_hessian(cam)
        Hg = nbv.view_hessian(cam).cpu().numpy().astype(np.float64)
        assert block_rel_err(Hg, Ho).max() < 1e-3


def test_empty_view_and_all_culled():
    cam = synth.simple_camera(40, 24, 50.0, dist=0.0)
    sc = scene_from_arrays([[0, 0, -1.0], [0, 0, 0.005]], [[-3] * 3] * 2, [[1, 0, 0, 0]] * 2, [0.5, 0.5], [[1, 1, 1]] * 2)
    nbv = _nbv(sc, bg=(0.1, 0.2, 0.3))
    r = {k: v.cpu().numpy() for k, v in nbv.render(cam).items()}
    assert np.all(r["ncontrib"] == 0) and np.all(r["T"] == 1.0) and np.all(r["depth"] == 0)
    np.testing.assert_allclose(r["rgb"], np.broadcast_to(np.float32([0.1, 0.2, 0.3]), r["rgb"].shape))
    off, ids = nbv.tile_lists(cam)
    assert int(off[-1]) == 0 and ids.numel() == 0
    assert float(nbv.view_hessian(cam).abs().sum()) == 0.0
    scores, best = nbv.score_candidates([cam, cam])
    assert np.all(scores.cpu().numpy() == 0) and int(best.item()) == 0  # tie -> lowest index


def test_clamped_opaque_gaussian_and_stacked_half_alphas():
    cam = synth.simple_camera(32, 32, 100.0, dist=0.0)
    f = 100.0
    on = lambda ix, iy, z: [((ix + 0.5) - 16) * z / f, ((iy + 0.5) - 16) * z / f, z]
    # third Gaussian far enough from the stacked pair (power < -6 there) that it is alone at its centre pixel
    sc = scene_from_arrays([on(16, 16, 1.0), on(16, 16, 2.0), on(2, 2, 1.5)], [[-3] * 3] * 3, [[1, 0, 0, 0]] * 3,
                           [0.5, 0.5, 0.999999], [[1, 0, 0], [0, 1, 0], [1, 1, 1]])
    scn = make_oracle_scene(sc, channel_mask=15)
    nbv = _nbv(sc, channel_mask=15)
    r = {k: v.cpu().numpy() for k, v in nbv.render(cam).items()}
    assert 1.0 - r["T"][16, 16] == pytest.approx(0.75, abs=2e-6)
    assert 1.0 - r["T"][2, 2] == pytest.approx(0.99, abs=1e-6)
    ro = scn.render(cam)
    np.testing.assert_array_equal(r["ncontrib"], ro["ncontrib"])
    np.testing.assert_allclose(r["rgb"], ro["rgb"], atol=1e-5, rtol=0)
    Ho = scn.view_hessian(cam)
    Hg = nbv.view_hessian(cam).cpu().numpy().astype(np.float64)
    assert block_rel_err(Hg, Ho).max() < 1e-3


def test_error_codes():
    from paper_2602_08266_b200 import api
    wl = synth.make_workload(0)
    n = api.NBV()
    with pytest.raises(api.NBVError) as e:
        n.accumulate_training(wl.train_cams)
    assert e.value.status == "NBV_ERR_NOT_LOADED"
    bad = wl.scene.subset(np.arange(10))
    bad.quat[3] = 0
    with pytest.raises(api.NBVError) as e:
        n.load_scene(bad)
    assert e.value.status == "NBV_ERR_BAD_DATA"
    bad = wl.scene.subset(np.arange(10))
    bad.opacity[2] = 1.0
    with pytest.raises(api.NBVError) as e:
        n.load_scene(bad)
    assert e.value.status == "NBV_ERR_BAD_DATA"
    n.load_scene(wl.scene)
    with pytest.raises(api.NBVError) as e:
        n.score_candidates(wl.cand_cams[:0])
    assert e.value.status == "NBV_ERR_EMPTY_CANDIDATES"
    with pytest.raises(api.NBVError) as e:
        n.score_candidates(wl.cand_cams, target_obj=3)
    assert e.value.status == "NBV_ERR_UNKNOWN_TARGET"
    cam = wl.cand_cams[:1].copy()
    cam["R"][0][0] = 2.0
    with pytest.raises(api.NBVError) as e:
        n.score_candidates(cam)
    assert e.value.status == "NBV_ERR_INVALID_ARG"
    with pytest.raises(api.NBVError):
        api.NBV(alpha_min=0.001)  # below 1/255: the support bound is built for 1/255


def test_mixed_image_sizes_and_batching_do_not_change_scores(wl):
    """One scoring call over cameras of two image sizes (the batches split at every size change, the tile-order table is
    rebuilt) and with 1 / 3 / 8 views in flight gives the scores of one-camera-at-a-time calls (up to the order of the
    floating-point atomics)."""
    rng = np.random.default_rng(9)
    big = synth.hemisphere_cameras(5, (0.6, 0.6), 200, 136, 170.0, 170.0, rng)        # 13 x 9 tiles, ragged
    small = synth.hemisphere_cameras(6, (0.6, 0.6), 64, 64, 55.43, 55.43, rng)
    cams = np.concatenate([small[:2], big[:3], small[2:], big[3:]])
    nbv = _nbv(wl.scene)
    nbv.accumulate_training(wl.train_cams)
    single = np.array([float(nbv.score_candidates(cams[i:i + 1])[0].item()) for i in range(len(cams))])
    for conc in (1, 3, 8):
        nbv.set_concurrency(conc)
        s, best = nbv.score_candidates(cams)
        np.testing.assert_allclose(s.cpu().numpy(), single, rtol=2e-5)
        assert int(best.item()) == int(np.argmax(single))
    ref = orc.score_candidates(make_oracle_scene(wl.scene), wl.train_cams, cams[[2, 7]])["scores"]
    np.testing.assert_allclose(single[[2, 7]], ref, rtol=1e-3, atol=1e-6)


@pytest.mark.parametrize("mode", [1, 2])
def test_weight_modes_match_the_oracle(wl, mode):
    """R2 / R3 readings of where the confidence acts (nbv_config.weight_mode), scores, per-Gaussian gains, arg-max, and the
    cached-block greedy path under the same mode."""
    scn = make_oracle_scene(wl.scene)
    nbv = _nbv(wl.scene, weight_mode=mode)
    nbv.accumulate_training(wl.train_cams)
    ref = orc.score_candidates(scn, wl.train_cams, wl.cand_cams, weight_mode=mode)
    s, best = nbv.score_candidates(wl.cand_cams)
    np.testing.assert_allclose(s.cpu().numpy(), ref["scores"], rtol=1e-3, atol=1e-6)
    assert int(best.item()) == ref["best"]
    g = nbv.gaussian_gains(wl.cand_cams[1]).cpu().numpy()
    np.testing.assert_allclose(g, ref["gains"][1], rtol=1e-3, atol=1e-6)
    base = orc.score_candidates(scn, wl.train_cams, wl.cand_cams, weight_mode=0)["scores"]
    assert not np.allclose(ref["scores"], base, rtol=1e-3)          # the readings really differ on this scene
    order, sc = nbv.select_greedy(wl.cand_cams, 1)
    np.testing.assert_allclose(sc.cpu().numpy()[0], ref["scores"], rtol=1e-3, atol=1e-6)
    assert order[0] == ref["best"]


# ------------------------------------------------------------------ the product's own chain rule, its own prior
def test_chain_rule_against_finite_differences_of_the_librarys_own_projection(wl):
    """nbv_chain (S5's d(mx,my,a,b,c,z)/d(mu,logscale,quat), derived from the factor U of Sigma2D = U U^T + blur I) against
    central differences of nbv_projected -- the library's own binary32 forward projection, not the oracle."""
    sub = wl.scene.subset(np.arange(400))
    cam = wl.cand_cams[1]
    nbv = _nbv(sub)
    G = nbv.chain(cam).cpu().numpy().astype(np.float64)
    vis0, rec0, _ = [t.cpu().numpy() for t in nbv.projected(cam)]
    cols = [("mean", 0), ("mean", 1), ("mean", 2), ("logscale", 0), ("logscale", 1), ("logscale", 2),
            ("quat", 0), ("quat", 1), ("quat", 2), ("quat", 3)]
    steps = dict(mean=2e-3, logscale=1e-2, quat=1e-2)
    out_idx = [0, 1, 6, 7, 8]                       # mx, my, a, b, c in the nbv_projected record
    FD = np.zeros((sub.N, 5, 10))
    FDz = np.zeros((sub.N, 3))
    ok = vis0.astype(bool).copy()
    for k, (name, j) in enumerate(cols):
        h = steps[name]
        recs = []
        for sgn in (+1, -1):
            pert = sub.subset(np.arange(sub.N))
            getattr(pert, name)[:, j] += np.float32(sgn * h)
            n2 = _nbv(pert)
            v, r, _ = [t.cpu().numpy() for t in n2.projected(cam)]
            ok &= v.astype(bool)
            recs.append((r.astype(np.float64), getattr(pert, name)[:, j].astype(np.float64)))
        dx = recs[0][1] - recs[1][1]               # the step actually taken in binary32
        FD[:, :, k] = (recs[0][0][:, out_idx] - recs[1][0][:, out_idx]) / dx[:, None]
        if name == "mean":
            FDz[:, j] = (recs[0][0][:, 5] - recs[1][0][:, 5]) / dx
    assert ok.sum() > 300
    Gm, dz = G[:, :50].reshape(-1, 5, 10), G[:, 50:]
    # scale of a row of the 5 x 10 matrix per parameter group; binary32 outputs differenced over a finite step: 1%
    for grp in (slice(0, 3), slice(3, 6), slice(6, 10)):
        ref = FD[ok][:, :, grp]
        scale = np.abs(ref).max(axis=2, keepdims=True) + 1e-9 * np.abs(ref).max()
        err = np.abs(Gm[ok][:, :, grp] - ref) / scale
        # centre rows do not depend on scale / rotation: exactly zero on both sides there
        assert np.nanmax(np.where(np.abs(ref).max(axis=2, keepdims=True) > 0, err, 0)) < 2e-2, grp
    np.testing.assert_allclose(dz[ok], FDz[ok], atol=2e-3)
    assert np.all(Gm[:, 0:2, 3:] == 0)            # the centre does not move with scale or rotation
    # the raw quaternion enters through q / |q|: no first-order change along q itself (R-10)
    q = sub.quat.astype(np.float64)
    radial = np.einsum("nek,nk->ne", Gm[:, :, 6:10], q)
    assert np.abs(radial[ok]).max() <= 1e-5 * np.abs(Gm[ok][:, :, 6:10]).max()


@pytest.mark.parametrize("prior", ["1e-2", "1e-4", "nonuniform"])
def test_prior_precisions_other_than_one(wl, prior):
    """Lambda is an API parameter (R-13).  S5/S6 run in binary64, so small and non-uniform priors hold the same tolerances:
    scores, per-Gaussian gains and the arg-max against the oracle."""
    lam = {"1e-2": np.full(14, 1e-2), "1e-4": np.full(14, 1e-4),
           "nonuniform": np.array([1e4, 1e4, 1e4, 1.0, 1.0, 1.0, 0.5, 0.5, 0.5, 0.5, 1e-2, 3.0, 3.0, 3.0])}[prior]
    scn = make_oracle_scene(wl.scene, channel_mask=15)
    nbv = _nbv(wl.scene, channel_mask=15, prior_precision=lam)
    train = np.concatenate([wl.train_cams, wl.cand_cams[3:4]])
    nbv.accumulate_training(train)
    ref = orc.score_candidates(scn, train, wl.cand_cams, prior=lam)
    s, best = nbv.score_candidates(wl.cand_cams)
    np.testing.assert_allclose(s.cpu().numpy(), ref["scores"], rtol=1e-3, atol=1e-6)
    assert int(best.item()) == ref["best"]
    g = nbv.gaussian_gains(wl.cand_cams[2]).cpu().numpy()
    np.testing.assert_allclose(g, ref["gains"][2], rtol=1e-3, atol=1e-6)


def test_tile_lists_longer_than_the_handover_capacity_take_the_fallback_path():
    """S3 hands S4 the first 1,024 entries of every tile's list (kernels.h: TL_CAP); a tile that walks more is processed by
    the S4 instantiation that filters the supertile list again.  3,000 faint Gaussians (sigma = 0.006: alpha barely above
    1/255, the transmittance needs ~1,500 of them to fall below 1e-4) stacked in the middle of a 48 x 40 image make the
    central tiles do that while the outer ones stay short, at two distances: images, counts, blocks, gains and scores against the oracle."""
    rng = np.random.default_rng(77)
    n = 3000
    mean = np.c_[rng.uniform(-0.02, 0.02, n), rng.uniform(-0.02, 0.02, n), rng.uniform(-0.05, 0.05, n)]
    sc = scene_from_arrays(mean, np.full((n, 3), -2.8), np.c_[np.ones(n), rng.normal(0, 0.2, (n, 3))], np.full(n, 0.006),
                           rng.uniform(0, 1, (n, 3)))
    cams = [synth.simple_camera(48, 40, 60.0, dist=0.5), synth.simple_camera(48, 40, 60.0, dist=3.0)]
    scn = make_oracle_scene(sc, channel_mask=15)
    nbv = _nbv(sc, channel_mask=15)
    walked, _ = [t.cpu().numpy() for t in nbv.tile_walk(cams[0])]
    assert walked.max() > 1024 and walked.min() <= 1024, (walked.min(), walked.max())      # both S4 instantiations have tiles
    for cam in cams:
        ro = scn.render(cam)
        rg = {k: v.cpu().numpy() for k, v in nbv.render(cam).items()}
        np.testing.assert_array_equal(rg["ncontrib"], ro["ncontrib"])
        np.testing.assert_allclose(rg["rgb"], ro["rgb"], atol=1e-5, rtol=0)
        Ho = scn.view_hessian(cam)
        Hg = nbv.view_hessian(cam).cpu().numpy().astype(np.float64)
        np.testing.assert_array_equal(np.abs(Hg).sum(axis=1) > 0, np.abs(Ho).sum(axis=1) > 0)
        assert block_rel_err(Hg, Ho).max() < 1e-3
    nbv.accumulate_training(cams[1:])
    ref = orc.score_candidates(scn, cams[1:], cams, -1)
    s, best = nbv.score_candidates(cams)
    np.testing.assert_allclose(s.cpu().numpy(), ref["scores"], rtol=1e-3, atol=1e-6)
    assert int(best.item()) == ref["best"]


def test_views_per_batch_choice(wl):
    """nbv_batch_views: 16 views per batch unless the 2 x 16 view slots (worst-case coarse lists, binary64 moment rows) would
    take more than a sixth of the device memory; a fixed concurrency wins; bad sizes give 0."""
    nbv = _nbv(wl.scene)
    assert nbv.batch_views(64, 64) == 16 and nbv.batch_views(1280, 720) == 16       # 800 Gaussians: a few MB per slot
    assert nbv.batch_views(0, 64) == 0 and nbv.batch_views(64, -1) == 0
    nbv.set_concurrency(5)
    assert nbv.batch_views(1280, 720) == 5
    nbv.set_concurrency(0)                                                           # back to the automatic choice
    assert nbv.batch_views(1280, 720) == 16
    with pytest.raises(Exception):
        nbv.set_concurrency(17)
    # a map whose slots cannot all fit: N x 60 supertiles x 12 B of coarse capacity alone is 7.2 GB per slot at 10M Gaussians
    big = synth.make_workload(0, n_gaussians=10_000_000)
    nb = _nbv(big.scene)
    assert nb.batch_views(1280, 720) == 8 and nb.batch_views(64, 64) == 16


def test_opt_in_fused_raster_launch_gives_the_same_numbers(wl, monkeypatch):
    """NBV_FUSED_RASTER=1 runs S3 and S4 of a tile back to back in one persistent launch (raster_kernel: S4 starts from the
    registers S3 ends with).  Not the default -- it measured slower -- but it is the same arithmetic in the same order per
    (tile, Gaussian), so scores, per-Gaussian gains, blocks and H_T agree with the two-launch path to the last bits."""
    ref = _nbv(wl.scene, channel_mask=15)
    monkeypatch.setenv("NBV_FUSED_RASTER", "1")
    fus = _nbv(wl.scene, channel_mask=15)
    monkeypatch.delenv("NBV_FUSED_RASTER")
    for n in (ref, fus):
        n.accumulate_training(wl.train_cams)
    np.testing.assert_array_equal(fus.training_hessian().cpu().numpy(), ref.training_hessian().cpu().numpy())
    sr, br = ref.score_candidates(wl.cand_cams)
    sf, bf = fus.score_candidates(wl.cand_cams)
    np.testing.assert_allclose(sf.cpu().numpy(), sr.cpu().numpy(), rtol=1e-9)
    assert int(bf.item()) == int(br.item())
    cam = wl.cand_cams[1]
    np.testing.assert_array_equal(fus.view_hessian(cam).cpu().numpy(), ref.view_hessian(cam).cpu().numpy())
    np.testing.assert_allclose(fus.gaussian_gains(cam).cpu().numpy(), ref.gaussian_gains(cam).cpu().numpy(), rtol=1e-9, atol=0)
    walked_f, last_f = fus.tile_walk(cam)
    walked_r, last_r = ref.tile_walk(cam)
    np.testing.assert_array_equal(walked_f.cpu().numpy(), walked_r.cpu().numpy())
    np.testing.assert_array_equal(last_f.cpu().numpy(), last_r.cpu().numpy())


def test_packed_exp_spec_is_the_specified_exp_spec_bit_for_bit():
    """The raster kernels take the last step of exp_spec (bits(p) + (k << 23)) as p * 2^k with 2^k from
    MUFU.EX2.  That is the same binary32 number only where ex2.approx is exact at integers and the product is normal: every
    argument the decision path can see, [-80, 80] -- checked here against the oracle's exp_spec on a grid that covers the
    whole footprint range [-6, 0] densely, every integer and half-integer multiple of ln 2 neighbourhood, and the clamp range."""
    import torch
    from paper_2602_08266_b200 import api
    rng = np.random.default_rng(3)
    ln2 = np.log(2.0)
    x = np.concatenate([np.linspace(-6.0, 0.0, 40001), rng.uniform(-80.0, 80.0, 20000), rng.uniform(-6.0, 0.0, 20000),
                        (np.arange(-115, 116)[:, None] * ln2 + np.linspace(-1e-4, 1e-4, 21)[None, :]).ravel(),
                        ((np.arange(-115, 116)[:, None] + 0.5) * ln2 + np.linspace(-1e-4, 1e-4, 21)[None, :]).ravel(),
                        [0.0, -0.0, -80.0, 80.0, -5.5412635, 1e-30, -1e-30]]).astype(np.float32)
    x = x[(x >= -80.0) & (x <= 80.0)]
    y = api.exp_spec_pairs(torch.as_tensor(x, device="cuda")).cpu().numpy()
    ref = orc.exp_spec(x)
    assert np.array_equal(y.view(np.uint32), ref.view(np.uint32)), int((y.view(np.uint32) != ref.view(np.uint32)).sum())
    # a parked pixel: -inf and NaN arguments give NaN, which fails every `>= alpha_min` test
    bad = api.exp_spec_pairs(torch.tensor([-np.inf, np.nan, 0.0], device="cuda")).cpu().numpy()
    assert np.isnan(bad[0]) and np.isnan(bad[1]) and bad[2] == 1.0
