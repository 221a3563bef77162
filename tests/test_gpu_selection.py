"""GPU-vs-oracle parity of per-output normalisation + fusion (Eq. 10-11) and greedy selection through the
C ABI: raw gains, denominators, fused scores, per-round scores 1e-3 relative (1e-6 abs floor); indices identical."""
import numpy as np
import pytest

from oracle import nbv_oracle as orc
from paper_2602_08266_b200 import synth
from conftest import make_oracle_scene

pytestmark = pytest.mark.gpu


def _workload(n_train, n_cand, W=96, H=80, n_gaussians=2000, seed=0):
    wl = synth.make_workload(0, n_gaussians=n_gaussians, seed=seed)
    rng = np.random.default_rng(123 + seed)
    f = 90.0
    wl.train_cams = synth.hemisphere_cameras(n_train, (0.6, 0.6), W, H, f, f, rng)
    wl.cand_cams = synth.hemisphere_cameras(n_cand, (0.5, 0.8), W, H, f, f, rng)
    return wl


def _nbv(scene, **kw):
    from paper_2602_08266_b200 import api
    n = api.NBV(**kw)
    n.load_scene(scene)
    return n


def _ctx(scene, mask, train):
    from paper_2602_08266_b200 import api
    n = api.NBV(channel_mask=mask)
    n.load_scene(scene)
    n.accumulate_training(train)
    return n


@pytest.mark.parametrize("target", [-1, 1])
def test_fused_scores_match_the_oracle(target):
    from paper_2602_08266_b200 import api
    wl = _workload(3, 10)                       # 10 candidates: two batches are not needed, ragged 96x80 image is
    nr, nd = _ctx(wl.scene, api.CH_RGB, wl.train_cams), _ctx(wl.scene, api.CH_DEPTH, wl.train_cams)
    out = api.score_candidates_fused(nr, nd, wl.train_cams, wl.cand_cams, target, 10.0)
    ref = orc.score_candidates_fused(make_oracle_scene(wl.scene, 7), make_oracle_scene(wl.scene, 8), wl.train_cams,
                                     wl.cand_cams, target, 10.0)
    np.testing.assert_allclose(out["raw"].cpu().numpy(), ref["raw"], rtol=1e-3, atol=1e-6)
    np.testing.assert_allclose(out["denom"].cpu().numpy(), ref["denom"], rtol=1e-3, atol=1e-6)
    np.testing.assert_allclose(out["fused"].cpu().numpy(), ref["fused"], rtol=1e-3, atol=1e-6)
    assert int(out["best"].item()) == ref["best"]
    # the property of Eq. 10 on the GPU side: the training views as candidates average to 1 + beta_d
    unit = api.score_candidates_fused(nr, nd, wl.train_cams, wl.train_cams, target, 10.0)
    assert float(unit["fused"].mean().item()) == pytest.approx(11.0, rel=1e-4)


def test_fused_shared_and_separate_rasterisation_agree():
    """The RGB and the depth context share S1-S3 of every batch when they composite with the same constants (the depth
    context sweeps the tile lists S3 left again); with different constants each context rasterises for itself.  A near plane
    moved by one part in 1e5 culls the same Gaussians, so both routes must give the same numbers -- and several batches."""
    from paper_2602_08266_b200 import api
    wl = _workload(3, 20)
    nr = _ctx(wl.scene, api.CH_RGB, wl.train_cams)
    nd = _ctx(wl.scene, api.CH_DEPTH, wl.train_cams)
    nd2 = api.NBV(channel_mask=api.CH_DEPTH, near_plane=0.0100001)
    nd2.load_scene(wl.scene)
    nd2.accumulate_training(wl.train_cams)
    for n in (nr, nd, nd2):
        n.set_concurrency(8)                                             # 20 candidates: batches of 8, 8, 4 on both raster streams
    shared = api.score_candidates_fused(nr, nd, wl.train_cams, wl.cand_cams, -1, 10.0)
    separate = api.score_candidates_fused(nr, nd2, wl.train_cams, wl.cand_cams, -1, 10.0)
    for k in ("raw", "denom", "fused"):
        np.testing.assert_allclose(shared[k].cpu().numpy(), separate[k].cpu().numpy(), rtol=1e-6, atol=0)
    assert int(shared["best"].item()) == int(separate["best"].item())
    # and the contexts are left as they were: a plain scoring call on the depth context alone gives its raw row
    sd, _ = nd.score_candidates(wl.cand_cams)
    np.testing.assert_allclose(sd.cpu().numpy(), shared["raw"][1].cpu().numpy(), rtol=1e-6, atol=0)


def test_fused_argument_errors():
    from paper_2602_08266_b200 import api
    wl = _workload(1, 2, n_gaussians=200)
    nr, nd = _ctx(wl.scene, api.CH_RGB, wl.train_cams), _ctx(wl.scene, api.CH_DEPTH, wl.train_cams)
    with pytest.raises(api.NBVError) as e:
        api.score_candidates_fused(nr, nd, wl.train_cams, wl.cand_cams[:0])
    assert e.value.status == "NBV_ERR_EMPTY_CANDIDATES"
    with pytest.raises(api.NBVError) as e:
        api.score_candidates_fused(nd, nr, wl.train_cams, wl.cand_cams)            # masks swapped
    assert e.value.status == "NBV_ERR_INVALID_ARG"
    with pytest.raises(api.NBVError) as e:
        api.score_candidates_fused(nr, nd, wl.train_cams[:0], wl.cand_cams)        # Eq. 10 needs |T| >= 1
    assert e.value.status == "NBV_ERR_INVALID_ARG"
    with pytest.raises(api.NBVError) as e:
        api.score_candidates_fused(nr, nd, wl.train_cams, wl.cand_cams, target_obj=99)
    assert e.value.status == "NBV_ERR_UNKNOWN_TARGET"


@pytest.mark.parametrize("cache_mb", ["4096", "0"])      # block cache / fallback that re-rasterises every round
def test_greedy_selection_matches_the_oracle(cache_mb, monkeypatch):
    from paper_2602_08266_b200 import api
    monkeypatch.setenv("NBV_GREEDY_CACHE_MB", cache_mb)
    wl = _workload(2, 12)
    nbv = _ctx(wl.scene, api.CH_RGB, wl.train_cams)
    order, scores = nbv.select_greedy(wl.cand_cams, 4)
    ref = orc.select_greedy(make_oracle_scene(wl.scene, 7), wl.train_cams, wl.cand_cams, 4)
    assert order.tolist() == ref["order"].tolist()
    s = scores.cpu().numpy()
    assert np.array_equal(np.isnan(s), np.isnan(ref["scores"]))
    m = ~np.isnan(s)
    np.testing.assert_allclose(s[m], ref["scores"][m], rtol=1e-3, atol=1e-6)
    # H_T now holds the training views plus the four selected ones (Eq. 6)
    H = nbv.training_hessian().cpu().numpy()
    scn = make_oracle_scene(wl.scene, 7)
    Ho = np.zeros((scn.N, 105))
    for cam in list(wl.train_cams) + [wl.cand_cams[i] for i in order]:
        scn.view_hessian(cam, out=Ho)
    Fo = orc.unpack_blocks(Ho)
    d = np.sqrt(np.maximum(np.einsum("nii->ni", Fo), 0))
    scale = orc.pack_blocks(d[:, :, None] * d[:, None, :])
    assert (np.abs(H - Ho) / (scale + 1e-3)).max() < 1e-3


def test_greedy_edge_cases():
    from paper_2602_08266_b200 import api
    wl = _workload(1, 3, n_gaussians=300)
    nbv = _ctx(wl.scene, api.CH_RGB, wl.train_cams)
    order, _ = nbv.select_greedy(wl.cand_cams, 3, want_scores=False)             # rounds == n: a permutation
    assert sorted(order.tolist()) == [0, 1, 2]
    with pytest.raises(api.NBVError) as e:
        nbv.select_greedy(wl.cand_cams, 4)
    assert e.value.status == "NBV_ERR_INVALID_ARG"
    with pytest.raises(api.NBVError) as e:
        nbv.select_greedy(wl.cand_cams[:0], 1)
    assert e.value.status == "NBV_ERR_EMPTY_CANDIDATES"


# ---- alternative criteria: nbv_config.criterion
def test_trace_and_det_criteria_match_the_oracle():
    from oracle import criteria as crit
    wl = synth.make_workload(0)
    scn = make_oracle_scene(wl.scene)
    for target in (-1, 1):
        ref = crit.score_candidates(scn, wl.train_cams, wl.cand_cams, crit.TRACE, target=target)
        nbv = _nbv(wl.scene, criterion=1)
        nbv.accumulate_training(wl.train_cams)
        s, best = nbv.score_candidates(wl.cand_cams, target_obj=target)
        np.testing.assert_allclose(s.cpu().numpy(), ref["scores"], rtol=1e-3, atol=0)
        assert int(best.item()) == ref["best"]
        d = nbv.gaussian_gains(wl.cand_cams[2], target_obj=target).cpu().numpy()      # per-Gaussian trace reductions D_g
        np.testing.assert_allclose(d, ref["terms"][2], rtol=1e-3, atol=1e-9)
    # greedy selection under the trace criterion: first round = plain scoring, S_T refreshed every round
    order, table = nbv.select_greedy(wl.cand_cams, 2, target_obj=1)
    np.testing.assert_allclose(table.cpu().numpy()[0], ref["scores"], rtol=1e-3)
    assert order[0] == ref["best"]
    # determinant criterion: carried in the log domain (R-17), the numbers of the log-det criterion
    nd, nl = _nbv(wl.scene, criterion=2), _nbv(wl.scene)
    for n in (nd, nl):
        n.accumulate_training(wl.train_cams)
    sd, bd = nd.score_candidates(wl.cand_cams)
    sl, bl = nl.score_candidates(wl.cand_cams)
    np.testing.assert_allclose(sd.cpu().numpy(), sl.cpu().numpy(), rtol=2e-6)
    assert int(bd.item()) == int(bl.item()) == crit.score_candidates(scn, wl.train_cams, wl.cand_cams, crit.DET)["best"]
    from paper_2602_08266_b200 import api
    with pytest.raises(api.NBVError):
        api.NBV(criterion=1, weight_mode=1)
    with pytest.raises(api.NBVError):
        api.NBV(criterion=3)
