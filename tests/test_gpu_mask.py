"""GPU-vs-oracle parity of the object-mask output (Eq. 1-2) through the
C ABI: mask image 1e-5 abs; blocks of 11 + K parameters 1e-3 relative to sqrt(H_kk H_ll) (1e-6 abs floor); gains and
scores 1e-3 relative; indices identical."""
import numpy as np
import pytest

from oracle import nbv_oracle as orc
from paper_2602_08266_b200 import synth
from conftest import make_oracle_scene

pytestmark = pytest.mark.gpu


def _scene(K, n=None, seed=0):
    n = (1500 if K <= 10 else 500) if n is None else n
    rng = np.random.default_rng(100 + seed)
    sc = synth.make_scene(n, K, -4.0, 0.5, rng)
    return sc


def _cams(n, W=80, H=64, seed=1):
    return synth.hemisphere_cameras(n, (0.55, 0.7), W, H, 75.0, 75.0, np.random.default_rng(seed))


def _mask_ctx(scene, **kw):
    from paper_2602_08266_b200 import api
    n = api.NBV(channel_mask=api.CH_MASK, **kw)
    n.load_scene(scene)
    return n


def _block_err(Hg, Ho, L):
    Fo = orc.unpack_blocks_L(Ho, L)
    d = np.sqrt(np.maximum(np.einsum("nii->ni", Fo), 0))
    iu = np.triu_indices(L)
    scale = (d[:, :, None] * d[:, None, :])[:, iu[0], iu[1]]
    return np.abs(Hg - Ho) / (scale + 1e-3)


@pytest.mark.parametrize("K,bg", [(3, 0), (6, 0), (6, 4), (9, 2), (22, 0), (50, 0), (52, 51)])      # K = 22: six groups; 50: config 4; 52 = NBV_MASK_KMAX
def test_mask_image_and_blocks(K, bg):
    sc = _scene(K)
    cam = _cams(1, seed=K)[0]
    scn = make_oracle_scene(sc)
    nbv = _mask_ctx(sc, mask_bg_channel=bg)
    L = 11 + K
    assert nbv.block_size() == L * (L + 1) // 2
    O = nbv.render_mask(cam).cpu().numpy()
    np.testing.assert_allclose(O, orc.render_mask(scn, cam, bg), atol=1e-5, rtol=0)
    np.testing.assert_allclose(O.sum(axis=2), 1.0, atol=1e-5)
    Hg = nbv.view_hessian(cam).cpu().numpy().astype(np.float64)
    Ho = orc.view_hessian_mask(scn, cam, bg)
    assert (np.abs(Ho).max(axis=1) > 0).sum() > 50
    assert np.array_equal(np.abs(Hg).max(axis=1) > 0, np.abs(Ho).max(axis=1) > 0)     # same set of touched Gaussians
    assert _block_err(Hg, Ho, L).max() < 1e-3


@pytest.mark.parametrize("target", [-1, 1])
def test_mask_scoring_and_training_accumulation(target):
    K = 6
    sc = _scene(K, seed=2)
    train, cands = _cams(3, seed=11), _cams(10, seed=12)            # 10 candidates: two batches (8 + 2)
    scn = make_oracle_scene(sc)
    nbv = _mask_ctx(sc)
    nbv.accumulate_training(train)
    ref = orc.score_candidates_mask(scn, train, cands, target)
    L = 11 + K
    assert _block_err(nbv.training_hessian().cpu().numpy().astype(np.float64), ref["H_T"], L).max() < 1e-3
    s, best = nbv.score_candidates(cands, target)
    np.testing.assert_allclose(s.cpu().numpy(), ref["scores"], rtol=1e-3, atol=1e-6)
    assert int(best.item()) == ref["best"]
    g = nbv.gaussian_gains(cands[0], target).cpu().numpy().astype(np.float64)
    conf = orc.confidence(scn.obj_logits, scn.opacity, 0.3, 0.3, target)
    go = orc.gaussian_gains_L(ref["H_T"], orc.view_hessian_mask(scn, cands[0]), conf, np.ones(L), L)
    np.testing.assert_allclose(g, go, rtol=1e-3, atol=1e-6)


def test_three_output_fusion_matches_the_oracle():
    from paper_2602_08266_b200 import api
    sc = _scene(5, seed=3)
    train, cands = _cams(2, seed=21), _cams(6, seed=22)
    ctxs = []
    for mask in (api.CH_RGB, api.CH_DEPTH, api.CH_MASK):
        n = api.NBV(channel_mask=mask)
        n.load_scene(sc)
        n.accumulate_training(train)
        ctxs.append(n)
    out = api.score_candidates_fused(ctxs[0], ctxs[1], train, cands, -1, 10.0, nbv_mask=ctxs[2], beta_o=1.0)
    ref = orc.score_candidates_fused(make_oracle_scene(sc, 7), make_oracle_scene(sc, 8), train, cands, -1, 10.0,
                                     scene_mask=make_oracle_scene(sc, 7), beta_o=1.0)
    np.testing.assert_allclose(out["raw"].cpu().numpy(), ref["raw"], rtol=1e-3, atol=1e-6)
    np.testing.assert_allclose(out["denom"].cpu().numpy(), ref["denom"], rtol=1e-3, atol=1e-6)
    np.testing.assert_allclose(out["fused"].cpu().numpy(), ref["fused"], rtol=1e-3, atol=1e-6)
    assert int(out["best"].item()) == ref["best"]


def test_mask_context_errors_and_greedy_fallback():
    from paper_2602_08266_b200 import api
    sc = _scene(4, n=300, seed=4)
    train, cands = _cams(1, seed=31), _cams(3, seed=32)
    nbv = _mask_ctx(sc)
    with pytest.raises(api.NBVError) as e:
        nbv.render(cands[0])
    assert e.value.status == "NBV_ERR_INVALID_ARG"
    with pytest.raises(api.NBVError) as e:
        _mask_ctx(sc, mask_bg_channel=4)                            # >= K
    assert e.value.status == "NBV_ERR_INVALID_ARG"
    rgb = api.NBV(channel_mask=api.CH_RGB); rgb.load_scene(sc)
    with pytest.raises(api.NBVError) as e:
        rgb.render_mask(cands[0])
    assert e.value.status == "NBV_ERR_INVALID_ARG"
    nbv.accumulate_training(train)
    order, _ = nbv.select_greedy(cands, 2)                           # mask contexts take the re-rasterising path
    first = orc.score_candidates_mask(make_oracle_scene(sc), train, cands)
    assert order[0] == first["best"] and len(set(order.tolist())) == 2


def test_mask_output_at_the_benchmarked_image_size_and_channel_count():
    """1280 x 720, K = 20 object channels (blocks of 31 parameters, five S4 channel groups), 20,000 Gaussians: training
    blocks, candidate blocks, per-Gaussian gains, scores and the arg-max against the oracle's stored values
    (tests/golden/mask_fullres.json, written by tests/golden/make_mask_golden.py from oracle/ alone)."""
    import importlib.util
    import json
    from pathlib import Path
    golden = Path(__file__).resolve().parent / "golden"
    spec = importlib.util.spec_from_file_location("make_mask_golden", golden / "make_mask_golden.py")
    mk = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mk)
    f = golden / "mask_fullres.json"
    assert f.exists(), "mask_fullres.json missing: run tests/golden/make_mask_golden.py"
    g = json.loads(f.read_text())
    wl = mk.workload()
    for k, v in mk.oracle_hashes().items():
        assert g[k] == v, "mask_fullres.json is stale (%s changed): regenerate it" % k
    assert g["input_sha256"] == mk.input_checksum(wl), "mask_fullres.json is stale (the synthetic inputs changed): regenerate it"
    K, L, step = g["K"], g["L"], g["block_step"]
    assert (K, L) == (wl.scene.K, 11 + wl.scene.K) and g["image"] == [1280, 720]
    nbv = _mask_ctx(wl.scene, mask_bg_channel=g["bg_channel"])
    nbv.accumulate_training(wl.train_cams)

    def check_blocks(Hg, touched, ref_blocks):
        touched = np.array(touched)
        assert np.array_equal(np.flatnonzero(np.abs(Hg).max(axis=1) > 0), touched)          # same set of touched Gaussians
        assert _block_err(Hg[touched[::step]], np.array(ref_blocks), L).max() < 1e-3

    check_blocks(nbv.training_hessian().cpu().numpy().astype(np.float64), g["train_touched"], g["train_blocks"])
    c0 = g["candidates"][0]
    check_blocks(nbv.view_hessian(wl.cand_cams[0]).cpu().numpy().astype(np.float64), c0["touched"], c0["blocks"])
    s, best = nbv.score_candidates(wl.cand_cams)
    np.testing.assert_allclose(s.cpu().numpy(), g["scores"], rtol=1e-3, atol=1e-6)
    assert int(best.item()) == g["best"]
    for i, c in enumerate(g["candidates"]):
        gg = nbv.gaussian_gains(wl.cand_cams[i]).cpu().numpy().astype(np.float64)
        t = np.array(c["touched"])
        np.testing.assert_allclose(gg[t], c["gains"], rtol=1e-3, atol=1e-6)
        rest = np.ones(len(gg), bool)
        rest[t] = False
        assert np.all(gg[rest] == 0)
