"""Pins for the oracle's per-pixel compositing (Eq. 1; readings R-4..R-8)."""
import json
import os

import numpy as np
import pytest

from oracle import nbv_oracle as orc
from paper_2602_08266_b200 import synth
from conftest import make_oracle_scene, scene_from_arrays

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "spec_examples.json")))


def _cam(W=32, H=32, f=100.0):
    return synth.simple_camera(W, H, f, dist=0.0)


def _on_pixel(cam, ix, iy, z):
    """world point (camera = identity) projecting exactly onto the centre of pixel (ix,iy)"""
    f = float(cam["fx"])
    return [((ix + 0.5) - float(cam["cx"])) * z / f, ((iy + 0.5) - float(cam["cy"])) * z / f, z]


def test_two_stacked_half_alpha_gaussians():
    cam = _cam()
    # pixel (16,16) centre is (16.5,16.5); cx = 16 -> offset 0.5 px
    pts = [_on_pixel(cam, 16, 16, 1.0), _on_pixel(cam, 16, 16, 2.0)]
    sc = scene_from_arrays(pts, [[-3] * 3] * 2, [[1, 0, 0, 0]] * 2, [0.5, 0.5], [[1, 0, 0], [0, 1, 0]])
    r = make_oracle_scene(sc, channel_mask=15).render(cam)
    g = GOLD["two_stacked_half_alpha"]
    # alpha = 0.5 * exp(power), power ~ 0 at the centre pixel (binary32 projection: |power| < 1e-6)
    assert 1.0 - r["T"][16, 16] == pytest.approx(g["total_alpha"], abs=2e-6)
    assert r["rgb"][16, 16, 0] == pytest.approx(0.5, abs=2e-6)
    assert r["rgb"][16, 16, 1] == pytest.approx(g["T_second"] * 0.5, abs=2e-6)
    assert r["depth"][16, 16] == pytest.approx(0.5 * 1.0 + 0.25 * 2.0, abs=5e-6)  # R-6: sum z alpha T
    assert r["ncontrib"][16, 16] == 2


def test_opaque_gaussian_is_capped_at_0_99():
    cam = _cam()
    sc = scene_from_arrays([_on_pixel(cam, 10, 12, 1.0)], [[-3] * 3], [[1, 0, 0, 0]], [0.999999], [[1, 1, 1]])
    r = make_oracle_scene(sc).render(cam)
    assert 1.0 - r["T"][12, 10] == pytest.approx(GOLD["alpha_cap"]["value"], abs=1e-7)
    assert r["rgb"][12, 10, 0] == pytest.approx(0.99, abs=1e-7)


def test_single_gaussian_pixel_values_follow_the_closed_form():
    cam = _cam(64, 64, 200.0)
    rho, z, sig = 0.02, 1.0, 0.7
    sc = scene_from_arrays([[0.013, -0.021, z]], [[np.log(rho)] * 3], [[1, 0, 0, 0]], [sig], [[0.2, 0.5, 0.9]])
    r = make_oracle_scene(sc).render(cam)
    f = 200.0
    mx, my = f * 0.013 / z + 32, f * (-0.021) / z + 32
    # off-axis isotropic Gaussian: Sigma2D = rho^2 J J^T + 0.3 I with the exact first-order J
    x, y = 0.013, -0.021
    J = np.array([[f / z, 0, -f * x / z**2], [0, f / z, -f * y / z**2]])
    S = rho**2 * J @ J.T + 0.3 * np.eye(2)
    Si = np.linalg.inv(S)
    X, Y = np.meshgrid(np.arange(64) + 0.5, np.arange(64) + 0.5)
    d = np.stack([X - mx, Y - my], -1)
    power = -0.5 * np.einsum("...i,ij,...j", d, Si, d)
    alpha = sig * np.exp(power)
    alpha[alpha < 1 / 255] = 0.0
    np.testing.assert_allclose(r["rgb"][..., 2], 0.9 * alpha, atol=3e-6)
    np.testing.assert_allclose(r["depth"], z * alpha, atol=3e-6)
    assert np.array_equal(r["ncontrib"] > 0, np.abs(alpha) > 0) or np.sum((r["ncontrib"] > 0) != (alpha > 0)) <= 2


def test_partition_of_unity_and_transmittance_invariants(wl0):
    # all colours 1 and background 1 -> every pixel renders exactly 1 = sum_i w_i + T_end (telescoping)
    s = wl0.scene
    ones = synth.Scene(s.mean, s.logscale, s.quat, s.opacity, np.ones_like(s.rgb), s.obj_logits, s.obj_id)
    scn = make_oracle_scene(ones, bg=(1.0, 1.0, 1.0))
    for cam in (wl0.train_cams[0], wl0.cand_cams[3]):
        r = scn.render(cam)
        np.testing.assert_allclose(r["rgb"], 1.0, atol=1e-12)
        assert r["T"].min() >= 1e-4 * (1 - 1e-5) and r["T32"].min() >= np.float32(1e-4)  # R-4: stop-before rule
        assert r["T"].max() <= 1.0
        np.testing.assert_allclose(r["T"], r["T32"], rtol=2e-5)
        assert np.all((r["ncontrib"] == 0) == (r["T"] == 1.0))


def test_trace_alphas_in_range_and_early_termination_invariant(wl0):
    """Every composited alpha is in [1/255, 0.99]; T is non-increasing along the ray; a pixel that stopped
    early did so because the next contributor would have crossed 1e-4."""
    scn = make_oracle_scene(wl0.scene)
    cam = wl0.train_cams[0]
    offsets, ids, clamped = scn.trace(cam)
    vis, rec, rect = scn.project(cam)
    order = scn.depth_order(cam)
    rank = np.full(wl0.scene.N, -1)
    rank[order] = np.arange(len(order))
    r = scn.render(cam)
    W = int(cam["width"])
    sig = wl0.scene.opacity.astype(np.float64)
    n_checked = 0
    for p in range(0, offsets.shape[0] - 1, 7):
        lst = ids[offsets[p]:offsets[p + 1]]
        if len(lst) == 0:
            continue
        assert np.all(np.diff(rank[lst]) > 0)  # front to back, each Gaussian once
        px, py = (p % W) + 0.5, (p // W) + 0.5
        dx, dy = px - rec[lst, 0].astype(np.float64), py - rec[lst, 1].astype(np.float64)
        power = rec[lst, 2] * dx * dx + rec[lst, 3] * dx * dy + rec[lst, 4] * dy * dy
        a = sig[lst] * np.exp(power)
        assert np.all(a >= (1 / 255) * (1 - 1e-5))
        a = np.minimum(a, 0.99)
        T = np.cumprod(1 - a)
        assert np.all(np.diff(T) <= 0) and T[-1] >= 1e-4 * (1 - 1e-5)
        assert T[-1] == pytest.approx(r["T"].reshape(-1)[p], rel=1e-9)
        n_checked += 1
    assert n_checked > 100
    # early termination: find pixels whose walk stopped before the list of candidates was exhausted
    stopped = 0
    for p in range(offsets.shape[0] - 1):
        lst = ids[offsets[p]:offsets[p + 1]]
        if len(lst) == 0:
            continue
        ix, iy = p % W, p // W
        later = order[rank[lst[-1]] + 1:]
        cover = later[(rect[later, 0] <= ix // 16) & (ix // 16 < rect[later, 2]) & (rect[later, 1] <= iy // 16) & (iy // 16 < rect[later, 3])]
        dx, dy = (ix + 0.5) - rec[cover, 0].astype(np.float64), (iy + 0.5) - rec[cover, 1].astype(np.float64)
        power = rec[cover, 2] * dx * dx + rec[cover, 3] * dx * dy + rec[cover, 4] * dy * dy
        a = np.minimum(sig[cover] * np.exp(power), 0.99)
        passing = np.flatnonzero(a >= (1 / 255) * (1 + 1e-5))
        if len(passing):
            nxt = passing[0]
            assert r["T"].reshape(-1)[p] * (1 - a[nxt]) < 1e-4 * (1 + 1e-5)
            stopped += 1
    assert stopped > 0


def test_brute_force_without_aabb_gives_the_same_image(wl0):
    """R-5: the conservative AABB never changes a result.  numpy brute force over ALL Gaussians in binary64."""
    scn = make_oracle_scene(wl0.scene, channel_mask=15)
    cam = wl0.cand_cams[0]
    vis, rec, _ = scn.project(cam)
    order = scn.depth_order(cam)
    r = scn.render(cam)
    W, H = int(cam["width"]), int(cam["height"])
    X, Y = np.meshgrid(np.arange(W) + 0.5, np.arange(H) + 0.5)
    T = np.ones((H, W))
    C = np.zeros((H, W, 3))
    D = np.zeros((H, W))
    done = np.zeros((H, W), dtype=bool)
    risky = np.zeros((H, W), dtype=bool)  # a decision within rounding distance of its threshold
    n = np.zeros((H, W), dtype=int)
    rec64 = rec.astype(np.float64)
    for g in order:
        dx, dy = X - rec64[g, 0], Y - rec64[g, 1]
        power = rec64[g, 2] * dx * dx + rec64[g, 3] * dx * dy + rec64[g, 4] * dy * dy
        a = float(wl0.scene.opacity[g]) * np.exp(power)
        risky |= (np.abs(a - 1 / 255) < 1e-7) & ~done
        ok = (a >= 1 / 255) & (power <= 0) & ~done
        a = np.minimum(a, float(np.float32(0.99)))
        Tn = T * (1 - a)
        risky |= ok & (np.abs(Tn - 1e-4) < 1e-9)
        stop = ok & (Tn < float(np.float32(1e-4)))
        done |= stop
        ok &= ~stop
        w = np.where(ok, a * T, 0.0)
        C += w[..., None] * wl0.scene.rgb[g].astype(np.float64)
        D += w * rec64[g, 5]
        T = np.where(ok, Tn, T)
        n += ok
    good = ~risky
    assert good.mean() > 0.99
    np.testing.assert_array_equal(r["ncontrib"][good], n[good])
    np.testing.assert_allclose(r["rgb"][good], C[good], atol=1e-9)
    np.testing.assert_allclose(r["depth"][good], D[good], atol=1e-9)
    np.testing.assert_allclose(r["T"][good], T[good], atol=1e-12)


def test_permutation_of_gaussians_leaves_the_image_identical(wl0):
    s = wl0.scene
    perm = np.random.default_rng(3).permutation(s.N)
    cam = wl0.cand_cams[2]
    r0 = make_oracle_scene(s).render(cam)
    r1 = make_oracle_scene(s.subset(perm)).render(cam)
    np.testing.assert_array_equal(r0["ncontrib"], r1["ncontrib"])
    np.testing.assert_array_equal(r0["rgb"], r1["rgb"])
    np.testing.assert_array_equal(r0["T32"], r1["T32"])


def test_monotone_occlusion():
    cam = _cam()
    pts = [_on_pixel(cam, 16, 16, 1.0), _on_pixel(cam, 16, 16, 2.0), _on_pixel(cam, 17, 16, 3.0)]
    Ts = []
    for front in (0.2, 0.5, 0.9):
        sc = scene_from_arrays(pts, [[-3.5] * 3] * 3, [[1, 0, 0, 0]] * 3, [front, 0.6, 0.6], [[1, 1, 1]] * 3)
        Ts.append(make_oracle_scene(sc).render(cam)["T"])
    assert np.all(Ts[1] <= Ts[0] + 1e-15) and np.all(Ts[2] <= Ts[1] + 1e-15)


def test_empty_view_renders_background():
    cam = _cam()
    sc = scene_from_arrays([[0, 0, -1.0]], [[-3] * 3], [[1, 0, 0, 0]], [0.5], [[1, 1, 1]])
    r = make_oracle_scene(sc, bg=(0.1, 0.2, 0.3)).render(cam)
    np.testing.assert_allclose(r["rgb"], np.broadcast_to(np.float32([0.1, 0.2, 0.3]).astype(np.float64), r["rgb"].shape))
    assert np.all(r["depth"] == 0) and np.all(r["T"] == 1) and np.all(r["ncontrib"] == 0)


def test_pixel_mask_renders_only_selected_pixels(wl0):
    scn = make_oracle_scene(wl0.scene)
    cam = wl0.cand_cams[1]
    full = scn.render(cam)
    mask = np.zeros((64, 64), dtype=np.uint8)
    mask[10:20, 30:44] = 1
    part = scn.render(cam, pixel_mask=mask)
    np.testing.assert_array_equal(part["rgb"][mask > 0], full["rgb"][mask > 0])
    assert np.all(part["ncontrib"][mask == 0] == 0)
