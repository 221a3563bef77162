"""Pins for the oracle's decision-path primitives and geometry (CPU only).

Each test checks the oracle against something other than itself: a closed form,
a library routine (numpy exp/log/eig), an invariant, or brute force.
Citations: S:Lnnn = /root/reference/SPEC.md, P:Lnnn = PAPER.md, R-n = DESIGN.md reading.
"""
import json
import os

import numpy as np
import pytest

from oracle import nbv_oracle as orc
from paper_2602_08266_b200 import synth
from conftest import make_oracle_scene, scene_from_arrays

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "spec_examples.json")))


# ------------------------------------------------------------------ exp_spec / log_bound (R-9)
def test_exp_spec_matches_library_exp_on_alpha_range():
    x = np.linspace(-6.0, 0.0, 20001).astype(np.float32)
    got = orc.exp_spec(x).astype(np.float64)
    ref = np.exp(x.astype(np.float64))
    assert np.max(np.abs(got / ref - 1.0)) < 2.5e-7
    assert orc.exp_spec(0.0)[0] == np.float32(1.0)
    assert np.all(got <= 1.0)  # sigma*G <= sigma: a Gaussian with sigma < 1/255 can never pass the alpha test
    assert np.all(np.diff(got) >= -1.2e-7 * got[1:])  # monotone up to 1 ulp


def test_exp_spec_wide_range_for_scales():
    x = np.linspace(-80.0, 80.0, 4001).astype(np.float32)
    got = orc.exp_spec(x).astype(np.float64)
    ref = np.exp(x.astype(np.float64))
    assert np.all(np.isfinite(got))
    assert np.max(np.abs(got / ref - 1.0)) < 3e-7


def test_log_bound_is_a_tight_upper_bound_of_ln_255_sigma():
    s = np.concatenate([np.linspace(1.0 / 255.0, 0.999999, 5000), [1e-6, 1e-3, 0.0039]]).astype(np.float32)
    got = orc.log_bound(s).astype(np.float64)
    ref = np.log(np.maximum(255.0 * s.astype(np.float64), 1.0))
    assert np.all(got >= ref - 1e-6)
    assert np.all(got <= ref + 0.08)
    assert np.all(got >= 0.0)


# ------------------------------------------------------------------ rotation / covariance
def _act(logscale, quat):
    sc = scene_from_arrays([[0, 0, 1]], [logscale], [quat], [0.5], [[1, 1, 1]])
    return make_oracle_scene(sc).activation()[0].reshape(3, 3).astype(np.float64)


def test_identity_quaternion_gives_diag_scales():
    M = _act([np.log(2.0), 0.0, np.log(0.5)], [1, 0, 0, 0])
    np.testing.assert_allclose(M, np.diag([2.0, 1.0, 0.5]), atol=3e-7)


def test_rotation_90deg_about_x_maps_y_to_z():
    c = np.cos(np.pi / 4)
    M = _act([0, 0, 0], [c, c, 0, 0])
    np.testing.assert_allclose(M @ np.array([0, 1.0, 0]), [0, 0, 1.0], atol=3e-7)
    np.testing.assert_allclose(M @ M.T, np.eye(3), atol=5e-7)  # orthonormal
    assert np.linalg.det(M) == pytest.approx(1.0, abs=1e-6)


def test_covariance_eigenvalues_are_squared_scales_and_sign_flip_invariant():
    rng = np.random.default_rng(1)
    for _ in range(20):
        q = rng.standard_normal(4)
        ls = rng.normal(-1, 0.5, 3)
        M = _act(ls, q)
        ev = np.sort(np.linalg.eigvalsh(M @ M.T))
        np.testing.assert_allclose(ev, np.sort(np.exp(2 * ls)), rtol=3e-6)
        M2 = _act(ls, -q)
        np.testing.assert_array_equal(M @ M.T, M2 @ M2.T)
        M3 = _act(ls, 3.7 * q)  # raw quaternion is normalised internally
        np.testing.assert_allclose(M3, M, atol=1e-6)


def test_zero_quaternion_and_bad_opacity_flag_bad_data():
    sc = scene_from_arrays([[0, 0, 1]], [[0, 0, 0]], [[0, 0, 0, 0]], [0.5], [[1, 1, 1]])
    assert make_oracle_scene(sc).bad_data
    sc = scene_from_arrays([[0, 0, 1]], [[0, 0, 0]], [[1, 0, 0, 0]], [1.0], [[1, 1, 1]])
    assert make_oracle_scene(sc).bad_data
    sc = scene_from_arrays([[0, 0, 1]], [[0, 0, 0]], [[1, 0, 0, 0]], [0.5], [[1, 1, 1]])
    assert not make_oracle_scene(sc).bad_data


# ------------------------------------------------------------------ projection
def _cam(W=640, H=480, f=500.0):
    return synth.simple_camera(W, H, f, dist=0.0)


def test_principal_point_projection():
    cam = _cam()
    sc = scene_from_arrays([[0, 0, 2.0]], [[-3, -3, -3]], [[1, 0, 0, 0]], [0.5], [[1, 1, 1]])
    vis, rec, _ = make_oracle_scene(sc).project(cam)
    assert vis[0] == 1
    assert rec[0, 0] == 320.0 and rec[0, 1] == 240.0 and rec[0, 5] == 2.0


def test_small_angle_isotropic_covariance_closed_form():
    cam = _cam()
    f, z = 500.0, 2.0
    for rho in (0.01, 0.05, 0.1):  # rho/z <= 0.05
        sc = scene_from_arrays([[0.1, -0.05, z]], [[np.log(rho)] * 3], [[0.3, 0.1, -0.2, 0.9]], [0.5], [[1, 1, 1]])
        _, rec, _ = make_oracle_scene(sc).project(cam)
        a, b, c = rec[0, 6:9]
        want = (f * rho / z) ** 2 + 0.3
        assert a == pytest.approx(want, rel=0.01) and c == pytest.approx(want, rel=0.01)
        assert abs(b) < 0.01 * want


def test_on_axis_isotropic_covariance_is_exact_and_conic_is_inverse():
    cam = _cam()
    f, z, rho = 500.0, 1.5, 0.03
    sc = scene_from_arrays([[0, 0, z]], [[np.log(rho)] * 3], [[1, 0, 0, 0]], [0.5], [[1, 1, 1]])
    _, rec, _ = make_oracle_scene(sc).project(cam)
    s2 = (f * rho / z) ** 2 + 0.3
    mx, my, qa, qb, qc, zz, a, b, c = rec[0].astype(np.float64)
    assert a == pytest.approx(s2, rel=1e-6) and c == pytest.approx(s2, rel=1e-6) and abs(b) < 1e-6
    assert -2 * qa == pytest.approx(1 / s2, rel=1e-6) and -2 * qc == pytest.approx(1 / s2, rel=1e-6)


def test_cov2d_symmetric_psd_with_blur_floor_and_conic_inverse():
    wl = synth.make_workload(0)
    scn = make_oracle_scene(wl.scene)
    vis, rec, _ = scn.project(wl.cand_cams[1])
    rec = rec[vis > 0].astype(np.float64)
    a, b, c = rec[:, 6], rec[:, 7], rec[:, 8]
    tr, det = a + c, a * c - b * b
    lam_min = tr / 2 - np.sqrt(np.maximum(tr * tr / 4 - det, 0))
    assert np.all(lam_min >= 0.3 * (1 - 1e-5))
    # conic = Sigma2D^-1: (A,B,C) = (-2qa, -qb, -2qc)
    A, B, Cc = -2 * rec[:, 2], -rec[:, 3], -2 * rec[:, 4]
    np.testing.assert_allclose(A * a + B * b, 1.0, rtol=0, atol=2e-4)
    np.testing.assert_allclose(A * b + B * c, 0.0, rtol=0, atol=2e-4 * np.sqrt(c / a).max())
    np.testing.assert_allclose(B * b + Cc * c, 1.0, rtol=0, atol=2e-4)


def test_sliding_along_the_ray_keeps_the_projected_centre():
    cam = synth.make_workload(0).train_cams[0]
    R = cam["R"].reshape(3, 3).astype(np.float64)
    t = cam["t"].astype(np.float64)
    centre = -R.T @ t
    mu = np.array([0.05, -0.02, 0.08])
    pts = [centre + s * (mu - centre) for s in (1.0, 1.3, 0.7)]
    sc = scene_from_arrays(pts, [[-4] * 3] * 3, [[1, 0, 0, 0]] * 3, [0.5] * 3, [[1, 1, 1]] * 3)
    _, rec, _ = make_oracle_scene(sc).project(cam)
    np.testing.assert_allclose(rec[1, :2], rec[0, :2], atol=2e-4)  # S:L70 (binary32 pixel coordinates)
    np.testing.assert_allclose(rec[2, :2], rec[0, :2], atol=2e-4)


def test_behind_camera_and_near_plane_are_culled():
    cam = _cam()
    sc = scene_from_arrays([[0, 0, -1.0], [0, 0, 0.01], [0, 0, 0.011]], [[-5] * 3] * 3, [[1, 0, 0, 0]] * 3, [0.5] * 3,
                           [[1, 1, 1]] * 3)
    vis, _, _ = make_oracle_scene(sc).project(cam)
    assert list(vis) == [0, 0, 1]  # S:L66, R-2: z <= near culled


def test_decision_projection_agrees_with_binary64_chain():
    wl = synth.make_workload(0)
    scn = make_oracle_scene(wl.scene)
    cam = wl.train_cams[0]
    vis, rec, _ = scn.project(cam)
    th = scn.theta()
    for g in np.flatnonzero(vis)[:200]:
        out6, _, _ = orc.chain(th[g], cam, scn.cfg)
        np.testing.assert_allclose(rec[g, [0, 1, 6, 7, 8, 5]], out6, rtol=2e-5, atol=2e-4)


def test_chain_matches_central_finite_differences():
    wl = synth.make_workload(0)
    scn = make_oracle_scene(wl.scene)
    cam = wl.cand_cams[2]
    th = scn.theta()
    rng = np.random.default_rng(0)
    for g in rng.choice(wl.scene.N, 12, replace=False):
        t0 = th[g].copy()
        t0[6:10] *= 1.7  # un-normalised raw quaternion: the chain goes through q/|q|
        _, G, dz = orc.chain(t0, cam, scn.cfg)
        for k in range(10):
            h = 1e-6 * max(1.0, abs(t0[k]))
            tp, tm = t0.copy(), t0.copy()
            tp[k] += h
            tm[k] -= h
            fp, _, _ = orc.chain(tp, cam, scn.cfg)
            fm, _, _ = orc.chain(tm, cam, scn.cfg)
            fd = (fp - fm) / (2 * h)
            scale = np.maximum(np.abs(G).max(axis=1), 1e-9)
            np.testing.assert_allclose(G[:, k] / scale, fd[:5] / scale, atol=2e-6)
            if k < 3:
                assert dz[k] == pytest.approx(fd[5], abs=1e-7)
            else:
                assert abs(fd[5]) < 1e-9


# ------------------------------------------------------------------ support rect, order, tile lists (R-5, R-7)
def test_rect_contains_every_pixel_that_can_pass_the_alpha_test():
    """Brute force in binary64 over every (pixel, Gaussian): alpha >= 1/255 * (1 - 1e-3) => pixel's tile in rect."""
    for cfg_i, cam_i in ((0, 0), (0, 3)):
        wl = synth.make_workload(cfg_i)
        scn = make_oracle_scene(wl.scene)
        cam = wl.cand_cams[cam_i]
        vis, rec, rect = scn.project(cam)
        W, H = int(cam["width"]), int(cam["height"])
        px = np.arange(W) + 0.5
        py = np.arange(H) + 0.5
        X, Y = np.meshgrid(px, py)
        TXi, TYi = np.meshgrid(np.arange(W) // 16, np.arange(H) // 16)
        for g in np.flatnonzero(vis):
            mx, my, qa, qb, qc = rec[g, :5].astype(np.float64)
            dx, dy = X - mx, Y - my
            power = qa * dx * dx + qb * dx * dy + qc * dy * dy
            alpha = float(wl.scene.opacity[g]) * np.exp(power)
            hit = alpha >= (1.0 / 255.0) * (1 - 1e-3)
            inside = (TXi >= rect[g, 0]) & (TXi < rect[g, 2]) & (TYi >= rect[g, 1]) & (TYi < rect[g, 3])
            assert not np.any(hit & ~inside)


def test_depth_order_sorts_by_z_then_index():
    wl = synth.make_workload(0)
    s = wl.scene
    # duplicate 50 Gaussians so that exact z ties exist
    idx = np.concatenate([np.arange(s.N), np.arange(50)])
    s2 = s.subset(idx)
    scn = make_oracle_scene(s2)
    cam = wl.train_cams[0]
    vis, rec, _ = scn.project(cam)
    order = scn.depth_order(cam)
    want = np.array(sorted(np.flatnonzero(vis), key=lambda g: (float(rec[g, 5]), g)))
    np.testing.assert_array_equal(order, want)
    z = rec[order, 5]
    assert np.all(np.diff(z) >= 0)
    ties = np.flatnonzero(np.diff(z) == 0)
    assert len(ties) >= 50 and np.all(order[ties] < order[ties + 1])  # R-7


def test_tile_lists_equal_the_definition():
    wl = synth.make_workload(0)
    scn = make_oracle_scene(wl.scene)
    for cam in (wl.train_cams[0], synth.hemisphere_cameras(1, (0.6, 0.6), 70, 50, 60.0, 60.0, np.random.default_rng(5))[0]):
        vis, rec, rect = scn.project(cam)
        order = scn.depth_order(cam)
        offsets, ids = scn.tile_lists(cam)
        TX = (int(cam["width"]) + 15) // 16
        TY = (int(cam["height"]) + 15) // 16
        assert offsets.shape[0] == TX * TY + 1 and offsets[-1] == len(ids)
        assert rect[vis > 0, 2].max() <= TX and rect[vis > 0, 3].max() <= TY
        for t in range(TX * TY):
            tx, ty = t % TX, t // TX
            want = [g for g in order if rect[g, 0] <= tx < rect[g, 2] and rect[g, 1] <= ty < rect[g, 3]]
            np.testing.assert_array_equal(ids[offsets[t]:offsets[t + 1]], want)


def test_golden_constants_of_the_spec():
    # SPEC.md worked examples reused as pins (tests/golden/spec_examples.json carries the citations)
    assert float(np.float32(0.99)) == pytest.approx(GOLD["alpha_cap"]["value"], abs=1e-7)
    assert 1.0 / 255.0 == pytest.approx(GOLD["alpha_skip"]["value"], rel=1e-12)
