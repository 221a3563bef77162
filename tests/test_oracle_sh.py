"""Pins of the SH degree 3 colour oracle (oracle/sh.py, oracle/nbv_oracle_ext.inc; reading R-18):
orthonormality and the addition theorem of the basis by quadrature, gradients by finite differences, reduction to the
degree-0 path, the structure of the coefficient rows, and J^T J from central differences of the smooth renderer."""
import numpy as np
import pytest

from oracle import nbv_oracle as orc
from oracle import sh
from paper_2602_08266_b200 import synth
from conftest import make_oracle_scene


def _sphere_quadrature(nt=24, nphi=48):
    x, w = np.polynomial.legendre.leggauss(nt)              # cos(theta) nodes: exact for the degree-6 products below
    phi = (np.arange(nphi) + 0.5) * 2 * np.pi / nphi
    ct, ph = np.meshgrid(x, phi, indexing="ij")
    st = np.sqrt(1 - ct ** 2)
    dirs = np.stack([st * np.cos(ph), st * np.sin(ph), ct], axis=-1).reshape(-1, 3)
    wts = np.repeat(w, nphi) * (2 * np.pi / nphi)
    return dirs, wts


def test_basis_is_orthonormal_and_obeys_the_addition_theorem():
    dirs, w = _sphere_quadrature()
    B = np.array([sh.basis(d)[0] for d in dirs])
    assert np.all(B[:, 0] == 1.0)                            # the direction-independent term is the stored rgb itself (R-8)
    gram = (B[:, 1:, None] * B[:, None, 1:] * w[:, None, None]).sum(axis=0)
    np.testing.assert_allclose(gram, np.eye(15), atol=1e-12)
    for lo, hi, l in ((1, 4, 1), (4, 9, 2), (9, 16, 3)):
        np.testing.assert_allclose((B[:, lo:hi] ** 2).sum(axis=1), (2 * l + 1) / (4 * np.pi), rtol=1e-12)
    # parity: degree l changes sign like (-1)^l under dir -> -dir
    Bm = np.array([sh.basis(-d)[0] for d in dirs[:50]])
    sign = np.array([1] + [-1] * 3 + [1] * 5 + [-1] * 7)
    np.testing.assert_allclose(Bm, B[:50] * sign, atol=1e-14)


def test_basis_gradient_by_finite_differences():
    rng = np.random.default_rng(0)
    for _ in range(5):
        d = rng.standard_normal(3); d /= np.linalg.norm(d)
        _, dB = sh.basis(d)
        # dB is the gradient of the polynomial in free (x,y,z): difference the polynomials along tangent directions
        for t in np.eye(3):
            t = t - d * (t @ d)
            h = 1e-6
            Bp, Bm = sh.basis(d + h * t)[0], sh.basis(d - h * t)[0]        # renormalised inside; tangent steps keep |d| to O(h^2)
            np.testing.assert_allclose((Bp - Bm) / (2 * h), dB @ t, atol=2e-8)


def _tiny(n=3, seed=3):
    sc = synth.micro_scene(n, seed)
    rng = np.random.default_rng(seed + 50)
    k = (0.3 * rng.standard_normal((n, 45))).astype(np.float32)
    cam = synth.hemisphere_cameras(1, (0.45, 0.45), 20, 16, 60.0, 60.0, rng, centre=np.zeros(3))[0]
    return sc, k, cam


def test_zero_coefficients_reduce_to_the_degree_0_path():
    wl = synth.make_workload(0, n_gaussians=400)
    scn = make_oracle_scene(wl.scene, channel_mask=15)
    cam = wl.cand_cams[0]
    k0 = np.zeros((400, 45), dtype=np.float32)
    r0, r = scn.render(cam), sh.render(scn, cam, k0)
    np.testing.assert_array_equal(r["ncontrib"], r0["ncontrib"])
    np.testing.assert_allclose(r["rgb"], r0["rgb"], atol=1e-15)
    np.testing.assert_allclose(sh.colours(scn, cam, k0), wl.scene.rgb, atol=0)
    H14 = orc.unpack_blocks(scn.view_hessian(cam))
    H59 = orc.unpack_blocks_L(sh.view_hessian(scn, cam, k0), 59)
    np.testing.assert_allclose(H59[:, :14, :14], H14, rtol=1e-12, atol=1e-300)
    # coefficient (j, ch) sees w B_j where rgb_ch sees w: its rows are B_j times the rgb rows (one view: B_j is a constant)
    vis, rec, _ = scn.project(cam)
    o = -np.asarray(cam["R"], dtype=np.float64).reshape(3, 3).T @ np.asarray(cam["t"], dtype=np.float64)
    g = int(np.argmax(np.abs(H14[:, 11, 11])))
    B, _ = sh.basis(wl.scene.mean[g].astype(np.float64) - o)
    for j in (1, 6, 12):
        for ch in range(3):
            np.testing.assert_allclose(H59[g, :14, 11 + 3 * j + ch], B[j] * H59[g, :14, 11 + ch], rtol=1e-10, atol=1e-12)
            np.testing.assert_allclose(H59[g, 11 + 3 * j + ch, 11 + 3 * j + ch], B[j] ** 2 * H59[g, 11 + ch, 11 + ch], rtol=1e-10)


def test_colour_depends_on_the_viewing_direction():
    sc, k, cam = _tiny()
    scn = make_oracle_scene(sc)
    c1 = sh.colours(scn, cam, k)
    cam2 = synth.hemisphere_cameras(1, (0.45, 0.45), 20, 16, 60.0, 60.0, np.random.default_rng(99), centre=np.zeros(3))[0]
    assert np.abs(c1 - sh.colours(scn, cam2, k)).max() > 1e-3
    o = -np.asarray(cam["R"], dtype=np.float64).reshape(3, 3).T @ np.asarray(cam["t"], dtype=np.float64)
    for g in range(sc.N):
        B, _ = sh.basis(sc.mean[g].astype(np.float64) - o)
        np.testing.assert_allclose(c1[g], sc.rgb[g] + B[1:] @ k[g].reshape(15, 3).astype(np.float64), rtol=1e-12)


@pytest.mark.parametrize("mask", [7, 15])
def test_blocks_equal_jtj_from_central_differences(mask):
    """59-wide rows: finite differences of the binary64 smooth renderer with frozen contributor sets, assembled into J^T J"""
    sc, k, cam = _tiny(3, 7)
    cfg = orc.default_config(mask, bg=(0.2, 0.1, 0.3), channel_weight=(1.0, 0.5, 2.0, 3.0))
    scn = orc.OracleScene(sc.mean, sc.logscale, sc.quat, sc.opacity, sc.rgb, sc.obj_logits, cfg)
    off, ids, cl = scn.trace(cam)
    th = sh.theta(scn, k)
    Han = orc.unpack_blocks_L(sh.view_hessian_smooth(th, cam, cfg, off, ids, cl), 59)
    om = np.array([1.0, 0.5, 2.0, 3.0]) * [(mask >> c) & 1 for c in range(4)]
    for g in range(sc.N):
        J = np.zeros((20 * 16 * 4, 59))
        for p in range(59):
            h = 1e-5 * max(1.0, abs(th[g, p]))
            tp, tm = th.copy(), th.copy()
            tp[g, p] += h; tm[g, p] -= h
            J[:, p] = ((sh.render_smooth(tp, cam, cfg, off, ids, cl) - sh.render_smooth(tm, cam, cfg, off, ids, cl)) / (2 * h)).reshape(-1)
        w = np.tile(om, 20 * 16)
        Hfd = (J * w[:, None]).T @ J
        assert np.linalg.norm(Han[g] - Hfd) <= 2e-6 * np.linalg.norm(Hfd), g
    # the analytic path of the normal mode is the same code: binary32-projected inputs agree with smooth mode to rounding
    Hn = orc.unpack_blocks_L(sh.view_hessian(scn, cam, k), 59)
    scale = np.sqrt(np.einsum("nii->ni", Han))[:, :, None] * np.sqrt(np.einsum("nii->ni", Han))[:, None, :]
    assert np.max(np.abs(Hn - Han) / (scale + 1e-9)) < 5e-4


def test_sh_gain_properties():
    wl = synth.make_workload(0, n_gaussians=300)
    scn = make_oracle_scene(wl.scene)
    k = (0.2 * np.random.default_rng(1).standard_normal((300, 45))).astype(np.float32)
    res = sh.score_candidates(scn, k, wl.train_cams, wl.cand_cams[:2])
    assert np.all(res["gains"] >= -1e-12) and res["scores"].min() > 0
    H = orc.unpack_blocks_L(res["H_T"], 59)
    assert np.linalg.eigvalsh(H[np.abs(res["H_T"]).sum(axis=1) > 0]).min() > -1e-6 * np.abs(H).max()      # PSD
    # a single view gives rank <= 3 in the 48 colour coefficients (one direction: B is one vector per channel)
    Hc = orc.unpack_blocks_L(sh.view_hessian(scn, wl.cand_cams[0], k), 59)
    g = int(np.argmax(np.einsum("nii->n", Hc)))
    assert np.linalg.matrix_rank(Hc[g][11:, 11:], tol=1e-9 * np.abs(Hc[g]).max()) <= 3
