"""Pins for the oracle's analytic Jacobians and per-Gaussian J^T J blocks
(PAPER.md L189-191 H ~= J^T J; L210 block-diagonal; L248 RGB + depth share geometry and opacity)."""
import numpy as np
import pytest
from scipy import special

from oracle import nbv_oracle as orc
from paper_2602_08266_b200 import synth
from conftest import make_oracle_scene, scene_from_arrays

P = 14


def _fd_blocks(theta, cam, cfg, offsets, ids, clamped, h=1e-6):
    """J^T J per Gaussian assembled column by column from central finite differences of the oracle's
    binary64 forward renderer with frozen contributor sets."""
    N = theta.shape[0]
    H = np.zeros((N, P, P))
    om = np.array([cfg.channel_weight[c] if (cfg.channel_mask >> c) & 1 else 0.0 for c in range(4)])
    for g in range(N):
        cols = []
        for k in range(P):
            tp, tm = theta.copy(), theta.copy()
            step = h * max(1.0, abs(theta[g, k]))
            tp[g, k] += step
            tm[g, k] -= step
            d = (orc.render_smooth(tp, cam, cfg, offsets, ids, clamped) - orc.render_smooth(tm, cam, cfg, offsets, ids, clamped)) / (2 * step)
            cols.append(d.reshape(-1, 4))
        J = np.stack(cols, axis=-1)  # (pixels, 4, 14)
        H[g] = np.einsum("pck,c,pcl->kl", J, om, J)
    return H


@pytest.mark.parametrize("n,seed,size,coord,mask", [(1, 0, 12, 0, 15), (2, 1, 8, 0, 15), (3, 2, 16, 1, 7), (5, 3, 16, 0, 15), (4, 4, 12, 0, 8)])
def test_analytic_blocks_equal_finite_difference_JtJ(n, seed, size, coord, mask):
    sc = synth.micro_scene(n, seed)
    sc.quat[:] *= np.float32(1.3)  # raw quaternions need not be unit: the chain goes through q/|q|
    cfg_kw = dict(opacity_coord=coord, bg=(0.3, 0.1, 0.2), channel_weight=(1.0, 0.5, 2.0, 3.0))
    scn = make_oracle_scene(sc, channel_mask=mask, **cfg_kw)
    cam = synth.simple_camera(size, size, 40.0, dist=0.5)
    offsets, ids, clamped = scn.trace(cam)
    assert len(ids) > 0
    th_logit = scn.theta()  # smooth mode always takes the opacity logit
    Han = orc.unpack_blocks(orc.view_hessian_smooth(th_logit, cam, scn.cfg, offsets, ids, clamped))
    # finite differences are taken w.r.t. the logit; convert to the sigma coordinate if requested
    cfg_fd = orc.default_config(mask, opacity_coord=0, bg=(0.3, 0.1, 0.2), channel_weight=(1.0, 0.5, 2.0, 3.0))
    Hfd = _fd_blocks(th_logit, cam, cfg_fd, offsets, ids, clamped)
    if coord == 1:
        s = sc.opacity.astype(np.float64)
        scale = np.ones((n, P))
        scale[:, 10] = 1.0 / (s * (1 - s))  # d/dsigma = d/dlogit / (sigma (1-sigma))
        Hfd = Hfd * scale[:, :, None] * scale[:, None, :]
    for g in range(n):
        num = np.linalg.norm(Han[g] - Hfd[g])
        den = np.linalg.norm(Hfd[g])
        assert den > 0
        assert num / den < 1e-6, (g, num / den)


def test_normal_mode_blocks_agree_with_smooth_mode(wl0):
    """value path on the binary32 splat (normal mode) vs all-binary64 smooth mode: same blocks to ~1e-5."""
    sc = wl0.scene.subset(np.arange(300))
    scn = make_oracle_scene(sc, channel_mask=15)
    cam = wl0.cand_cams[0]
    offsets, ids, clamped = scn.trace(cam)
    Hs = orc.view_hessian_smooth(scn.theta(), cam, scn.cfg, offsets, ids, clamped)
    Hn = scn.view_hessian(cam)
    d = np.sqrt(np.abs(orc.unpack_blocks(Hs)[:, np.arange(P), np.arange(P)]))
    scale = orc.pack_blocks(d[:, :, None] * d[:, None, :])
    assert np.max(np.abs(Hn - Hs) / (scale + 1e-12)) < 2e-4


def _closed_form_single_isotropic(f, z, rho, sig, rgb, coord, mask, omega):
    """Continuum limit (pixel sums -> integrals) for one isotropic Gaussian on the optical axis, identity
    camera, background 0 (derivation: DESIGN.md 'closed form').  alpha = sig exp(-t/2), t = |d|^2/s2 <= Q."""
    a0 = (f * rho / z) ** 2
    s2 = a0 + 0.3
    Q = 2 * np.log(255 * sig)
    kappa = (1 - sig) if coord == 0 else 1 / sig

    def mono(i, j):  # integral of alpha^2 ux^i uy^j over the disc, u = d/s2
        if i % 2 or j % 2:
            return 0.0
        n = (i + j) // 2
        radial = special.gammainc(n + 1, Q) * special.gamma(n + 1)  # int_0^Q t^n e^-t dt
        ang = 2 * special.gamma((i + 1) / 2) * special.gamma((j + 1) / 2) / special.gamma((i + j) / 2 + 1)
        return sig**2 * (s2 / 2) * s2 ** (-n) * radial * ang

    # dalpha/dtheta_k = alpha * poly_k(ux,uy); polys as {(i,j): coeff}
    g1 = f / z
    poly = [dict() for _ in range(P)]
    poly[0] = {(1, 0): g1}
    poly[1] = {(0, 1): g1}
    poly[2] = {(2, 0): -a0 / z, (0, 2): -a0 / z}
    poly[3] = {(2, 0): a0}
    poly[4] = {(0, 2): a0}
    poly[10] = {(0, 0): kappa}
    v = [rgb[0], rgb[1], rgb[2], z]
    H = np.zeros((P, P))
    for c in range(4):
        if not (mask >> c) & 1:
            continue
        rows = []
        for k in range(P):
            pk = {m: v[c] * co for m, co in poly[k].items()}  # beta_c = v_c (nothing behind, bg 0)
            if c < 3 and k == 11 + c:
                pk[(0, 0)] = pk.get((0, 0), 0.0) + 1.0  # + w e_c, w = alpha
            if c == 3 and k == 2:
                pk[(0, 0)] = pk.get((0, 0), 0.0) + 1.0  # dz/dmu_z = 1
            rows.append(pk)
        for k in range(P):
            for l in range(P):
                acc = 0.0
                for (i1, j1), c1 in rows[k].items():
                    for (i2, j2), c2 in rows[l].items():
                        acc += c1 * c2 * mono(i1 + i2, j1 + j2)
                H[k, l] += omega[c] * acc
    return H


@pytest.mark.parametrize("coord,mask", [(0, 7), (1, 15), (0, 8)])
def test_single_isotropic_gaussian_closed_form(coord, mask):
    f, z, rho, sig = 300.0, 1.0, 0.04, 0.6
    rgb = (0.3, 0.7, 0.5)
    omega = (1.0, 1.0, 1.0, 2.0)
    W = 129  # odd: the principal point 64.5 is the centre of pixel 64
    cam = synth.simple_camera(W, W, f, dist=0.0)
    sc = scene_from_arrays([[0, 0, z]], [[np.log(rho)] * 3], [[1, 0, 0, 0]], [sig], [rgb])
    scn = make_oracle_scene(sc, channel_mask=mask, opacity_coord=coord, channel_weight=omega)
    Hor = orc.unpack_blocks(scn.view_hessian(cam))[0]
    Hcf = _closed_form_single_isotropic(f, z, rho, sig, rgb, coord, mask, omega)
    d = np.sqrt(np.diag(Hcf))
    live = d > 0
    # every entry, relative to the natural scale sqrt(H_kk H_ll): pixel sum vs integral at sqrt(s2) = 12 px
    err = np.abs(Hor - Hcf)[np.ix_(live, live)] / np.outer(d[live], d[live])
    assert err.max() < 3e-4, err.max()
    # rows/columns the closed form says are exactly zero: log-scale z, quaternion, and (RGB only) nothing else
    dead = ~live
    assert np.all(np.abs(Hor[dead][:, dead]) <= 1e-9 * np.abs(Hor).max())
    assert np.all(np.abs(Hor[np.ix_(dead, live)]) <= 1e-6 * np.outer(np.ones(dead.sum()), d[live]) * np.sqrt(np.abs(Hor).max()))


def test_blocks_are_psd_and_annihilate_the_quaternion_direction(wl0):
    scn = make_oracle_scene(wl0.scene, channel_mask=15)
    H = scn.view_hessian(wl0.train_cams[0])
    F = orc.unpack_blocks(H)
    ev = np.linalg.eigvalsh(F)
    tr = np.trace(F, axis1=1, axis2=2)
    assert np.all(ev[:, 0] >= -1e-9 * np.maximum(tr, 1e-300))  # PSD
    # the rendering is invariant to scaling the raw quaternion: H (0,..,q,..,0) = 0 (reading R-10)
    q = np.zeros((wl0.scene.N, P))
    q[:, 6:10] = wl0.scene.quat
    Hq = np.einsum("nij,nj->ni", F, q)
    scale = np.sqrt(np.maximum(np.einsum("nii->ni", F), 0)) * np.sqrt(np.maximum(F[:, 6:10, 6:10].trace(axis1=1, axis2=2), 0))[:, None]
    assert np.all(np.abs(Hq) <= 1e-7 * scale + 1e-12)
    assert np.all(np.linalg.matrix_rank(F[tr > 0][:50]) <= 13)


def test_invisible_gaussians_have_zero_blocks_and_visible_ones_do_not(wl0):
    scn = make_oracle_scene(wl0.scene)
    cam = wl0.train_cams[0]
    offsets, ids, _ = scn.trace(cam)
    H = scn.view_hessian(cam)
    seen = np.zeros(wl0.scene.N, dtype=bool)
    seen[ids] = True
    assert np.all(H[~seen] == 0)  # S:L294 (culled or fully occluded)
    assert np.all(np.abs(H[seen]).sum(axis=1) > 0)
    assert 0 < seen.sum() < wl0.scene.N


def test_two_identical_views_double_every_block(wl0):
    scn = make_oracle_scene(wl0.scene)
    cam = wl0.train_cams[0]
    H1 = scn.view_hessian(cam)
    H2 = scn.view_hessian(cam, out=H1.copy())
    # S:L315; the band-ordered accumulation is run-to-run deterministic, and x + x = 2x exactly
    assert np.array_equal(H2, 2 * H1)
    assert np.array_equal(scn.view_hessian(cam), H1)


def test_channel_additivity_rgb_plus_depth(wl0):
    cam = wl0.cand_cams[1]
    Hrgb = make_oracle_scene(wl0.scene, channel_mask=7).view_hessian(cam)
    Hd = make_oracle_scene(wl0.scene, channel_mask=8).view_hessian(cam)
    Hall = make_oracle_scene(wl0.scene, channel_mask=15).view_hessian(cam)
    np.testing.assert_allclose(Hrgb + Hd, Hall, rtol=1e-12, atol=1e-14)
    # depth uses no colour parameter: its rgb rows/cols are zero
    F = orc.unpack_blocks(Hd)
    assert np.all(F[:, 11:, :] == 0)


def test_doubling_resolution_quadruples_the_trace():
    sc = scene_from_arrays([[0.0, 0.0, 1.0]], [[np.log(0.05)] * 3], [[0.9, 0.1, 0.3, 0.2]], [0.5], [[0.4, 0.6, 0.8]])
    # derivatives w.r.t. opacity and colour are resolution independent per pixel -> their diagonal sums scale with pixel count
    tr = []
    for W, f in ((64, 100.0), (128, 200.0)):
        cam = synth.simple_camera(W, W, f, dist=0.0)
        F = orc.unpack_blocks(make_oracle_scene(sc).view_hessian(cam))[0]
        tr.append(np.trace(F[10:, 10:]))
    assert 3.0 < tr[1] / tr[0] < 5.0


def test_rank_is_bounded_by_channels_times_pixels():
    sc = scene_from_arrays([[0.0, 0.0, 1.0]], [[np.log(0.01)] * 3], [[1, 0, 0, 0]], [0.5], [[0.4, 0.6, 0.8]])
    cam = synth.simple_camera(2, 2, 20.0, dist=0.0)  # 4 pixels, RGB -> rank <= 12
    F = orc.unpack_blocks(make_oracle_scene(sc).view_hessian(cam))[0]
    assert np.linalg.matrix_rank(F) <= 12
    mask = np.zeros((2, 2), dtype=np.uint8)
    mask[0, 0] = 1
    F1 = orc.unpack_blocks(make_oracle_scene(sc).view_hessian(cam, pixel_mask=mask))[0]
    assert 0 < np.linalg.matrix_rank(F1) <= 3
