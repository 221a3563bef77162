"""Seeded synthetic inputs: Gaussian clouds with object vectors, and hemisphere cameras.

This module serves BOTH the CUDA path (tests, bench) and the CPU oracle.  It
holds none of the method's arithmetic: it only draws random arrays with the
shapes and value distributions BASELINE.json's five configs state and builds
look-at camera poses.  numpy only.

The inputs stand in for the paper's workloads (BlenderProc+BOP synthetic
scenes, GraspNet scenes with a 1280x720 RealSense-class camera, and
robot-captured scenes; section IV.A.1), none of which is in
this container.  Recipe:

  scene box        [-0.3,0.3]^2 x [0,0.2] m
  object centres   c_k ~ U(box)
  object id        ~ U{0..K-1} per Gaussian
  mean             ~ N(c_k, 0.05^2 I)
  log-scale        ~ N(ls_mean, ls_std^2)^3
  quaternion       N(0,1)^4 normalised (w,x,y,z)
  opacity          sigmoid(N(0,1))
  RGB              U(0,1)^3
  object logits    N(0,1)^K, +3 on the Gaussian's own object id
  cameras          on a hemisphere about (0,0,0.1): azimuth U[0,2pi),
                   elevation U[15deg,75deg], radius as the config says,
                   looking at the centre, up = +z, OpenCV axes
"""
from __future__ import annotations

import dataclasses
import numpy as np

# Host-side camera record; same field order as `nbv_camera` in include/nbv.h
# (width, height, fx, fy, cx, cy, R_cw[9] row-major world->camera, t_cw[3]).
CAMERA_DTYPE = np.dtype(
    [
        ("width", "<i4"),
        ("height", "<i4"),
        ("fx", "<f4"),
        ("fy", "<f4"),
        ("cx", "<f4"),
        ("cy", "<f4"),
        ("R", "<f4", (9,)),
        ("t", "<f4", (3,)),
    ]
)
assert CAMERA_DTYPE.itemsize == 72

CH_RGB = 7
CH_RGBD = 15


@dataclasses.dataclass
class Scene:
    """Gaussian map G with object vectors (section III.A.1), SH degree 0."""

    mean: np.ndarray  # (N,3) f32
    logscale: np.ndarray  # (N,3) f32
    quat: np.ndarray  # (N,4) f32 w,x,y,z
    opacity: np.ndarray  # (N,)  f32 in (0,1)
    rgb: np.ndarray  # (N,3) f32
    obj_logits: np.ndarray  # (N,K) f32
    obj_id: np.ndarray  # (N,)  i32  generator's ground-truth id (not an input of the method)

    @property
    def N(self) -> int:
        return int(self.mean.shape[0])

    @property
    def K(self) -> int:
        return int(self.obj_logits.shape[1])

    def subset(self, idx) -> "Scene":
        return Scene(*(getattr(self, f.name)[idx].copy() for f in dataclasses.fields(self)))


@dataclasses.dataclass
class Workload:
    name: str
    scene: Scene
    train_cams: np.ndarray  # CAMERA_DTYPE (T,)
    cand_cams: np.ndarray  # CAMERA_DTYPE (C,)
    channel_mask: int  # CH_RGB or CH_RGBD
    target_obj: int  # -1 = whole scene
    seed: int


CONFIGS = {
    # index: BASELINE.json configs[index]
    0: dict(name="tiny", N=2_000, K=3, W=64, H=64, fx=None, fov_deg=60.0, T=1, C=4,
            radius=(0.6, 0.6), ls=(-4.0, 0.5), channels=CH_RGB, target=False),
    1: dict(name="tabletop", N=50_000, K=10, W=640, H=480, fx=None, fov_deg=60.0, T=10, C=20,
            radius=(0.5, 0.8), ls=(-4.0, 0.5), channels=CH_RGB, target=False),
    2: dict(name="graspnet", N=200_000, K=20, W=1280, H=720, fx=910.0, fov_deg=None, T=20, C=64,
            radius=(0.5, 0.8), ls=(-4.0, 0.5), channels=CH_RGBD, target=False),
    3: dict(name="object_centric", N=200_000, K=20, W=1280, H=720, fx=910.0, fov_deg=None, T=20, C=64,
            radius=(0.5, 0.8), ls=(-4.0, 0.5), channels=CH_RGBD, target=True),
    4: dict(name="stress", N=1_000_000, K=50, W=1280, H=720, fx=910.0, fov_deg=None, T=50, C=256,
            radius=(0.5, 0.8), ls=(-5.0, 0.7), channels=CH_RGB, target=False),
}

BOX_LO = np.array([-0.3, -0.3, 0.0])
BOX_HI = np.array([0.3, 0.3, 0.2])
LOOK_AT = np.array([0.0, 0.0, 0.1])


def make_scene(N: int, K: int, ls_mean: float, ls_std: float, rng: np.random.Generator,
               centres: np.ndarray | None = None, cluster_std: np.ndarray | None = None) -> Scene:
    if centres is None:
        centres = rng.uniform(BOX_LO, BOX_HI, size=(K, 3))
    if cluster_std is None:
        cluster_std = np.full(K, 0.05)
    obj_id = rng.integers(0, K, size=N)
    mean = centres[obj_id] + rng.standard_normal((N, 3)) * cluster_std[obj_id, None]
    logscale = ls_mean + ls_std * rng.standard_normal((N, 3))
    q = rng.standard_normal((N, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    opacity = 1.0 / (1.0 + np.exp(-rng.standard_normal(N)))
    rgb = rng.uniform(0.0, 1.0, size=(N, 3))
    logits = rng.standard_normal((N, K))
    logits[np.arange(N), obj_id] += 3.0
    f32 = np.float32
    opacity = np.clip(opacity.astype(f32), f32(1e-6), f32(1.0 - 1e-6))
    return Scene(mean.astype(f32), logscale.astype(f32), q.astype(f32), opacity,
                 rgb.astype(f32), logits.astype(f32), obj_id.astype(np.int32))


def look_at_camera(pos, target, W: int, H: int, fx: float, fy: float, cx: float, cy: float) -> np.ndarray:
    """One CAMERA_DTYPE record: OpenCV axes (+x right, +y down, +z forward), world up = +z."""
    pos = np.asarray(pos, dtype=np.float64)
    fwd = np.asarray(target, dtype=np.float64) - pos
    fwd /= np.linalg.norm(fwd)
    up = np.array([0.0, 0.0, 1.0])
    right = np.cross(fwd, up)
    nr = np.linalg.norm(right)
    if nr < 1e-9:  # looking straight down/up: any horizontal right vector
        right = np.array([1.0, 0.0, 0.0])
    else:
        right /= nr
    down = np.cross(fwd, right)
    R = np.stack([right, down, fwd])  # rows: camera axes in world coordinates
    t = -R @ pos
    cam = np.zeros((), dtype=CAMERA_DTYPE)
    cam["width"], cam["height"] = W, H
    cam["fx"], cam["fy"], cam["cx"], cam["cy"] = fx, fy, cx, cy
    cam["R"] = R.reshape(9)
    cam["t"] = t
    return cam


def hemisphere_cameras(n: int, radius, W: int, H: int, fx: float, fy: float,
                       rng: np.random.Generator, centre=LOOK_AT) -> np.ndarray:
    cams = np.zeros(n, dtype=CAMERA_DTYPE)
    for i in range(n):
        az = rng.uniform(0.0, 2.0 * np.pi)
        el = np.deg2rad(rng.uniform(15.0, 75.0))
        r = rng.uniform(radius[0], radius[1]) if radius[1] > radius[0] else radius[0]
        pos = centre + r * np.array([np.cos(el) * np.cos(az), np.cos(el) * np.sin(az), np.sin(el)])
        cams[i] = look_at_camera(pos, centre, W, H, fx, fy, W / 2.0, H / 2.0)
    return cams


def _intrinsics(c) -> float:
    if c["fx"] is not None:
        return float(c["fx"])
    return float((c["W"] / 2.0) / np.tan(np.deg2rad(c["fov_deg"]) / 2.0))


def make_workload(config: int, seed: int | None = None, n_gaussians: int | None = None,
                  n_train: int | None = None, n_cand: int | None = None) -> Workload:
    """BASELINE.json configs[config]; the optional overrides shrink it for tests/samples."""
    c = CONFIGS[config]
    # config 3 is "the scene of config 2" -> same stream as config 2 unless a seed is given
    seed = (2 if config == 3 else config) if seed is None else seed
    rng = np.random.default_rng(seed)
    N = c["N"] if n_gaussians is None else n_gaussians
    K = c["K"]
    target = -1
    centres = rng.uniform(BOX_LO, BOX_HI, size=(K, 3))
    cluster_std = np.full(K, 0.05)
    if c["target"]:
        # object-centric NBV: a small target cluster (< 3% of the 1280x720 pixels at
        # 0.5-0.8 m: +-2 sigma = 0.08 m ~ 110 px across) with three other objects
        # overlapping it from above / outside, so it is partly occluded.
        trng = np.random.default_rng(seed + 1000)
        target = int(trng.integers(0, K))
        cluster_std[target] = 0.02
        centres[target] = np.array([trng.uniform(-0.1, 0.1), trng.uniform(-0.1, 0.1), 0.03])
        others = [k for k in range(K) if k != target][:3]
        for j, k in enumerate(others):
            ang = 2.0 * np.pi * j / 3.0 + trng.uniform(0.0, 0.5)
            d = trng.uniform(0.06, 0.10)
            centres[k] = centres[target] + np.array([d * np.cos(ang), d * np.sin(ang), trng.uniform(0.04, 0.08)])
    scene = make_scene(N, K, c["ls"][0], c["ls"][1], rng, centres, cluster_std)
    f = _intrinsics(c)
    T = c["T"] if n_train is None else n_train
    C = c["C"] if n_cand is None else n_cand
    # cameras always drawn for the full config so that shrinking T/C keeps a prefix
    train = hemisphere_cameras(c["T"], c["radius"], c["W"], c["H"], f, f, rng)[:T]
    cand = hemisphere_cameras(c["C"], c["radius"], c["W"], c["H"], f, f, rng)[:C]
    return Workload(c["name"], scene, train, cand, c["channels"], target, seed)


def micro_scene(n: int, seed: int, spread: float = 0.03, ls_mean: float = -3.5, K: int = 2) -> Scene:
    """A handful of Gaussians near the origin, for finite-difference and edge-case tests."""
    rng = np.random.default_rng(seed)
    centres = np.zeros((K, 3))
    return make_scene(n, K, ls_mean, 0.3, rng, centres, np.full(K, spread))


def simple_camera(W: int, H: int, f: float, dist: float = 0.5) -> np.ndarray:
    """Camera on the +z axis side looking at the origin along -z_world... expressed as identity
    rotation with the scene pushed `dist` in front: R = I, t = (0,0,dist)."""
    cam = np.zeros((), dtype=CAMERA_DTYPE)
    cam["width"], cam["height"] = W, H
    cam["fx"], cam["fy"], cam["cx"], cam["cy"] = f, f, W / 2.0, H / 2.0
    cam["R"] = np.eye(3).reshape(9)
    cam["t"] = (0.0, 0.0, dist)
    return cam
