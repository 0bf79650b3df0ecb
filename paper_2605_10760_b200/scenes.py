"""Seeded synthetic input generators (numpy only) shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NONE of the method's arithmetic (no projection, no compositing, no gradients): it only draws the
inputs of the hot path -- Gaussians (mu, s, q, opacity, colour/SH; Eq. 19), a pinhole
camera with a world-to-camera pose T_k (intrinsics PAPER.md:420) and upstream image gradients -- with
the shapes of BASELINE.json `configs` (recipes restated in DESIGN.md "Input recipe").  The paper's Replica-derived
data are not available; these scenes stand in for them (only the shapes 1200x680 / HFOV 90 deg => f = 600 are taken).

Every array is float32, C-contiguous, drawn from one numpy Generator(PCG64(seed)) in a fixed order.
"""
from __future__ import annotations

import dataclasses
import numpy as np

SH_C0 = 0.5 / np.sqrt(np.pi)  # degree-0 real SH basis value, used only to turn a drawn RGB into a DC coefficient


@dataclasses.dataclass
class Camera:
    width: int
    height: int
    fx: float
    fy: float
    cx: float
    cy: float
    T_cw: np.ndarray  # float32 [3,4] row-major [R|t], p_c = R p_w + t  (world-to-camera)
    near_z: float = 0.2

    def copy(self) -> "Camera":
        return dataclasses.replace(self, T_cw=self.T_cw.copy())


@dataclasses.dataclass
class Scene:
    means: np.ndarray      # [N,3]
    scales: np.ndarray     # [N,3] activated (linear, > 0)
    quats: np.ndarray      # [N,4] (w,x,y,z), not normalised
    opacities: np.ndarray  # [N]   activated, in (0,1)
    sh: np.ndarray         # [N,K,3], K = (sh_degree+1)^2
    sh_degree: int
    camera: Camera
    bg: np.ndarray         # [3]
    name: str = ""

    @property
    def N(self) -> int:
        return int(self.means.shape[0])


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _sigmoid(x):
    return 1.0 / (1.0 + np.exp(-x))


def identity_pose() -> np.ndarray:
    T = np.zeros((3, 4), dtype=np.float32)
    T[0, 0] = T[1, 1] = T[2, 2] = 1.0
    return T


def look_at(eye, target, up=(0.0, 0.0, 1.0)) -> np.ndarray:
    """World-to-camera [R|t] for a camera at `eye` looking at `target`; x right, y down, z forward."""
    eye = np.asarray(eye, dtype=np.float64)
    fwd = np.asarray(target, dtype=np.float64) - eye
    fwd /= np.linalg.norm(fwd)
    right = np.cross(fwd, np.asarray(up, dtype=np.float64))
    right /= np.linalg.norm(right)
    down = np.cross(fwd, right)
    R = np.stack([right, down, fwd], axis=0)
    T = np.concatenate([R, (-R @ eye)[:, None]], axis=1)
    return _f32(T)


def se3_exp(xi) -> tuple[np.ndarray, np.ndarray]:
    """(R, V rho) of Exp(xi^), xi = (rho, phi); used only to PERTURB input poses (config 4 recipe)."""
    xi = np.asarray(xi, dtype=np.float64)
    rho, phi = xi[:3], xi[3:]
    th = np.linalg.norm(phi)
    K = np.array([[0, -phi[2], phi[1]], [phi[2], 0, -phi[0]], [-phi[1], phi[0], 0]])
    if th < 1e-8:
        A, B, C = 1.0 - th * th / 6, 0.5 - th * th / 24, 1.0 / 6 - th * th / 120
    else:
        A, B, C = np.sin(th) / th, (1 - np.cos(th)) / th**2, (th - np.sin(th)) / th**3
    R = np.eye(3) + A * K + B * K @ K
    V = np.eye(3) + B * K + C * K @ K
    return R, V @ rho


def perturb_pose(T_cw: np.ndarray, xi) -> np.ndarray:
    """T <- Exp(xi^) T (left-multiplicative twist on the world-to-camera pose)."""
    R, t = se3_exp(xi)
    W = T_cw[:, :3].astype(np.float64)
    tt = T_cw[:, 3].astype(np.float64)
    return _f32(np.concatenate([R @ W, (R @ tt + t)[:, None]], axis=1))


def rgb_to_sh0(rgb):
    return (rgb - 0.5) / SH_C0


# ----------------------------------------------------------------------------------------------------------------
# config 1: tiny scene
# ----------------------------------------------------------------------------------------------------------------
def tiny_scene(seed: int = 1, N: int = 256, size: int = 64) -> Scene:
    rng = np.random.Generator(np.random.PCG64(seed))
    xy = rng.uniform(-1.0, 1.0, size=(N, 2))
    z = rng.uniform(2.0, 4.0, size=(N, 1))
    means = np.concatenate([xy, z], axis=1)
    scales = np.exp(rng.normal(-3.0, 0.3, size=(N, 3)))
    quats = rng.normal(size=(N, 4))
    opac = _sigmoid(rng.normal(0.0, 1.0, size=N))
    rgb = rng.uniform(0.0, 1.0, size=(N, 3))
    cam = Camera(size, size, float(size), float(size), size / 2.0, size / 2.0, identity_pose())
    return Scene(_f32(means), _f32(scales), _f32(quats), _f32(opac), _f32(rgb_to_sh0(rgb)[:, None, :]), 0, cam,
                 np.zeros(3, np.float32), name=f"tiny{N}_{size}x{size}_seed{seed}")


# ----------------------------------------------------------------------------------------------------------------
# config 2: monocular keyframe mapping
# ----------------------------------------------------------------------------------------------------------------
def mono_scene(seed: int = 2, N: int = 50_000, width: int = 640, height: int = 480, f: float = 525.0) -> Scene:
    rng = np.random.Generator(np.random.PCG64(seed))
    cx, cy = width / 2.0, height / 2.0
    u = rng.uniform(0.0, width, size=N)
    v = rng.uniform(0.0, height, size=N)
    z = rng.uniform(0.5, 6.0, size=N)
    means = np.stack([(u - cx) * z / f, (v - cy) * z / f, z], axis=1)
    scales = np.exp(rng.normal(-4.0, 0.5, size=(N, 3)))
    quats = rng.normal(size=(N, 4))
    opac = _sigmoid(rng.normal(0.0, 1.5, size=N))
    rgb = rng.uniform(0.0, 1.0, size=(N, 3))
    cam = Camera(width, height, f, f, cx, cy, identity_pose())
    return Scene(_f32(means), _f32(scales), _f32(quats), _f32(opac), _f32(rgb_to_sh0(rgb)[:, None, :]), 0, cam,
                 np.zeros(3, np.float32), name=f"mono{N}_{width}x{height}_seed{seed}")


def mono_targets(seed: int, width: int, height: int):
    """Seeded random targets of config 2: RGB ~ U[0,1], depth ~ U[0.5,6]."""
    rng = np.random.Generator(np.random.PCG64(seed + 7919))
    return _f32(rng.uniform(0.0, 1.0, size=(3, height, width))), _f32(rng.uniform(0.5, 6.0, size=(height, width)))


# ----------------------------------------------------------------------------------------------------------------
# config 3 (and the Gaussian sets of configs 4, 5): Replica-shaped room
# ----------------------------------------------------------------------------------------------------------------
ROOM = np.array([8.0, 6.0, 3.0])


def _unit(v):
    return v / np.linalg.norm(v, axis=-1, keepdims=True)


def _replica_gaussians(rng, N: int, sh_degree: int, patches: int = 64):
    centres = rng.uniform(0.0, 1.0, size=(patches, 3)) * ROOM
    normals = _unit(rng.normal(size=(patches, 3)))
    helper = np.where(np.abs(normals[:, :1]) < 0.9, np.array([[1.0, 0, 0]]), np.array([[0, 1.0, 0]]))
    t1 = _unit(np.cross(normals, helper))
    t2 = np.cross(normals, t1)
    pid = np.arange(N) % patches
    g = rng.normal(size=(N, 3))
    means = centres[pid] + 0.3 * (g[:, :1] * t1[pid] + g[:, 1:2] * t2[pid]) + 0.01 * g[:, 2:3] * normals[pid]
    scales = np.exp(rng.normal(-4.5, 0.5, size=(N, 3)))
    quats = rng.normal(size=(N, 4))
    opac = _sigmoid(rng.normal(1.0, 1.0, size=N))
    K = (sh_degree + 1) ** 2
    sh = rng.normal(0.0, 0.2, size=(N, K, 3))
    return means, scales, quats, opac, sh, centres


def _replica_camera(rng, centres, width, height, f):
    eye = (0.25 + 0.5 * rng.uniform(0.0, 1.0, size=3)) * ROOM
    target = centres[int(rng.integers(0, centres.shape[0]))]
    return Camera(width, height, f, f, (width - 1) / 2.0, (height - 1) / 2.0, look_at(eye, target))


def replica_scene(seed: int = 30, N: int = 300_000, width: int = 1200, height: int = 680, f: float = 600.0,
                  sh_degree: int = 3) -> Scene:
    rng = np.random.Generator(np.random.PCG64(seed))
    means, scales, quats, opac, sh, centres = _replica_gaussians(rng, N, sh_degree)
    cam = _replica_camera(rng, centres, width, height, f)
    return Scene(_f32(means), _f32(scales), _f32(quats), _f32(opac), _f32(sh), sh_degree, cam,
                 np.zeros(3, np.float32), name=f"replica{N}_{width}x{height}_sh{sh_degree}_seed{seed}")


def tracking_perturbation(seed: int):
    """Config 4: twist with |rho| = 2 cm (random direction) and |phi| = 1 degree (random axis)."""
    rng = np.random.Generator(np.random.PCG64(seed + 104729))
    rho = _unit(rng.normal(size=3)) * 0.02
    phi = _unit(rng.normal(size=3)) * np.deg2rad(1.0)
    return np.concatenate([rho, phi])


def fused_scene(seed: int = 50, N_sub: int = 500_000, submaps: int = 4, views: int = 8, width: int = 1200,
                height: int = 680, f: float = 600.0, sh_degree: int = 3):
    """Config 5: union of `submaps` Replica-shaped submaps, each already mapped by a Sim(3) (Eq. 19, PAPER.md:239:
    mu' = s R mu + t, s_i' = s s_i, rotation composed into the quaternion; opacity and colour unchanged), and `views`
    cameras.  Returns (scene_with_first_camera, [cameras])."""
    rng = np.random.Generator(np.random.PCG64(seed))
    parts, all_centres = [], []
    centre = ROOM / 2.0
    for _ in range(submaps):
        means, scales, quats, opac, sh, centres = _replica_gaussians(rng, N_sub, sh_degree)
        s = float(np.exp(rng.uniform(np.log(0.5), np.log(2.0))))
        yaw = float(rng.uniform(-np.pi, np.pi))
        t = rng.uniform(-1.0, 1.0, size=3) * np.array([1.0, 1.0, 0.25])
        c, sn = np.cos(yaw), np.sin(yaw)
        R = np.array([[c, -sn, 0.0], [sn, c, 0.0], [0.0, 0.0, 1.0]])
        means = (s * (means - centre) @ R.T) + centre + t
        centres = (s * (centres - centre) @ R.T) + centre + t
        scales = s * scales
        qy = np.array([np.cos(yaw / 2), 0.0, 0.0, np.sin(yaw / 2)])  # yaw quaternion composed on the left
        w1, x1, y1, z1 = qy
        w2, x2, y2, z2 = quats.T
        quats = np.stack([w1 * w2 - x1 * x2 - y1 * y2 - z1 * z2, w1 * x2 + x1 * w2 + y1 * z2 - z1 * y2,
                          w1 * y2 - x1 * z2 + y1 * w2 + z1 * x2, w1 * z2 + x1 * y2 - y1 * x2 + z1 * w2], axis=1)
        parts.append((means, scales, quats, opac, sh))
        all_centres.append(centres)
    cat = [np.concatenate([p[k] for p in parts], axis=0) for k in range(5)]
    centres = np.concatenate(all_centres, axis=0)
    cams = [_replica_camera(rng, centres, width, height, f) for _ in range(views)]
    scene = Scene(_f32(cat[0]), _f32(cat[1]), _f32(cat[2]), _f32(cat[3]), _f32(cat[4]), sh_degree, cams[0],
                  np.zeros(3, np.float32), name=f"fused{submaps}x{N_sub}_{views}views_seed{seed}")
    return scene, cams


def upstream_gradients(seed: int, width: int, height: int):
    """Upstream dL/dRGB [3,H,W], dL/dDepth [H,W] ~ N(0,1) (configs 1 and 3); dL/dAlpha = 0."""
    rng = np.random.Generator(np.random.PCG64(seed + 15485863))
    return _f32(rng.normal(size=(3, height, width))), _f32(rng.normal(size=(height, width)))
