"""ctypes front-end of the fp64 CPU oracle (oracle/gso.cpp).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.  It imports
nothing from paper_2605_10760_b200 (scenes are passed in duck-typed: any object with means/scales/quats/opacities/sh/
sh_degree/camera/bg attributes, camera with width/height/fx/fy/cx/cy/near_z/T_cw).
"""
from __future__ import annotations

import ctypes as C
import dataclasses
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None


class _Camera(C.Structure):
    _fields_ = [("width", C.c_int32), ("height", C.c_int32), ("fx", C.c_double), ("fy", C.c_double),
                ("cx", C.c_double), ("cy", C.c_double), ("near_z", C.c_double), ("T_cw", C.c_double * 12)]


class _Options(C.Structure):
    _fields_ = [("dilation", C.c_double), ("alpha_min", C.c_double), ("alpha_max", C.c_double), ("T_min", C.c_double),
                ("tile", C.c_int32), ("brute_force", C.c_int32), ("max_threads", C.c_int32), ("reserved", C.c_int32)]


@dataclasses.dataclass
class Options:
    dilation: float = 0.3
    alpha_min: float = 1.0 / 255.0
    alpha_max: float = 0.99
    T_min: float = 1e-4
    tile: int = 16
    brute_force: bool = False
    max_threads: int = 0

    @staticmethod
    def no_cutoffs(**kw) -> "Options":
        """Thresholds disabled (alpha_min 0, no clamp, no early exit): the smooth function used by FD pins."""
        return Options(alpha_min=0.0, alpha_max=float("inf"), T_min=0.0, **kw)

    def c(self) -> _Options:
        return _Options(self.dilation, self.alpha_min, self.alpha_max, self.T_min, self.tile, int(self.brute_force),
                        self.max_threads, 0)


def lib():
    global _LIB
    if _LIB is None:
        from . import build as _b
        _LIB = C.CDLL(_b.build())
        _LIB.gso_bin.restype = C.c_int64
    return _LIB


def _cam(cam, T_cw64=None) -> _Camera:
    """Camera struct; intrinsics and pose are the float32 values the GPU path receives, promoted to double.
    T_cw64 (3x4 float64) overrides the pose without float32 rounding (finite-difference tests only)."""
    c = _Camera()
    c.width, c.height = int(cam.width), int(cam.height)
    c.fx, c.fy = float(np.float32(cam.fx)), float(np.float32(cam.fy))
    c.cx, c.cy = float(np.float32(cam.cx)), float(np.float32(cam.cy))
    c.near_z = float(np.float32(cam.near_z))
    T = np.asarray(cam.T_cw, dtype=np.float32).astype(np.float64) if T_cw64 is None else np.asarray(T_cw64, np.float64)
    for k, v in enumerate(T.reshape(-1)[:12]):
        c.T_cw[k] = float(v)
    return c


def _p(a, ty):
    return None if a is None else a.ctypes.data_as(C.POINTER(ty))


def _f64(a):
    """Parameters go to the oracle as doubles: float32 arrays are promoted exactly; fp64 arrays (FD tests) pass through."""
    return np.ascontiguousarray(a, dtype=np.float64)


def num_threads(opt: Options = Options()) -> int:
    o = opt.c()
    return int(lib().gso_num_threads(C.byref(o)))


def sh_basis(deg: int, n):
    n = np.ascontiguousarray(n, dtype=np.float64)
    B = np.zeros(16)
    dB = np.zeros((16, 3))
    lib().gso_sh_basis(int(deg), _p(n, C.c_double), _p(B, C.c_double), _p(dB, C.c_double))
    return B, dB


def quat_to_R(q):
    q = np.ascontiguousarray(q, dtype=np.float64)
    R = np.zeros((3, 3))
    lib().gso_quat_to_R(_p(q, C.c_double), _p(R, C.c_double))
    return R


def se3_exp(xi):
    xi = np.ascontiguousarray(xi, dtype=np.float64)
    R = np.zeros((3, 3))
    t = np.zeros(3)
    lib().gso_se3_exp(_p(xi, C.c_double), _p(R, C.c_double), _p(t, C.c_double))
    return R, t


def pose_apply(xi, T_cw):
    xi = np.ascontiguousarray(xi, dtype=np.float64)
    Ti = np.ascontiguousarray(np.asarray(T_cw, dtype=np.float64).reshape(3, 4))
    To = np.zeros((3, 4))
    lib().gso_pose_apply(_p(xi, C.c_double), _p(Ti, C.c_double), _p(To, C.c_double))
    return To


def preprocess(scene, opt: Options = Options(), camera=None, T_cw64=None) -> dict:
    """Reading C1 steps 1-6, 8: per-Gaussian features in fp64 + exact pixel/tile rects + fp32 depth keys."""
    cam = camera if camera is not None else scene.camera
    N = int(scene.means.shape[0])
    out = dict(visible=np.zeros(N, np.uint8), pc=np.zeros((N, 3)), mean2d=np.zeros((N, 2)), cov2d=np.zeros((N, 3)),
               conic=np.zeros((N, 3)), color=np.zeros((N, 3)), z=np.zeros(N), z32=np.zeros(N, np.float32),
               rect_px=np.zeros((N, 4), np.int32), rect_tile=np.zeros((N, 4), np.int32))
    c, o = _cam(cam, T_cw64), opt.c()
    rc = lib().gso_preprocess(C.c_int64(N), int(scene.sh_degree), _p(_f64(scene.means), C.c_double),
                              _p(_f64(scene.scales), C.c_double), _p(_f64(scene.quats), C.c_double),
                              _p(_f64(scene.opacities), C.c_double), _p(_f64(scene.sh), C.c_double), C.byref(c),
                              C.byref(o), _p(out["visible"], C.c_uint8), _p(out["pc"], C.c_double),
                              _p(out["mean2d"], C.c_double), _p(out["cov2d"], C.c_double),
                              _p(out["conic"], C.c_double), _p(out["color"], C.c_double), _p(out["z"], C.c_double),
                              _p(out["z32"], C.c_float), _p(out["rect_px"], C.c_int32),
                              _p(out["rect_tile"], C.c_int32))
    if rc != 0:
        raise RuntimeError(f"gso_preprocess failed: {rc}")
    return out


def bin_tiles(rect_tile, z32, tiles_x: int, tiles_y: int):
    """Reading C1 step 8 / Q13: (tile, bits(z32), index)-ordered instance list and per-tile ranges."""
    rect_tile = np.ascontiguousarray(rect_tile, dtype=np.int32)
    z32 = np.ascontiguousarray(z32, dtype=np.float32)
    N = rect_tile.shape[0]
    I = lib().gso_bin(C.c_int64(N), _p(rect_tile, C.c_int32), _p(z32, C.c_float), tiles_x, tiles_y, C.c_int64(0),
                      None, None, None)
    if I < 0:
        raise RuntimeError("gso_bin: rect outside the tile grid")
    keys = np.zeros(I, np.uint64)
    ids = np.zeros(I, np.uint32)
    ranges = np.zeros((tiles_x * tiles_y, 2), np.uint32)
    lib().gso_bin(C.c_int64(N), _p(rect_tile, C.c_int32), _p(z32, C.c_float), tiles_x, tiles_y, C.c_int64(I),
                  _p(keys, C.c_uint64), _p(ids, C.c_uint32), _p(ranges, C.c_uint32))
    return keys, ids, ranges


def render(feat: dict, opacities, cam, bg, opt: Options = Options(), d_rgb=None, d_depth=None, d_alpha=None) -> dict:
    """Reading C1 step 7 (+ C2 when d_rgb is given).  `feat` holds visible, mean2d, cov2d, conic, color, z, z32."""
    N = int(feat["visible"].shape[0])
    H, W = int(cam.height), int(cam.width)
    out = dict(rgb=np.zeros((3, H, W)), depth=np.zeros((H, W)), alpha=np.zeros((H, W)),
               n_blended=np.zeros((H, W), np.int32), margin=np.zeros((H, W)))
    bwd = d_rgb is not None
    g = {}
    if bwd:
        d_rgb = np.ascontiguousarray(d_rgb, dtype=np.float64)
        d_depth = None if d_depth is None else np.ascontiguousarray(d_depth, dtype=np.float64)
        d_alpha = None if d_alpha is None else np.ascontiguousarray(d_alpha, dtype=np.float64)
        g = dict(g_mean2d=np.zeros((N, 2)), g_conic=np.zeros((N, 3)), g_opac=np.zeros(N), g_color=np.zeros((N, 3)),
                 g_z=np.zeros(N))
    c, o = _cam(cam), opt.c()
    bg64 = np.ascontiguousarray(bg, dtype=np.float64)
    d = C.c_double
    f = {k: np.ascontiguousarray(feat[k]) for k in ("visible", "mean2d", "cov2d", "conic", "color", "z", "z32")}
    rc = lib().gso_render(C.c_int64(N), _p(f["visible"], C.c_uint8), _p(f["mean2d"], d), _p(f["cov2d"], d),
                          _p(f["conic"], d), _p(_f64(opacities), C.c_double), _p(f["color"], d), _p(f["z"], d),
                          _p(f["z32"], C.c_float), C.byref(c), C.byref(o), _p(bg64, d), _p(out["rgb"], d),
                          _p(out["depth"], d), _p(out["alpha"], d), _p(out["n_blended"], C.c_int32),
                          _p(out["margin"], d), _p(d_rgb, d) if bwd else None, _p(d_depth, d), _p(d_alpha, d),
                          _p(g.get("g_mean2d"), d), _p(g.get("g_conic"), d), _p(g.get("g_opac"), d),
                          _p(g.get("g_color"), d), _p(g.get("g_z"), d))
    if rc != 0:
        raise RuntimeError(f"gso_render failed: {rc}")
    out.update(g)
    return out


def preprocess_bwd(scene, g2d: dict, opt: Options = Options(), camera=None, T_cw64=None) -> dict:
    """Readings C3 + C4: dense parameter gradients and the 6-DoF pose gradient from the 2D gradients."""
    cam = camera if camera is not None else scene.camera
    N = int(scene.means.shape[0])
    K = (int(scene.sh_degree) + 1) ** 2
    out = dict(g_means=np.zeros((N, 3)), g_scales=np.zeros((N, 3)), g_quats=np.zeros((N, 4)), g_opacities=np.zeros(N),
               g_sh=np.zeros((N, K, 3)), g_twist=np.zeros(6), g_W=np.zeros((3, 3)), g_pc_sum=np.zeros(3),
               g_v_sum=np.zeros(3))
    c, o = _cam(cam, T_cw64), opt.c()
    d = C.c_double
    gin = {k: np.ascontiguousarray(g2d[k], dtype=np.float64) for k in ("g_mean2d", "g_conic", "g_opac", "g_color", "g_z")}
    rc = lib().gso_preprocess_bwd(C.c_int64(N), int(scene.sh_degree), _p(_f64(scene.means), C.c_double),
                                  _p(_f64(scene.scales), C.c_double), _p(_f64(scene.quats), C.c_double),
                                  _p(_f64(scene.opacities), C.c_double), _p(_f64(scene.sh), C.c_double), C.byref(c),
                                  C.byref(o), _p(gin["g_mean2d"], d), _p(gin["g_conic"], d), _p(gin["g_opac"], d),
                                  _p(gin["g_color"], d), _p(gin["g_z"], d), _p(out["g_means"], d),
                                  _p(out["g_scales"], d), _p(out["g_quats"], d), _p(out["g_opacities"], d),
                                  _p(out["g_sh"], d), _p(out["g_twist"], d), _p(out["g_W"], d),
                                  _p(out["g_pc_sum"], d), _p(out["g_v_sum"], d))
    if rc != 0:
        raise RuntimeError(f"gso_preprocess_bwd failed: {rc}")
    return out


def forward(scene, opt: Options = Options(), camera=None, T_cw64=None) -> dict:
    """Whole forward: features + image.  Returns the feature dict with the image entries merged in."""
    cam = camera if camera is not None else scene.camera
    feat = preprocess(scene, opt, cam, T_cw64)
    img = render(feat, scene.opacities, cam, scene.bg, opt)
    return {**feat, **img}


def forward_backward(scene, d_rgb, d_depth, d_alpha=None, opt: Options = Options(), camera=None) -> dict:
    """Whole fwd+bwd: image, 2D gradients, dense parameter gradients, pose gradient."""
    cam = camera if camera is not None else scene.camera
    feat = preprocess(scene, opt, cam)
    img = render(feat, scene.opacities, cam, scene.bg, opt, d_rgb, d_depth, d_alpha)
    grads = preprocess_bwd(scene, img, opt, cam)
    return {**feat, **img, **grads}
