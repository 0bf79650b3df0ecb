"""Thin ctypes binding of libgs.so (include/gs.h).  Argument marshalling only: every step of the hot path runs in the
CUDA kernels of csrc/.  torch is used for device memory and streams, nothing else.  There is no CPU fallback: if the
library is missing or no CUDA device is present the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

GS_ACCUMULATE = 1
GS_POSE_ONLY = 2
GS_SPARSE_GRADS = 4
GS_TILE = 16

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgs.so")
_lib = None

STATUS = {0: "GS_OK", -1: "GS_E_INVALID", -2: "GS_E_ORDER", -3: "GS_E_CUDA", -4: "GS_E_NOMEM", -5: "GS_E_OVERFLOW",
          -6: "GS_E_TOO_LARGE"}

EXPORTS = ["gs_create", "gs_destroy", "gs_last_error", "gs_preprocess", "gs_bin_tiles", "gs_rasterize_fwd",
           "gs_rasterize_bwd", "gs_pose_grad", "gs_get_counts", "gs_get_binning", "gs_get_features", "gs_poll",
           "gs_aux_l1_grad", "gs_aux_pose_step", "gs_fwd_bwd_host", "gs_fwd_bwd_host_async", "gs_profile_enable", "gs_profile_read",
           "gs_get_launch_count", "gs_get_workload", "gs_loss_map", "gs_loss_iso", "gs_sim3_apply", "gs_measure_peaks", "gs_loss_refine", "gs_voxel_set_clear", "gs_voxel_insert_boxes",
           "gs_voxel_insert_rays", "gs_voxel_retain", "gs_adam_step", "gs_prune_mask", "gs_compact_work_bytes",
           "gs_compact_plan", "gs_compact_rows", "gs_loss_normal", "gs_set_option", "gs_refine_views", "gs_visible_ids", "gs_adam_step_sparse", "gs_get_visible_ids",
           "gs_compact_plan_static", "gs_compact_plan_static_max"]
GS_OPT_EXACT_TILE_CULL = 1
GS_OPT_VIEW_STREAMS = 2
PEAKS = ["fma_tlanes", "issue_twarp", "ex2_tlanes", "lds128_bcast_twarp", "lds128_twarp", "lds32_bcast_twarp",
         "lds64_bcast_twarp", "red_glanes", "hbm_read_gbs", "hbm_write_gbs", "hbm_copy_gbs", "sm_count", "sm_mhz_max"]
STAGES = ["preprocess", "tile_scan", "emit", "tile_sort", "raster_fwd", "raster_bwd", "gauss_bwd", "pose_grad"]


class GsError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{STATUS.get(code, code)}: {msg}")
        self.code = code


class gs_camera(C.Structure):
    _fields_ = [("width", C.c_int32), ("height", C.c_int32), ("fx", C.c_float), ("fy", C.c_float), ("cx", C.c_float),
                ("cy", C.c_float), ("near_z", C.c_float), ("T_cw", C.c_float * 12)]


class gs_gaussians(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in ("means", "scales", "quats", "opacities", "sh")]


class gs_refine_batch(C.Structure):
    _fields_ = [("n_views", C.c_int32), ("cams", C.POINTER(gs_camera)), ("T_cw_dev", C.c_void_p), ("target_rgb", C.c_void_p),
                ("target_depth", C.c_void_p), ("normal_prior", C.c_void_p), ("ab", C.c_void_p), ("alpha_p", C.c_float),
                ("lambda_", C.c_float), ("beta", C.c_float), ("lambda_n", C.c_float)]


class gs_adam_config(C.Structure):
    _fields_ = [("lr_means", C.c_float), ("lr_scales", C.c_float), ("lr_quats", C.c_float), ("lr_opacities", C.c_float),
                ("lr_sh", C.c_float), ("beta1", C.c_float), ("beta2", C.c_float), ("eps", C.c_float), ("step", C.c_int32)]


def load_library():
    """Loads libgs.so (no build, no fallback).  Raises if it is missing: build it with paper_2605_10760_b200/build.py."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2605_10760_b200.build` (nvcc, sm_100a). "
                           "There is no CPU fallback.")
    lib = C.CDLL(LIB_PATH)
    vp, i64, u32, f = C.c_void_p, C.c_int64, C.c_uint32, C.c_float
    lib.gs_create.argtypes = [C.POINTER(vp), C.c_int]
    lib.gs_destroy.argtypes = [vp]
    lib.gs_last_error.argtypes = [vp]
    lib.gs_last_error.restype = C.c_char_p
    lib.gs_preprocess.argtypes = [vp, vp, i64, C.c_int, vp, vp, vp, vp, vp, C.POINTER(gs_camera), vp]
    lib.gs_bin_tiles.argtypes = [vp, vp]
    lib.gs_rasterize_fwd.argtypes = [vp, vp, C.POINTER(f * 3), vp, vp, vp]
    lib.gs_rasterize_bwd.argtypes = [vp, vp, vp, vp, vp, u32, vp, vp, vp, vp, vp]
    lib.gs_pose_grad.argtypes = [vp, vp, u32, vp]
    lib.gs_get_counts.argtypes = [vp, vp, C.POINTER(i64), C.POINTER(i64)]
    lib.gs_get_binning.argtypes = [vp, vp, vp, vp, vp]
    lib.gs_get_features.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp]
    lib.gs_poll.argtypes = [vp]
    lib.gs_set_option.argtypes = [vp, C.c_int, C.c_int]
    lib.gs_aux_l1_grad.argtypes = [vp, i64, vp, vp, f, vp]
    lib.gs_aux_pose_step.argtypes = [vp, vp, vp, f]
    lib.gs_loss_map.argtypes = [vp, C.c_int32, C.c_int32, vp, vp, vp, vp, f, f, vp, vp, vp]
    lib.gs_loss_iso.argtypes = [vp, i64, vp, f, vp, vp]
    lib.gs_loss_refine.argtypes = [vp, C.c_int32, C.c_int32, vp, vp, vp, vp, vp, f, f, f, vp, vp, vp, vp, vp]
    lib.gs_sim3_apply.argtypes = [vp, i64, f, C.POINTER(f * 9), C.POINTER(f * 3), vp, vp, vp, vp, vp, vp]
    lib.gs_profile_enable.argtypes = [vp, C.c_int]
    lib.gs_profile_read.argtypes = [vp, C.POINTER(f * 8)]
    lib.gs_get_launch_count.argtypes = [vp, C.POINTER(C.c_uint64)]
    lib.gs_get_workload.argtypes = [vp, vp, C.POINTER(C.c_uint64 * 7)]
    lib.gs_voxel_set_clear.argtypes = [vp, vp, i64]
    lib.gs_voxel_insert_boxes.argtypes = [vp, vp, i64, f, f, i64, vp, vp, vp]
    lib.gs_voxel_insert_rays.argtypes = [vp, vp, i64, f, C.POINTER(gs_camera), vp, C.c_int32, vp]
    lib.gs_voxel_retain.argtypes = [vp, vp, i64, vp, i64, f, i64, vp, vp]
    lib.gs_adam_step.argtypes = [vp, i64, C.c_int, C.POINTER(gs_adam_config), C.POINTER(gs_gaussians), C.POINTER(gs_gaussians),
                                 C.POINTER(gs_gaussians), C.POINTER(gs_gaussians), vp]
    lib.gs_prune_mask.argtypes = [vp, i64, vp, f, vp]
    lib.gs_compact_work_bytes.argtypes = [i64]
    lib.gs_compact_plan.argtypes = [vp, i64, vp, vp, vp, vp]
    lib.gs_compact_rows.argtypes = [vp, i64, C.c_int32, vp, vp, vp]
    lib.gs_compact_plan_static.argtypes = [vp, i64, vp, vp, vp]
    lib.gs_compact_plan_static_max.argtypes = []
    lib.gs_loss_normal.argtypes = [vp, C.c_int32, C.c_int32, f, f, f, f, vp, vp, f, vp, vp, vp]
    lib.gs_visible_ids.argtypes = [vp, C.POINTER(vp), C.POINTER(vp)]
    lib.gs_get_visible_ids.argtypes = [vp, vp, vp]
    lib.gs_adam_step_sparse.argtypes = [vp, i64, C.c_int, C.POINTER(gs_adam_config), C.POINTER(gs_gaussians), C.POINTER(gs_gaussians),
                                        C.POINTER(gs_gaussians), C.POINTER(gs_gaussians), vp, vp, i64]
    lib.gs_refine_views.argtypes = [vp, vp, i64, C.c_int, C.POINTER(gs_gaussians), C.POINTER(gs_refine_batch), C.POINTER(f * 3),
                                    C.POINTER(gs_gaussians), vp, vp, vp, vp]
    lib.gs_measure_peaks.argtypes = [C.c_int, vp, C.POINTER(C.c_double * len(PEAKS))]
    lib.gs_fwd_bwd_host.argtypes = [vp, vp, i64, C.c_int, vp, vp, vp, vp, vp, C.POINTER(gs_camera), C.POINTER(f * 3)] + [vp] * 11
    lib.gs_fwd_bwd_host_async.argtypes = lib.gs_fwd_bwd_host.argtypes
    for name in EXPORTS:
        if name not in ("gs_last_error", "gs_compact_work_bytes", "gs_compact_plan_static_max"):
            getattr(lib, name).restype = C.c_int
    lib.gs_compact_work_bytes.restype = C.c_int64
    lib.gs_compact_plan_static_max.restype = C.c_int64
    _lib = lib
    return lib


def camera_struct(cam) -> gs_camera:
    c = gs_camera()
    c.width, c.height = int(cam.width), int(cam.height)
    c.fx, c.fy, c.cx, c.cy, c.near_z = float(cam.fx), float(cam.fy), float(cam.cx), float(cam.cy), float(cam.near_z)
    T = np.asarray(cam.T_cw, dtype=np.float32).reshape(-1)
    for k in range(12):
        c.T_cw[k] = float(T[k])
    return c


def _ptr(t, dtype=None):
    """Device pointer of a contiguous CUDA tensor (or None)."""
    if t is None:
        return None
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda or not t.is_contiguous():
        raise TypeError("expected a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise TypeError(f"expected dtype {dtype}, got {t.dtype}")
    return C.c_void_p(t.data_ptr())


def _stream(stream=None):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _bg(bg):
    if bg is None:
        return None
    b = np.asarray(bg, dtype=np.float32).reshape(3)
    return (C.c_float * 3)(float(b[0]), float(b[1]), float(b[2]))


class Context:
    """Owns a gs_ctx.  The five calls below carry the names and argument order of include/gs.h."""

    def __init__(self, device: int = 0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: the 3DGS path runs only in the sm_100a kernels of libgs.so (no CPU fallback)")
        self.lib = load_library()
        self.device = device
        self._h = C.c_void_p()
        rc = self.lib.gs_create(C.byref(self._h), device)
        if rc != 0:
            raise GsError(rc, "gs_create failed")
        self._keep = None

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self.lib.gs_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc):
        if rc != 0:
            raise GsError(rc, self.lib.gs_last_error(self._h).decode())

    # -- the five calls ------------------------------------------------------------------------------------------
    def gs_preprocess(self, means, scales, quats, opacities, sh, sh_degree, cam, T_cw_dev=None, stream=None):
        import torch
        N = int(means.shape[0])
        self._keep = (means, scales, quats, opacities, sh, T_cw_dev)  # retained until the backward (gs.h)
        c = cam if isinstance(cam, gs_camera) else camera_struct(cam)
        f32 = torch.float32
        self._check(self.lib.gs_preprocess(self._h, _stream(stream), N, int(sh_degree), _ptr(means, f32),
                                           _ptr(scales, f32), _ptr(quats, f32), _ptr(opacities, f32), _ptr(sh, f32),
                                           C.byref(c), _ptr(T_cw_dev, f32)))
        self.N, self.K, self.W, self.H = N, (int(sh_degree) + 1) ** 2, c.width, c.height

    def gs_bin_tiles(self, stream=None):
        self._check(self.lib.gs_bin_tiles(self._h, _stream(stream)))

    def gs_rasterize_fwd(self, bg, rgb, depth, alpha, stream=None):
        import torch
        f32 = torch.float32
        self._check(self.lib.gs_rasterize_fwd(self._h, _stream(stream), _bg(bg), _ptr(rgb, f32), _ptr(depth, f32),
                                              _ptr(alpha, f32)))

    def gs_rasterize_bwd(self, d_rgb, d_depth, d_alpha, flags, g_means, g_scales, g_quats, g_opacities, g_sh, stream=None):
        import torch
        f32 = torch.float32
        self._check(self.lib.gs_rasterize_bwd(self._h, _stream(stream), _ptr(d_rgb, f32), _ptr(d_depth, f32),
                                              _ptr(d_alpha, f32), int(flags), _ptr(g_means, f32), _ptr(g_scales, f32),
                                              _ptr(g_quats, f32), _ptr(g_opacities, f32), _ptr(g_sh, f32)))

    def gs_pose_grad(self, flags, g_twist, stream=None):
        import torch
        self._check(self.lib.gs_pose_grad(self._h, _stream(stream), int(flags), _ptr(g_twist, torch.float32)))

    def gs_refine_views(self, params, sh_degree, cams, target_rgb, target_depth, ab, weights, bg, grads, g_twist, g_ab, loss,
                        normal_prior=None, T_cw_dev=None, visible=None, stream=None):
        """One Eq. 23 iteration over the views (include/gs.h).  params / grads: dicts of CUDA tensors; cams: list of cameras;
        target_rgb [V,3,H,W], target_depth [V,H,W], ab [V,2]; weights = (alpha', lambda, beta, lambda_n)."""
        import torch
        V = len(cams)
        arr = (gs_camera * V)(*[c if isinstance(c, gs_camera) else camera_struct(c) for c in cams])
        p = lambda t: None if t is None else t.data_ptr()
        batch = gs_refine_batch(V, arr, p(T_cw_dev), p(target_rgb), p(target_depth), p(normal_prior), p(ab), float(weights[0]),
                                float(weights[1]), float(weights[2]), float(weights[3]))
        gp, gg = _gaussians(params), _gaussians(grads)
        self._keep = (params, grads, target_rgb, target_depth, ab, normal_prior, T_cw_dev, arr)
        self._check(self.lib.gs_refine_views(self._h, _stream(stream), int(params["means"].shape[0]), int(sh_degree), C.byref(gp),
                                             C.byref(batch), _bg(bg), C.byref(gg), _ptr(g_twist, torch.float32),
                                             _ptr(g_ab, torch.float32), _ptr(loss, torch.float64),
                                             None if visible is None else C.c_void_p(visible.data_ptr())))

    # -- introspection -------------------------------------------------------------------------------------------
    def gs_get_counts(self, stream=None):
        nv, ni = C.c_int64(0), C.c_int64(0)
        self._check(self.lib.gs_get_counts(self._h, _stream(stream), C.byref(nv), C.byref(ni)))
        return int(nv.value), int(ni.value)

    def gs_get_binning(self, stream=None):
        import torch
        _, I = self.gs_get_counts(stream)
        tiles = ((self.W + GS_TILE - 1) // GS_TILE) * ((self.H + GS_TILE - 1) // GS_TILE)
        dev = torch.device("cuda", self.device)
        keys = torch.empty(I, dtype=torch.int64, device=dev)
        ids = torch.empty(I, dtype=torch.int32, device=dev)
        ranges = torch.empty((tiles, 2), dtype=torch.int32, device=dev)
        self._check(self.lib.gs_get_binning(self._h, _stream(stream), _ptr(keys), _ptr(ids), _ptr(ranges)))
        torch.cuda.current_stream().synchronize()
        return (keys.cpu().numpy().view(np.uint64), ids.cpu().numpy().view(np.uint32),
                ranges.cpu().numpy().view(np.uint32))

    def gs_get_features(self, stream=None):
        import torch
        dev = torch.device("cuda", self.device)
        N = self.N
        out = dict(mean2d=torch.empty((N, 2), dtype=torch.float64, device=dev),
                   conic=torch.empty((N, 3), dtype=torch.float32, device=dev),
                   color=torch.empty((N, 3), dtype=torch.float32, device=dev),
                   depth=torch.empty(N, dtype=torch.float32, device=dev),
                   depth_key=torch.empty(N, dtype=torch.int32, device=dev),
                   rect=torch.empty((N, 4), dtype=torch.int32, device=dev))
        self._check(self.lib.gs_get_features(self._h, _stream(stream), _ptr(out["mean2d"]), _ptr(out["conic"]),
                                             _ptr(out["color"]), _ptr(out["depth"]), _ptr(out["depth_key"]),
                                             _ptr(out["rect"])))
        torch.cuda.current_stream().synchronize()
        res = {k: v.cpu().numpy() for k, v in out.items()}
        res["depth_key"] = res["depth_key"].view(np.uint32)
        return res

    def gs_visible_ids(self):
        """(ids_ptr, n_visible_ptr): raw DEVICE addresses (ints) of the visible-Gaussian index list and its count."""
        a, b = C.c_void_p(), C.c_void_p()
        self._check(self.lib.gs_visible_ids(self._h, C.byref(a), C.byref(b)))
        return int(a.value), int(b.value)

    def gs_get_visible_ids(self, stream=None):
        """int32 CUDA tensor [N] holding the visible-Gaussian indices in slot order (first n_visible entries valid)."""
        import torch
        out = torch.empty(max(self.N, 1), dtype=torch.int32, device=torch.device("cuda", self.device))
        self._check(self.lib.gs_get_visible_ids(self._h, _stream(stream), _ptr(out)))
        return out[:self.N]

    def gs_set_option(self, option: int, value: int):
        self._check(self.lib.gs_set_option(self._h, int(option), int(value)))

    def gs_poll(self):
        self._check(self.lib.gs_poll(self._h))

    def gs_profile_enable(self, on: bool):
        self._check(self.lib.gs_profile_enable(self._h, int(bool(on))))

    def gs_profile_read(self) -> dict:
        ms = (C.c_float * 8)()
        self._check(self.lib.gs_profile_read(self._h, C.byref(ms)))
        return {k: float(ms[i]) for i, k in enumerate(STAGES)}

    def gs_get_launch_count(self) -> int:
        n = C.c_uint64(0)
        self._check(self.lib.gs_get_launch_count(self._h, C.byref(n)))
        return int(n.value)

    def gs_get_workload(self, stream=None) -> dict:
        w = (C.c_uint64 * 7)()
        self._check(self.lib.gs_get_workload(self._h, _stream(stream), C.byref(w)))
        return dict(evaluated=int(w[0]), blended=int(w[1]), last_pos_sum=int(w[2]), list_len_x_pixels=int(w[3]),
                    region_entries=int(w[4]), evaluated_bwd=int(w[5]), region_entries_bwd=int(w[6]))

    # -- host-buffer path (numpy arrays in / out; copies inside) ---------------------------------------------------
    def gs_fwd_bwd_host(self, scene_arrays, sh_degree, cam, bg, d_rgb, d_depth, out, stream=None, sync=True):
        """scene_arrays = (means, scales, quats, opacities, sh) float32 numpy (ideally pinned); out = dict of float32
        numpy arrays rgb, depth, alpha, g_means, g_scales, g_quats, g_opacities, g_sh, g_twist (any may be absent)."""
        def hp(a):
            if a is None:
                return None
            assert a.dtype == np.float32 and a.flags["C_CONTIGUOUS"]
            return C.c_void_p(a.ctypes.data)
        means, scales, quats, opac, sh = scene_arrays
        c = cam if isinstance(cam, gs_camera) else camera_struct(cam)
        fn = self.lib.gs_fwd_bwd_host if sync else self.lib.gs_fwd_bwd_host_async   # async: the caller synchronises
        self._check(fn(
            self._h, _stream(stream), int(means.shape[0]), int(sh_degree), hp(means), hp(scales), hp(quats), hp(opac),
            hp(sh), C.byref(c), _bg(bg), hp(d_rgb), hp(d_depth), hp(out.get("rgb")), hp(out.get("depth")),
            hp(out.get("alpha")), hp(out.get("g_means")), hp(out.get("g_scales")), hp(out.get("g_quats")),
            hp(out.get("g_opacities")), hp(out.get("g_sh")), hp(out.get("g_twist"))))


def gs_aux_l1_grad(pred, target, weight, grad, stream=None):
    import torch
    lib = load_library()
    rc = lib.gs_aux_l1_grad(_stream(stream), int(pred.numel()), _ptr(pred, torch.float32), _ptr(target, torch.float32),
                            float(weight), _ptr(grad, torch.float32))
    if rc != 0:
        raise GsError(rc, "gs_aux_l1_grad")


def gs_loss_map(rgb, depth, target_rgb, target_depth, alpha, beta, d_rgb, d_depth, loss, stream=None):
    """Eq. 4 photometric + depth L1 terms: writes the upstream gradients and double loss[4] (device; the last is scratch)."""
    import torch
    f32 = torch.float32
    H, W = depth.shape
    rc = load_library().gs_loss_map(_stream(stream), int(W), int(H), _ptr(rgb, f32), _ptr(depth, f32), _ptr(target_rgb, f32),
                                    _ptr(target_depth, f32), float(alpha), float(beta), _ptr(d_rgb, f32), _ptr(d_depth, f32),
                                    _ptr(loss, torch.float64))
    if rc != 0:
        raise GsError(rc, "gs_loss_map")


def gs_loss_refine(rgb, depth, target_rgb, target_depth, ab, alpha_p, lam, beta, d_rgb, d_depth, g_ab, work, loss, stream=None):
    """Eq. 23 (without the normal term) on the exposure-compensated render: writes the upstream gradients, (dL/da, dL/db)
    and double loss[8] (device).  work: float scratch of 9 H W elements."""
    import torch
    f32 = torch.float32
    H, W = depth.shape
    assert work.numel() >= 9 * H * W
    rc = load_library().gs_loss_refine(_stream(stream), int(W), int(H), _ptr(rgb, f32), _ptr(depth, f32), _ptr(target_rgb, f32),
                                       _ptr(target_depth, f32), _ptr(ab, f32), float(alpha_p), float(lam), float(beta),
                                       _ptr(d_rgb, f32), _ptr(d_depth, f32), _ptr(g_ab, f32), _ptr(work, f32),
                                       _ptr(loss, torch.float64))
    if rc != 0:
        raise GsError(rc, "gs_loss_refine")


def gs_loss_normal(cam, depth, normal_prior, lambda_n, normals_out, d_depth, loss, stream=None):
    """Depth-induced normals (normals_out, optional) and lambda_n L_normal; its depth gradient is ADDED into d_depth."""
    import torch
    f32 = torch.float32
    H, W = depth.shape
    rc = load_library().gs_loss_normal(_stream(stream), int(W), int(H), float(cam.fx), float(cam.fy), float(cam.cx), float(cam.cy),
                                       _ptr(depth, f32), _ptr(normal_prior, f32), float(lambda_n), _ptr(normals_out, f32),
                                       _ptr(d_depth, f32), _ptr(loss, torch.float64))
    if rc != 0:
        raise GsError(rc, "gs_loss_normal")


def gs_loss_iso(scales, lambda_s, g_scales, loss, stream=None):
    """Eq. 4 isotropy regulariser: adds its gradient into g_scales, writes double loss[2] (device)."""
    import torch
    f32 = torch.float32
    rc = load_library().gs_loss_iso(_stream(stream), int(scales.shape[0]), _ptr(scales, f32), float(lambda_s),
                                    _ptr(g_scales, f32), _ptr(loss, torch.float64))
    if rc != 0:
        raise GsError(rc, "gs_loss_iso")


def gs_sim3_apply(s, R, t, means, scales, quats, means_out=None, scales_out=None, quats_out=None, stream=None):
    """Eq. 19: Sim(3) correction (s, R, t) of Gaussians on the device; in place unless outputs are given."""
    import torch
    f32 = torch.float32
    Rm = np.asarray(R, np.float32).reshape(9); tv = np.asarray(t, np.float32).reshape(3)
    Rc = (C.c_float * 9)(*[float(x) for x in Rm]); tc = (C.c_float * 3)(*[float(x) for x in tv])
    mo = means if means_out is None else means_out
    so = scales if scales_out is None else scales_out
    qo = quats if quats_out is None else quats_out
    rc = load_library().gs_sim3_apply(_stream(stream), int(means.shape[0]), float(s), Rc, tc, _ptr(means, f32),
                                      _ptr(scales, f32), _ptr(quats, f32), _ptr(mo, f32), _ptr(so, f32), _ptr(qo, f32))
    if rc != 0:
        raise GsError(rc, "gs_sim3_apply")


PARAM_KEYS = ("means", "scales", "quats", "opacities", "sh")


def _gaussians(d) -> gs_gaussians:
    import torch
    g = gs_gaussians()
    for k in PARAM_KEYS:
        t = d[k]
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous() and t.dtype == torch.float32):
            raise TypeError(f"{k}: expected a contiguous float32 CUDA tensor")
        setattr(g, k, t.data_ptr())
    return g


def gs_adam_step(params, grads, m, v, lrs, step, visible=None, beta1=0.9, beta2=0.999, eps=1e-15, stream=None):
    """One fused Adam step in place (include/gs.h).  params / grads / m / v: dicts of CUDA tensors keyed means, scales, quats,
    opacities, sh; lrs: dict of learning rates; visible: optional int32/uint32 CUDA tensor [N]."""
    import torch
    N = int(params["means"].shape[0])
    K = int(params["sh"].shape[1])
    deg = int(round(K ** 0.5)) - 1
    cfg = gs_adam_config(float(lrs["means"]), float(lrs["scales"]), float(lrs["quats"]), float(lrs["opacities"]), float(lrs["sh"]),
                         float(beta1), float(beta2), float(eps), int(step))
    gp, gg, gm, gv = _gaussians(params), _gaussians(grads), _gaussians(m), _gaussians(v)
    vis = None if visible is None else C.c_void_p(visible.data_ptr())
    rc = load_library().gs_adam_step(_stream(stream), N, deg, C.byref(cfg), C.byref(gp), C.byref(gg), C.byref(gm), C.byref(gv), vis)
    if rc != 0:
        raise GsError(rc, "gs_adam_step")


def gs_adam_step_sparse(params, grads, m, v, lrs, step, ids_ptr, n_rows_ptr, max_rows, beta1=0.9, beta2=0.999, eps=1e-15,
                        stream=None):
    """gs_adam_step on GS_SPARSE_GRADS gradients; ids_ptr / n_rows_ptr: device addresses from Context.gs_visible_ids()."""
    N = int(params["means"].shape[0])
    K = int(params["sh"].shape[1])
    deg = int(round(K ** 0.5)) - 1
    cfg = gs_adam_config(float(lrs["means"]), float(lrs["scales"]), float(lrs["quats"]), float(lrs["opacities"]), float(lrs["sh"]),
                         float(beta1), float(beta2), float(eps), int(step))
    gp, gg, gm, gv = _gaussians(params), _gaussians(grads), _gaussians(m), _gaussians(v)
    rc = load_library().gs_adam_step_sparse(_stream(stream), N, deg, C.byref(cfg), C.byref(gp), C.byref(gg), C.byref(gm),
                                            C.byref(gv), C.c_void_p(ids_ptr), C.c_void_p(n_rows_ptr), int(max_rows))
    if rc != 0:
        raise GsError(rc, "gs_adam_step_sparse")


def gs_prune_mask(opacities, min_opacity, keep, stream=None):
    import torch
    rc = load_library().gs_prune_mask(_stream(stream), int(opacities.numel()), _ptr(opacities, torch.float32), float(min_opacity),
                                      _ptr(keep, torch.uint8))
    if rc != 0:
        raise GsError(rc, "gs_prune_mask")


def gs_compact(keep, arrays, stream=None):
    """Order-preserving compaction of a dict of [N,...] float32 CUDA tensors by the uint8 mask `keep`.  Returns (dict of
    compacted tensors [n_kept,...], index tensor [N] (destination row or 0xFFFFFFFF))."""
    import torch
    lib = load_library()
    N = int(keep.numel())
    dev = keep.device
    index = torch.empty(N, dtype=torch.int32, device=dev)
    n_kept = torch.zeros(1, dtype=torch.int64, device=dev)
    work = torch.empty(max(1, int(lib.gs_compact_work_bytes(N))), dtype=torch.uint8, device=dev)
    rc = lib.gs_compact_plan(_stream(stream), N, _ptr(keep, torch.uint8), _ptr(index), _ptr(n_kept), _ptr(work))
    if rc != 0:
        raise GsError(rc, "gs_compact_plan")
    n = int(n_kept.item())                                # the one host read: sizes the outputs
    out = {}
    for k, a in arrays.items():
        width = int(a.numel() // max(N, 1)) if N else 1
        o = torch.empty((n,) + tuple(a.shape[1:]), dtype=torch.float32, device=dev)
        rc = lib.gs_compact_rows(_stream(stream), N, width, _ptr(index), _ptr(a, torch.float32), _ptr(o, torch.float32))
        if rc != 0:
            raise GsError(rc, "gs_compact_rows")
        out[k] = o
    return out, index


def gs_compact_plan_static(keep, index, n_kept, stream=None):
    """gs_compact_plan_static of include/gs.h: the compaction plan of the uint8 mask `keep` written into the caller's
    `index` (int32/uint32 [N]) and `n_kept` (int64 [1]) CUDA tensors, with the scratch taken from a fixed 64 KiB array
    inside libgs.so instead of a fresh device allocation.  It is meant for code that cannot allocate where it compacts: an
    agent whose device memory was all handed out at start-up, or a pruning / fusion step running beside tracking streams
    that a cudaMalloc would stall.  Nothing is allocated here either (the caller brings every tensor), and N above
    gs_compact_plan_static_max() (16 Mi Gaussians) raises GS_E_TOO_LARGE.  Calls on one device share the scratch, so two
    calls that may overlap on the GPU race; make the first call on a device during set-up."""
    import torch
    lib = load_library()
    N = int(keep.numel())
    if N > int(lib.gs_compact_plan_static_max()):
        raise GsError(-6, f"gs_compact_plan_static: N = {N} exceeds the fixed scratch of {int(lib.gs_compact_plan_static_max())} "
                          "Gaussians; use gs_compact_plan with caller scratch")
    assert index.numel() == N and index.element_size() == 4 and n_kept.dtype == torch.int64 and n_kept.numel() == 1
    rc = lib.gs_compact_plan_static(_stream(stream), N, _ptr(keep, torch.uint8), _ptr(index), _ptr(n_kept))
    if rc != 0:
        raise GsError(rc, "gs_compact_plan_static")


class VoxelSet:
    """Hash set of 64-bit voxel keys in device memory (include/gs.h, Eqs. 20-22)."""

    def __init__(self, capacity: int, device: int = 0):
        import torch
        assert capacity >= 2 and capacity & (capacity - 1) == 0
        dev = torch.device("cuda", device)
        self.capacity = capacity
        self.table = torch.empty(capacity, dtype=torch.int64, device=dev)
        self.overflow = torch.zeros(1, dtype=torch.int32, device=dev)
        self.clear()

    def clear(self, stream=None):
        rc = load_library().gs_voxel_set_clear(_stream(stream), _ptr(self.table), self.capacity)
        if rc != 0:
            raise GsError(rc, "gs_voxel_set_clear")
        self.overflow.zero_()

    def insert_boxes(self, means, scales, voxel, k, stream=None):
        import torch
        rc = load_library().gs_voxel_insert_boxes(_stream(stream), _ptr(self.table), self.capacity, float(voxel), float(k),
                                                  int(means.shape[0]), _ptr(means, torch.float32), _ptr(scales, torch.float32),
                                                  _ptr(self.overflow))
        if rc != 0:
            raise GsError(rc, "gs_voxel_insert_boxes")

    def insert_rays(self, cam, depth, voxel, stride=1, stream=None):
        import torch
        c = cam if isinstance(cam, gs_camera) else camera_struct(cam)
        rc = load_library().gs_voxel_insert_rays(_stream(stream), _ptr(self.table), self.capacity, float(voxel), C.byref(c),
                                                 _ptr(depth, torch.float32), int(stride), _ptr(self.overflow))
        if rc != 0:
            raise GsError(rc, "gs_voxel_insert_rays")

    def keys(self):
        """Sorted numpy uint64 array of the stored keys (test / inspection helper; synchronises)."""
        t = self.table.cpu().numpy().view(np.uint64)
        return np.sort(t[t != np.uint64(0xFFFFFFFFFFFFFFFF)])


def gs_voxel_retain(occ, free, voxel, means, retain, stream=None):
    import torch
    rc = load_library().gs_voxel_retain(_stream(stream), _ptr(occ.table) if occ else None, occ.capacity if occ else 0,
                                        _ptr(free.table) if free else None, free.capacity if free else 0, float(voxel),
                                        int(means.shape[0]), _ptr(means, torch.float32), _ptr(retain, torch.uint8))
    if rc != 0:
        raise GsError(rc, "gs_voxel_retain")


def gs_measure_peaks(device: int = 0, stream=None) -> dict:
    """Measured machine peaks (include/gs.h): the roofline denominators.  Synchronous, ~0.2 s."""
    out = (C.c_double * len(PEAKS))()
    rc = load_library().gs_measure_peaks(int(device), _stream(stream), C.byref(out))
    if rc != 0:
        raise GsError(rc, "gs_measure_peaks")
    return {k: float(out[i]) for i, k in enumerate(PEAKS)}


def gs_aux_pose_step(T_cw_dev, g_twist, step, stream=None):
    import torch
    lib = load_library()
    rc = lib.gs_aux_pose_step(_stream(stream), _ptr(T_cw_dev, torch.float32), _ptr(g_twist, torch.float32), float(step))
    if rc != 0:
        raise GsError(rc, "gs_aux_pose_step")


# ---------------------------------------------------------------------------------------------------------------
# Convenience wrapper used by the tests, smoke() and bench.py: device tensors for one scene + one fwd/bwd iteration.
# ---------------------------------------------------------------------------------------------------------------
class DeviceScene:
    def __init__(self, scene, device: int = 0):
        import torch
        dev = torch.device("cuda", device)
        t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to(dev)
        self.means, self.scales, self.quats = t(scene.means), t(scene.scales), t(scene.quats)
        self.opacities, self.sh = t(scene.opacities), t(scene.sh)
        self.sh_degree = int(scene.sh_degree)
        self.N = int(scene.means.shape[0])
        self.K = (self.sh_degree + 1) ** 2
        self.bg = np.asarray(scene.bg, dtype=np.float32)
        self.dev = dev

    def alloc_outputs(self, W, H):
        import torch
        z = lambda *s: torch.zeros(s, dtype=torch.float32, device=self.dev)
        return dict(rgb=z(3, H, W), depth=z(H, W), alpha=z(H, W), g_means=z(self.N, 3), g_scales=z(self.N, 3),
                    g_quats=z(self.N, 4), g_opacities=z(self.N), g_sh=z(self.N, self.K, 3), g_twist=z(6))


def forward(ctx: Context, ds: DeviceScene, cam, out, T_cw_dev=None):
    ctx.gs_preprocess(ds.means, ds.scales, ds.quats, ds.opacities, ds.sh, ds.sh_degree, cam, T_cw_dev)
    ctx.gs_bin_tiles()
    ctx.gs_rasterize_fwd(ds.bg, out["rgb"], out["depth"], out["alpha"])


def backward(ctx: Context, out, d_rgb, d_depth, d_alpha=None, flags=0, pose=True):
    if flags & GS_POSE_ONLY:
        ctx.gs_rasterize_bwd(d_rgb, d_depth, d_alpha, flags, None, None, None, None, None)
    else:
        ctx.gs_rasterize_bwd(d_rgb, d_depth, d_alpha, flags, out["g_means"], out["g_scales"], out["g_quats"],
                             out["g_opacities"], out["g_sh"])
    if pose:
        ctx.gs_pose_grad(flags & GS_ACCUMULATE, out["g_twist"])
