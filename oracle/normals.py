"""Oracle of the depth-induced normals and the normal term of Eqs. 4 / 23.  TEST INFRASTRUCTURE (plain numpy, fp64): only
tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this module; it shares no code with
paper_2605_10760_b200/csrc.

Paper: "The normal term L_normal = sum_k |1 - N^_k^T N-_k| is a cosine embedding loss between the depth-induced
normal N^_k and the monocular normal prior N-_k"; rendered normals are shown in PAPER.md:133 (Fig. 3) and PAPER.md:393 (Fig. 7).
How the normal is induced from the depth is not stated.  Reading Q22: back-project the rendered depth D^ (reading
Q8: camera-space z, un-normalised) with the pinhole model, p(u,v) = ((u - cx) D / fx, (v - cy) D / fy, D); forward differences
t_x = p(u+1,v) - p(u,v), t_y = p(u,v+1) - p(u,v); N^ = (t_y x t_x) / |t_y x t_x| (faces the camera: (0,0,-1) for a
fronto-parallel plane).  A pixel has a normal iff it is not in the last column / row and the three depths involved are > 0;
the prior is valid where it is non-zero.  L_normal = (1 / H W) sum over pixels with a normal and a valid prior of
|1 - N^ . N-| (mean reduction as in reading Q18; sign(0) = 0); pixels without contribute nothing.
"""
from __future__ import annotations

import numpy as np


def _point(depth, x, y, fx, fy, cx, cy):
    z = depth[y, x]
    return np.array([(x - cx) * z / fx, (y - cy) * z / fy, z])


def normal_at(depth, x, y, fx, fy, cx, cy):
    """Depth-induced unit normal of pixel (x, y), or None."""
    H, W = depth.shape
    if x + 1 >= W or y + 1 >= H or not (depth[y, x] > 0 and depth[y, x + 1] > 0 and depth[y + 1, x] > 0):
        return None
    p = _point(depth, x, y, fx, fy, cx, cy)
    tx = _point(depth, x + 1, y, fx, fy, cx, cy) - p
    ty = _point(depth, x, y + 1, fx, fy, cx, cy) - p
    n = np.cross(ty, tx)
    ln = np.linalg.norm(n)
    return None if not ln > 0 else n / ln


def normals(depth, fx, fy, cx, cy):
    """[3,H,W] normal map (zeros where undefined) and the [H,W] validity mask."""
    depth = np.asarray(depth, np.float64)
    H, W = depth.shape
    out = np.zeros((3, H, W)); ok = np.zeros((H, W), bool)
    for y in range(H):
        for x in range(W):
            n = normal_at(depth, x, y, float(fx), float(fy), float(cx), float(cy))
            if n is not None:
                out[:, y, x] = n; ok[y, x] = True
    return out, ok


def normal_loss(depth, prior, fx, fy, cx, cy):
    """L_normal (unweighted) and dL/dD^ [H,W].  prior: [3,H,W] unit normals (zero vector = no prior at that pixel)."""
    depth = np.asarray(depth, np.float64); prior = np.asarray(prior, np.float64)
    H, W = depth.shape
    fx, fy, cx, cy = float(fx), float(fy), float(cx), float(cy)
    loss, g = 0.0, np.zeros((H, W))
    for y in range(H - 1):
        for x in range(W - 1):
            nb = prior[:, y, x]
            if not nb.any():
                continue
            if not (depth[y, x] > 0 and depth[y, x + 1] > 0 and depth[y + 1, x] > 0):
                continue
            p0 = _point(depth, x, y, fx, fy, cx, cy)
            tx = _point(depth, x + 1, y, fx, fy, cx, cy) - p0
            ty = _point(depth, x, y + 1, fx, fy, cx, cy) - p0
            c = np.cross(ty, tx); ln = np.linalg.norm(c)
            if not ln > 0:
                continue
            n = c / ln
            e = 1.0 - n @ nb
            loss += abs(e)
            gn = -np.sign(e) * nb                      # dL/dn
            gc = (gn - n * (n @ gn)) / ln                # through the normalisation
            gty = np.cross(tx, gc)                       # c = ty x tx:  dL/dty = tx x gc,  dL/dtx = gc x ty
            gtx = np.cross(gc, ty)
            # p(u,v) = ray(u,v) * D with ray = ((u-cx)/fx, (v-cy)/fy, 1): dL/dD = ray . dL/dp
            ray = lambda xx, yy: np.array([(xx - cx) / fx, (yy - cy) / fy, 1.0])
            g[y, x + 1] += ray(x + 1, y) @ gtx
            g[y + 1, x] += ray(x, y + 1) @ gty
            g[y, x] -= ray(x, y) @ (gtx + gty)
    return loss / (H * W), g / (H * W)
