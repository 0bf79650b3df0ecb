"""Oracle of Eq. 19: applying a submap's Sim(3) correction C = (s, R, t) to its Gaussians.
TEST INFRASTRUCTURE (plain numpy, fp64): only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import
this module; it shares no code with paper_2605_10760_b200/csrc.

    mu' = s R mu + t,   Sigma' = s^2 R Sigma R^T,   s' = s s_i,   "with unchanged opacity and color".

Sigma = Rq diag(s_i^2) Rq^T with Rq the rotation of the Gaussian's unit quaternion, so Sigma' is obtained by scaling the
three scales by s and left-multiplying the rotation: Rq' = R Rq, i.e. q' = q_R (x) q (Hamilton product, (w,x,y,z)).  The
quaternion is only defined up to sign and (for the raw, unnormalised parametrisation of the ABI) up to a positive factor:
the oracle returns q_R (x) q with q_R the unit quaternion of R with w >= 0 (first non-zero component positive).
"""
from __future__ import annotations

import numpy as np


def quat_of_rotation(R):
    """Unit quaternion (w,x,y,z) of a rotation matrix, by the eigenvector of the 4x4 Davenport matrix (branch-free)."""
    R = np.asarray(R, np.float64)
    K = np.array([[R[0, 0] + R[1, 1] + R[2, 2], R[2, 1] - R[1, 2], R[0, 2] - R[2, 0], R[1, 0] - R[0, 1]],
                  [R[2, 1] - R[1, 2], R[0, 0] - R[1, 1] - R[2, 2], R[0, 1] + R[1, 0], R[0, 2] + R[2, 0]],
                  [R[0, 2] - R[2, 0], R[0, 1] + R[1, 0], R[1, 1] - R[0, 0] - R[2, 2], R[1, 2] + R[2, 1]],
                  [R[1, 0] - R[0, 1], R[0, 2] + R[2, 0], R[1, 2] + R[2, 1], R[2, 2] - R[0, 0] - R[1, 1]]]) / 3.0
    w, v = np.linalg.eigh(K)
    q = v[:, np.argmax(w)]
    k = np.flatnonzero(np.abs(q) > 1e-12)[0]
    return q * np.sign(q[k])


def rotation_of_quat(q):
    q = np.asarray(q, np.float64)
    w, x, y, z = q / np.linalg.norm(q)
    return np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y)],
                     [2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x)],
                     [2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)]])


def sim3_apply(means, scales, quats, s, R, t):
    """Eq. 19, Gaussian by Gaussian.  Returns (means', scales', quats') in fp64; opacity and colour are untouched."""
    means = np.asarray(means, np.float64); scales = np.asarray(scales, np.float64); quats = np.asarray(quats, np.float64)
    R = np.asarray(R, np.float64); t = np.asarray(t, np.float64)
    qr = quat_of_rotation(R)
    m2 = np.empty_like(means); s2 = np.empty_like(scales); q2 = np.empty_like(quats)
    for i in range(means.shape[0]):
        m2[i] = s * (R @ means[i]) + t
        s2[i] = s * scales[i]
        w1, x1, y1, z1 = qr
        w, x, y, z = quats[i]
        q2[i] = [w1 * w - x1 * x - y1 * y - z1 * z, w1 * x + x1 * w + y1 * z - z1 * y,
                 w1 * y - x1 * z + y1 * w + z1 * x, w1 * z + x1 * y - y1 * x + z1 * w]
    return m2, s2, q2


def covariance(scales_i, quat_i):
    Rq = rotation_of_quat(quat_i)
    return Rq @ np.diag(np.asarray(scales_i, np.float64) ** 2) @ Rq.T


# ----------------------------------------------------------------------------------------------------------------------
# Eqs. 20-22: occupancy-aware fusion on "a frustum-aware occupancy grid of voxel size v"
#   O_occ  = U_i   { kappa(x) : x in [mu_i - k s_i, mu_i + k s_i] }                      (Eq. 20, target Gaussians)
#   O_free = U_u,k { kappa(c_k + t (r_k(u) - c_k)) : t in [0, 1) }                       (Eq. 21, keyframe depth maps)
#   a borrowed Gaussian j is retained iff kappa(mu_j) not in O_occ and not in O_free       (Eq. 22)
# "We pack each voxel index kappa(.) into a 64-bit spatial-hash key".
# Readings (Q21): kappa(x) = floor(x / v) per axis (fp64 division of the fp32 inputs); key = three 21-bit
# fields (index + 2^20) packed x | y << 21 | z << 42; the box of Eq. 20 is axis-aligned in world coordinates with half
# extents k s_i component-wise (the paper's interval notation; the Gaussian's rotation is ignored); r_k(u) is the
# back-projection of pixel u (integer-centred, Q7) at its depth D_k(u) (camera-space z), c_k the camera centre; pixels with
# depth <= 0 cast no ray; v and k are arguments (unpublished).  The voxel set of a ray is computed by the 3-D DDA
# (Amanatides & Woo) in fp64; `ray_voxels_by_definition` is the independent plain definition used to pin it.  Which voxels
# a ray meets is decided by comparisons of crossing parameters; where two crossings coincide to within rounding (a ray
# through a voxel edge, a surface point on a voxel face) the set is not determined by the mathematics: `free_keys`
# reports those voxels separately (`ambiguous`), and a second implementation is compared with this one up to them.
# ----------------------------------------------------------------------------------------------------------------------
KEY_BIAS = 1 << 20


def pack_key(ix, iy, iz):
    ix = np.asarray(ix, np.int64) + KEY_BIAS; iy = np.asarray(iy, np.int64) + KEY_BIAS; iz = np.asarray(iz, np.int64) + KEY_BIAS
    assert ((ix >= 0) & (ix < (1 << 21)) & (iy >= 0) & (iy < (1 << 21)) & (iz >= 0) & (iz < (1 << 21))).all()
    return (ix | (iy << 21) | (iz << 42)).astype(np.uint64)


def kappa(x, v):
    """Voxel index of points x [...,3]: floor(x / v) in fp64."""
    return np.floor(np.asarray(x, np.float64) / np.float64(v)).astype(np.int64)


def occupied_set(means, scales, v, k):
    """Eq. 20 as a Python set of packed keys: every voxel meeting the closed box [mu - k s, mu + k s]."""
    means = np.asarray(means, np.float64); scales = np.asarray(scales, np.float64)
    out = set()
    for i in range(means.shape[0]):
        lo = kappa(means[i] - np.float64(k) * scales[i], v)
        hi = kappa(means[i] + np.float64(k) * scales[i], v)
        for iz in range(lo[2], hi[2] + 1):
            for iy in range(lo[1], hi[1] + 1):
                for ix in range(lo[0], hi[0] + 1):
                    out.add(int(pack_key(ix, iy, iz)))
    return out


def ray_voxels(c, r, v):
    """Voxels met by the half-open segment c + t (r - c), t in [0, 1): 3-D DDA in fp64.  Returns a list of (ix,iy,iz)."""
    c = np.asarray(c, np.float64); r = np.asarray(r, np.float64); v = np.float64(v)
    d = r - c
    idx = np.floor(c / v).astype(np.int64)
    step = np.zeros(3, np.int64); t_max = np.full(3, np.inf); t_delta = np.full(3, np.inf)
    for a in range(3):
        if d[a] > 0:
            step[a] = 1
            t_max[a] = ((np.float64(idx[a]) + 1.0) * v - c[a]) / d[a]
            t_delta[a] = v / d[a]
        elif d[a] < 0:
            step[a] = -1
            t_max[a] = (np.float64(idx[a]) * v - c[a]) / d[a]
            t_delta[a] = -v / d[a]
    out = [tuple(int(q) for q in idx)]
    while True:
        a = 0                                  # axis of the nearest boundary; ties -> lowest axis
        if t_max[1] < t_max[a]:
            a = 1
        if t_max[2] < t_max[a]:
            a = 2
        if not (t_max[a] < 1.0):               # the next boundary lies at t >= 1: outside the half-open segment
            break
        idx[a] += step[a]
        t_max[a] = t_max[a] + t_delta[a]
        out.append(tuple(int(q) for q in idx))
    return out


def ray_voxels_by_definition(c, r, v):
    """The plain definition of Eq. 21 for one ray: kappa at the midpoints between consecutive boundary crossings of the
    open parameter interval (0, 1) (and at t -> 0+).  Equals ray_voxels except on measure-zero ties."""
    c = np.asarray(c, np.float64); r = np.asarray(r, np.float64); d = r - c
    ts = [0.0, 1.0]
    for a in range(3):
        if d[a] != 0:
            lo, hi = sorted((c[a], r[a]))
            for m in range(int(np.floor(lo / v)) - 1, int(np.floor(hi / v)) + 2):
                t = (m * v - c[a]) / d[a]
                if 0.0 < t < 1.0:
                    ts.append(t)
    ts = sorted(set(ts))
    return {tuple(int(q) for q in np.floor((c + 0.5 * (t0 + t1) * d) / v)) for t0, t1 in zip(ts[:-1], ts[1:])}


def backproject(depth, fx, fy, cx, cy, T_cw, stride=1):
    """Camera centre c_k = -R^T t and world-space surface points r_k(u) = R^T (p_c - t) of the pixels (every `stride`-th in
    x and y, row by row) with depth > 0, p_c = ((u - cx) z / fx, (v - cy) z / fy, z)   (world-to-camera pose)."""
    depth = np.asarray(depth, np.float64)
    T = np.asarray(T_cw, np.float64).reshape(3, 4)
    R, t = T[:, :3], T[:, 3]
    fx, fy, cx, cy = np.float64(fx), np.float64(fy), np.float64(cx), np.float64(cy)
    c = -(R.T @ t)
    H, W = depth.shape
    ys, xs = np.meshgrid(np.arange(0, H, stride), np.arange(0, W, stride), indexing="ij")
    z = depth[ys, xs]
    ok = z > 0.0
    xs, ys, z = xs[ok].astype(np.float64), ys[ok].astype(np.float64), z[ok]
    pc = np.stack([(xs - cx) * z / fx, (ys - cy) * z / fy, z], axis=1)
    return c, (pc - t) @ R          # row i: R^T (p_c,i - t)


def free_set(depth, fx, fy, cx, cy, T_cw, v, stride=1):
    """Eq. 21 for one keyframe as a Python set of packed keys."""
    c, pts = backproject(depth, fx, fy, cx, cy, T_cw, stride)
    out = set()
    for r in pts:
        for (ix, iy, iz) in ray_voxels(c, r, v):
            out.add(int(pack_key(ix, iy, iz)))
    return out


def retain_mask(means, occ, free, v):
    """Eq. 22: True where kappa(mu_j) is in neither set."""
    idx = kappa(means, v)
    keys = pack_key(idx[:, 0], idx[:, 1], idx[:, 2])
    return np.array([(int(q) not in occ) and (int(q) not in free) for q in keys], dtype=bool)



# ----------------------------------------------------------------------------------------------------------------------
# The same sets for inputs of the paper's size (a 1200 x 680 depth map, 5 x 10^5 Gaussians): identical definitions, written
# over arrays of rays / Gaussians instead of Python loops over them.  Pinned against the per-item functions above
# (tests/test_oracle_fusion_occupancy_pins.py).
# ----------------------------------------------------------------------------------------------------------------------
def occupied_keys(means, scales, v, k):
    """Eq. 20 as a sorted array of unique packed keys: offsets (dx, dy, dz) >= 0 from the lowest voxel of every box, kept
    where they stay inside that Gaussian's box."""
    means = np.asarray(means, np.float64); scales = np.asarray(scales, np.float64)
    if means.shape[0] == 0:
        return np.zeros(0, np.uint64)
    lo = kappa(means - np.float64(k) * scales, v)
    hi = kappa(means + np.float64(k) * scales, v)
    n = hi - lo + 1
    out = []
    small = (n <= 8).all(axis=1)                      # the bulk: one pass per offset; the few large boxes one by one
    ls, ns = lo[small], n[small]
    if ls.shape[0]:
        m = ns.max(axis=0)
        for dz in range(m[2]):
            for dy in range(m[1]):
                for dx in range(m[0]):
                    w = (dx < ns[:, 0]) & (dy < ns[:, 1]) & (dz < ns[:, 2])
                    if w.any():
                        out.append(np.unique(pack_key(ls[w, 0] + dx, ls[w, 1] + dy, ls[w, 2] + dz)))
    for l, h in zip(lo[~small], hi[~small]):
        gx, gy, gz = np.meshgrid(*(np.arange(l[a], h[a] + 1) for a in range(3)), indexing="ij")
        out.append(pack_key(gx.ravel(), gy.ravel(), gz.ravel()))
    return np.unique(np.concatenate(out))


_EPS = np.finfo(np.float64).eps


def free_keys(c, pts, v):
    """Eq. 21 for rays c -> pts[i]: the 3-D DDA of `ray_voxels`, all rays stepped together.  Returns (keys, ambiguous):
    sorted unique packed keys of the voxels met, and the keys whose membership hinges on a comparison that rounding can
    turn -- two boundary crossings closer than the crossing parameters are known (either order is a valid walk and the
    voxel in between differs), or a crossing that close to t = 1 (the end voxel is entered or not).  A crossing parameter
    t = (boundary - c_a) / d_a computed from c, r that are themselves a few ulp uncertain is known to about
    tol_a = 64 eps ((|c_a| + |r_a| + v) / |d_a| + 1) + 4 eps n after n steps of accumulation."""
    c = np.asarray(c, np.float64); r = np.asarray(pts, np.float64).reshape(-1, 3); v = np.float64(v)
    M = r.shape[0]
    if M == 0:
        return np.zeros(0, np.uint64), np.zeros(0, np.uint64)
    d = r - c
    idx = np.repeat(np.floor(c / v).astype(np.int64)[None, :], M, axis=0)
    step = np.sign(d).astype(np.int64)
    with np.errstate(divide="ignore", invalid="ignore"):
        nxt = np.where(d > 0, (idx + 1).astype(np.float64) * v, idx.astype(np.float64) * v)
        t_max = np.where(d != 0, (nxt - c) / d, np.inf)
        t_delta = np.where(d != 0, v / np.abs(d), np.inf)
        tol = np.where(d != 0, 64 * _EPS * ((np.abs(c) + np.abs(r) + v) / np.abs(d) + 1.0), 0.0)
    frac = c / v - np.floor(c / v)
    start_fragile = bool(((frac < 64 * _EPS * (1 + np.abs(c / v))) | (1 - frac < 64 * _EPS * (1 + np.abs(c / v)))).any())
    keys = [np.unique(pack_key(idx[:1, 0], idx[:1, 1], idx[:1, 2]))]
    amb = []
    alive = np.arange(M)
    n = 0
    rows = None
    while alive.size:
        tm = t_max[alive]
        a = np.argmin(tm, axis=1)                    # ties -> lowest axis
        rows = np.arange(alive.size)
        t_a = tm[rows, a]
        slack = tol[alive] + 4 * _EPS * n
        go = t_a < 1.0
        # crossings that rounding could reorder or move across t = 1
        near_end = np.abs(t_a - 1.0) <= slack[rows, a]
        tm2 = tm.copy(); tm2[rows, a] = np.inf
        b = np.argmin(tm2, axis=1)
        t_b = tm2[rows, b]
        near_tie = go & np.isfinite(t_b) & (t_b - t_a <= slack[rows, a] + slack[rows, b])
        for sel, ax in ((near_end, a), (near_tie, a), (near_tie, b)):
            if sel.any():
                q = idx[alive[sel]].copy()
                q[np.arange(q.shape[0]), ax[sel]] += step[alive[sel], ax[sel]]
                amb.append(pack_key(q[:, 0], q[:, 1], q[:, 2]))
        alive, a = alive[go], a[go]
        if not alive.size:
            break
        rows = np.arange(alive.size)
        idx[alive, a] += step[alive, a]
        t_max[alive, a] = t_max[alive, a] + t_delta[alive, a]
        keys.append(np.unique(pack_key(idx[alive, 0], idx[alive, 1], idx[alive, 2])))
        n += 1
        if len(keys) >= 16:
            keys = [np.unique(np.concatenate(keys))]
    keys = np.unique(np.concatenate(keys))
    amb = np.unique(np.concatenate(amb)) if amb else np.zeros(0, np.uint64)
    if start_fragile:      # the camera centre sits on a voxel face: every ray's first voxel is undetermined
        amb = keys
    return keys, amb
