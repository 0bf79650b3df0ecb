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
