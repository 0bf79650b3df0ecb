"""Pins of the depth-induced normal / L_normal oracle (oracle/normals.py): planes with known normals, the cosine
loss on hand-built cases, central finite differences, invalid-pixel rules."""
import numpy as np

from oracle import normals as on


def _plane_depth(n, d0, W, H, fx, fy, cx, cy):
    """Depth map of the plane n . p = n_z d0 (passing through (0,0,d0)): z = n_z d0 / (n . ray)."""
    ys, xs = np.mgrid[0:H, 0:W]
    ray = np.stack([(xs - cx) / fx, (ys - cy) / fy, np.ones_like(xs, float)])
    return n[2] * d0 / np.tensordot(n, ray, 1)


def test_fronto_parallel_and_tilted_planes_give_their_normals():
    fx, fy, cx, cy, W, H = 50.0, 55.0, 7.5, 5.0, 16, 11
    nm, ok = on.normals(np.full((H, W), 2.0), fx, fy, cx, cy)
    assert ok[:-1, :-1].all() and not ok[-1].any() and not ok[:, -1].any()
    assert np.allclose(nm[:, :-1, :-1], np.array([0, 0, -1.0])[:, None, None], atol=1e-14)    # faces the camera
    for nrm in ([0.3, -0.2, -1.0], [-0.5, 0.1, -0.8]):
        n = np.array(nrm) / np.linalg.norm(nrm)
        nm, ok = on.normals(_plane_depth(n, 3.0, W, H, fx, fy, cx, cy), fx, fy, cx, cy)
        assert np.allclose(nm[:, :-1, :-1], n[:, None, None], atol=1e-12)                     # exact for a plane: p is linear on it


def test_loss_values_by_hand_and_invalid_pixels():
    fx = fy = 40.0; cx = cy = 2.0; W = H = 5
    depth = np.full((H, W), 2.0)
    prior = np.zeros((3, H, W)); prior[2] = -1.0                   # prior = rendered normal everywhere -> loss 0
    l, g = on.normal_loss(depth, prior, fx, fy, cx, cy)
    assert abs(l) < 1e-15
    prior[:, 1, 1] = [0.0, 0.6, -0.8]                              # one pixel: 1 - (0,0,-1).(0,.6,-.8) = 0.2
    prior[:, 2, 2] = [0.0, 0.0, 1.0]                               # opposite: |1 - (-1)| = 2
    l, _ = on.normal_loss(depth, prior, fx, fy, cx, cy)
    assert np.isclose(l, (0.2 + 2.0) / 25)
    prior[:, 2, 2] = 0.0                                           # zero prior = no prior
    depth2 = depth.copy(); depth2[1, 2] = 0.0                      # invalid depth kills the normals that use it: (1,1), (1,2), (0,2)
    l, g = on.normal_loss(depth2, prior, fx, fy, cx, cy)
    assert abs(l) < 1e-15 and not g.any()
    assert on.normal_at(depth2, 1, 1, fx, fy, cx, cy) is None and on.normal_at(depth2, 2, 0, fx, fy, cx, cy) is None
    assert on.normal_at(depth2, 0, 1, fx, fy, cx, cy) is not None


def test_gradient_by_central_finite_differences():
    r = np.random.Generator(np.random.PCG64(5))
    fx, fy, cx, cy, W, H = 30.0, 33.0, 6.2, 4.1, 13, 9
    depth = 2.0 + 0.3 * r.normal(size=(H, W))
    depth[3, 4] = 0.0
    prior = r.normal(size=(3, H, W)); prior /= np.linalg.norm(prior, axis=0)
    prior[:, 5, 5] = 0.0
    l, g = on.normal_loss(depth, prior, fx, fy, cx, cy)
    assert l > 0.3
    for trial in range(8):
        u = r.normal(size=depth.shape) if trial < 4 else np.zeros(depth.shape)
        if trial >= 4:
            u.flat[r.integers(u.size)] = 1.0
        u[3, 4] = 0.0
        h = 1e-6
        fd = (on.normal_loss(depth + h * u, prior, fx, fy, cx, cy)[0] - on.normal_loss(depth - h * u, prior, fx, fy, cx, cy)[0]) / (2 * h)
        assert abs(fd - (g * u).sum()) <= 1e-7 * max(1.0, abs(fd))
    # scaling the depth map leaves the normals (and the loss) unchanged: the gradient is orthogonal to the depth itself
    assert abs((g * depth).sum()) < 1e-12
    assert np.isclose(on.normal_loss(1.7 * depth, prior, fx, fy, cx, cy)[0], l)
