"""Pins of oracle/fusion.py (Eq. 19): the covariance law Sigma' = s^2 R Sigma R^T written out with matrices,
identity, composition of two corrections, scipy's rotation conversions, and -- through the renderer -- invariance of the
image when the camera is moved by the same similarity.  CPU only."""
import numpy as np
from scipy.spatial.transform import Rotation

from oracle import fusion as of


def _rand(seed, N=50):
    r = np.random.default_rng(seed)
    return r.normal(size=(N, 3)), np.exp(r.normal(-3, 0.5, (N, 3))), r.normal(size=(N, 4))


def _rot(seed):
    return Rotation.random(random_state=seed).as_matrix()


def test_covariance_law_and_centres():
    means, scales, quats = _rand(1)
    s, R, t = 1.7, _rot(2), np.array([0.3, -1.2, 0.5])
    m2, s2, q2 = of.sim3_apply(means, scales, quats, s, R, t)
    for i in range(len(means)):
        assert np.allclose(m2[i], s * R @ means[i] + t, atol=1e-14)
        Sig = of.covariance(scales[i], quats[i])
        assert np.allclose(of.covariance(s2[i], q2[i]), s * s * R @ Sig @ R.T, rtol=1e-12, atol=1e-18)
    assert np.allclose(s2, s * scales)


def test_identity_and_composition():
    means, scales, quats = _rand(3)
    m2, s2, q2 = of.sim3_apply(means, scales, quats, 1.0, np.eye(3), np.zeros(3))
    assert np.allclose(m2, means) and np.allclose(s2, scales) and np.allclose(q2, quats)
    sa, Ra, ta = 0.6, _rot(4), np.array([1.0, 2.0, -0.5])
    sb, Rb, tb = 1.9, _rot(5), np.array([-0.2, 0.1, 0.7])
    m1, s1, q1 = of.sim3_apply(means, scales, quats, sa, Ra, ta)
    mb, sbb, qb = of.sim3_apply(m1, s1, q1, sb, Rb, tb)
    # C_b o C_a = (sb sa, Rb Ra, sb Rb ta + tb)
    mc, sc, qc = of.sim3_apply(means, scales, quats, sb * sa, Rb @ Ra, sb * Rb @ ta + tb)
    assert np.allclose(mb, mc, atol=1e-12) and np.allclose(sbb, sc)
    for i in range(len(means)):   # quaternions agree up to sign: compare the rotations
        assert np.allclose(of.rotation_of_quat(qb[i]), of.rotation_of_quat(qc[i]), atol=1e-12)


def test_quaternion_conversions_against_scipy():
    for seed in range(8):
        R = _rot(10 + seed)
        q = of.quat_of_rotation(R)                       # (w,x,y,z)
        assert abs(np.linalg.norm(q) - 1) < 1e-12
        assert np.allclose(of.rotation_of_quat(q), R, atol=1e-12)
        qs = Rotation.from_matrix(R).as_quat()           # scipy: (x,y,z,w)
        qs = np.array([qs[3], qs[0], qs[1], qs[2]])
        assert np.allclose(q, qs * np.sign(qs[np.flatnonzero(np.abs(qs) > 1e-12)[0]]), atol=1e-12)
    # 180-degree rotation (w = 0): the trace-based textbook formula breaks down here, the eigenvector form does not
    R = np.diag([1.0, -1.0, -1.0])
    assert np.allclose(of.rotation_of_quat(of.quat_of_rotation(R)), R, atol=1e-12)


def test_rendered_image_is_invariant_when_the_camera_moves_with_the_similarity(oracle):
    """Eq. 19 with s = 1 is a rigid motion of the map; composing the camera with its inverse (Eq. 15) must
    reproduce the image (degree-0 colour: 'unchanged color' does not rotate SH)."""
    from paper_2605_10760_b200 import scenes
    sc = scenes.tiny_scene()
    ref = oracle.forward(sc)
    R, t = _rot(21), np.array([0.2, -0.1, 0.3])
    m2, s2, q2 = of.sim3_apply(sc.means, sc.scales, sc.quats, 1.0, R, t)
    import copy
    sc2 = copy.copy(sc)
    sc2.means = m2.astype(np.float32); sc2.scales = s2.astype(np.float32); sc2.quats = q2.astype(np.float32)
    cam = sc.camera.copy()
    W, tc = sc.camera.T_cw[:, :3].astype(np.float64), sc.camera.T_cw[:, 3].astype(np.float64)
    T2 = np.zeros((3, 4)); T2[:, :3] = W @ R.T; T2[:, 3] = tc - W @ R.T @ t   # p_c = W R^T (p' - t) + t_c
    cam.T_cw = T2.astype(np.float32)
    got = oracle.forward(sc2, camera=cam)
    assert np.abs(got["rgb"] - ref["rgb"]).max() < 2e-5 and np.abs(got["depth"] - ref["depth"]).max() < 2e-5
