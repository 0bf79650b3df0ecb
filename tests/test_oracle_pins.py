"""Pins of the fp64 oracle (oracle/gso.cpp) to things other than itself: library routines (scipy), closed forms,
invariants, brute force and central finite differences.  The paper prints no worked numeric example for the renderer
(SURVEY.md section 4), so no tests/golden value comes from it; every pin below is mathematical.  CPU only.
"""
import copy
import types

import numpy as np
import pytest
from scipy.spatial.transform import Rotation

from paper_2605_10760_b200 import scenes


def as64(sc):
    """Scene copy with float64 parameter arrays (the oracle takes doubles; FD tests perturb below fp32 resolution)."""
    s = copy.copy(sc)
    for k in ("means", "scales", "quats", "opacities", "sh"):
        setattr(s, k, np.asarray(getattr(sc, k), dtype=np.float64).copy())
    return s


def small_scene(seed, N=12, size=12, sh_degree=3, pose=True):
    rng = np.random.default_rng(seed)
    means = np.concatenate([rng.uniform(-0.8, 0.8, (N, 2)), rng.uniform(2.0, 4.0, (N, 1))], axis=1)
    scales = np.exp(rng.normal(-1.6, 0.4, (N, 3)))
    quats = rng.normal(size=(N, 4))
    opac = 1 / (1 + np.exp(-rng.normal(0, 1, N)))
    K = (sh_degree + 1) ** 2
    sh = rng.normal(0, 0.4, (N, K, 3))
    cam = scenes.Camera(size, size, float(size), float(size), (size - 1) / 2, (size - 1) / 2, scenes.identity_pose())
    if pose:
        xi = np.concatenate([rng.normal(0, 0.1, 3), rng.normal(0, 0.15, 3)])
        cam.T_cw = scenes.perturb_pose(cam.T_cw, xi)
    sc = scenes.Scene(means, scales, quats, opac, sh, sh_degree, cam, rng.uniform(0, 1, 3), name="small")
    return as64(sc)


# ------------------------------------------------------------------------------------------------------------------
# quaternion -> R, SE(3) exponential
# ------------------------------------------------------------------------------------------------------------------
def test_quat_to_R_matches_scipy_and_rodrigues(oracle):
    rng = np.random.default_rng(0)
    for _ in range(50):
        q = rng.normal(size=4) * rng.uniform(0.1, 5)
        R = oracle.quat_to_R(q)
        assert np.allclose(R @ R.T, np.eye(3), atol=1e-14)
        assert abs(np.linalg.det(R) - 1) < 1e-14
        Rs = Rotation.from_quat([q[1], q[2], q[3], q[0]]).as_matrix()  # scipy is scalar-last
        assert np.allclose(R, Rs, atol=1e-14)
        assert np.allclose(oracle.quat_to_R(-q), R, atol=1e-15)
    # axis-angle (Rodrigues): q = (cos(th/2), sin(th/2) axis)
    axis = np.array([1.0, 2.0, -0.5]); axis /= np.linalg.norm(axis); th = 0.7
    K = np.array([[0, -axis[2], axis[1]], [axis[2], 0, -axis[0]], [-axis[1], axis[0], 0]])
    Rrod = np.eye(3) + np.sin(th) * K + (1 - np.cos(th)) * K @ K
    assert np.allclose(oracle.quat_to_R(np.concatenate([[np.cos(th / 2)], np.sin(th / 2) * axis])), Rrod, atol=1e-15)


def test_se3_exp_matches_matrix_exponential(oracle):
    from scipy.linalg import expm
    rng = np.random.default_rng(1)
    for scale in (1.0, 1e-3, 1e-9, 0.0):
        xi = rng.normal(size=6) * np.array([1, 1, 1, scale, scale, scale])
        R, t = oracle.se3_exp(xi)
        A = np.zeros((4, 4))
        A[:3, :3] = [[0, -xi[5], xi[4]], [xi[5], 0, -xi[3]], [-xi[4], xi[3], 0]]
        A[:3, 3] = xi[:3]
        E = expm(A)
        assert np.allclose(R, E[:3, :3], atol=1e-13) and np.allclose(t, E[:3, 3], atol=1e-13)
    T = np.concatenate([Rotation.from_rotvec([0.1, -0.2, 0.3]).as_matrix(), [[0.5], [-1], [2]]], axis=1)
    xi = rng.normal(size=6) * 0.3
    R, t = oracle.se3_exp(xi)
    To = oracle.pose_apply(xi, T)
    assert np.allclose(To[:, :3], R @ T[:, :3], atol=1e-14) and np.allclose(To[:, 3], R @ T[:, 3] + t, atol=1e-14)


# ------------------------------------------------------------------------------------------------------------------
# real spherical harmonics
# ------------------------------------------------------------------------------------------------------------------
def _sphere_quadrature(nth=24, nph=48):
    x, w = np.polynomial.legendre.leggauss(nth)  # x = cos(theta)
    ph = (np.arange(nph) + 0.5) * 2 * np.pi / nph
    ct, phg = np.meshgrid(x, ph, indexing="ij")
    st = np.sqrt(1 - ct * ct)
    n = np.stack([st * np.cos(phg), st * np.sin(phg), ct], axis=-1).reshape(-1, 3)
    wt = np.repeat(w, nph) * (2 * np.pi / nph)
    return n, wt


def test_sh_orthonormal_on_the_sphere(oracle):
    n, wt = _sphere_quadrature()
    B = np.stack([oracle.sh_basis(3, v)[0] for v in n])
    G = (B * wt[:, None]).T @ B
    assert np.allclose(G, np.eye(16), atol=1e-13)
    assert abs(oracle.sh_basis(0, n[0])[0][0] - 0.28209479177387814) < 1e-16  # 1/(2 sqrt(pi))
    # lower degrees are prefixes, zero-padded
    for deg, K in ((0, 1), (1, 4), (2, 9)):
        Bd = oracle.sh_basis(deg, n[5])[0]
        assert np.allclose(Bd[:K], B[5, :K], atol=0) and np.all(Bd[K:] == 0)


def test_sh_matches_scipy_complex_harmonics(oracle):
    """Real SH from scipy's complex Y_l^m (Condon-Shortley); the oracle's basis is the real form with sign (-1)^m."""
    from scipy.special import sph_harm_y
    rng = np.random.default_rng(2)
    for _ in range(20):
        v = rng.normal(size=3); v /= np.linalg.norm(v)
        theta, phi = np.arccos(v[2]), np.arctan2(v[1], v[0])
        B = oracle.sh_basis(3, v)[0]
        k = 0
        for l in range(4):
            for m in range(-l, l + 1):
                Y = sph_harm_y(l, abs(m), theta, phi)
                if m == 0:
                    ref = Y.real
                elif m > 0:
                    ref = np.sqrt(2) * (-1) ** m * Y.real
                else:
                    ref = np.sqrt(2) * (-1) ** m * Y.imag
                assert abs(B[k] - (-1) ** m * ref) < 1e-13, (l, m)
                k += 1


def test_sh_jacobian_and_homogeneity(oracle):
    rng = np.random.default_rng(3)
    v = rng.normal(size=3)
    B, dB = oracle.sh_basis(3, v)
    h = 1e-6
    for j in range(3):
        e = np.zeros(3); e[j] = h
        fd = (oracle.sh_basis(3, v + e)[0] - oracle.sh_basis(3, v - e)[0]) / (2 * h)
        assert np.allclose(fd, dB[:, j], rtol=1e-8, atol=1e-8)
    lam = 1.7
    Bl = oracle.sh_basis(3, lam * v)[0]
    deg = np.array([0] + [1] * 3 + [2] * 5 + [3] * 7)
    assert np.allclose(Bl, lam ** deg * B, rtol=1e-13)


# ------------------------------------------------------------------------------------------------------------------
# EWA projection
# ------------------------------------------------------------------------------------------------------------------
def _one_gaussian(mu, s, q, o, rgb, size=33, f=40.0, T=None):
    cam = scenes.Camera(size, size, f, f, (size - 1) / 2, (size - 1) / 2, scenes.identity_pose() if T is None else T)
    sh = scenes.rgb_to_sh0(np.asarray(rgb, dtype=np.float64))[None, None, :]
    sc = scenes.Scene(np.array([mu], float), np.array([s], float), np.array([q], float), np.array([o], float), sh, 0,
                      cam, np.zeros(3), name="one")
    return sc


def test_ewa_isotropic_on_axis_closed_form(oracle):
    sigma, z0, f = 0.05, 2.5, 40.0
    sc = _one_gaussian([0, 0, z0], [sigma] * 3, [0.3, -0.5, 0.2, 0.7], 0.8, [0.2, 0.5, 0.9], f=f)
    ft = oracle.preprocess(sc)
    v = (f * sigma / z0) ** 2 + 0.3
    assert np.allclose(ft["cov2d"][0], [v, 0, v], atol=1e-13)
    assert np.allclose(ft["conic"][0], [1 / v, 0, 1 / v], atol=1e-13)
    assert np.allclose(ft["mean2d"][0], [16, 16]) and ft["z32"][0] == np.float32(z0)
    assert np.allclose(ft["color"][0], [0.2, 0.5, 0.9], atol=1e-15)


def test_ewa_matches_monte_carlo_projection(oracle):
    """Sample N(mu, Sigma) with a tiny Sigma, push the samples through the pinhole, compare the empirical covariance
    with J W Sigma W^T J^T (+ 0.3 I removed)."""
    rng = np.random.default_rng(4)
    mu = np.array([0.4, -0.3, 3.0]); s = np.array([2e-3, 5e-3, 1e-3]); q = rng.normal(size=4)
    T = scenes.perturb_pose(scenes.identity_pose(), [0.1, -0.2, 0.05, 0.2, -0.1, 0.3]).astype(np.float64)
    sc = _one_gaussian(mu, s, q, 0.9, [0.5] * 3, f=300.0, size=400, T=T.astype(np.float32))
    T = sc.camera.T_cw.astype(np.float64)
    ft = oracle.preprocess(sc)
    assert ft["visible"][0]
    R = Rotation.from_quat([q[1], q[2], q[3], q[0]]).as_matrix()
    L = R @ np.diag(s)
    pts = mu + rng.normal(size=(400000, 3)) @ L.T
    pc = pts @ T[:, :3].T + T[:, 3]
    uv = np.stack([300.0 * pc[:, 0] / pc[:, 2], 300.0 * pc[:, 1] / pc[:, 2]], axis=1)
    emp = np.cov(uv.T)
    got = np.array([[ft["cov2d"][0, 0] - 0.3, ft["cov2d"][0, 1]], [ft["cov2d"][0, 1], ft["cov2d"][0, 2] - 0.3]])
    assert np.allclose(emp, got, rtol=2e-2, atol=1e-3 * np.abs(got).max())
    assert np.allclose(uv.mean(0) + [sc.camera.cx, sc.camera.cy], ft["mean2d"][0], atol=1e-2)


# ------------------------------------------------------------------------------------------------------------------
# single-Gaussian closed form (north_star pin 1)
# ------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("o", [0.6, 0.9999])
def test_single_gaussian_image_closed_form(oracle, o):
    sigma, z0, f, size = 0.3, 2.0, 40.0, 33
    col = np.array([0.2, 0.5, 0.9])
    sc = _one_gaussian([0, 0, z0], [sigma] * 3, [1, 0, 0, 0], o, col, size=size, f=f)
    sc.bg = np.array([0.1, 0.2, 0.3])
    out = oracle.forward(sc)
    v = (f * sigma / z0) ** 2 + 0.3
    yy, xx = np.mgrid[0:size, 0:size].astype(float)
    G = np.exp(-0.5 * ((xx - 16) ** 2 + (yy - 16) ** 2) / v)
    alpha = np.minimum(0.99, o * G)
    alpha = np.where(alpha >= 1 / 255, alpha, 0.0)
    assert np.allclose(out["alpha"], alpha, atol=1e-15)
    assert np.allclose(out["depth"], z0 * alpha, atol=1e-15)
    for ch in range(3):
        assert np.allclose(out["rgb"][ch], col[ch] * alpha + (1 - alpha) * sc.bg[ch], atol=1e-15)
    assert (out["n_blended"] == (alpha > 0)).all()
    # closed-form gradients for L = sum(gC*rgb) with bg = 0: dL/do = sum gC.col G [unclamped], dL/dcol = sum gC alpha
    sc.bg = np.zeros(3)
    rng = np.random.default_rng(5)
    gC = rng.normal(size=(3, size, size)); gD = rng.normal(size=(size, size))
    r = oracle.forward_backward(sc, gC, gD)
    live = (alpha > 0) & (o * G <= 0.99)
    w = np.einsum("c,chw->hw", col, gC) + z0 * gD
    assert np.isclose(r["g_opacities"][0], (w * G * live).sum(), rtol=1e-12)
    assert np.allclose(r["g_color"][0], (gC * alpha).sum(axis=(1, 2)), rtol=1e-12)
    assert np.isclose(r["g_z"][0], (gD * alpha).sum(), rtol=1e-12)
    # d/dv of o exp(-r2/(2v)) = alpha r2/(2 v^2); conic a = c = 1/v  ->  dL/da = -1/2 sum w alpha dx^2 on live pixels
    assert np.isclose(r["g_conic"][0, 0], (-0.5 * w * o * G * (xx - 16) ** 2 * live).sum(), rtol=1e-12)
    assert np.isclose(r["g_conic"][0, 2], (-0.5 * w * o * G * (yy - 16) ** 2 * live).sum(), rtol=1e-12)


def test_opacity_below_threshold_is_culled(oracle):
    sc = _one_gaussian([0, 0, 2], [0.3] * 3, [1, 0, 0, 0], 1 / 255 - 1e-6, [1, 1, 1])
    out = oracle.forward(sc)
    assert not out["visible"][0] and out["alpha"].max() == 0
    sc.opacities[0] = 1 / 255 + 1e-6
    out = oracle.forward(sc)
    assert out["visible"][0] and out["n_blended"].sum() == 1  # only the centre pixel reaches 1/255


# ------------------------------------------------------------------------------------------------------------------
# occlusion (pin 2), monotone transmittance / convexity (pin 3)
# ------------------------------------------------------------------------------------------------------------------
def test_three_opaque_near_gaussians_occlude_everything_behind(oracle):
    sc = small_scene(6, N=40, size=16, sh_degree=1, pose=False)
    sc.bg = np.zeros(3)
    wall = dict(means=np.tile([[0.0, 0.0, 1.0]], (3, 1)) + np.array([[0, 0, 0.0], [0, 0, 1e-3], [0, 0, 2e-3]]),
                scales=np.full((3, 3), 5.0), quats=np.tile([[1.0, 0, 0, 0]], (3, 1)), opacities=np.full(3, 0.999999),
                sh=np.zeros((3, 4, 3)))
    both = copy.copy(sc)
    for k, v in wall.items():
        setattr(both, k, np.concatenate([v, getattr(sc, k)], axis=0))
    only = copy.copy(sc)
    for k, v in wall.items():
        setattr(only, k, v)
    rng = np.random.default_rng(7)
    gC, gD = rng.normal(size=(3, 16, 16)), rng.normal(size=(16, 16))
    a = oracle.forward_backward(both, gC, gD)
    b = oracle.forward_backward(only, gC, gD)
    assert np.allclose(a["alpha"], 1 - 1e-6, atol=1e-12)  # T = 0.01^3 = 1e-6 < 1e-4
    for k in ("rgb", "depth", "alpha"):
        assert np.array_equal(a[k], b[k])
    assert (a["n_blended"] == 3).all()
    for k in ("g_means", "g_scales", "g_quats", "g_opacities", "g_sh"):
        assert np.all(a[k][3:] == 0), k


def test_transmittance_monotone_and_colour_in_hull(oracle):
    sc = as64(scenes.tiny_scene())
    out = oracle.forward(sc)
    assert out["alpha"].min() >= 0 and out["alpha"].max() <= 1
    # prefixes of the depth-ordered list: alpha (= 1 - T) never decreases as Gaussians are appended back to front
    order = np.lexsort((np.arange(sc.N), out["z32"].view(np.uint32)))
    prev = np.zeros_like(out["alpha"])
    for n in (1, 8, 64, 256):
        keep = order[:n]
        sub = copy.copy(sc)
        for k in ("means", "scales", "quats", "opacities", "sh"):
            setattr(sub, k, getattr(sc, k)[keep])
        a = oracle.forward(sub)["alpha"]
        assert (a >= prev - 1e-15).all()
        prev = a
    assert np.allclose(prev, out["alpha"], atol=1e-15)
    # sum of blending weights = alpha: white Gaussians on a black background render alpha in every channel
    white = copy.copy(sc)
    white.sh = scenes.rgb_to_sh0(np.ones((sc.N, 1, 3)))
    w = oracle.forward(white)
    for ch in range(3):
        assert np.allclose(w["rgb"][ch], out["alpha"], atol=1e-14)
    # colour inside alpha * [min col, max col]; depth inside alpha * [min z, max z]
    vis = out["visible"].astype(bool)
    for ch in range(3):
        lo, hi = out["color"][vis][:, ch].min(), out["color"][vis][:, ch].max()
        assert (out["rgb"][ch] >= out["alpha"] * lo - 1e-12).all() and (out["rgb"][ch] <= out["alpha"] * hi + 1e-12).all()
    assert (out["depth"] >= out["alpha"] * 2.0 - 1e-12).all() and (out["depth"] <= out["alpha"] * 4.0 + 1e-12).all()


# ------------------------------------------------------------------------------------------------------------------
# hand-built one-pixel stacks: termination rule Q3(b), clamp gradient Q2, alpha threshold Q1
# ------------------------------------------------------------------------------------------------------------------
def _stack(oracle, alphas, cols, zs, opt=None, gC=(1.0, 0.0, 0.0), gD=0.0, bg=(0, 0, 0), mean2d=None):
    """Gaussians centred on the single pixel (0,0) of a 1x1 image with G = 1 there, so alpha_i = min(.99, o_i)
    (`mean2d` moves the centres: unit conic, so G = exp(-|mean|^2 / 2) at the pixel)."""
    n = len(alphas)
    feat = dict(visible=np.ones(n, np.uint8), mean2d=np.zeros((n, 2)) if mean2d is None else np.asarray(mean2d, float).reshape(n, 2), cov2d=np.tile([[1.0, 0, 1.0]], (n, 1)),
                conic=np.tile([[1.0, 0, 1.0]], (n, 1)), color=np.asarray(cols, float).reshape(n, 3),
                z=np.asarray(zs, float), z32=np.asarray(zs, np.float32))
    cam = types.SimpleNamespace(width=1, height=1, fx=1.0, fy=1.0, cx=0.0, cy=0.0, near_z=0.2,
                                T_cw=scenes.identity_pose())
    return oracle.render(feat, np.asarray(alphas, float), cam, np.asarray(bg, float), opt or oracle.Options(),
                         np.asarray(gC, float).reshape(3, 1, 1), np.full((1, 1), gD), None)


def test_stack_values_by_hand(oracle):
    r = _stack(oracle, [0.5, 0.5], [[1, 0, 0], [0, 1, 0]], [1.0, 2.0], bg=(0, 0, 1))
    assert np.allclose(r["rgb"].ravel(), [0.5, 0.25, 0.25]) and np.isclose(r["depth"][0, 0], 0.5 * 1 + 0.25 * 2)
    assert np.isclose(r["alpha"][0, 0], 0.75)
    # order is by depth, not by input position
    r2 = _stack(oracle, [0.5, 0.5], [[0, 1, 0], [1, 0, 0]], [2.0, 1.0], bg=(0, 0, 1))
    assert np.allclose(r2["rgb"].ravel(), [0.5, 0.25, 0.25])
    # equal depth: lower index first (Q13)
    r3 = _stack(oracle, [0.5, 0.5], [[1, 0, 0], [0, 1, 0]], [1.0, 1.0])
    assert np.allclose(r3["rgb"].ravel(), [0.5, 0.25, 0.0])


def test_termination_rule_blend_iff_T_in_front_at_least_1e_minus_4(oracle):
    # alphas .99,.99 -> T = 1e-4 after two; float: 0.01*0.01 = 1.0000000000000002e-4 >= 1e-4 -> third IS blended
    a = [0.999, 0.999, 0.5, 0.5]
    r = _stack(oracle, a, [[1, 1, 1]] * 4, [1, 2, 3, 4])
    T2 = (1 - 0.99) * (1 - 0.99)
    assert r["n_blended"][0, 0] == (4 if T2 * 0.5 >= 1e-4 else 3)
    # T = 0.01 * 0.005 = 5e-5 < 1e-4 in front of the third -> it is dropped
    r = _stack(oracle, [0.999, 0.999, 0.5], [[1, 0, 0], [1, 0, 0], [0, 1, 0]], [1, 2, 3],
               opt=oracle.Options(alpha_max=0.995))
    assert r["n_blended"][0, 0] == 2 and r["rgb"][1, 0, 0] == 0.0
    assert np.isclose(r["alpha"][0, 0], 1 - 0.005 * 0.005)
    # T in front = 0.01 >= 1e-4 -> blended even though T afterwards is 1e-4 * ...
    r = _stack(oracle, [0.999, 0.9999], [[1, 0, 0], [0, 1, 0]], [1, 2])
    assert r["n_blended"][0, 0] == 2 and np.isclose(r["rgb"][1, 0, 0], 0.01 * 0.99)


def test_alpha_threshold_and_clamp_gradient(oracle):
    # alpha = 1/255 exactly is kept (skip iff alpha < 1/255); just below is skipped
    assert _stack(oracle, [1 / 255], [[1, 1, 1]], [1])["n_blended"][0, 0] == 1
    assert _stack(oracle, [np.nextafter(1 / 255, 0)], [[1, 1, 1]], [1])["n_blended"][0, 0] == 0
    # clamped Gaussian: colour/depth gradients flow (alpha = .99), opacity/conic/mean get nothing (Q2)
    r = _stack(oracle, [0.995, 0.5], [[1, 0, 0], [1, 0, 0]], [1, 2], gC=(1, 0, 0), gD=2.0)
    assert r["g_opac"][0] == 0 and np.all(r["g_conic"][0] == 0) and np.all(r["g_mean2d"][0] == 0)
    assert np.isclose(r["g_color"][0, 0], 0.99) and np.isclose(r["g_z"][0], 2 * 0.99)
    # the unclamped one behind it: dL/dalpha_2 = T_2 w_2 with w = gC.col + gD z = 1 + 4, T_2 = 0.01 ; G = 1 -> dL/do
    assert np.isclose(r["g_opac"][1], 0.01 * 5.0)
    # unclamped pair by hand: L = w1 a1 + w2 a2 (1-a1): dL/da1 = w1 - w2 a2 ; dL/da2 = w2 (1-a1)
    r = _stack(oracle, [0.3, 0.6], [[1, 0, 0], [0.5, 0, 0]], [1, 3], gC=(1, 0, 0), gD=0.5)
    w1, w2 = 1 + 0.5 * 1, 0.5 + 0.5 * 3
    assert np.isclose(r["g_opac"][0], w1 - w2 * 0.6) and np.isclose(r["g_opac"][1], w2 * 0.7)


def test_margin_values_by_hand(oracle):
    """`margin` (C6) decides which pixels the GPU parity tests hold to 1e-5 and which to 1e-2, so its value
    is pinned on one-pixel stacks where it can be computed by hand:
    margin = min( min_i |alpha_i / (1/255) - 1| over evaluated Gaussians, |T / 1e-4 - 1| at every exit test )."""
    # one Gaussian just above the alpha threshold: alpha = (1 + 3e-5)/255 -> 3e-5 (the exit test gives |1/1e-4 - 1|)
    r = _stack(oracle, [(1 + 3e-5) / 255], [[1, 1, 1]], [1])
    assert r["n_blended"][0, 0] == 1 and np.isclose(r["margin"][0, 0], 3e-5, rtol=1e-9, atol=0)
    # just below (opacity 0.5, pixel at the distance where o G = (1 - 3e-5)/255, inside the oracle's padded box):
    # skipped, and the margin is the same distance on the other side
    d = np.sqrt(-2.0 * np.log((1 - 3e-5) / 255 / 0.5))
    r = _stack(oracle, [0.5], [[1, 1, 1]], [1], mean2d=[[d, 0.0]])
    assert r["n_blended"][0, 0] == 0 and np.isclose(r["margin"][0, 0], 3e-5, rtol=1e-6, atol=0)
    r = _stack(oracle, [0.5], [[1, 1, 1]], [1], mean2d=[[0.0, -np.sqrt(-2.0 * np.log((1 + 3e-5) / 255 / 0.5))]])
    assert r["n_blended"][0, 0] == 1 and np.isclose(r["margin"][0, 0], 3e-5, rtol=1e-6, atol=0)
    # a far-from-threshold Gaussian: alpha = 0.5 -> |127.5 - 1| from the alpha test, |1e4 - 1| from the exit test
    r = _stack(oracle, [0.5], [[1, 1, 1]], [1])
    assert np.isclose(r["margin"][0, 0], 126.5, rtol=1e-12)
    # transmittance in front of the third entry = 1e-4 (1 +- delta): margin = delta; + side blends it, - side exits
    opt = oracle.Options(alpha_max=0.99999)
    for delta, blended in ((+1e-3, 3), (-1e-3, 2), (+2.5e-5, 3), (-2.5e-5, 2)):
        a2 = 1.0 - 1e-3 * (1.0 + delta)      # (1 - 0.9)(1 - a2) = 1e-4 (1 + delta)
        r = _stack(oracle, [0.9, a2, 0.5], [[1, 0, 0], [0, 1, 0], [0, 0, 1]], [1, 2, 3], opt=opt)
        T3 = (1.0 - 0.9) * (1.0 - a2)
        assert r["n_blended"][0, 0] == blended
        assert np.isclose(r["margin"][0, 0], abs(T3 / 1e-4 - 1.0), rtol=1e-9) and np.isclose(r["margin"][0, 0], abs(delta), rtol=1e-6)
    # the exit test is only taken for Gaussians that pass the alpha test: a sub-threshold Gaussian at T ~ 1e-4 adds
    # its alpha distance, not its T distance
    d = np.sqrt(-2.0 * np.log(0.0039 / 0.5))   # third Gaussian: opacity 0.5, alpha = 0.0039 < 1/255 at the pixel
    r = _stack(oracle, [0.9, 1.0 - 1e-3 * (1 + 1e-3), 0.5], [[1, 0, 0]] * 3, [1, 2, 3], opt=opt, mean2d=[[0, 0], [0, 0], [d, 0]])
    assert r["n_blended"][0, 0] == 2 and np.isclose(r["margin"][0, 0], abs(0.0039 * 255 - 1.0), rtol=1e-6)
    # a pixel that no Gaussian reaches: +inf (empty list), and >= 1 - tiny when the only Gaussian is far away
    r = _stack(oracle, [], np.zeros((0, 3)), [])
    assert np.isinf(r["margin"][0, 0]) and r["margin"][0, 0] > 0
    n = 1
    feat = dict(visible=np.ones(n, np.uint8), mean2d=np.full((n, 2), 40.0), cov2d=np.tile([[1.0, 0, 1.0]], (n, 1)),
                conic=np.tile([[1.0, 0, 1.0]], (n, 1)), color=np.ones((n, 3)), z=np.ones(n), z32=np.ones(n, np.float32))
    cam = types.SimpleNamespace(width=1, height=1, fx=1.0, fy=1.0, cx=0.0, cy=0.0, near_z=0.2, T_cw=scenes.identity_pose())
    for brute in (False, True):
        r = oracle.render(feat, np.array([0.9]), cam, np.zeros(3), oracle.Options(brute_force=brute))
        assert r["n_blended"][0, 0] == 0 and r["margin"][0, 0] >= 1.0 - 1e-12


# ------------------------------------------------------------------------------------------------------------------
# analytic gradients vs central finite differences (pin 4), incl. the pose; pose <-> means consistency
# ------------------------------------------------------------------------------------------------------------------
def _loss(oracle, sc, gC, gD, gA, opt, T64=None):
    out = oracle.forward(sc, opt, T_cw64=T64)
    return float((gC * out["rgb"]).sum() + (gD * out["depth"]).sum() + (gA * out["alpha"]).sum()), out


def _analytic(oracle, sc, gC, gD, gA, opt, T64=None):
    feat = oracle.preprocess(sc, opt, T_cw64=T64)
    cam = copy.copy(sc.camera)
    img = oracle.render(feat, sc.opacities, cam, sc.bg, opt, gC, gD, gA) if T64 is None else None
    return feat, img


@pytest.mark.parametrize("cutoffs", [False, True])
def test_gradients_match_central_finite_differences(oracle, cutoffs):
    opt = oracle.Options() if cutoffs else oracle.Options.no_cutoffs()
    rng = np.random.default_rng(11)
    for seed in range(40):
        sc = small_scene(100 + seed, N=12, size=12, sh_degree=3)
        if cutoffs:  # need every threshold decision to sit well away from its boundary
            if oracle.forward(sc, opt)["margin"].min() < 1e-3:
                continue
        break
    else:
        pytest.fail("no scene with margin > 1e-3 found")
    H = W = 12
    gC, gD, gA = rng.normal(size=(3, H, W)), rng.normal(size=(H, W)), rng.normal(size=(H, W))
    feat = oracle.preprocess(sc, opt)
    img = oracle.render(feat, sc.opacities, sc.camera, sc.bg, opt, gC, gD, gA)
    g = oracle.preprocess_bwd(sc, img, opt)
    if cutoffs:  # the cut-offs are live in this scene: some pixel blends fewer Gaussians than are visible
        assert (img["n_blended"] < feat["visible"].sum()).any()
    names = dict(means="g_means", scales="g_scales", quats="g_quats", opacities="g_opacities", sh="g_sh")
    for pname, gname in names.items():
        base = getattr(sc, pname)
        for trial in range(6):
            u = rng.normal(size=base.shape)
            if trial >= 3:  # single-element directions
                u = np.zeros(base.size); u[rng.integers(base.size)] = 1.0; u = u.reshape(base.shape)
            h = 1e-6
            sp, sm = copy.copy(sc), copy.copy(sc)
            setattr(sp, pname, base + h * u); setattr(sm, pname, base - h * u)
            fd = (_loss(oracle, sp, gC, gD, gA, opt)[0] - _loss(oracle, sm, gC, gD, gA, opt)[0]) / (2 * h)
            an = float((g[gname] * u).sum())
            scale = max(abs(an), np.abs(g[gname]).max() * 1e-3, 1e-9)
            assert abs(fd - an) / scale < 2e-6, (pname, trial, fd, an)
    # pose: T <- Exp(h xi) T in full double precision
    T0 = sc.camera.T_cw.astype(np.float64)
    for trial in range(8):
        xi = rng.normal(size=6)
        if trial >= 2:
            xi = np.zeros(6); xi[trial - 2] = 1.0
        h = 1e-6
        Lp = _loss(oracle, sc, gC, gD, gA, opt, oracle.pose_apply(h * xi, T0))[0]
        Lm = _loss(oracle, sc, gC, gD, gA, opt, oracle.pose_apply(-h * xi, T0))[0]
        fd, an = (Lp - Lm) / (2 * h), float(g["g_twist"] @ xi)
        scale = max(abs(an), np.abs(g["g_twist"]).max() * 1e-3)
        assert abs(fd - an) / scale < 2e-6, (trial, fd, an)
    # rigid-translation equivalence: dL/drho = W sum_i dL/dmu_i  (holds with SH colour); exact for orthonormal W, the
    # float32-rounded pose is orthonormal to ~3e-8 only
    Wm = T0[:, :3]
    assert np.allclose(g["g_twist"][:3], Wm @ g["g_means"].sum(0), rtol=0, atol=1e-6 * np.abs(g["g_twist"]).max())


def test_quaternion_gradient_is_tangential_and_scales_inversely(oracle):
    sc = small_scene(12, N=6, size=10, sh_degree=0)
    rng = np.random.default_rng(12)
    gC, gD = rng.normal(size=(3, 10, 10)), rng.normal(size=(10, 10))
    g1 = oracle.forward_backward(sc, gC, gD)
    assert np.allclose((g1["g_quats"] * sc.quats).sum(1), 0, atol=1e-9 * np.abs(g1["g_quats"]).max())
    s2 = copy.copy(sc); s2.quats = sc.quats * 3.0
    g2 = oracle.forward_backward(s2, gC, gD)
    assert np.allclose(g2["g_quats"] * 3.0, g1["g_quats"], rtol=1e-10, atol=1e-12)
    assert np.allclose(g2["rgb"], g1["rgb"], atol=1e-14)


# ------------------------------------------------------------------------------------------------------------------
# Eq. 19 + Eq. 15: Sim(3) on the Gaussians, inverse on the right of the camera pose
# ------------------------------------------------------------------------------------------------------------------
def _apply_sim3(sc, s, Rm, t):
    out = copy.copy(sc)
    out.means = s * sc.means @ Rm.T + t
    out.scales = s * sc.scales
    rq = Rotation.from_matrix(Rm) * Rotation.from_quat(sc.quats[:, [1, 2, 3, 0]])
    out.quats = rq.as_quat()[:, [3, 0, 1, 2]]
    return out


def test_rigid_transform_of_map_and_camera_leaves_image_unchanged(oracle):
    sc = small_scene(13, N=30, size=24, sh_degree=0)
    Rm = Rotation.from_rotvec([0.4, -0.7, 0.2]).as_matrix(); t = np.array([0.3, -1.2, 0.8])
    moved = _apply_sim3(sc, 1.0, Rm, t)
    T = sc.camera.T_cw.astype(np.float64)
    Tn = np.concatenate([T[:, :3] @ Rm.T, (T[:, 3] - T[:, :3] @ Rm.T @ t)[:, None]], axis=1)  # T o C^-1
    a = oracle.forward(sc, T_cw64=T)
    b = oracle.forward(moved, T_cw64=Tn)
    for k in ("rgb", "depth", "alpha"):
        assert np.allclose(a[k], b[k], atol=1e-11), k


def test_scale_covariance_depth_scales_rgb_alpha_do_not(oracle):
    sc = small_scene(14, N=30, size=24, sh_degree=2)
    lam = 1.7
    opt = oracle.Options(dilation=0.0)
    T = sc.camera.T_cw.astype(np.float64)
    big = _apply_sim3(sc, lam, np.eye(3), np.zeros(3))
    big.camera = sc.camera.copy(); big.camera.near_z = sc.camera.near_z * lam
    Tn = T.copy(); Tn[:, 3] *= lam
    a = oracle.forward(sc, opt, T_cw64=T)
    b = oracle.forward(big, opt, T_cw64=Tn)
    assert np.allclose(a["rgb"], b["rgb"], atol=1e-11) and np.allclose(a["alpha"], b["alpha"], atol=1e-11)
    assert np.allclose(lam * a["depth"], b["depth"], atol=1e-10)


# ------------------------------------------------------------------------------------------------------------------
# bounding boxes are conservative; binning by brute force
# ------------------------------------------------------------------------------------------------------------------
def test_boxed_rendering_equals_brute_force(oracle):
    rng = np.random.default_rng(15)
    for sc in (scenes.tiny_scene(), scenes.replica_scene(seed=31, N=5000, width=160, height=120, f=80.0)):
        gC = rng.normal(size=(3, sc.camera.height, sc.camera.width)); gD = rng.normal(size=gC.shape[1:])
        a = oracle.forward_backward(sc, gC, gD)
        b = oracle.forward_backward(sc, gC, gD, opt=oracle.Options(brute_force=True))
        assert a["visible"].sum() > 50
        for k in ("rgb", "depth", "alpha", "n_blended", "g_means", "g_scales", "g_quats", "g_opacities", "g_sh",
                  "g_twist"):
            assert np.array_equal(a[k], b[k]), k


def test_exact_rect_is_tight_and_conservative(oracle):
    """Every pixel with alpha >= 1/255 lies inside rect_px; each rect edge row/column holds such a pixel or the
    ellipse's extreme point falls between pixel centres (so shrinking by one full pixel would cut the ellipse)."""
    sc = scenes.replica_scene(seed=32, N=3000, width=160, height=120, f=80.0)
    ft = oracle.preprocess(sc)
    yy, xx = np.mgrid[0:120, 0:160].astype(float)
    n_checked = 0
    for i in np.flatnonzero(ft["visible"])[:400]:
        a, b, c = ft["conic"][i]; mx, my = ft["mean2d"][i]
        dx, dy = xx - mx, yy - my
        al = sc.opacities[i] * np.exp(-0.5 * (a * dx * dx + c * dy * dy) - b * dx * dy)
        ys, xs = np.nonzero(al >= 1 / 255)
        x0, y0, x1, y1 = ft["rect_px"][i]
        if len(xs):
            assert xs.min() >= x0 and xs.max() < x1 and ys.min() >= y0 and ys.max() < y1
        # exact half widths: rho sqrt(cov)
        rho = np.sqrt(2 * np.log(sc.opacities[i] * 255.0))
        assert x0 == max(0, int(np.ceil(mx - rho * np.sqrt(ft["cov2d"][i, 0]))))
        assert y1 == min(120, int(np.floor(my + rho * np.sqrt(ft["cov2d"][i, 2]))) + 1)
        tx0, ty0, tx1, ty1 = ft["rect_tile"][i]
        assert (tx0, ty0, tx1, ty1) == (x0 // 16, y0 // 16, (x1 - 1) // 16 + 1, (y1 - 1) // 16 + 1)
        n_checked += 1
    assert n_checked > 100


def test_binning_matches_brute_force_lists(oracle):
    sc = scenes.replica_scene(seed=33, N=4000, width=160, height=120, f=80.0)
    ft = oracle.preprocess(sc)
    tx, ty = 10, 8
    keys, ids, ranges = oracle.bin_tiles(ft["rect_tile"], ft["z32"], tx, ty)
    bits = ft["z32"].view(np.uint32)
    pos = 0
    for t in range(tx * ty):
        cx, cy = t % tx, t // tx
        r = ft["rect_tile"]
        members = [i for i in range(sc.N) if r[i, 0] <= cx < r[i, 2] and r[i, 1] <= cy < r[i, 3]]
        members.sort(key=lambda i: (int(bits[i]), i))
        n = len(members)
        assert list(ids[pos:pos + n]) == members
        assert all(int(k) == (t << 32 | int(bits[i])) for k, i in zip(keys[pos:pos + n], members))
        assert tuple(ranges[t]) == ((pos, pos + n) if n else (0, 0))
        pos += n
    assert pos == len(keys) and len(keys) == int(((ft["rect_tile"][:, 2] - ft["rect_tile"][:, 0]) *
                                                 (ft["rect_tile"][:, 3] - ft["rect_tile"][:, 1])).sum())
    assert np.all(np.diff(keys.astype(np.uint64)) >= 0)


def test_depth_key_is_the_canonical_fp32_fma_chain(oracle):
    sc = scenes.replica_scene(seed=34, N=2000, width=160, height=120, f=80.0)
    ft = oracle.preprocess(sc)
    T = sc.camera.T_cw.astype(np.float32)
    mu = sc.means.astype(np.float32)

    def fma32(a, b, c):  # exact product and sum in double, rounded once to fp32 (= fmaf; 24+24 < 53 bits)
        return np.float32(np.float64(a) * np.float64(b) + np.float64(c))
    for i in range(0, 2000, 37):
        ref = fma32(T[2, 0], mu[i, 0], fma32(T[2, 1], mu[i, 1], fma32(T[2, 2], mu[i, 2], T[2, 3])))
        assert ft["z32"][i] == ref
