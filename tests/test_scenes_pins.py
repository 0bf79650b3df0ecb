"""CPU pins of the one piece of arithmetic the input-generator module carries: scenes.se3_exp / scenes.perturb_pose, the
left-multiplicative twist used to PERTURB input poses (config 4 target pose, test cameras; reading Q14 / C4 of DESIGN.md,
PAPER.md:317 "per-keyframe pose deltas").  It never checks a result, but both sides are fed with what it produces, so it
is pinned like an oracle function: against the matrix exponential of the 4x4 twist (scipy), and against the oracle's own
statement of the same map (gso.pose_apply, which test_oracle_pins.py pins separately)."""
import numpy as np
import pytest
from scipy.linalg import expm

from paper_2605_10760_b200 import scenes


def _hat(xi):
    rho, phi = xi[:3], xi[3:]
    M = np.zeros((4, 4))
    M[:3, :3] = [[0, -phi[2], phi[1]], [phi[2], 0, -phi[0]], [-phi[1], phi[0], 0]]
    M[:3, 3] = rho
    return M


@pytest.mark.parametrize("scale", [0.0, 1e-10, 1e-4, 0.05, 1.0, 3.0])
def test_perturb_pose_is_expm_of_the_twist_times_the_pose(scale, oracle):
    r = np.random.Generator(np.random.PCG64(5))
    for trial in range(5):
        xi = r.normal(0, 1, 6) * scale
        T = scenes.perturb_pose(scenes.look_at(r.uniform(-2, 2, 3), r.uniform(3, 5, 3)), r.normal(0, 0.3, 6)).astype(np.float64)
        T4 = np.vstack([T, [0, 0, 0, 1]])
        want = (expm(_hat(xi)) @ T4)[:3]
        got = scenes.perturb_pose(T.astype(np.float32), xi).astype(np.float64)
        assert np.abs(got - want).max() <= 2e-7 * (1 + np.abs(want).max())          # float32 output
        R, t = scenes.se3_exp(xi)
        assert np.abs(R - expm(_hat(xi))[:3, :3]).max() <= 1e-12 and np.abs(t - expm(_hat(xi))[:3, 3]).max() <= 1e-12
        assert np.abs(R @ R.T - np.eye(3)).max() <= 1e-12
        # the oracle's statement of the same update
        assert np.abs(oracle.pose_apply(xi, T) - want).max() <= 1e-12 * (1 + np.abs(want).max())


def test_perturb_pose_translation_and_rotation_parts_are_not_swapped():
    T = np.concatenate([np.eye(3), np.zeros((3, 1))], 1).astype(np.float32)
    assert np.allclose(scenes.perturb_pose(T, [0.1, 0.2, 0.3, 0, 0, 0]), np.concatenate([np.eye(3), [[0.1], [0.2], [0.3]]], 1))
    Rz = scenes.perturb_pose(T, [0, 0, 0, 0, 0, np.pi / 2])        # quarter turn about z: x -> y
    assert np.allclose(Rz[:, :3] @ [1, 0, 0], [0, 1, 0], atol=1e-7) and np.allclose(Rz[:, 3], 0)
