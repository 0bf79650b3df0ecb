"""GPU parity of gs_sim3_apply (Eq. 19) against oracle/fusion.py on the same seeded inputs: centres and
scales within fp32 rounding of the fp64 result, rotations compared as matrices (quaternions are sign-ambiguous), in place
and out of place, including a 180-degree rotation (w = 0 branch of the host quaternion conversion)."""
import numpy as np
import pytest
from scipy.spatial.transform import Rotation

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("case", ["random", "half_turn", "identity"])
def test_sim3_apply_matches_oracle(case):
    import torch
    from oracle import fusion as of
    from paper_2605_10760_b200 import binding as b
    r = np.random.Generator(np.random.PCG64(77))
    N = 100_003
    means = r.uniform(-4, 4, (N, 3)).astype(np.float32)
    scales = np.exp(r.normal(-4.5, 0.5, (N, 3))).astype(np.float32)
    quats = r.normal(size=(N, 4)).astype(np.float32)
    if case == "random":
        s, R, t = 1.37, Rotation.random(random_state=5).as_matrix(), np.array([0.4, -1.1, 0.25])
    elif case == "half_turn":
        s, R, t = 0.5, np.diag([-1.0, 1.0, -1.0]), np.array([1.0, 2.0, 3.0])
    else:
        s, R, t = 1.0, np.eye(3), np.zeros(3)
    R32 = R.astype(np.float32); t32 = t.astype(np.float32)
    rm, rs, rq = of.sim3_apply(means[:2000], scales[:2000], quats[:2000], np.float32(s), R32, t32)   # oracle on a sample
    dm, dsc, dq = (torch.from_numpy(a).cuda() for a in (means, scales, quats))
    om, os_, oq = torch.empty_like(dm), torch.empty_like(dsc), torch.empty_like(dq)
    b.gs_sim3_apply(s, R32, t32, dm, dsc, dq, om, os_, oq)
    torch.cuda.synchronize()
    gm, gs_, gq = om.cpu().numpy(), os_.cpu().numpy(), oq.cpu().numpy()
    assert np.abs(gm[:2000] - rm).max() <= 4e-6 * (1 + np.abs(rm).max())
    assert np.abs(gs_[:2000] / rs - 1).max() <= 2e-7
    for i in range(0, 2000, 37):
        assert np.abs(of.rotation_of_quat(gq[i].astype(np.float64)) - of.rotation_of_quat(rq[i])).max() < 5e-6
        # covariance law Sigma' = s^2 R Sigma R^T, end to end on the GPU outputs
        lhs = of.covariance(gs_[i], gq[i])
        rhs = float(np.float32(s)) ** 2 * R32.astype(np.float64) @ of.covariance(scales[i], quats[i]) @ R32.astype(np.float64).T
        assert np.abs(lhs - rhs).max() <= 2e-5 * np.abs(rhs).max()
    # in place gives the same bits
    b.gs_sim3_apply(s, R32, t32, dm, dsc, dq)
    torch.cuda.synchronize()
    assert torch.equal(dm, om) and torch.equal(dsc, os_) and torch.equal(dq, oq)
    if case == "identity":
        assert np.array_equal(gm, means) and np.array_equal(gs_, scales) and np.array_equal(gq, quats)
