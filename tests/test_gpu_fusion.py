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


# ----------------------------------------------------------------------------------------------------------------------
# Eqs. 20-22: occupancy sets and the retain test against oracle/fusion.py (set contents as sorted key lists, retain
# masks, order-preserving compaction).  O_occ, retain masks and index lists are bit-exact.  O_free is compared up to the
# voxels the oracle reports as undetermined by the mathematics (two boundary crossings, or a crossing and t = 1, closer
# than rounding resolves: free_keys' `ambiguous`): the symmetric difference must lie inside that set, and the set must be
# tiny -- on generic inputs it is empty, so the comparison is exact in practice and says so when it is not.
# ----------------------------------------------------------------------------------------------------------------------
def _f32(x):
    return np.ascontiguousarray(x, np.float32)


def _assert_equal_up_to_ties(got, keys, amb, rays):
    diff = np.setxor1d(got, keys)
    print(f"free set: {len(keys)} keys, {len(amb)} ambiguous, {len(diff)} differ")
    assert np.isin(diff, amb).all(), (len(diff), len(amb))
    # a ray steps ~10^2 times and a step is ambiguous with probability ~10^-12 (tolerance / spread of the crossing
    # parameters): anything beyond a handful means the tolerance or one of the two walks is wrong
    assert len(amb) <= 8 + rays // 100_000


def test_occupied_set_matches_oracle_bit_exact():
    import torch
    from oracle import fusion as of
    from paper_2605_10760_b200 import binding as b, scenes
    sc = scenes.replica_scene(seed=61, N=3000, width=64, height=48, f=32.0, sh_degree=0)
    v, k = np.float32(0.02), np.float32(1.5)
    want = np.array(sorted(of.occupied_set(sc.means, sc.scales, float(v), float(k))), np.uint64)
    vs = b.VoxelSet(1 << 17)
    vs.insert_boxes(torch.from_numpy(sc.means).cuda(), torch.from_numpy(sc.scales).cuda(), v, k)
    torch.cuda.synchronize()
    assert int(vs.overflow.item()) == 0
    assert np.array_equal(vs.keys(), want) and len(want) > 3000
    # inserting the same Gaussians again changes nothing; a table that is too small reports the overflow
    vs.insert_boxes(torch.from_numpy(sc.means).cuda(), torch.from_numpy(sc.scales).cuda(), v, k)
    torch.cuda.synchronize()
    assert np.array_equal(vs.keys(), want)
    small = b.VoxelSet(1 << 10)
    small.insert_boxes(torch.from_numpy(sc.means).cuda(), torch.from_numpy(sc.scales).cuda(), v, k)
    torch.cuda.synchronize()
    assert int(small.overflow.item()) > 0 and len(small.keys()) == 1 << 10


@pytest.mark.parametrize("stride", [1, 3])
def test_free_set_matches_oracle_bit_exact(stride):
    import torch
    from oracle import fusion as of
    from paper_2605_10760_b200 import binding as b, scenes
    r = np.random.Generator(np.random.PCG64(62 + stride))
    W, H = 37, 23          # ragged against the stride and the CTA size
    cam = scenes.Camera(W, H, 30.0, 31.0, 18.25, 11.0, scenes.perturb_pose(scenes.look_at([1.0, 2.0, 1.2], [4.0, 3.0, 1.0]),
                                                                               r.normal(0, 0.05, 6)))
    depth = _f32(r.uniform(0.4, 3.0, (H, W)))
    depth[r.uniform(size=(H, W)) < 0.15] = 0.0       # invalid pixels cast no ray
    v = np.float32(0.05)
    c, pts = of.backproject(depth, np.float32(cam.fx), np.float32(cam.fy), np.float32(cam.cx), np.float32(cam.cy),
                            _f32(cam.T_cw), stride)
    keys, amb = of.free_keys(c, pts, float(v))
    vs = b.VoxelSet(1 << 18)
    vs.insert_rays(cam, torch.from_numpy(depth).cuda(), v, stride)
    torch.cuda.synchronize()
    assert int(vs.overflow.item()) == 0
    _assert_equal_up_to_ties(vs.keys(), keys, amb, len(pts))


def test_retain_and_compaction_config5_shaped():
    """Config-5 shape: a target submap and three borrowed submaps mapped by Eq. 19 into its frame (reduced to 4 x 20k
    Gaussians so that the pure-Python oracle finishes in seconds); Eq. 22 retain masks bit-exact, retained Gaussians compacted
    in their original order."""
    import torch
    from oracle import fusion as of
    from paper_2605_10760_b200 import binding as b, scenes
    sc, cams = scenes.fused_scene(seed=63, N_sub=20_000, submaps=4, views=2, width=48, height=32, f=24.0, sh_degree=0)
    n = 20_000
    tgt_m, tgt_s = sc.means[:n], sc.scales[:n]
    src_m = sc.means[n:]
    v, k = np.float32(0.04), np.float32(1.0)
    occ_o = of.occupied_set(tgt_m, tgt_s, float(v), float(k))
    depth = _f32(np.random.Generator(np.random.PCG64(64)).uniform(1.0, 4.0, (32, 48)))
    free_o = set()
    for cam in cams:
        free_o |= of.free_set(depth, np.float32(cam.fx), np.float32(cam.fy), np.float32(cam.cx), np.float32(cam.cy),
                              _f32(cam.T_cw), float(v), 1)
    want = of.retain_mask(src_m, occ_o, free_o, float(v))
    occ, free = b.VoxelSet(1 << 19), b.VoxelSet(1 << 19)
    occ.insert_boxes(torch.from_numpy(tgt_m).cuda(), torch.from_numpy(tgt_s).cuda(), v, k)
    for cam in cams:
        free.insert_rays(cam, torch.from_numpy(depth).cuda(), v, 1)
    src = torch.from_numpy(np.ascontiguousarray(src_m)).cuda()
    retain = torch.empty(src.shape[0], dtype=torch.uint8, device="cuda")
    b.gs_voxel_retain(occ, free, v, src, retain)
    torch.cuda.synchronize()
    assert int(occ.overflow.item()) == 0 and int(free.overflow.item()) == 0
    assert np.array_equal(occ.keys(), np.array(sorted(occ_o), np.uint64))
    assert np.array_equal(free.keys(), np.array(sorted(free_o), np.uint64))
    got = retain.cpu().numpy().astype(bool)
    assert np.array_equal(got, want) and 0 < want.sum() < len(want)
    # one-set variants (either table may be NULL)
    b.gs_voxel_retain(occ, None, v, src, retain)
    torch.cuda.synchronize()
    assert np.array_equal(retain.cpu().numpy().astype(bool), of.retain_mask(src_m, occ_o, set(), float(v)))
    # compaction keeps the original order: fused set = target + retained borrowed Gaussians
    b.gs_voxel_retain(occ, free, v, src, retain)
    out, index = b.gs_compact(retain, dict(means=src, quats=torch.from_numpy(np.ascontiguousarray(sc.quats[n:])).cuda()))
    torch.cuda.synchronize()
    assert np.array_equal(out["means"].cpu().numpy(), src_m[want]) and np.array_equal(out["quats"].cpu().numpy(), sc.quats[n:][want])
    idx = index.cpu().numpy().view(np.uint32)
    assert np.array_equal(idx[want], np.arange(want.sum(), dtype=np.uint32)) and (idx[~want] == 0xFFFFFFFF).all()


def _box_keys(of, means, scales, v, k):
    """Eq. 20 by its definition, vectorised: per Gaussian every voxel index between kappa(mu - k s) and kappa(mu + k s)."""
    out = []
    for m, s in zip(np.asarray(means, np.float64), np.asarray(scales, np.float64)):
        lo, hi = of.kappa(m - np.float64(k) * s, v), of.kappa(m + np.float64(k) * s, v)
        gx, gy, gz = np.meshgrid(*(np.arange(lo[a], hi[a] + 1) for a in range(3)), indexing="ij")
        out.append(of.pack_key(gx.ravel(), gy.ravel(), gz.ravel()))
    return np.unique(np.concatenate(out))


def test_large_boxes_are_inserted_completely():
    """Background-sized Gaussians (10^4..10^5 voxels per box: the warp-cooperative path of vox_boxes_kernel) mixed with
    ordinary ones: the set is the definition's, bit for bit."""
    import torch
    from oracle import fusion as of
    from paper_2605_10760_b200 import binding as b
    r = np.random.Generator(np.random.PCG64(66))
    N = 300
    means = _f32(r.uniform(-2, 2, (N, 3)))
    scales = _f32(np.exp(r.normal(-4.0, 0.5, (N, 3))))
    big = [3, 64, 65, 131, 299]            # two of them in one warp, one in the last (ragged) warp
    scales[big] = _f32([[0.3, 0.2, 0.1], [0.05, 0.4, 0.05], [0.2, 0.2, 0.2], [0.011, 0.013, 0.6], [0.25, 0.1, 0.3]])
    v, k = np.float32(0.02), np.float32(3.0)
    want = _box_keys(of, means, scales, float(v), float(k))
    assert np.array_equal(_box_keys(of, means[:40], scales[:40], float(v), float(k)),
                          np.array(sorted(of.occupied_set(means[:40], scales[:40], float(v), float(k))), np.uint64))
    vs = b.VoxelSet(1 << 21)
    vs.insert_boxes(torch.from_numpy(means).cuda(), torch.from_numpy(scales).cuda(), v, k)
    torch.cuda.synchronize()
    assert int(vs.overflow.item()) == 0
    got = vs.keys()
    assert len(want) > 400_000 and np.array_equal(got, want)


def test_full_table_and_runaway_scales_end_promptly_with_overflow():
    """An undersized table and Gaussians with metre-sized scales must end in an overflow report, not in a kernel that
    probes the whole table per key or walks 10^8 voxels in one thread."""
    import torch
    from paper_2605_10760_b200 import binding as b, scenes
    r = np.random.Generator(np.random.PCG64(67))
    v, k = np.float32(0.02), np.float32(3.0)
    N = 5_000
    means = _f32(r.uniform(-3, 3, (N, 3)))
    scales = _f32(np.exp(r.normal(-3.5, 0.4, (N, 3))))
    scales[::500] = 2.0                     # (2 * 3 * 2 m / 2 cm)^3 = 2e8 voxels each: beyond the per-box limit
    scales[7::500] = 0.5                    # 3.4e6 voxels each: warp path, abandoned once the overflow is known
    small = b.VoxelSet(1 << 12)
    dm, dsc = torch.from_numpy(means).cuda(), torch.from_numpy(scales).cuda()
    depth = torch.from_numpy(_f32(r.uniform(1.0, 5.0, (480, 640)))).cuda()
    cam = scenes.Camera(640, 480, 300.0, 300.0, 320.0, 240.0, scenes.look_at([0.0, 0.0, 0.0], [1.0, 0.2, 0.1]))
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0.record()
    small.insert_boxes(dm, dsc, v, k)
    small.insert_rays(cam, depth, v, 1)     # 307 200 rays of ~100 steps each into the full table
    t1.record()
    torch.cuda.synchronize()
    assert int(small.overflow.item()) >= 10 and len(small.keys()) == 1 << 12
    assert t0.elapsed_time(t1) < 2000.0, t0.elapsed_time(t1)
    # a roomy table still refuses the 2e8-voxel boxes (counted once each) and stores everything else
    roomy = b.VoxelSet(1 << 24)
    keep = np.ones(N, bool); keep[7::500] = False          # leave the 3.4e6-voxel boxes out of this part
    roomy.insert_boxes(torch.from_numpy(means[keep]).cuda(), torch.from_numpy(scales[keep]).cuda(), v, k)
    torch.cuda.synchronize()
    assert int(roomy.overflow.item()) == len(range(0, N, 500)) and 100_000 < len(roomy.keys()) < 1 << 23


def test_non_finite_gaussians_are_counted_and_never_retained():
    import torch
    from oracle import fusion as of
    from paper_2605_10760_b200 import binding as b
    r = np.random.Generator(np.random.PCG64(68))
    N = 1000
    means = _f32(r.uniform(-1, 1, (N, 3)))
    scales = _f32(np.exp(r.normal(-4.0, 0.3, (N, 3))))
    v, k = np.float32(0.05), np.float32(1.0)
    bad = np.zeros(N, bool); bad[[0, 17, 500, 999]] = True
    m2, s2 = means.copy(), scales.copy()
    m2[0, 1] = np.nan; m2[17, 0] = np.inf; s2[500, 2] = np.nan; m2[999] = -np.inf
    want = _box_keys(of, means[~bad], scales[~bad], float(v), float(k))
    vs = b.VoxelSet(1 << 16)
    vs.insert_boxes(torch.from_numpy(m2).cuda(), torch.from_numpy(s2).cuda(), v, k)
    torch.cuda.synchronize()
    assert int(vs.overflow.item()) == 4 and np.array_equal(vs.keys(), want)     # voxel 0 was not invented for the NaNs
    # retain against an EMPTY pair of sets: everything finite is retained, nothing non-finite is
    retain = torch.empty(N, dtype=torch.uint8, device="cuda")
    b.gs_voxel_retain(b.VoxelSet(1 << 4), None, v, torch.from_numpy(m2).cuda(), retain)
    torch.cuda.synchronize()
    finite = np.isfinite(m2).all(1)
    assert np.array_equal(retain.cpu().numpy().astype(bool), finite) and (~finite).sum() == 3


def test_free_set_of_a_full_size_depth_map():
    """Eq. 21 at the paper's keyframe size: every pixel of a 1200 x 680 depth map casts a ray (stride 1)."""
    import torch
    from oracle import fusion as of
    from paper_2605_10760_b200 import binding as b, scenes
    r = np.random.Generator(np.random.PCG64(71))
    W, H = 1200, 680
    cam = scenes.Camera(W, H, 600.0, 600.0, 599.5, 339.5,
                        scenes.perturb_pose(scenes.look_at([0.3, -0.2, 1.4], [4.0, 1.0, 1.1]), r.normal(0, 0.05, 6)))
    # a room-like depth: smooth walls 2..6 m away, objects in front of them, pixel noise, 5 % invalid pixels
    yy, xx = np.meshgrid(np.linspace(-1, 1, H), np.linspace(-1, 1, W), indexing="ij")
    depth = 4.0 + 1.5 * np.sin(2.1 * xx + 0.3) * np.cos(1.3 * yy) + 0.4 * xx * yy
    depth[(np.abs(xx - 0.2) < 0.25) & (np.abs(yy + 0.1) < 0.4)] = 1.3
    depth = _f32(depth + r.normal(0, 0.01, depth.shape))
    depth[r.uniform(size=depth.shape) < 0.05] = 0.0
    v = np.float32(0.08)
    c, pts = of.backproject(depth, np.float32(cam.fx), np.float32(cam.fy), np.float32(cam.cx), np.float32(cam.cy), _f32(cam.T_cw), 1)
    keys, amb = of.free_keys(c, pts, float(v))
    assert len(pts) > 0.9 * W * H and len(keys) > 50_000
    vs = b.VoxelSet(1 << 21)
    vs.insert_rays(cam, torch.from_numpy(depth).cuda(), v, 1)
    torch.cuda.synchronize()
    assert int(vs.overflow.item()) == 0
    _assert_equal_up_to_ties(vs.keys(), keys, amb, len(pts))


def test_occupied_set_of_half_a_million_gaussians_and_a_nearly_full_table():
    """Eq. 20 for a config-4-sized map (500 k Gaussians, Replica-shaped scales), bit-exact; then the same keys into a table
    only ~1.2 x their number: either everything fits within the probe window (exact set, no overflow) or the overflow is
    reported and nothing foreign was stored."""
    import torch
    from oracle import fusion as of
    from paper_2605_10760_b200 import binding as b, scenes
    sc = scenes.replica_scene(seed=69, N=500_000)
    v, k = np.float32(0.04), np.float32(2.0)
    want = of.occupied_keys(sc.means, sc.scales, float(v), float(k))
    dm, dsc = torch.from_numpy(sc.means).cuda(), torch.from_numpy(sc.scales).cuda()
    vs = b.VoxelSet(1 << 20)                         # load factor ~0.4
    vs.insert_boxes(dm, dsc, v, k)
    torch.cuda.synchronize()
    assert 300_000 < len(want) < 500_000
    assert int(vs.overflow.item()) == 0 and np.array_equal(vs.keys(), want)
    tight = b.VoxelSet(1 << 19)                      # load factor ~0.8: probe windows of 128 slots start to fill up
    tight.insert_boxes(dm, dsc, v, k)
    torch.cuda.synchronize()
    got, ov = tight.keys(), int(tight.overflow.item())
    print(f"nearly full table: {len(got)} of {len(want)} keys stored, overflow {ov}")
    assert np.isin(got, want).all()
    assert (ov == 0 and np.array_equal(got, want)) or (ov > 0 and len(got) < len(want))
    # the retain test against the roomy set: bit-exact for 500 k borrowed Gaussians (vectorised form of Eq. 22)
    src = _f32(sc.means + np.random.Generator(np.random.PCG64(70)).normal(0, 0.05, sc.means.shape))
    idx = of.kappa(src, float(v))
    want_retain = ~np.isin(of.pack_key(idx[:, 0], idx[:, 1], idx[:, 2]), want)
    retain = torch.empty(src.shape[0], dtype=torch.uint8, device="cuda")
    b.gs_voxel_retain(vs, None, v, torch.from_numpy(src).cuda(), retain)
    torch.cuda.synchronize()
    assert np.array_equal(retain.cpu().numpy().astype(bool), want_retain) and 0.05 < want_retain.mean() < 0.95
