"""Pins of the occupancy-aware fusion oracle (oracle/fusion.py, Eqs. 20-22): hand-built voxel scenes,
box-count closed form, a ray through known voxels, the DDA against the plain definition of Eq. 21, key packing."""
import numpy as np

from oracle import fusion as of


def test_key_packing_is_injective_and_ordered_fields():
    assert int(of.pack_key(0, 0, 0)) == (1 << 20) | (1 << 41) | (1 << 62)
    a = of.pack_key(np.array([-3, 5]), np.array([7, -1]), np.array([0, 2]))
    for key, (x, y, z) in zip(a, [(-3, 7, 0), (5, -1, 2)]):
        k = int(key)
        assert (k & 0x1FFFFF) - (1 << 20) == x and ((k >> 21) & 0x1FFFFF) - (1 << 20) == y and (k >> 42) - (1 << 20) == z
    r = np.random.Generator(np.random.PCG64(1))
    idx = r.integers(-1000, 1000, (5000, 3))
    keys = of.pack_key(idx[:, 0], idx[:, 1], idx[:, 2])
    assert len(set(map(int, keys))) == len({tuple(i) for i in idx})


def test_kappa_is_floor_division_with_negative_coordinates():
    assert np.array_equal(of.kappa([[0.0, -0.0, 0.019], [-0.001, 0.02, -0.02]], 0.02), [[0, 0, 0], [-1, 1, -1]])


def test_box_voxel_count_closed_form():
    # one Gaussian: the box [mu - k s, mu + k s] meets prod_a (floor((mu_a + k s_a)/v) - floor((mu_a - k s_a)/v) + 1) voxels
    mu, s, v, k = np.array([[0.013, -0.204, 1.0]]), np.array([[0.03, 0.011, 0.05]]), 0.02, 1.5
    want = 1
    for a in range(3):
        want *= int(np.floor((mu[0, a] + k * s[0, a]) / v) - np.floor((mu[0, a] - k * s[0, a]) / v)) + 1
    occ = of.occupied_set(mu, s, v, k)
    # by hand: x in [-0.032, 0.058] -> voxels -2..2 (5); y in [-0.2205, -0.1875] -> -12..-10 (3); z in [0.925, 1.075] -> 46..53 (8)
    assert len(occ) == want == 5 * 3 * 8
    # a point-like Gaussian occupies exactly its own voxel; two Gaussians in the same voxel give one key
    occ = of.occupied_set(np.array([[0.05, 0.05, 0.05], [0.051, 0.049, 0.0501]]), np.full((2, 3), 1e-6), 0.02, 1.0)
    assert occ == {int(of.pack_key(2, 2, 2))}


def test_ray_through_known_voxels():
    v = 1.0
    # along +x from the centre of voxel (0,0,0) to the centre of voxel (3,0,0): voxels 0..3 (the end voxel is entered at t<1)
    assert of.ray_voxels([0.5, 0.5, 0.5], [3.5, 0.5, 0.5], v) == [(0, 0, 0), (1, 0, 0), (2, 0, 0), (3, 0, 0)]
    # ending exactly ON the boundary x = 3: t in [0,1) never reaches voxel 3
    assert of.ray_voxels([0.5, 0.5, 0.5], [3.0, 0.5, 0.5], v) == [(0, 0, 0), (1, 0, 0), (2, 0, 0)]
    # negative direction and a diagonal in the xy plane that crosses x first, then y
    assert of.ray_voxels([0.5, 0.5, 0.5], [-1.5, 0.5, 0.5], v) == [(0, 0, 0), (-1, 0, 0), (-2, 0, 0)]
    assert of.ray_voxels([0.9, 0.5, 0.5], [1.5, 1.4, 0.5], v) == [(0, 0, 0), (1, 0, 0), (1, 1, 0)]
    # zero-length ray: only the camera's own voxel
    assert of.ray_voxels([0.2, 0.2, 0.2], [0.2, 0.2, 0.2], v) == [(0, 0, 0)]


def test_dda_equals_the_plain_definition_on_random_rays():
    r = np.random.Generator(np.random.PCG64(2))
    for trial in range(300):
        v = float(r.uniform(0.02, 0.3))
        c = r.uniform(-2, 2, 3); p = c + r.normal(0, 1.5, 3)
        if trial % 7 == 0:
            p[int(r.integers(3))] = c[int(r.integers(3))]   # axis-parallel components
        got = of.ray_voxels(c, p, v)
        assert len(got) == len(set(got))                       # the DDA never revisits a voxel
        assert set(got) == of.ray_voxels_by_definition(c, p, v)
        for a, b in zip(got[:-1], got[1:]):                     # consecutive voxels are face neighbours
            assert sum(abs(x - y) for x, y in zip(a, b)) == 1


def test_free_set_and_retain_on_a_hand_built_scene():
    # a 2x1 depth map looking down +z from the origin with f = 1: pixel (0,0) -> ray to (0,0,2.5), pixel (1,0) invalid
    depth = np.array([[2.5, 0.0]])
    T = np.array([[1, 0, 0, 0], [0, 1, 0, 0], [0, 0, 1, 0]], float)
    free = of.free_set(depth, 1.0, 1.0, 0.0, 0.0, T, 1.0)
    assert free == {int(of.pack_key(0, 0, z)) for z in (0, 1, 2)}
    # camera moved to world (10, 0, 0) (t = -R c): the same ray, shifted
    T2 = T.copy(); T2[0, 3] = -10.0
    free2 = of.free_set(depth, 1.0, 1.0, 0.0, 0.0, T2, 1.0)
    assert free2 == {int(of.pack_key(10, 0, z)) for z in (0, 1, 2)}
    occ = of.occupied_set(np.array([[5.5, 0.5, 0.5]]), np.array([[0.1, 0.1, 0.1]]), 1.0, 1.0)
    means = np.array([[0.5, 0.5, 1.5],     # inside the carved free space -> dropped
                      [5.2, 0.9, 0.1],     # in the occupied voxel       -> dropped
                      [0.5, 0.5, 3.5],     # behind the observed surface -> kept
                      [-0.5, 0.5, 1.5]])   # beside the ray              -> kept
    assert np.array_equal(of.retain_mask(means, occ, free, 1.0), [False, False, True, True])


def test_backprojection_inverts_the_pinhole_model():
    r = np.random.Generator(np.random.PCG64(3))
    from scipy.spatial.transform import Rotation
    R = Rotation.random(random_state=4).as_matrix(); t = r.normal(size=3)
    T = np.concatenate([R, t[:, None]], 1)
    depth = r.uniform(0.5, 3, (4, 5))
    c, pts = of.backproject(depth, 7.0, 8.0, 2.0, 1.5, T)
    assert np.allclose(R @ c + t, 0, atol=1e-12)
    pc = (R @ pts.T).T + t
    uu = 7.0 * pc[:, 0] / pc[:, 2] + 2.0; vv = 8.0 * pc[:, 1] / pc[:, 2] + 1.5
    assert np.allclose(uu.reshape(4, 5), np.arange(5)[None, :], atol=1e-10) and np.allclose(vv.reshape(4, 5), np.arange(4)[:, None], atol=1e-10)
    assert np.allclose(pc[:, 2].reshape(4, 5), depth)


# ----------------------------------------------------------------------------------------------------------------------
# The array forms used at the paper's sizes (occupied_keys, free_keys) against the per-item definitions, and the tie
# analysis of free_keys on rays built to be degenerate.
# ----------------------------------------------------------------------------------------------------------------------
def test_occupied_keys_equals_the_per_gaussian_definition():
    r = np.random.Generator(np.random.PCG64(11))
    m = r.uniform(-1, 1, (400, 3)); s = np.exp(r.normal(-4, 0.6, (400, 3)))
    s[3] = [0.3, 0.2, 0.1]; s[77] = [0.001, 0.5, 0.001]                    # large boxes take the one-by-one branch
    for v, k in ((0.02, 1.5), (0.05, 3.0), (1.0, 0.0)):
        want = np.array(sorted(of.occupied_set(m, s, v, k)), np.uint64)
        assert np.array_equal(of.occupied_keys(m, s, v, k), want)
    assert of.occupied_keys(np.zeros((0, 3)), np.zeros((0, 3)), 0.02, 1.0).size == 0


def test_free_keys_equals_the_per_ray_dda_and_the_plain_definition():
    from scipy.spatial.transform import Rotation
    r = np.random.Generator(np.random.PCG64(12))
    R = Rotation.random(random_state=13).as_matrix(); t = r.normal(size=3)
    depth = r.uniform(0.4, 3.0, (19, 31)); depth[r.uniform(size=depth.shape) < 0.2] = 0.0
    for stride, v in ((1, 0.05), (3, 0.11)):
        c, pts = of.backproject(depth, 30.0, 31.0, 15.25, 9.0, np.concatenate([R, t[:, None]], 1), stride)
        keys, amb = of.free_keys(c, pts, v)
        per_ray, by_def = set(), set()
        for p in pts:
            per_ray |= {int(of.pack_key(*q)) for q in of.ray_voxels(c, p, v)}
            by_def |= {int(of.pack_key(*q)) for q in of.ray_voxels_by_definition(c, p, v)}
        assert set(map(int, keys)) == per_ray == by_def and amb.size == 0      # generic rays: nothing hinges on rounding
    k0, a0 = of.free_keys(np.zeros(3), np.zeros((0, 3)), 0.1)
    assert k0.size == 0 and a0.size == 0


def test_free_keys_reports_the_voxels_that_hinge_on_a_tie():
    key = lambda *q: int(of.pack_key(*q))
    # through the voxel edge x = 1, y = 1 (both crossings at t = 0.25): the walk goes (0,0,0) -> (1,0,0) -> (1,1,0) -> ...
    # but (0,1,0) instead of (1,0,0) is as valid; both are reported, the unambiguous voxels are not
    keys, amb = of.free_keys([0.5, 0.5, 0.5], [[2.5, 2.5, 0.5]], 1.0)
    assert {key(0, 0, 0), key(1, 1, 0), key(2, 2, 0)} <= set(map(int, keys))
    assert {key(1, 0, 0), key(0, 1, 0)} <= set(map(int, amb)) and key(0, 0, 0) not in set(map(int, amb))
    # surface point exactly on the face x = 3 (t = 1 there): the end voxel (3,0,0) is not entered, and is reported
    keys, amb = of.free_keys([0.5, 0.5, 0.5], [[3.0, 0.5, 0.5]], 1.0)
    assert set(map(int, keys)) == {key(0, 0, 0), key(1, 0, 0), key(2, 0, 0)} and set(map(int, amb)) == {key(3, 0, 0)}
    # the same two rays moved off the degenerate position by 1e-6: nothing is reported
    keys, amb = of.free_keys([0.5, 0.5, 0.5], [[2.5, 2.5 + 1e-6, 0.5], [3.0 - 1e-6, 0.5, 0.5]], 1.0)
    assert amb.size == 0
    # a camera centre on a voxel face makes every first voxel undetermined
    keys, amb = of.free_keys([1.0, 0.5, 0.5], [[2.5, 0.7, 0.5]], 1.0)
    assert np.array_equal(keys, amb)


def test_backprojection_is_the_matrix_form():
    """c = -R^T t and r = R^T (p_c - t) written with matrix products equal the component sums (to rounding)."""
    from scipy.spatial.transform import Rotation
    r = np.random.Generator(np.random.PCG64(14))
    R = Rotation.random(random_state=15).as_matrix(); t = r.normal(size=3)
    depth = r.uniform(0.5, 3, (6, 7)); depth[2, 3] = 0.0; depth[5, 6] = -1.0
    c, pts = of.backproject(depth, 7.0, 8.0, 2.0, 1.5, np.concatenate([R, t[:, None]], 1), 2)
    want = []
    for y in range(0, 6, 2):
        for x in range(0, 7, 2):
            z = depth[y, x]
            if z > 0:
                pc = np.array([(x - 2.0) * z / 7.0, (y - 1.5) * z / 8.0, z])
                want.append([sum(R[b, a] * (pc[b] - t[b]) for b in range(3)) for a in range(3)])
    assert pts.shape == (len(want), 3) and np.allclose(pts, want, rtol=0, atol=1e-14)
    assert np.allclose(c, [-sum(R[b, a] * t[b] for b in range(3)) for a in range(3)], rtol=0, atol=1e-15)
