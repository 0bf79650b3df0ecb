"""Pins of oracle/loss.py (Eq. 4 terms) against what the mathematics fixes: closed forms on constant
images, central finite differences away from the kinks, exact zeros of the isotropy term, its invariances, and the
paper's weights.  CPU only."""
import numpy as np

from oracle import loss as ol


def _images(seed, H=7, W=9):
    r = np.random.default_rng(seed)
    rgb = r.uniform(0, 1, (3, H, W)); trgb = r.uniform(0, 1, (3, H, W))
    d = r.uniform(0.5, 6, (H, W)); td = r.uniform(0.5, 6, (H, W))
    return rgb, d, trgb, td


def test_l1_closed_form_on_constant_images():
    H, W = 4, 6
    rgb = np.full((3, H, W), 0.75); trgb = np.full((3, H, W), 0.25)
    d = np.full((H, W), 2.0); td = np.full((H, W), 3.5)
    lr, ld, gr, gd = ol.l1_terms(rgb, d, trgb, td)
    assert abs(lr - 0.5) < 1e-15 and abs(ld - 1.5) < 1e-15          # means of constant absolute differences
    assert np.allclose(gr, 1.0 / (3 * H * W)) and np.allclose(gd, -1.0 / (H * W))
    total, g_rgb, g_d = ol.map_loss(rgb, d, trgb, td)                # Eq. 4 weights alpha = 0.95, beta = 0.25
    assert abs(total - (0.95 * 0.5 + 0.25 * 1.5)) < 1e-15
    assert np.allclose(g_rgb, 0.95 / (3 * H * W)) and np.allclose(g_d, -0.25 / (H * W))


def test_l1_gradient_by_finite_differences():
    rgb, d, trgb, td = _images(3)
    _, g_rgb, g_d = ol.map_loss(rgb, d, trgb, td)
    h = 1e-6
    r = np.random.default_rng(4)
    for _ in range(20):
        c, y, x = r.integers(3), r.integers(rgb.shape[1]), r.integers(rgb.shape[2])
        p, m = rgb.copy(), rgb.copy(); p[c, y, x] += h; m[c, y, x] -= h
        fd = (ol.map_loss(p, d, trgb, td)[0] - ol.map_loss(m, d, trgb, td)[0]) / (2 * h)
        assert abs(fd - g_rgb[c, y, x]) < 1e-9
        p, m = d.copy(), d.copy(); p[y, x] += h; m[y, x] -= h
        fd = (ol.map_loss(rgb, p, trgb, td)[0] - ol.map_loss(rgb, m, trgb, td)[0]) / (2 * h)
        assert abs(fd - g_d[y, x]) < 1e-9


def test_invalid_depth_pixels_and_exact_matches_contribute_nothing():
    rgb, d, trgb, td = _images(5)
    td[2, 3] = 0.0; td[0, 0] = -1.0          # no target depth there (reading Q18)
    d[4, 4] = td[4, 4]; rgb[1, 1, 1] = trgb[1, 1, 1]   # exact matches: sign(0) = 0
    lr, ld, gr, gd = ol.l1_terms(rgb, d, trgb, td)
    assert gd[2, 3] == 0.0 and gd[0, 0] == 0.0 and gd[4, 4] == 0.0 and gr[1, 1, 1] == 0.0
    d2 = d.copy(); d2[2, 3] += 100.0
    assert ol.l1_terms(rgb, d2, trgb, td)[1] == ld
    H, W = d.shape
    valid = td > 0
    assert abs(ld - np.abs(d - td)[valid].sum() / (H * W)) < 1e-15


def test_iso_zero_for_isotropic_and_hand_values():
    s = np.array([[0.3, 0.3, 0.3], [1.0, 2.0, 3.0]])
    loss, g = ol.iso_loss(s, lambda_s=10.0)
    # second Gaussian: mean 2 -> |1-2| + 0 + |3-2| = 2; lambda_s = 10
    assert abs(loss - 20.0) < 1e-14
    assert np.all(g[0] == 0.0)
    # signs (-1, 0, +1), their mean 0 -> gradient 10 * (-1, 0, 1)
    assert np.allclose(g[1], [-10.0, 0.0, 10.0])


def test_iso_gradient_by_finite_differences_and_invariances():
    r = np.random.default_rng(6)
    s = np.exp(r.normal(-4.5, 0.5, (40, 3)))
    loss, g = ol.iso_loss(s)
    h = 1e-9
    for _ in range(30):
        i, j = r.integers(40), r.integers(3)
        p, m = s.copy(), s.copy(); p[i, j] += h; m[i, j] -= h
        fd = (ol.iso_loss(p)[0] - ol.iso_loss(m)[0]) / (2 * h)
        assert abs(fd - g[i, j]) < 1e-5 * max(1.0, abs(g[i, j]))
    # the gradient of every Gaussian sums to zero (the loss is invariant to a common shift of its three scales) ...
    assert np.abs(g.sum(axis=1)).max() < 1e-12
    assert abs(ol.iso_loss(s + 0.01)[0] - loss) < 1e-10
    # ... the loss is 1-homogeneous in the scales and invariant to a permutation of the axes
    assert abs(ol.iso_loss(3.0 * s)[0] - 3.0 * loss) < 1e-9
    assert abs(ol.iso_loss(s[:, [2, 0, 1]])[0] - loss) < 1e-12
