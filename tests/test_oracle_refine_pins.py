"""Pins of the Eq. 23 refinement-loss oracle (oracle/loss.py: exposure compensation + SSIM): closed
forms, brute force on a tiny image, symmetry / invariance identities, central finite differences."""
import numpy as np

from oracle import loss as ol


def _imgs(seed, H, W):
    r = np.random.Generator(np.random.PCG64(seed))
    return r.uniform(0, 1, (3, H, W)), r.uniform(0, 1, (3, H, W)), r.uniform(0.5, 6, (H, W)), r.uniform(0.5, 6, (H, W))


def test_window_is_the_normalised_gaussian():
    w = ol.ssim_window()
    assert w.shape == (11, 11) and abs(w.sum() - 1) < 1e-15 and np.allclose(w, w.T) and np.allclose(w, w[::-1, ::-1])
    assert np.isclose(w[5, 6] / w[5, 5], np.exp(-1 / (2 * 1.5 ** 2)))


def test_ssim_of_an_image_with_itself_is_one_and_is_symmetric():
    x, y, _, _ = _imgs(1, 20, 23)
    s, _ = ol.ssim_mean(x, x)
    assert abs(s - 1.0) < 1e-12
    sxy, _ = ol.ssim_mean(x, y)
    syx, _ = ol.ssim_mean(y, x)
    assert abs(sxy - syx) < 1e-14 and sxy < 0.5     # unrelated noise images are dissimilar


def test_constant_images_closed_form_in_the_interior():
    # interior pixels (window inside the image): mu = c, sigma = 0  =>  s = (2 c1 c2 + C1) / (c1^2 + c2^2 + C1)
    c1, c2 = 0.3, 0.7
    s, _, _, _ = ol.ssim_terms(np.full((25, 25), c1), np.full((25, 25), c2))
    want = (2 * c1 * c2 + ol.SSIM_C1) / (c1 * c1 + c2 * c2 + ol.SSIM_C1)
    assert np.allclose(s[5:-5, 5:-5], want, atol=1e-14)
    # at the corner pixel the window sees zeros: mu = c * m with m = (sum of the 6x6 quadrant weights)
    w = ol.ssim_window(); m = w[5:, 5:].sum()
    m1, m2 = c1 * m, c2 * m
    v1, v2, v12 = c1 * c1 * m - m1 * m1, c2 * c2 * m - m2 * m2, c1 * c2 * m - m1 * m2
    corner = (2 * m1 * m2 + ol.SSIM_C1) * (2 * v12 + ol.SSIM_C2) / ((m1 * m1 + m2 * m2 + ol.SSIM_C1) * (v1 + v2 + ol.SSIM_C2))
    assert abs(s[0, 0] - corner) < 1e-14


def test_ssim_map_against_brute_force_loops():
    r = np.random.Generator(np.random.PCG64(3))
    x, y = r.uniform(0, 1, (13, 14)), r.uniform(0, 1, (13, 14))
    s, _, _, _ = ol.ssim_terms(x, y)
    g = np.exp(-((np.arange(11) - 5) ** 2) / 4.5); g /= g.sum()
    for (py, px) in ((0, 0), (6, 7), (12, 13), (3, 11)):
        acc = np.zeros(5)
        for dy in range(-5, 6):
            for dx in range(-5, 6):
                yy, xx = py + dy, px + dx
                if 0 <= yy < 13 and 0 <= xx < 14:
                    wgt = g[dy + 5] * g[dx + 5]
                    acc += wgt * np.array([x[yy, xx], y[yy, xx], x[yy, xx] ** 2, y[yy, xx] ** 2, x[yy, xx] * y[yy, xx]])
        m1, m2, e11, e22, e12 = acc
        want = (2 * m1 * m2 + 1e-4) * (2 * (e12 - m1 * m2) + 9e-4) / ((m1 * m1 + m2 * m2 + 1e-4) * (e11 - m1 * m1 + e22 - m2 * m2 + 9e-4))
        assert abs(s[py, px] - want) < 1e-13


def test_ssim_gradient_by_central_finite_differences():
    x, y, _, _ = _imgs(5, 14, 17)
    _, g = ol.ssim_mean(x, y)
    r = np.random.Generator(np.random.PCG64(6))
    for trial in range(6):
        u = r.normal(size=x.shape) if trial < 3 else np.zeros(x.shape)
        if trial >= 3:
            u.flat[r.integers(u.size)] = 1.0
        h = 1e-6
        fd = (ol.ssim_mean(x + h * u, y)[0] - ol.ssim_mean(x - h * u, y)[0]) / (2 * h)
        an = float((g * u).sum())
        assert abs(fd - an) <= 1e-7 * max(1.0, abs(an) * 1e3) and abs(fd - an) <= 2e-6 * max(abs(an), 1e-6)


def test_refine_loss_terms_weights_and_exposure_gradients():
    rgb, tgt, d, td = _imgs(7, 12, 15)
    a, b = 0.13, -0.04
    out = ol.refine_loss(rgb, d, tgt, td, a, b)
    it = np.exp(a) * rgb + b
    # the terms are the plain definitions on the exposure-compensated image, with the paper's weights
    assert np.isclose(out["l1_rgb"], np.abs(it - tgt).mean()) and np.isclose(out["l1_depth"], np.abs(d - td).mean())
    assert np.isclose(out["total"], 1.75 * out["l1_rgb"] + 0.2 * (1 - out["ssim"]) + 0.25 * out["l1_depth"])
    assert np.isclose(1.75, (1 - 0.2) + 0.95)                 # alpha' = (1 - lambda) + alpha
    # identity exposure reduces to the unexposed loss; target equal to the exposed render gives zero photometric loss
    o0 = ol.refine_loss(rgb, d, tgt, td, 0.0, 0.0)
    assert np.isclose(o0["l1_rgb"], np.abs(rgb - tgt).mean())
    oz = ol.refine_loss(rgb, d, it, d, a, b)
    assert abs(oz["l1_rgb"]) < 1e-15 and abs(oz["ssim"] - 1) < 1e-12 and abs(oz["total"]) < 1e-12
    # finite differences in a, b and in the rendered image / depth
    f = lambda aa, bb, im=rgb, dd=d: ol.refine_loss(im, dd, tgt, td, aa, bb)["total"]
    h = 1e-6
    assert abs((f(a + h, b) - f(a - h, b)) / (2 * h) - out["g_a"]) < 1e-6 * max(1, abs(out["g_a"]))
    assert abs((f(a, b + h) - f(a, b - h)) / (2 * h) - out["g_b"]) < 1e-6 * max(1, abs(out["g_b"]))
    r = np.random.Generator(np.random.PCG64(8))
    u = r.normal(size=rgb.shape)
    fd = (f(a, b, rgb + h * u) - f(a, b, rgb - h * u)) / (2 * h)
    assert abs(fd - (out["d_rgb"] * u).sum()) < 1e-6 * max(1, abs(fd))
    ud = r.normal(size=d.shape)
    fd = (f(a, b, rgb, d + h * ud) - f(a, b, rgb, d - h * ud)) / (2 * h)
    assert abs(fd - (out["d_depth"] * ud).sum()) < 1e-6 * max(1, abs(fd))
    # dL/da = sum dL/dI~ e^a I^ and dL/db = sum dL/dI~  (chain rule through I~ = e^a I^ + b)
    g_it = out["d_rgb"] / np.exp(a)
    assert np.isclose(out["g_b"], g_it.sum()) and np.isclose(out["g_a"], (g_it * np.exp(a) * rgb).sum())
