"""Oracle of the mapping-loss terms of Eq. 4 that need no dataset: the photometric and depth L1 terms and the isotropy
regulariser.  TEST INFRASTRUCTURE (plain numpy, fp64): only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline
leg may import this module; it shares no code with paper_2605_10760_b200/csrc.

Paper (Eq. 4):
    L_map = alpha L1(I^, I) + beta L1(D^, D) + lambda_n L_normal + lambda_s L_iso,
    alpha = 0.95, beta = 0.25, lambda_s = 10,  L_iso = sum_i |s_i - mean(s_i)|.
"The photometric and depth terms reduce to per-keyframe L1 errors" -- the reduction is not stated.  Reading Q18
(DESIGN.md): mean over pixels (and channels) of |I^ - I|; mean over ALL pixels of |D^ - D| restricted to pixels with a
valid target depth D > 0 (invalid pixels contribute 0 to the sum and to the gradient); |.| of a 3-vector in L_iso is the
1-norm over the three scale components; sign(0) = 0 in every sub-gradient.  L_normal needs the normal prior: out of scope.
"""
from __future__ import annotations

import numpy as np


def l1_terms(rgb, depth, target_rgb, target_depth):
    """Returns (L1 rgb, L1 depth, dL1rgb/drgb [3,H,W], dL1depth/ddepth [H,W]), unweighted (fp64)."""
    rgb = np.asarray(rgb, np.float64); depth = np.asarray(depth, np.float64)
    trgb = np.asarray(target_rgb, np.float64); td = np.asarray(target_depth, np.float64)
    C, H, W = rgb.shape
    assert C == 3 and depth.shape == (H, W) and trgb.shape == rgb.shape and td.shape == depth.shape
    loss_rgb = 0.0
    g_rgb = np.zeros_like(rgb)
    for c in range(3):                      # sum over channels and pixels, then the mean
        d = rgb[c] - trgb[c]
        loss_rgb += np.abs(d).sum()
        g_rgb[c] = np.sign(d)
    loss_rgb /= 3.0 * H * W
    g_rgb /= 3.0 * H * W
    valid = td > 0.0
    dd = np.where(valid, depth - td, 0.0)
    loss_d = np.abs(dd).sum() / (H * W)
    g_d = np.sign(dd) / (H * W)
    return loss_rgb, loss_d, g_rgb, g_d


def map_loss(rgb, depth, target_rgb, target_depth, alpha=0.95, beta=0.25):
    """alpha L1(I^, I) + beta L1(D^, D) of Eq. 4 and its gradients w.r.t. the rendered images."""
    lr, ld, gr, gd = l1_terms(rgb, depth, target_rgb, target_depth)
    return alpha * lr + beta * ld, alpha * gr, beta * gd


def iso_loss(scales, lambda_s=10.0):
    """lambda_s sum_i |s_i - mean(s_i)|_1 and its gradient w.r.t. the (activated) scales [N,3] (fp64)."""
    s = np.asarray(scales, np.float64)
    loss = 0.0
    g = np.zeros_like(s)
    for i in range(s.shape[0]):             # Gaussian by Gaussian, as the sum is written
        sbar = (s[i, 0] + s[i, 1] + s[i, 2]) / 3.0
        sg = np.sign(s[i] - sbar)
        loss += np.abs(s[i] - sbar).sum()
        g[i] = sg - sg.sum() / 3.0            # d/ds_ij sum_k |s_ik - sbar| with dsbar/ds_ij = 1/3
    return lambda_s * loss, lambda_s * g


# ----------------------------------------------------------------------------------------------------------------------
# Eq. 23: the refinement loss of the fused map on the exposure-compensated render
#     I~(u) = e^{a_k} I^(u) + b_k,     L_rf = alpha' L1(I~, I) + lambda (1 - SSIM(I~, I)) + beta L1(D^, D-)  [+ lambda'_n L_normal]
# with alpha' = (1 - lambda) + alpha = 1.75, lambda = 0.2 (lambda_n is garbled there -- reading Q16 -- and the
# normal term is oracle/normals.py).  The paper does not define SSIM beyond its name.  Reading Q19: the
# standard structural similarity index with an 11 x 11 Gaussian window of sigma 1.5 (normalised to sum 1), constants
# C1 = 0.01^2, C2 = 0.03^2 (dynamic range 1), windowed moments by correlation with ZERO padding outside the image
# (window always 11 x 11, so border pixels see zeros), computed per colour channel; SSIM(I~, I) = mean of the SSIM map
# over all pixels and channels.
# ----------------------------------------------------------------------------------------------------------------------
SSIM_C1, SSIM_C2 = 0.01 ** 2, 0.03 ** 2


def ssim_window(size=11, sigma=1.5):
    g = np.exp(-((np.arange(size) - size // 2) ** 2) / (2.0 * sigma * sigma))
    g /= g.sum()
    return np.outer(g, g)


def _win(img, w):
    from scipy.signal import correlate2d
    return correlate2d(img, w, mode="same", boundary="fill", fillvalue=0.0)


def ssim_terms(x, y):
    """SSIM map of one channel pair [H,W] and the partial derivatives of the map w.r.t. the windowed moments of x:
    returns (s, ds/dm1, ds/de11, ds/de12) with m1 = W*x, e11 = W*x^2, e12 = W*(x y)."""
    w = ssim_window()
    m1, m2 = _win(x, w), _win(y, w)
    e11, e22, e12 = _win(x * x, w), _win(y * y, w), _win(x * y, w)
    n1, n2 = 2 * m1 * m2 + SSIM_C1, 2 * (e12 - m1 * m2) + SSIM_C2
    d1, d2 = m1 * m1 + m2 * m2 + SSIM_C1, (e11 - m1 * m1) + (e22 - m2 * m2) + SSIM_C2
    s = n1 * n2 / (d1 * d2)
    ds_dm1 = (2 * m2 * n2 - 2 * m2 * n1) / (d1 * d2) - s * (2 * m1 / d1 - 2 * m1 / d2)
    ds_de11 = -s / d2
    ds_de12 = 2 * n1 / (d1 * d2)
    return s, ds_dm1, ds_de11, ds_de12


def ssim_mean(x, y):
    """Mean SSIM over pixels and channels of [3,H,W] images, and its gradient w.r.t. x (plain chain rule: every moment is
    a correlation with the symmetric window, whose adjoint under zero padding is the same correlation)."""
    x = np.asarray(x, np.float64); y = np.asarray(y, np.float64)
    C, H, W = x.shape
    w = ssim_window()
    total, g = 0.0, np.zeros_like(x)
    for c in range(C):
        s, a, b11, b12 = ssim_terms(x[c], y[c])
        total += s.sum()
        g[c] = _win(a, w) + 2.0 * x[c] * _win(b11, w) + y[c] * _win(b12, w)
    n = C * H * W
    return total / n, g / n


def refine_loss(rgb, depth, target_rgb, target_depth, a, b, alpha_p=1.75, lam=0.2, beta=0.25):
    """Eq. 23 without the normal term.  Returns a dict: the terms, the total, dL/dI^ [3,H,W], dL/dD^ [H,W], dL/da, dL/db."""
    rgb = np.asarray(rgb, np.float64)
    ea = float(np.exp(a))
    it = ea * rgb + float(b)                                   # I~ = e^a I^ + b
    l1, ld, g1, gd = l1_terms(it, depth, target_rgb, target_depth)
    sm, gs = ssim_mean(it, np.asarray(target_rgb, np.float64))
    g_it = alpha_p * g1 - lam * gs                             # dL / dI~
    total = alpha_p * l1 + lam * (1.0 - sm) + beta * ld
    return dict(l1_rgb=l1, ssim=sm, l1_depth=ld, total=total, d_rgb=ea * g_it, d_depth=beta * gd,
                g_a=float((g_it * ea * rgb).sum()), g_b=float(g_it.sum()))
