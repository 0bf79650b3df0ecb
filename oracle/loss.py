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
