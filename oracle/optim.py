"""Oracle of the optimiser step and pruning of the map refinement ("optimized ... by gradient descent", PAPER.md:322
"2,000 iterations at half the per-agent learning rate and prunes Gaussians with opacity below 0.005").  TEST
INFRASTRUCTURE (plain numpy, fp64): only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this
module; it shares no code with paper_2605_10760_b200/csrc.

The paper names neither the optimiser nor the parametrisation.  Reading Q20: Adam (Kingma & Ba, Algorithm 1, with
bias correction), one learning rate per parameter group, on the parametrisation of the 3DGS lineage: centres, raw quaternions
and SH coefficients directly, scales through theta_s = log s, opacities through theta_o = logit(o) -- so that the
activated values the C-ABI works with (Q12) stay in (0, inf) and (0, 1).  The gradients handed in are w.r.t. the ACTIVATED
values (what gs_rasterize_bwd returns); the chain rule dL/dtheta_s = s dL/ds, dL/dtheta_o = o (1 - o) dL/do is part of the step.
Only Gaussians with a non-zero `visible` entry are touched (moments included), as in the lineage's sparse Adam; None = all.
"""
from __future__ import annotations

import numpy as np


def adam_update(theta, g, m, v, lr, t, beta1=0.9, beta2=0.999, eps=1e-15):
    """Kingma & Ba, Algorithm 1, one step (t is 1-based).  Returns (theta', m', v')."""
    m = beta1 * m + (1.0 - beta1) * g
    v = beta2 * v + (1.0 - beta2) * g * g
    mhat = m / (1.0 - beta1 ** t)
    vhat = v / (1.0 - beta2 ** t)
    return theta - lr * mhat / (np.sqrt(vhat) + eps), m, v


def adam_step(params, grads, m, v, lrs, t, visible=None, beta1=0.9, beta2=0.999, eps=1e-15):
    """params / grads / m / v: dicts with keys means, scales, quats, opacities, sh (fp64 arrays of the ABI shapes; scales
    and opacities ACTIVATED).  Returns new (params, m, v) dicts."""
    N = params["means"].shape[0]
    vis = np.ones(N, bool) if visible is None else (np.asarray(visible) != 0)
    out_p, out_m, out_v = {}, {}, {}
    for key in ("means", "scales", "quats", "opacities", "sh"):
        p = np.asarray(params[key], np.float64); g = np.asarray(grads[key], np.float64)
        if key == "scales":
            theta, gt = np.log(p), g * p
        elif key == "opacities":
            theta, gt = np.log(p) - np.log1p(-p), g * p * (1.0 - p)
        else:
            theta, gt = p, g
        th2, m2, v2 = adam_update(theta, gt, np.asarray(m[key], np.float64), np.asarray(v[key], np.float64), lrs[key], t,
                                  beta1, beta2, eps)
        if key == "scales":
            p2 = np.exp(th2)
        elif key == "opacities":
            p2 = 1.0 / (1.0 + np.exp(-th2))
        else:
            p2 = th2
        sel = vis.reshape((N,) + (1,) * (p.ndim - 1))
        out_p[key] = np.where(sel, p2, p)
        out_m[key] = np.where(sel, m2, np.asarray(m[key], np.float64))
        out_v[key] = np.where(sel, v2, np.asarray(v[key], np.float64))
    return out_p, out_m, out_v


def prune(arrays, opacities, min_opacity=0.005):
    """Keeps the Gaussians with opacity >= min_opacity, in their original order.  `arrays`: dict of [N,...] arrays.
    Returns (kept dict, indices of the kept Gaussians)."""
    keep = np.flatnonzero(np.asarray(opacities) >= np.float32(min_opacity))
    return {k: np.asarray(a)[keep] for k, a in arrays.items()}, keep
