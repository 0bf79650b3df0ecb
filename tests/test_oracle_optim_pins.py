"""Pins of the optimiser / pruning oracle (oracle/optim.py): textbook Adam closed forms, the activated-
parameter chain rule against an explicit raw-parameter optimisation, sparse-visibility semantics, pruning."""
import numpy as np

from oracle import optim as oo


def test_first_adam_step_is_minus_lr_sign_g_and_bias_correction():
    g = np.array([0.3, -2.0, 1e-4])
    th, m, v = oo.adam_update(np.zeros(3), g, np.zeros(3), np.zeros(3), lr=0.01, t=1, eps=0.0)
    assert np.allclose(th, -0.01 * np.sign(g), rtol=1e-12)           # mhat / sqrt(vhat) = g / |g| at t = 1
    assert np.allclose(m, 0.1 * g) and np.allclose(v, 0.001 * g * g)
    # constant gradient: every step moves by lr (bias-corrected moments stay g and g^2)
    th, m, v = np.zeros(1), np.zeros(1), np.zeros(1)
    for t in range(1, 6):
        th, m, v = oo.adam_update(th, np.array([0.7]), m, v, lr=0.02, t=t, eps=0.0)
    assert np.allclose(th, -5 * 0.02, rtol=1e-12)
    # hand-computed second step with a different gradient
    g1, g2 = 1.0, -3.0
    m2 = 0.9 * 0.1 * g1 + 0.1 * g2; v2 = 0.999 * 0.001 * g1 * g1 + 0.001 * g2 * g2
    want = -0.1 - 0.1 * (m2 / (1 - 0.81)) / np.sqrt(v2 / (1 - 0.999 ** 2))
    th, m, v = oo.adam_update(np.zeros(1), np.array([g1]), np.zeros(1), np.zeros(1), 0.1, 1, eps=0.0)
    th, m, v = oo.adam_update(th, np.array([g2]), m, v, 0.1, 2, eps=0.0)
    assert np.allclose(th, want, rtol=1e-12)


def _state(seed, N=7, K=4):
    r = np.random.Generator(np.random.PCG64(seed))
    p = dict(means=r.normal(size=(N, 3)), scales=np.exp(r.normal(-3, 0.5, (N, 3))), quats=r.normal(size=(N, 4)),
             opacities=1 / (1 + np.exp(-r.normal(0, 1, N))), sh=r.normal(0, 0.2, (N, K, 3)))
    g = {k: r.normal(size=a.shape) for k, a in p.items()}
    z = {k: np.zeros_like(a) for k, a in p.items()}
    return p, g, z


def test_activated_parametrisation_equals_raw_parameter_adam():
    p, g, z = _state(1)
    lrs = dict(means=1e-3, scales=5e-3, quats=1e-3, opacities=5e-2, sh=2.5e-3)
    p2, m2, v2 = oo.adam_step(p, g, z, z, lrs, t=1)
    # explicit raw parameters: theta_s = log s, theta_o = logit o, gradient by the chain rule
    ths, _, _ = oo.adam_update(np.log(p["scales"]), g["scales"] * p["scales"], 0, 0, lrs["scales"], 1)
    assert np.allclose(p2["scales"], np.exp(ths), rtol=1e-13) and (p2["scales"] > 0).all()
    o = p["opacities"]
    tho, _, _ = oo.adam_update(np.log(o / (1 - o)), g["opacities"] * o * (1 - o), 0, 0, lrs["opacities"], 1)
    assert np.allclose(p2["opacities"], 1 / (1 + np.exp(-tho)), rtol=1e-13)
    assert ((p2["opacities"] > 0) & (p2["opacities"] < 1)).all()
    thm, _, _ = oo.adam_update(p["means"], g["means"], 0, 0, lrs["means"], 1)
    assert np.allclose(p2["means"], thm)
    # a huge learning rate still cannot leave the domains
    p3, _, _ = oo.adam_step(p, g, z, z, {k: 50.0 for k in lrs}, t=1)
    assert (p3["scales"] > 0).all() and ((p3["opacities"] >= 0) & (p3["opacities"] <= 1)).all()


def test_visibility_mask_freezes_parameters_and_moments():
    p, g, z = _state(2)
    lrs = {k: 1e-2 for k in p}
    vis = np.array([1, 0, 1, 1, 0, 0, 1])
    m0 = {k: np.full_like(a, 0.25) for k, a in p.items()}
    p2, m2, v2 = oo.adam_step(p, g, m0, z, lrs, t=3, visible=vis)
    for k in p:
        assert np.array_equal(p2[k][vis == 0], p[k][vis == 0]) and np.array_equal(m2[k][vis == 0], m0[k][vis == 0])
        assert not np.allclose(p2[k][vis == 1], p[k][vis == 1])
    pa, _, _ = oo.adam_step(p, g, m0, z, lrs, t=3)
    for k in p:
        assert np.array_equal(p2[k][vis == 1], pa[k][vis == 1])


def test_prune_keeps_order_and_the_paper_threshold():
    o = np.array([0.5, 0.004, 0.005, 0.0049999, 0.9, 0.0], np.float32)
    kept, idx = oo.prune(dict(a=np.arange(6) * 10, b=np.arange(12).reshape(6, 2)), o)   # opacity below 0.005 is pruned
    assert np.array_equal(idx, [0, 2, 4]) and np.array_equal(kept["a"], [0, 20, 40]) and np.array_equal(kept["b"][1], [4, 5])
