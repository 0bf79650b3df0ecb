"""GPU parity of the optimiser step and pruning (gs_adam_step, gs_prune_mask, gs_compact_*) against
oracle/optim.py: parameters within 1e-6 relative after several steps, moments within 1e-6, untouched Gaussians bit-identical,
pruning index lists bit-exact and order-preserving."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

KEYS = ("means", "scales", "quats", "opacities", "sh")


def _state(seed, N, K):
    r = np.random.Generator(np.random.PCG64(seed))
    f = lambda a: np.ascontiguousarray(a, np.float32)
    p = dict(means=f(r.normal(size=(N, 3))), scales=f(np.exp(r.normal(-3, 0.5, (N, 3)))), quats=f(r.normal(size=(N, 4))),
             opacities=f(1 / (1 + np.exp(-r.normal(0, 1.5, N)))), sh=f(r.normal(0, 0.2, (N, K, 3))))
    return p, r


@pytest.mark.parametrize("N,deg,masked", [(1000, 3, True), (4097, 0, False), (1, 1, True), (0, 2, False)])
def test_adam_steps_match_oracle(N, deg, masked):
    import torch
    from oracle import optim as oo
    from paper_2605_10760_b200 import binding as b
    K = (deg + 1) ** 2
    p, r = _state(70 + N, N, K)
    lrs = dict(means=1.6e-4, scales=5e-3, quats=1e-3, opacities=5e-2, sh=2.5e-3)
    dp = {k: torch.from_numpy(a.copy()).cuda() for k, a in p.items()}
    dm = {k: torch.zeros_like(t) for k, t in dp.items()}
    dv = {k: torch.zeros_like(t) for k, t in dp.items()}
    op = {k: a.astype(np.float64) for k, a in p.items()}
    om = {k: np.zeros_like(a) for k, a in op.items()}
    ov = {k: np.zeros_like(a) for k, a in op.items()}
    for t in range(1, 6):
        g = {k: np.ascontiguousarray(r.normal(size=a.shape) * (10.0 if k == "opacities" else 1.0), np.float32) for k, a in p.items()}
        vis = (r.uniform(size=N) < 0.4).astype(np.int32) if masked else None
        dg = {k: torch.from_numpy(a).cuda() for k, a in g.items()}
        if N == 0:
            b.gs_adam_step(dp, dg, dm, dv, lrs, t, None)
            continue
        b.gs_adam_step(dp, dg, dm, dv, lrs, t, None if vis is None else torch.from_numpy(vis).cuda())
        # the oracle steps from the GPU's own fp32 state (one step of rounding, not five accumulated), as the kernel does
        prev = {k: dp_k for k, dp_k in op.items()}
        # the constants are the float32 values the C-ABI receives, promoted
        f32 = lambda x: float(np.float32(x))
        op, om, ov = oo.adam_step(op, {k: a.astype(np.float64) for k, a in g.items()}, om, ov, {k: f32(x) for k, x in lrs.items()},
                                  t, vis, beta1=f32(0.9), beta2=f32(0.999), eps=f32(1e-15))
        torch.cuda.synchronize()
        for k in KEYS:
            got = dp[k].cpu().numpy().astype(np.float64)
            assert np.allclose(got, op[k], rtol=2e-6, atol=1e-9), (k, t, np.abs(got / op[k] - 1).max())
            # m is a signed sum (two fp32 roundings of terms up to max|g| / 10): absolute bound; v is a sum of squares: relative
            assert np.allclose(dm[k].cpu().numpy(), om[k], rtol=2e-6, atol=2e-7 * max(1.0, float(np.abs(g[k]).max())))
            assert np.allclose(dv[k].cpu().numpy(), ov[k], rtol=2e-6, atol=1e-14)
            if vis is not None:   # untouched Gaussians: bit-identical parameters
                assert np.array_equal(dp[k].cpu().numpy()[vis == 0], prev[k].astype(np.float32)[vis == 0])
        assert (dp["scales"] > 0).all() and ((dp["opacities"] > 0) & (dp["opacities"] < 1)).all()
        op = {k: dp[k].cpu().numpy().astype(np.float64) for k in KEYS}
        om = {k: dm[k].cpu().numpy().astype(np.float64) for k in KEYS}
        ov = {k: dv[k].cpu().numpy().astype(np.float64) for k in KEYS}


@pytest.mark.parametrize("N", [0, 1, 1023, 1024, 1025, 300_000, 2_000_003])
def test_prune_and_compaction_bit_exact(N):
    import torch
    from oracle import optim as oo
    from paper_2605_10760_b200 import binding as b
    r = np.random.Generator(np.random.PCG64(80 + N % 97))
    o = np.ascontiguousarray(r.uniform(0, 0.02, N), np.float32)
    if N > 4:
        o[1], o[2], o[3] = np.float32(0.005), np.nextafter(np.float32(0.005), np.float32(0)), 0.0
    means = np.ascontiguousarray(r.normal(size=(N, 3)), np.float32)
    sh = np.ascontiguousarray(r.normal(size=(N, 4, 3)), np.float32)
    kept, idx = oo.prune(dict(means=means, sh=sh, opacities=o), o, 0.005)
    do = torch.from_numpy(o).cuda()
    keep = torch.empty(N, dtype=torch.uint8, device="cuda")
    b.gs_prune_mask(do, 0.005, keep)
    out, index = b.gs_compact(keep, dict(means=torch.from_numpy(means).cuda(), sh=torch.from_numpy(sh).cuda(), opacities=do))
    torch.cuda.synchronize()
    want_keep = np.zeros(N, bool); want_keep[idx] = True
    assert np.array_equal(keep.cpu().numpy().astype(bool), want_keep)
    for k in kept:
        assert np.array_equal(out[k].cpu().numpy(), kept[k]), k
    ix = index.cpu().numpy().view(np.uint32)
    assert np.array_equal(ix[want_keep], np.arange(len(idx), dtype=np.uint32)) and (ix[~want_keep] == 0xFFFFFFFF).all()


def test_sparse_gradients_and_sparse_adam(oracle):
    """GS_SPARSE_GRADS: one gradient row per visible Gaussian, in the order of gs_visible_ids -- against the oracle's dense
    gradients gathered at those indices; gs_adam_step_sparse on them == gs_adam_step with the visibility mask, bit for bit."""
    import torch
    from paper_2605_10760_b200 import binding as b, scenes
    sc = scenes.replica_scene(seed=39, N=20000, width=300, height=170, f=150.0, sh_degree=2)
    gC, gD = scenes.upstream_gradients(39, 300, 170)
    ref = oracle.forward_backward(sc, gC, gD)
    ctx = b.Context(0)
    ds = b.DeviceScene(sc)
    out = ds.alloc_outputs(300, 170)
    b.forward(ctx, ds, sc.camera, out)
    nv, _ = ctx.gs_get_counts()
    for k in ("g_means", "g_scales", "g_quats", "g_opacities", "g_sh"):
        out[k].fill_(123.0)                       # rows beyond n_visible must stay untouched
    b.backward(ctx, out, torch.from_numpy(gC).cuda(), torch.from_numpy(gD).cuda(), None, flags=b.GS_SPARSE_GRADS)
    torch.cuda.synchronize()
    ids_ptr, n_ptr = ctx.gs_visible_ids()
    holder = ctx.gs_get_visible_ids()[:nv].clone()
    ids_h = holder.cpu().numpy().astype(np.int64)
    assert len(set(ids_h.tolist())) == nv and (ref["visible"][ids_h] == 1).all()
    for gk, rk in (("g_means", "g_means"), ("g_scales", "g_scales"), ("g_quats", "g_quats"), ("g_opacities", "g_opacities"), ("g_sh", "g_sh")):
        got = out[gk].cpu().numpy()
        want = ref[rk][ids_h]
        rel = np.linalg.norm(got[:nv].astype(np.float64) - want) / np.linalg.norm(want)
        assert rel <= 1e-3, (gk, rel)
        assert (got[nv:] == 123.0).all(), gk
    assert np.linalg.norm(out["g_twist"].cpu().numpy() - ref["g_twist"]) <= 1e-3 * np.linalg.norm(ref["g_twist"])
    with pytest.raises(b.GsError, match="GS_E_INVALID"):
        b.backward(ctx, out, torch.from_numpy(gC).cuda(), torch.from_numpy(gD).cuda(), None, flags=b.GS_SPARSE_GRADS | b.GS_ACCUMULATE)
    # sparse Adam == masked dense Adam, bit for bit
    keys = ("means", "scales", "quats", "opacities", "sh")
    pa = dict(means=ds.means.clone(), scales=ds.scales.clone(), quats=ds.quats.clone(), opacities=ds.opacities.clone(), sh=ds.sh.clone())
    pb = {k: t.clone() for k, t in pa.items()}
    ma = {k: torch.zeros_like(t) for k, t in pa.items()}; va = {k: torch.zeros_like(t) for k, t in pa.items()}
    mb = {k: torch.zeros_like(t) for k, t in pa.items()}; vb = {k: torch.zeros_like(t) for k, t in pa.items()}
    sparse = dict(means=out["g_means"], scales=out["g_scales"], quats=out["g_quats"], opacities=out["g_opacities"], sh=out["g_sh"])
    dense = {k: torch.zeros_like(t) for k, t in pa.items()}
    idt = holder.long()
    for k in keys:
        dense[k][idt] = sparse[k][:nv]
    mask = torch.zeros(sc.N, dtype=torch.int32, device="cuda"); mask[idt] = 1
    lrs = dict(means=1.6e-4, scales=5e-3, quats=1e-3, opacities=5e-2, sh=2.5e-3)
    b.gs_adam_step_sparse(pa, sparse, ma, va, lrs, 1, ids_ptr, n_ptr, sc.N)
    b.gs_adam_step(pb, dense, mb, vb, lrs, 1, mask)
    torch.cuda.synchronize()
    for k in keys:
        assert torch.equal(pa[k], pb[k]) and torch.equal(ma[k], mb[k]) and torch.equal(va[k], vb[k]), k
        assert not torch.equal(pa[k], getattr(ds, k))
    ctx.close()
