"""gs_refine_views: one whole Eq. 23 iteration over a batch of keyframe views in one C call -- forward,
exposure-compensated L1 + SSIM + depth (+ normal) loss, backward with gradients accumulated over the views, pose and
exposure gradients per keyframe -- against the same composition of the oracles (gso + oracle/loss.py + oracle/normals.py)."""
import numpy as np
import pytest

from paper_2605_10760_b200 import scenes

pytestmark = pytest.mark.gpu


def _rel(a, b):
    a = np.asarray(a, np.float64); b = np.asarray(b, np.float64)
    n = np.linalg.norm(b)
    return np.linalg.norm(a - b) / n if n > 0 else np.linalg.norm(a - b)


@pytest.mark.parametrize("with_normals,view_streams", [(False, 1), (True, 1), (True, 2), (False, 3)])
def test_refine_views_matches_the_composed_oracles(oracle, with_normals, view_streams):
    import torch
    from oracle import loss as ol, normals as on
    from paper_2605_10760_b200 import binding as b
    W, H, V = 96, 64, 3
    sc, cams = scenes.fused_scene(seed=90, N_sub=4000, submaps=2, views=V, width=W, height=H, f=48.0, sh_degree=1)
    r = np.random.Generator(np.random.PCG64(91))
    trgb = r.uniform(0, 1, (V, 3, H, W)).astype(np.float32)
    tdep = r.uniform(0.5, 5, (V, H, W)).astype(np.float32)
    ab = np.stack([r.normal(0, 0.1, V), r.normal(0, 0.05, V)], 1).astype(np.float32)
    prior = r.normal(size=(V, 3, H, W)); prior[:, 2] = -np.abs(prior[:, 2]) - 0.5
    prior = (prior / np.linalg.norm(prior, axis=1, keepdims=True)).astype(np.float32)
    wts = (1.75, 0.2, 0.25, 0.1 if with_normals else 0.0)
    # oracle composition, view by view
    names = ("g_means", "g_scales", "g_quats", "g_opacities", "g_sh")
    acc, tw, gab, losses = None, [], [], []
    for v in range(V):
        img = oracle.forward(sc, camera=cams[v])
        lo = ol.refine_loss(img["rgb"], img["depth"], trgb[v], tdep[v], ab[v, 0], ab[v, 1], *wts[:3])
        d_depth = lo["d_depth"].copy()
        ln = 0.0
        if with_normals:
            c = cams[v]
            ln, gn = on.normal_loss(img["depth"], prior[v], np.float32(c.fx), np.float32(c.fy), np.float32(c.cx), np.float32(c.cy))
            d_depth += wts[3] * gn
        g = oracle.forward_backward(sc, lo["d_rgb"], d_depth, camera=cams[v])
        acc = {k: g[k].copy() for k in names} if acc is None else {k: acc[k] + g[k] for k in names}
        tw.append(g["g_twist"]); gab.append([lo["g_a"], lo["g_b"]]); losses.append([lo["l1_rgb"], lo["ssim"], lo["l1_depth"], lo["total"], wts[3] * ln])
    # GPU: one call
    ctx = b.Context(0)
    # view_streams > 1: the views run concurrently on sub-contexts / streams and all ACCUMULATE into zeroed arrays
    ctx.gs_set_option(b.GS_OPT_VIEW_STREAMS, view_streams)
    ds = b.DeviceScene(sc)
    params = dict(means=ds.means, scales=ds.scales, quats=ds.quats, opacities=ds.opacities, sh=ds.sh)
    grads = {k: torch.full_like(t, 3.0) for k, t in params.items()}      # view 0 overwrites whatever is there
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    g_twist = torch.zeros(V, 6, device="cuda"); g_ab = torch.zeros(V, 2, device="cuda")
    loss = torch.zeros(V, 10, dtype=torch.float64, device="cuda"); vis = torch.full((sc.N,), 7, dtype=torch.int32, device="cuda")
    args = (params, 1, cams, t(trgb), t(tdep), t(ab), wts, sc.bg, grads, g_twist, g_ab, loss)
    for attempt in range(3):
        try:
            ctx.gs_refine_views(*args, normal_prior=t(prior) if with_normals else None, visible=vis)
            torch.cuda.synchronize(); ctx.gs_poll()
            break
        except b.GsError as e:
            if e.code != -5 or attempt == 2:
                raise
    for k, gk in zip(("means", "scales", "quats", "opacities", "sh"), names):
        assert _rel(grads[k].cpu().numpy(), acc[gk]) <= 1e-3, (k, _rel(grads[k].cpu().numpy(), acc[gk]))
    got_l = loss.cpu().numpy()
    for v in range(V):
        assert _rel(g_twist[v].cpu().numpy(), tw[v]) <= 1e-3
        assert np.allclose(g_ab[v].cpu().numpy(), gab[v], rtol=1e-4, atol=1e-6)
        assert np.allclose(got_l[v, :4], losses[v][:4], rtol=1e-5) and np.isclose(got_l[v, 8], losses[v][4], rtol=1e-4, atol=1e-12)
    seen = np.zeros(sc.N, bool)
    for v in range(V):
        seen |= oracle.preprocess(sc, camera=cams[v])["visible"].astype(bool)
    gv = vis.cpu().numpy()
    assert set(np.unique(gv)) <= {0, 1} and (gv[seen] == 1).all() and gv.sum() <= seen.sum() * 1.01 + 2
    ctx.close()


def test_overflow_on_a_view_sub_context_is_reported_by_gs_poll():
    """GS_OPT_VIEW_STREAMS = 2: view 1 runs on a context-owned sub-context.  If only THAT context's instance capacity
    overflows (its calibration view saw almost nothing, the next call's view sees the whole scene), gs_poll on the parent
    after the stream sync must say so -- the accumulated gradients are missing a view -- and the re-issued call must agree
    with a single-stream context."""
    import torch
    from paper_2605_10760_b200 import binding as b
    W, H = 300, 170
    sc = scenes.replica_scene(seed=36, N=20000, width=W, height=H, f=150.0, sh_degree=1)
    near = sc.camera
    away = near.copy()
    away.T_cw = near.T_cw.copy()
    away.T_cw[2, 3] -= 1000.0                         # the whole scene lies far behind this camera: no instances at all
    r = np.random.Generator(np.random.PCG64(95))
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    trgb = t(r.uniform(0, 1, (2, 3, H, W)).astype(np.float32)); tdep = t(r.uniform(0.5, 5, (2, H, W)).astype(np.float32))
    ab = t(np.zeros((2, 2), np.float32))
    ds = b.DeviceScene(sc)
    params = dict(means=ds.means, scales=ds.scales, quats=ds.quats, opacities=ds.opacities, sh=ds.sh)
    wts = (1.75, 0.2, 0.25, 0.0)

    def run(ctx, cams):
        grads = {k: torch.zeros_like(v) for k, v in params.items()}
        g_twist = torch.zeros(2, 6, device="cuda"); g_ab = torch.zeros(2, 2, device="cuda")
        loss = torch.zeros(2, 10, dtype=torch.float64, device="cuda")
        ctx.gs_refine_views(params, 1, cams, trgb, tdep, ab, wts, sc.bg, grads, g_twist, g_ab, loss)
        torch.cuda.synchronize()
        return grads, g_twist

    ctx = b.Context(0)
    ctx.gs_set_option(b.GS_OPT_VIEW_STREAMS, 2)
    run(ctx, [near, away])                 # calibration: the sub-context (view 1) sizes itself for an almost empty view
    ctx.gs_poll()
    run(ctx, [near, near])                 # view 1 overflows the sub-context; the parent (same view as before) does not
    with pytest.raises(b.GsError, match="GS_E_OVERFLOW") as e:
        ctx.gs_poll()
    assert "view stream 1" in str(e.value)
    ctx.gs_poll()                          # reported once; both contexts are clean (and the sub-context has grown)
    grads, g_twist = run(ctx, [near, near])
    ctx.gs_poll()
    # left unpolled, the same overflow is caught at the ENTRY of the next gs_refine_views, before anything is enqueued
    ctx2 = b.Context(0)
    ctx2.gs_set_option(b.GS_OPT_VIEW_STREAMS, 2)
    run(ctx2, [near, away]); run(ctx2, [near, near])
    with pytest.raises(b.GsError, match="GS_E_OVERFLOW"):
        run(ctx2, [near, near])
    ctx2.close()
    one = b.Context(0)
    want, want_twist = run(one, [near, near])
    one.gs_poll()
    for k in params:
        assert _rel(grads[k].cpu().numpy(), want[k].cpu().numpy()) <= 1e-5, k
        assert float(want[k].abs().max()) > 0
    assert _rel(g_twist.cpu().numpy(), want_twist.cpu().numpy()) <= 1e-5
    ctx.close(); one.close()
