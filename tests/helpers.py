"""Shared helpers of the GPU parity tests: drive libcs through its Python binding and the oracle on the same
seeded Workload, and apply the tolerance rules T1-T4.  Nothing here computes any
expected value itself."""
import numpy as np

import gen
import oracle


# Context options applied by new_ctx / make_ctx; the `path` fixture of the GPU tests switches them so that every parity
# case runs on the sorted layout (sorted-cell kernel) and in place (direct kernel).
CTX_OPTIONS = {}


def new_ctx(freqs, npix, units=0, options=None):
    import paper_2604_08463_b200 as cs
    return cs.Context(freqs, npix, units=units, options=CTX_OPTIONS if options is None else options)


def make_ctx(w, d_dev=None, device="cuda:0", units=0, options=None):
    """Context with the workload's clusters, data and batch set.  Returns (ctx, d_dev)."""
    import torch
    ctx = new_ctx(w.freqs, w.npix, units=units, options=options)
    ctx.set_clusters(w.maps, w.Kmap, w.cfg_maps, w.region_idx, w.nregion)
    if d_dev is None:
        d_dev = torch.from_numpy(w.data()).to(device)
    ctx.set_data(d_dev, w.ninv)
    ctx.set_batch(w.cfg_of, w.data_of)
    return ctx, d_dev


def gpu_eval(ctx, params, want_grad=True):
    """nll [B,nregion], grad [nparam] as numpy fp64."""
    import torch
    p = torch.from_numpy(np.ascontiguousarray(params, dtype=np.float64)).cuda()
    nll = torch.full((ctx.batch * ctx.nregion,), float("nan"), dtype=torch.float64, device="cuda")
    grad = torch.full_like(p, float("nan")) if want_grad else None
    ctx.build_sed_tables(p)
    ctx.spectral_like_grad(nll, grad)
    torch.cuda.synchronize()
    return nll.cpu().numpy().reshape(ctx.batch, ctx.nregion), (grad.cpu().numpy() if want_grad else None)


def gpu_maps(ctx, params, entries=None, npix=None):
    import torch
    p = torch.from_numpy(np.ascontiguousarray(params, dtype=np.float64)).cuda()
    nsel = ctx.batch if entries is None else len(entries)
    s = torch.full((nsel, 3, 2, ctx.npix), float("nan"), dtype=torch.float32, device="cuda")
    ctx.build_sed_tables(p)
    ctx.component_maps(s, entries)
    torch.cuda.synchronize()
    return s.cpu().numpy()


def oracle_entry(w, params, e, model=None, want_maps=False, data=None):
    """The oracle on batch entry e (dict of oracle.nll_grad, with tolerance scales)."""
    model = model or oracle.Model(w.freqs)
    off = w.param_offsets()
    c = int(w.cfg_of[e])
    d = (data if data is not None else w.data())[int(w.data_of[e])]
    return oracle.nll_grad(model, d, w.ninv, w.maps[w.cfg_maps[c]], w.K_of_cfg(c), params[off[e]:off[e + 1]],
                           region=w.region_idx, nregion=w.nregion, want_maps=want_maps, want_tol=True)


def check_T1(nll_gpu, nll_ref, rtol=1e-5):
    """T1: |nll_gpu - nll_ref| <= 1e-5 |nll_ref| (per entry and region)."""
    nll_gpu, nll_ref = np.asarray(nll_gpu), np.asarray(nll_ref)
    err = np.abs(nll_gpu - nll_ref)
    assert np.all(err <= rtol * np.abs(nll_ref) + 1e-300), (float(err.max()), nll_gpu, nll_ref)
    return float((err / np.maximum(np.abs(nll_ref), 1e-300)).max())


def grad_errors_unfloored(g_gpu, ref, K):
    """What the T2 bounds hide: per parameter block ||dg||_2 / ||g_ref||_2 (no floor), and the worst single cluster
    |dg_k| / |g_ref_k|.  north_star's literal "1e-4 on gradients" is the block figure; it holds away from optima."""
    g_ref = ref["grad"]
    o, blocks = 0, []
    for k in K:
        sl = slice(o, o + k)
        blocks.append(float(np.linalg.norm(g_gpu[sl] - g_ref[sl]) / max(np.linalg.norm(g_ref[sl]), 1e-300)))
        o += k
    nz = np.abs(g_ref) > 0
    worst = float(np.max(np.abs(g_gpu - g_ref)[nz] / np.abs(g_ref)[nz])) if nz.any() else 0.0
    return blocks, worst


def check_T2(g_gpu, ref, K, rtol=1e-4, floor=1e-6):
    """T2: per parameter block ||dg||_2 <= 1e-4 ||g_ref||_2 + 1e-6 ||Gscale||_2 and per cluster
    |dg_k| <= 1e-4 sum_p |g_p| + 1e-6 Gscale_k.  Failure messages carry the unfloored errors too."""
    g_ref, absg, gs = ref["grad"], ref["absg"], ref["gscale"]
    dg = np.abs(g_gpu - g_ref)
    bad = dg > rtol * absg + floor * gs
    blocks, worst_rel = grad_errors_unfloored(g_gpu, ref, K)
    info = {"block ||dg||/||g_ref|| (no floor)": blocks, "worst cluster |dg|/|g_ref|": worst_rel}
    assert not bad.any(), (np.flatnonzero(bad)[:8], dg[bad][:8], (rtol * absg + floor * gs)[bad][:8], info)
    o = 0
    worst = 0.0
    for k in K:
        sl = slice(o, o + k)
        lhs = np.linalg.norm(g_gpu[sl] - g_ref[sl])
        rhs = rtol * np.linalg.norm(g_ref[sl]) + floor * np.linalg.norm(gs[sl])
        assert lhs <= rhs, (o, lhs, rhs, info)
        worst = max(worst, lhs / max(rhs, 1e-300))
        o += k
    return worst


def check_T3(s_gpu, s_ref, rtol=1e-5):
    """T3: per component ||ds||_2 <= 1e-5 ||s_ref||_2 and max|ds| <= 1e-5 max|s_ref|."""
    worst = 0.0
    for c in range(3):
        ds = s_gpu[c].astype(np.float64) - s_ref[c]
        l2, mx = np.linalg.norm(ds) / np.linalg.norm(s_ref[c]), np.abs(ds).max() / np.abs(s_ref[c]).max()
        assert l2 <= rtol and mx <= rtol, (c, l2, mx)
        worst = max(worst, l2, mx)
    return worst
