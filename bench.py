#!/usr/bin/env python
"""bench.py -- pixel-evals/s of the fused -logL + gradient hot path (BASELINE.json `metric`) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload c3h|c5|c4|c3|c2] [--batch B]

A step = one pass of the hot path over one batch: cs_build_sed_tables (a1) + cs_spectral_like_grad (a2 + a3,
value and gradient) for every batch entry.  The default workload "c3h" is the shape the metric is quoted on
("nside=64 with batch >= 1024", BASELINE.json north_star): nside 64, K = (500, 50, 100), 1024 entries each with its
own noise realisation, so that the data stream (6.04 GB per step) is larger than L2 and has to come from HBM.
Inputs are seeded and synthetic (gen/); see DESIGN.md "Input recipe".

--gpus N > 1 without a torchrun environment re-launches itself under torch.distributed.run with one rank per GPU
(batch-sharded replicas, no collective on the data path: DESIGN.md "Multi-GPU"); NCCL is used for the timing barrier
and the max over ranks only.

Prints ONE JSON line (rank 0).  Keys beyond the base contract: `roofline`, `cpu_baseline`, `e2e`, `clocks`,
`gpu_launches`, `parity` (GPU vs oracle on the cpu_baseline sample), `extras` (every other BASELINE configuration, the
cell-size sweep, f2, f3) and, as the LAST key, `configs`: one short array per configuration (summary_of).
"""
import argparse
import json
import os
import socket
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import gen  # noqa: E402

METRIC = "pixel-evals/s of fused -logL+grad (batch x npix)"
UNIT = "pixel-evals/s"
BYTES_PER_PIXEL_EVAL = 120.0   # 15 bands x (Q,U) x fp32: the compulsory d stream


def make_workload(name, batch, rank=0):
    """Workload for this rank.  Noise realisations are offset by rank so that ranks hold distinct data."""
    if name == "c3h":
        B = batch or 1024
        w = gen.make_config(1, ndata=B)
        desc = f"C3-H: nside 64, K=(500,50,100), {B} entries x distinct noise realisations"
    elif name == "c5":
        B = batch or 256
        w = gen.make_config(4, ndata=B)
        desc = f"C5: nside 128, K=(2000,200,400), {B} noise realisations"
    elif name == "c3":
        B = batch or 1024
        w = gen.make_config(2, batch=B)
        desc = f"C3: nside 64 clustering scan, {B} configurations sharing one data set"
    elif name == "c4":
        w = gen.make_config(3, batch=batch or None)
        desc = f"C4: nside 64, 3 latitude regions, 64 configurations x 100 noise realisations ({w.batch} entries, 100 data sets)"
    elif name == "kmax":
        # the shape of the paper's own optimum (Table 2: beta_d per pixel, K_Td = 2500, K_bs = 150): every pixel
        # is its own cell, the configuration stays in place on the direct kernel
        B = batch or 256
        w = gen.make_config(1, ndata=B, K=(49152, 2500, 150))
        desc = f"Kmax: nside 64, K=(npix,2500,150) (beta_d per pixel, PAPER.md Table 2), {B} entries x distinct noise realisations"
    elif name == "c2":
        w = gen.make_config(1)
        desc = "C2: nside 64, K=(500,50,100), one entry"
    else:
        raise SystemExit(f"unknown workload {name}")
    if rank:
        w.realizations = tuple(r + rank * w.ndata for r in w.realizations)
    return w, desc


class ClockSampler:
    """Samples SM clocks and throttle reasons with nvidia-smi while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, smax, reasons, power = [], None, set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for t, line in self.rows:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                mhz, mx = float(f[0]), float(f[1])
            except ValueError:
                continue
            smax = mx
            if t0 - 0.05 <= t <= t1 + 0.05:
                sm.append(mhz)
                try:
                    power.append(float(f[2]))
                except ValueError:
                    pass
                for nm, v in zip(names, f[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
        if not sm and self.rows:   # region shorter than the sampling period: take the nearest sample
            f = [x.strip() for x in min(self.rows, key=lambda r: abs(r[0] - t0))[1].split(",")]
            try:
                sm = [float(f[0])]
            except ValueError:
                sm = []
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": smax, "reasons": sorted(reasons),
                "power_w_max": max(power) if power else None, "samples": len(sm)}


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def oracle_sample(w, params, budget_s=12.0, min_entries=2, max_entries=64, threads=None):
    """Times the oracle, as it stands, on the first entries of the workload until `budget_s` is used.
    Returns (pixel-evals/s, threads, entries, per-entry results)."""
    import oracle
    all_threads = oracle.num_threads()
    if threads:
        oracle.set_num_threads(threads)
    model = oracle.Model(w.freqs)
    off = w.param_offsets()
    d = w.data()
    res, t_used, n = [], 0.0, 0
    while n < min(max_entries, w.batch) and (n < min_entries or t_used < budget_s):
        c = int(w.cfg_of[n])
        t0 = time.perf_counter()
        r = oracle.nll_grad(model, d[int(w.data_of[n])], w.ninv, w.maps[w.cfg_maps[c]], w.K_of_cfg(c),
                            params[off[n]:off[n + 1]], region=w.region_idx, nregion=w.nregion, want_tol=True)
        t_used += time.perf_counter() - t0
        res.append(r)
        n += 1
    used = oracle.num_threads()
    if threads:
        oracle.set_num_threads(all_threads)
    return n * w.npix / t_used, used, n, res


def run_reference(args, rank, world):
    """--impl reference: the CPU fp64 oracle on a bounded sample of the same workload (tier framing (4))."""
    if rank != 0:
        return
    import oracle
    name = args.workload
    # the oracle only needs a few entries: build a small slice of the workload
    w, desc = make_workload(name, min(args.batch or 8, 8))
    params = w.params_jittered(seed=7)
    per_step = 2
    for _ in range(args.warmup):
        oracle_sample(w, params, budget_s=0.0, min_entries=1, max_entries=1)
    t0 = time.perf_counter()
    done = 0
    for s in range(args.steps):
        sub_t, _, n, _ = oracle_sample(w, params, budget_s=0.0, min_entries=per_step, max_entries=per_step)
        done += n
    dt = time.perf_counter() - t0
    val = done * w.npix / dt
    cores = oracle.num_threads()
    out = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(args.steps, 1), "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": desc, "sample": f"{per_step} entries per step"},
           "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle",
                            "sample": f"{per_step} entries x {w.npix} pixels per step, {args.steps} steps"},
           "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(out), flush=True)


def kernel_name(ctx, w, nfreq):
    """The fused kernel(s) the batch runs on: a property of each configuration's layout (cs_layout_info)."""
    kinds = {ctx.layout_info(int(c))[0] for c in np.unique(w.cfg_of)}
    names = [f"k_like_sc<{15 if nfreq == 15 else 16},GRAD> (sorted-cell kernel, private cell-sorted copies)" if k else
             f"k_like_direct<{15 if nfreq == 15 else 16},GRAD> (direct kernel, in place)" for k in sorted(kinds, reverse=True)]
    return " + ".join(names)


def copies_bytes(ctx, w):
    """Bytes of the private cell-sorted copies of the batch: one per distinct (sorted configuration, data set) pair, its
    tiles x 512 positions x nfreq x (Q, U) x fp32."""
    info = {int(c): ctx.layout_info(int(c)) for c in np.unique(w.cfg_of)}
    pairs = {(int(c), int(d)) for c, d in zip(w.cfg_of, w.data_of) if info[int(c)][0]}
    return sum(info[c][1] * 512 * w.nfreq * 2 * 4 for c, _ in pairs)


def time_hot_path(ctx, w, params, steps, warmup, dev, stream, barrier=None):
    """W warm-up steps, then K timed steps of (tables + likelihood/gradient) with CUDA events on `stream`.
    Returns dict(ms, kernel_ms (fused kernels per step), launches, nll, grad)."""
    import torch
    p_dev = torch.from_numpy(params).to(dev)
    nll = torch.zeros(w.batch * w.nregion, dtype=torch.float64, device=dev)
    grad = torch.zeros_like(p_dev)

    def step():
        ctx.build_sed_tables(p_dev, stream)
        ctx.spectral_like_grad(nll, grad, stream)

    sync = barrier or torch.cuda.synchronize
    for _ in range(warmup):
        step()
    sync()
    if ctx.check() != 0:
        raise SystemExit("device error bit set during warm-up")
    ctx.profile(True)
    l0 = ctx.kernel_launches()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sync()
    t0 = time.time()
    ev0.record(stream)
    for _ in range(steps):
        step()
    ev1.record(stream)
    sync()
    t1 = time.time()
    ms = ev0.elapsed_time(ev1)
    launches = ctx.kernel_launches() - l0
    k_ms, k_n = ctx.profile_read()
    ctx.profile(False)
    return {"ms": ms, "kernel_ms_per_step": k_ms / max(steps, 1), "kernel_launches_per_step": k_n / max(steps, 1),
            "launches": launches, "nll": nll, "grad": grad, "p_dev": p_dev, "t0": t0, "t1": t1}


def extra_workload(cs, name, batch, steps, dev, stream, peak, prefixes=None):
    """Short runs of another BASELINE configuration for `extras`: the whole batch, or (prefixes) its first b entries for
    every b in `prefixes` on the same context and data (the batch sweep of config 5).  Returns {key: result}."""
    import torch
    t0 = time.time()
    w, desc = make_workload(name, batch)
    d_dev = torch.from_numpy(w.data()).to(dev)
    t_gen = time.time() - t0
    t0 = time.time()
    ctx = cs.Context(w.freqs, w.npix)
    ctx.set_clusters(w.maps, w.Kmap, w.cfg_maps, w.region_idx, w.nregion)
    ctx.set_data(d_dev, w.ninv)
    torch.cuda.synchronize()
    t_setup = time.time() - t0
    res = {}
    params_all = w.params_jittered(seed=7)
    off = w.param_offsets()
    for b in (prefixes or [w.batch]):
        import dataclasses
        wb = dataclasses.replace(w, cfg_of=w.cfg_of[:b], data_of=w.data_of[:b])
        t0 = time.time()
        ctx.set_batch(wb.cfg_of, wb.data_of)
        torch.cuda.synchronize()
        t_batch = time.time() - t0
        r = time_hot_path(ctx, wb, params_all[:off[b]], steps, 3, dev, stream)
        pe = float(b) * w.npix
        ms_step = r["ms"] / steps
        sorted_cfgs = sum(1 for c in np.unique(wb.cfg_of) if ctx.layout_info(int(c))[0])
        streams = len({(int(c), int(d)) for c, d in zip(wb.cfg_of, wb.data_of)}) if sorted_cfgs else len(np.unique(wb.data_of))
        res[b] = {"workload": desc if b == w.batch else f"{desc}: first {b} entries", "batch": b, "npix": w.npix, "steps": steps,
                  "ms_per_step": ms_step, "pixel_evals_per_s": pe / (ms_step * 1e-3),
                  "fused_kernel_ms_per_step": r["kernel_ms_per_step"], "kernel": kernel_name(ctx, wb, w.nfreq),
                  # d-stream accounting (120 B per pixel-eval): every entry streams its own (private) data
                  "roofline_frac_of_measured_peak": BYTES_PER_PIXEL_EVAL * pe / (r["kernel_ms_per_step"] * 1e-3) / 1e9 / peak
                  if r["kernel_ms_per_step"] > 0 else None,
                  "distinct_data_sets": int(len(np.unique(wb.data_of))),
                  "configurations_sorted": sorted_cfgs, "configurations": int(len(np.unique(wb.cfg_of))),
                  "streams_read_per_step": streams, "workspace_GB": ctx.workspace_bytes() / 1e9, "copies_GB": copies_bytes(ctx, wb) / 1e9,
                  "datagen_s": round(t_gen, 1), "set_clusters_and_data_s": round(t_setup, 1), "set_batch_s": round(t_batch, 3)}
    ctx.close()
    del d_dev
    torch.cuda.empty_cache()
    return res


def extra_cells(cs, name, batch, steps, dev, stream):
    """f3 on a workload: cs_cell_moments once, then steps of tables + cs_spectral_like_grad_cells.  Reported under its
    own metric: pixel-evals-equivalent/s = batch x npix / step time (no pixel is touched in the step)."""
    import torch
    w, desc = make_workload(name, batch)
    d_dev = torch.from_numpy(w.data()).to(dev)
    ctx = cs.Context(w.freqs, w.npix, options={"layout": cs.LAYOUT_SORTED})
    ctx.set_clusters(w.maps, w.Kmap, w.cfg_maps, w.region_idx, w.nregion)
    ctx.set_data(d_dev, w.ninv)
    ctx.set_batch(w.cfg_of, w.data_of)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record(stream)
    ctx.cell_moments(stream)
    e1.record(stream)
    torch.cuda.synchronize()
    mom_ms = e0.elapsed_time(e1)
    p_dev = torch.from_numpy(w.params_jittered(seed=7)).to(dev)
    nll = torch.zeros(w.batch * w.nregion, dtype=torch.float64, device=dev)
    grad = torch.zeros_like(p_dev)
    for _ in range(3):
        ctx.build_sed_tables(p_dev, stream)
        ctx.spectral_like_grad_cells(nll, grad, stream)
    torch.cuda.synchronize()
    e0.record(stream)
    for _ in range(steps):
        ctx.build_sed_tables(p_dev, stream)
        ctx.spectral_like_grad_cells(nll, grad, stream)
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    nll_pp = torch.zeros_like(nll)
    ctx.spectral_like_grad(nll_pp, None, stream)
    torch.cuda.synchronize()
    rel = float(((nll - nll_pp).abs() / nll_pp.abs()).max().item())
    out = {"metric": "f3 cell-compressed likelihood: pixel-evals-equivalent/s (batch x npix / step time)",
           "workload": desc, "batch": w.batch, "ms_per_step": ms, "pixel_evals_equivalent_per_s": w.batch * w.npix / (ms * 1e-3),
           "cell_moments_ms_once": mom_ms, "max_rel_diff_nll_vs_per_pixel_path": rel, "workspace_GB": ctx.workspace_bytes() / 1e9}
    ctx.close()
    del d_dev
    torch.cuda.empty_cache()
    return out


def extra_kmeans(cs, dev):
    """f2: the 32 distinct cluster maps of the C3 scan (nside 64, K = 1 .. 1000, 10 Lloyd iterations) in one batched call."""
    import torch
    from gen import kmeans as gk
    vecs = gen.pix2vec_ring(64)
    specs = sorted({(prm, int(k[prm])) for k in gen.c3_grid() for prm in range(3)})
    probs = [(prm, K) for prm, K in specs if 1 < K < vecs.shape[0]]
    cent0 = np.concatenate([gk.initial_centroids(vecs, K, gen.rng_for("kmeans", (prm * 1_000_003 + K) * 16)) for prm, K in probs])
    v_d = torch.from_numpy(vecs).to(dev)
    lab = torch.zeros((len(probs), vecs.shape[0]), dtype=torch.int32, device=dev)
    Ks = [K for _, K in probs]
    times = []
    for _ in range(2):
        cent = torch.from_numpy(cent0.copy()).to(dev)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        cs.spherical_kmeans(v_d, Ks, cent, lab, iters=10)
        torch.cuda.synchronize()
        times.append(time.perf_counter() - t0)
    return {"workload": f"{len(probs)} K-means problems of the C3 scan, nside 64, K = {min(Ks)} .. {max(Ks)}, 10 Lloyd iterations",
            "ms": 1e3 * min(times), "dot_products_per_s": 11 * vecs.shape[0] * float(sum(Ks)) / min(times)}


# K = (K_bd, K_Td, K_bs) of the cell-size sweep: from the paper's own optimum (beta_d per pixel, Table 2) through
# the upper half of its grid (Table 1: K up to 10000 on regions of ~9800 pixels, i.e. 1-5 pixels per cell on
# the full nside-64 sky at the same densities) down to the bench configuration.
SWEEP_K = [(49152, 2500, 150), (25000, 5000, 1500), (12500, 2500, 750), (5000, 1500, 750), (3000, 1000, 600),
           (2000, 800, 500), (1000, 500, 500), (500, 50, 100)]


def extra_cellsweep(cs, dev, stream, peak, ndata=256, steps=5):
    """Pixel-evals/s against the mean cell size (pixels per distinct cluster triple), nside 64, `ndata` entries with
    their own noise realisation, on each layout: in place (direct kernel), sorted (sorted-cell kernel) and the
    library's own choice (CS_OPT_MIN_FILL).  The patch maps come from the library's own K-means (cs_spherical_kmeans,
    seeded starts from gen): the numpy generator would need minutes for K = 25000."""
    import dataclasses
    import torch
    from gen import kmeans as gk
    w0 = gen.make_config(1, ndata=ndata)
    vecs = gen.pix2vec_ring(w0.nside)
    npix = w0.npix
    specs = sorted({(prm, int(K[prm])) for K in SWEEP_K for prm in range(3) if 1 < K[prm] < npix})
    cent0 = np.concatenate([gk.initial_centroids(vecs, K, gen.rng_for("kmeans", (prm * 1_000_003 + K) * 16)) for prm, K in specs])
    lab = torch.zeros((len(specs), npix), dtype=torch.int32, device=dev)
    cs.spherical_kmeans(torch.from_numpy(vecs).to(dev), [K for _, K in specs], torch.from_numpy(cent0).to(dev), lab, iters=10)
    torch.cuda.synchronize()
    lab = lab.cpu().numpy()
    maps_of = {s: lab[i] for i, s in enumerate(specs)}
    d_dev = torch.from_numpy(w0.data()).to(dev)
    rows = []
    for K in SWEEP_K:
        maps = np.stack([np.arange(npix, dtype=np.int32) if K[prm] >= npix else maps_of[(prm, int(K[prm]))] for prm in range(3)])
        Kmap = np.array([min(k, npix) for k in K], dtype=np.int32)
        w = dataclasses.replace(w0, maps=np.ascontiguousarray(maps), Kmap=Kmap)
        params = w.params_jittered(seed=7)
        ncell = len(np.unique(maps[0].astype(np.int64) * (int(Kmap[1]) * int(Kmap[2])) + maps[1].astype(np.int64) * int(Kmap[2]) + maps[2]))
        row = {"K": list(K), "pixels_per_cell": npix / ncell}
        for key, layout in (("inplace", cs.LAYOUT_INPLACE), ("sorted", cs.LAYOUT_SORTED), ("auto", cs.LAYOUT_AUTO)):
            try:
                ctx = cs.Context(w.freqs, w.npix, options={"layout": layout})
                ctx.set_clusters(w.maps, w.Kmap, w.cfg_maps, w.region_idx, w.nregion)
                ctx.set_data(d_dev, w.ninv)
                ctx.set_batch(w.cfg_of, w.data_of)
                r = time_hot_path(ctx, w, params, steps, 3, dev, stream)
                srt, _, fill = ctx.layout_info(0)
                row[key] = float(w.batch) * npix / (r["ms"] / steps * 1e-3)
                if key == "sorted":
                    row["fill"] = fill
                    row["copies_GB"] = copies_bytes(ctx, w) / 1e9
                if key == "auto":
                    row["auto_kernel"] = "sc" if srt else "direct"
                ctx.close()
            except Exception as exc:
                row[key] = None
                row[key + "_error"] = repr(exc)
            torch.cuda.empty_cache()
        rows.append(row)
    del d_dev
    torch.cuda.empty_cache()
    return {"workload": f"nside 64, {ndata} entries x distinct noise realisations, K swept", "steps": steps, "rows": rows}


def _short_kernel(name):
    return "+".join(k for k, tag in (("sc", "k_like_sc"), ("direct", "k_like_direct")) if tag in (name or ""))


def summary_of(out, peak):
    """Every configuration on one screen, as the LAST key of the line (a record that keeps only the tail of the line
    still shows it).  Per configuration: [ms per step, G pixel-evals/s, fraction of the measured HBM peak counting the
    bytes each entry streams (120 B per pixel-eval: every entry reads its own, private or distinct, data), the same
    fraction counting only the DISTINCT data bytes of the step (the compulsory traffic: for a scan of configurations
    over shared data the streamed bytes are replicas, not algorithmic bytes), kernel]."""
    ex = out.get("extras", {})
    s = {"fmt": "[ms/step, G pixel-evals/s, frac of HBM peak by streamed per-entry bytes, frac by distinct-data bytes, kernel]"}
    rf = out["roofline"]
    s["c3h"] = [round(out["ms_per_step"], 4), round(out["value"] / out["n_gpus"] / 1e9, 2), round(rf["frac"], 3), round(rf["frac"], 3), _short_kernel(rf["kernel"])]
    for key in ("c3", "c4", "kmax", "c5_batch1", "c5_batch16", "c5_batch64", "c5_batch256"):
        e = ex.get(key)
        if not e or "error" in e:
            continue
        fr = e.get("roofline_frac_of_measured_peak")
        s[key] = [round(e["ms_per_step"], 4), round(e["pixel_evals_per_s"] / 1e9, 2), None if fr is None else round(fr, 3),
                  None if fr is None else round(fr * e["distinct_data_sets"] / e["batch"], 4), _short_kernel(e["kernel"])]
    c2 = ex.get("c2")
    if c2:
        s["c2"] = {"like_grad_call_us": round(c2["like_grad_call_us"], 1), "adatopk_200_iters_ms": round(c2["optimize_200_iters_ms"], 2),
                   "lbfgs_100_iters_ms": round(c2["lbfgs_100_iters_ms"], 2)}
    sw = ex.get("cellsweep")
    if sw and "rows" in sw:
        g = lambda v: None if v is None else round(v / 1e9, 1)
        s["cellsweep_fmt"] = "[pixels per cell, sorted fill, G pixel-evals/s in place, sorted, auto, auto's kernel]"
        s["cellsweep"] = [[round(r["pixels_per_cell"], 2), round(r.get("fill") or 0, 3), g(r.get("inplace")), g(r.get("sorted")), g(r.get("auto")),
                           r.get("auto_kernel")] for r in sw["rows"]]
    for key in ("f3_cells_c3", "f3_cells_c3h", "f3_cells_c4"):
        e = ex.get(key)
        if e and "error" not in e:
            s[key] = [round(e["ms_per_step"], 4), round(e["pixel_evals_equivalent_per_s"] / 1e9, 1), round(e["workspace_GB"], 2)]
    if "f2_kmeans" in ex and "ms" in ex["f2_kmeans"]:
        s["f2_kmeans_ms"] = round(ex["f2_kmeans"]["ms"], 2)
    if "component_maps_GBps" in ex:
        s["maps_GBps"] = round(ex["component_maps_GBps"], 0)
    return s


def relaunch_multi_gpu(args):
    """python bench.py --gpus N (N > 1) without a torchrun environment: start N ranks of this script."""
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")          # communicator set-up lines: one per rank
    env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
    sys.exit(subprocess.call(cmd, env=env))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c3h")
    ap.add_argument("--batch", type=int, default=0)
    ap.add_argument("--layout", default="auto", choices=["auto", "inplace", "sorted"],
                    help="CS_OPT_LAYOUT of the headline context (default: the library's own choice)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-extras", action="store_true")
    args = ap.parse_args()
    if args.impl == "ours" and args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        relaunch_multi_gpu(args)
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    args.warmup = max(args.warmup, 3)

    import torch
    import paper_2604_08463_b200 as cs
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libcs has no CPU path")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    w, desc = make_workload(args.workload, args.batch, rank)
    t_gen = time.time()
    d_host = torch.from_numpy(w.data())
    t_gen = time.time() - t_gen
    params = w.params_jittered(seed=7)

    ctx = cs.Context(w.freqs, w.npix, options={"layout": {"auto": cs.LAYOUT_AUTO, "inplace": cs.LAYOUT_INPLACE,
                                                          "sorted": cs.LAYOUT_SORTED}[args.layout]})
    ctx.set_clusters(w.maps, w.Kmap, w.cfg_maps, w.region_idx, w.nregion)
    d_dev = d_host.to(dev)
    ctx.set_data(d_dev, w.ninv)
    torch.cuda.synchronize()
    t_batch = time.perf_counter()
    ctx.set_batch(w.cfg_of, w.data_of)          # allocates and gathers the private sorted copies (synchronous)
    torch.cuda.synchronize()
    t_batch = time.perf_counter() - t_batch
    stream = torch.cuda.current_stream()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local_rank)
    sampler.start()
    time.sleep(0.25)
    r = time_hot_path(ctx, w, params, args.steps, args.warmup, dev, stream, barrier)
    clocks = sampler.stop(r["t0"], r["t1"])
    ms, nll, grad, p_dev = r["ms"], r["nll"], r["grad"], r["p_dev"]

    ms_t = torch.tensor([ms], dtype=torch.float64, device=dev)
    if dist is not None:
        dist.all_reduce(ms_t, op=dist.ReduceOp.MAX)
    ms_max = float(ms_t.item())
    pe_step = float(w.batch) * w.npix                   # pixel-evals per step on this rank
    value = pe_step * world * args.steps / (ms_max * 1e-3)

    # roofline of the dominant kernel (fused per-pixel kernel, gradient mode): algorithmic bytes of one launch
    # (120 B x pixel-evals of the launch) over its average duration, measured live with CUDA events on its stream
    peak, peak_src = peaks()
    n_launch = max(r["kernel_launches_per_step"], 1e-9)
    k_avg_ms = r["kernel_ms_per_step"] / n_launch
    alg_bytes = BYTES_PER_PIXEL_EVAL * pe_step / n_launch
    achieved = alg_bytes / (k_avg_ms * 1e-3) / 1e9 if k_avg_ms > 0 else 0.0
    kname = kernel_name(ctx, w, w.nfreq)
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": None, "traffic_source": None, "kernel": kname, "kernel_ms": k_avg_ms,
                "kernel_launches_per_step": n_launch,
                "kernel_share_of_step": r["kernel_ms_per_step"] * args.steps / ms if ms else None,
                "peak_source": peak_src, "frac_of_8TBps_nominal": achieved / 8000.0,
                "algorithmic_bytes_per_launch": alg_bytes}
    # dram__bytes_read.sum + dram__bytes_write.sum of one launch of that kernel, from the committed ncu --set full
    # capture; only quoted when the capture was taken on this workload, batch and kernel
    traffic_file = os.path.join(ROOT, "profiles", "r02_traffic.csv")
    if os.path.exists(traffic_file):
        try:
            import csv
            with open(traffic_file) as fh:
                for row in csv.DictReader(fh):
                    if row["workload"] == args.workload and int(row["batch"]) == w.batch and row["kernel"] in kname:
                        roofline["traffic"] = int(row["dram_bytes_per_launch"])
                        roofline["traffic_source"] = f"profiles/r02_traffic.csv ({row['capture']}): one ncu --set full capture, not this run"
        except Exception:
            pass

    fills = [ctx.layout_info(int(c)) for c in np.unique(w.cfg_of)]
    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f32 (fp64 tables and reductions)", "data": "synthetic",
           "config": {"workload": desc, "nside": w.nside, "npix": w.npix, "batch_per_gpu": w.batch, "nfreq": w.nfreq,
                      "l2": "inputs larger than L2 (no flush)" if d_dev.numel() * 4 > 2 * 126e6 else "inputs fit in L2: L2-resident by design of this workload",
                      "step": "cs_build_sed_tables + cs_spectral_like_grad(value+grad); the fused kernel reads private cell-sorted "
                              "copies of d made once per data set in cs_set_batch / cs_set_data (relayout_ms_once, outside the "
                              "timed region; inside it in e2e)",
                      "datagen_s": round(t_gen, 1), "sorted_configurations": sum(1 for f in fills if f[0]),
                      "configurations": len(fills), "fill_min": min(f[2] for f in fills),
                      "relayout_ms_once": round(1e3 * t_batch, 2), "workspace_GB": ctx.workspace_bytes() / 1e9,
                      "copies_GB": copies_bytes(ctx, w) / 1e9},
           "roofline": roofline, "clocks": clocks, "gpu_launches": int(r["launches"])}

    # ---- end to end through the C ABI with host buffers (H2D of d and params, D2H of nll and grad inside); every
    #      rank runs it on its own batch, the time is the max over ranks
    if not args.no_e2e:
        d_pin = d_host.pin_memory()
        p_pin = torch.from_numpy(params).pin_memory()
        nll_pin = torch.zeros(w.batch * w.nregion, dtype=torch.float64).pin_memory()
        grad_pin = torch.zeros(params.shape[0], dtype=torch.float64).pin_memory()
        ninv_h = np.ascontiguousarray(w.ninv)
        n_e2e = max(1, min(args.steps, 3))
        ctx.eval_host(d_pin, ninv_h, p_pin, nll_pin, grad_pin)       # warm-up (allocates the staging buffer)
        barrier()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            ctx.eval_host(d_pin, ninv_h, p_pin, nll_pin, grad_pin)
        torch.cuda.synchronize()
        dt_t = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device=dev)
        if dist is not None:
            dist.all_reduce(dt_t, op=dist.ReduceOp.MAX)
        dt = float(dt_t.item())
        same = bool(np.array_equal(nll_pin.numpy(), nll.cpu().numpy()))
        out["e2e"] = {"value": pe_step * world * n_e2e / dt, "unit": UNIT,
                      "h2d_bytes_per_step": int(d_pin.numel() * 4 + p_pin.numel() * 8) * world,
                      "d2h_bytes_per_step": int(nll_pin.numel() * 8 + grad_pin.numel() * 8) * world,
                      "steps": n_e2e, "ms_per_step": 1e3 * dt / n_e2e, "bitwise_equal_to_device_path": same}
        # optimizer-shaped end to end: the data go up once (H2D + cs_set_data, which gathers the sorted copies), then K
        # steps each upload their parameters and read nll and grad back
        K_res = 20
        barrier()
        t0 = time.perf_counter()
        d_dev.copy_(d_pin, non_blocking=True)
        ctx.set_data(d_dev, w.ninv)
        for _ in range(K_res):
            p_dev.copy_(p_pin, non_blocking=True)
            ctx.build_sed_tables(p_dev, stream)
            ctx.spectral_like_grad(nll, grad, stream)
            nll_pin.copy_(nll, non_blocking=True)
            grad_pin.copy_(grad, non_blocking=True)
            torch.cuda.synchronize()
        dt_t = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device=dev)
        if dist is not None:
            dist.all_reduce(dt_t, op=dist.ReduceOp.MAX)
        dt = float(dt_t.item())
        out["e2e"]["upload_once_then_K_steps"] = {
            "value": pe_step * world * K_res / dt, "unit": UNIT, "K": K_res, "total_ms": 1e3 * dt,
            "h2d_bytes_once": int(d_pin.numel() * 4) * world,
            "h2d_bytes_per_step": int(p_pin.numel() * 8) * world,
            "d2h_bytes_per_step": int(nll_pin.numel() * 8 + grad_pin.numel() * 8) * world}
        del d_pin

    if rank == 0 and world == 1:
        # ---- parity sample + CPU baseline: the oracle on the first entries of the same workload
        if not args.no_cpu:
            nll_h = nll.cpu().numpy().reshape(w.batch, w.nregion)
            grad_h = grad.cpu().numpy()
            val, cores, n, res = oracle_sample(w, params)
            val1, cores1, n1, _ = oracle_sample(w, params, budget_s=3.0, min_entries=1, max_entries=8, threads=1)
            off = w.param_offsets()
            e_nll, e_g, blk, worst_cluster, binds = 0.0, 0.0, [0.0, 0.0, 0.0], 0.0, "relative (1e-4 sum|g_p|)"
            for e, rr in enumerate(res):
                e_nll = max(e_nll, float(np.max(np.abs(nll_h[e] - rr["nll"]) / np.abs(rr["nll"]))))
                g = grad_h[off[e]:off[e + 1]]
                dg = np.abs(g - rr["grad"])
                rel_term, floor_term = 1e-4 * rr["absg"], 1e-6 * rr["gscale"]
                ratio = dg / (rel_term + floor_term)
                if ratio.max() > e_g:
                    e_g = float(ratio.max())
                    k = int(np.argmax(ratio))
                    binds = "floor (1e-6 Gscale)" if floor_term[k] > rel_term[k] else "relative (1e-4 sum|g_p|)"
                nz = np.abs(rr["grad"]) > 0
                worst_cluster = max(worst_cluster, float(np.max(dg[nz] / np.abs(rr["grad"][nz]))))
                o = 0
                for t, kk in enumerate(w.K_of_cfg(int(w.cfg_of[e]))):
                    sl = slice(o, o + kk)
                    blk[t] = max(blk[t], float(np.linalg.norm(g[sl] - rr["grad"][sl]) / np.linalg.norm(rr["grad"][sl])))
                    o += kk
            out["cpu_baseline"] = {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle",
                                   "sample": f"first {n} entries x {w.npix} pixels of the same workload",
                                   "value_1thread": val1, "sample_1thread": f"first {n1} entries x {w.npix} pixels, {cores1} thread"}
            out["parity"] = {"entries": n, "max_rel_err_nll": e_nll,
                             "grad_block_rel_l2_beta_d": blk[0], "grad_block_rel_l2_T_d": blk[1], "grad_block_rel_l2_beta_s": blk[2],
                             "grad_block_rel_l2_unfloored (beta_d, T_d, beta_s): max ||dg||_2 / ||g_ref||_2": blk,
                             "grad_worst_cluster_rel_unfloored: max |dg_k| / |g_ref_k|": worst_cluster,
                             "max_grad_err_over_T2_bound": e_g, "T2_term_binding_at_the_worst_cluster": binds,
                             "north_star_literal_1e-4_on_block_norms_holds": bool(max(blk) <= 1e-4),
                             "pass": bool(e_nll <= 1e-5 and e_g <= 1.0)}
        # ---- extras: component maps, the one-entry configuration with its optimizer run, and every other
        #      BASELINE configuration (short runs)
        if not args.no_extras:
            nsel = min(w.batch, 256)     # 1.2 GB of maps; measured: 64 entries 4.4 TB/s, 256 entries 5.4 TB/s (longer walk per CTA)
            s = torch.empty((nsel, 3, 2, w.npix), dtype=torch.float32, device=dev)
            ent = np.arange(nsel, dtype=np.int32)
            ctx.build_sed_tables(p_dev, stream)
            ctx.component_maps(s, ent, stream)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(5):
                ctx.component_maps(s, ent, stream)
            e1.record(stream)
            torch.cuda.synchronize()
            mms = e0.elapsed_time(e1) / 5
            out["extras"] = {"component_maps_pixel_evals_per_s": nsel * w.npix / (mms * 1e-3),
                             "component_maps_GBps": nsel * w.npix * 144.0 / (mms * 1e-3) / 1e9, "component_maps_entries": nsel}
            del s
            ctx.close()
            del d_dev
            torch.cuda.empty_cache()
            # config 2 of BASELINE.json: one entry, K=(500,50,100), 200 AdaTopK iterations from (1.54, 20, -3)
            w2 = gen.make_config(1)
            c2 = cs.Context(w2.freqs, w2.npix)
            c2.set_clusters(w2.maps, w2.Kmap, w2.cfg_maps, w2.region_idx, w2.nregion)
            d2 = torch.from_numpy(w2.data()).to(dev)
            c2.set_data(d2, w2.ninv)
            c2.set_batch(w2.cfg_of, w2.data_of)
            K2 = w2.K_of_cfg(0)
            lo = torch.from_numpy(np.concatenate([np.full(K2[0], 0.5), np.full(K2[1], 8.0), np.full(K2[2], -5.0)])).to(dev)
            hi = torch.from_numpy(np.concatenate([np.full(K2[0], 3.0), np.full(K2[1], 40.0), np.full(K2[2], -1.0)])).to(dev)
            nf = torch.zeros(1, dtype=torch.float64, device=dev)
            times = []
            for _ in range(2):
                p2 = torch.from_numpy(w2.params_const()).to(dev)
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                c2.optimize(p2, lo, hi, cs.opt_defaults(iters=200), nf, stream)
                torch.cuda.synchronize()
                times.append(time.perf_counter() - t0)
            # the same problem with the L-BFGS back-end (f4(i)), 100 iterations
            p3 = torch.from_numpy(w2.params_const()).to(dev)
            nf3 = torch.zeros(1, dtype=torch.float64, device=dev)
            t_lb = []
            for _ in range(2):
                p3.copy_(torch.from_numpy(w2.params_const()).to(dev))
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                c2.optimize(p3, lo, hi, cs.opt_defaults(iters=100, method=cs.METHOD_LBFGS), nf3, stream)
                torch.cuda.synchronize()
                t_lb.append(time.perf_counter() - t0)
            n1 = torch.zeros(1, dtype=torch.float64, device=dev)
            g1 = torch.zeros_like(p2)
            e0.record(stream)
            for _ in range(20):
                c2.build_sed_tables(p2, stream)
                c2.spectral_like_grad(n1, g1, stream)
            e1.record(stream)
            torch.cuda.synchronize()
            out["extras"]["c2"] = {"workload": "C2: nside 64, K=(500,50,100), one entry",
                                   "optimize_200_iters_ms": 1e3 * min(times), "final_nll": float(nf.item()),
                                   "lbfgs_100_iters_ms": 1e3 * min(t_lb), "lbfgs_final_nll": float(nf3.item()),
                                   "like_grad_call_us": 1e3 * e0.elapsed_time(e1) / 20,
                                   "pixel_evals_per_s": w2.npix / (e0.elapsed_time(e1) / 20 * 1e-3)}
            c2.close()
            del d2
            try:   # the shape of the paper's own optimum (Table 2): beta_d per pixel, in place on the direct kernel
                out["extras"]["kmax"] = extra_workload(cs, "kmax", 256, 5, dev, stream, peak, None)[256]
            except Exception as exc:
                out["extras"]["kmax"] = {"error": repr(exc)}
            for nm, prefixes in (("c3", None), ("c4", None), ("c5", [1, 16, 64, 256])):
                try:
                    for b, res in extra_workload(cs, nm, 0, 5, dev, stream, peak, prefixes).items():
                        out["extras"][nm if prefixes is None else f"{nm}_batch{b}"] = res
                except Exception as exc:   # a failed extra must not lose the headline line
                    out["extras"][nm] = {"error": repr(exc)}
            for key, fn in (("f3_cells_c3", lambda: extra_cells(cs, "c3", 0, 5, dev, stream)),
                            ("f3_cells_c3h", lambda: extra_cells(cs, "c3h", 256, 5, dev, stream)),
                            ("f3_cells_c4", lambda: extra_cells(cs, "c4", 0, 5, dev, stream)),
                            ("f2_kmeans", lambda: extra_kmeans(cs, dev)),
                            ("cellsweep", lambda: extra_cellsweep(cs, dev, stream, peak))):
                try:
                    out["extras"][key] = fn()
                except Exception as exc:
                    out["extras"][key] = {"error": repr(exc)}
    if rank == 0:
        out["configs"] = summary_of(out, peak)     # last key on purpose
        print(json.dumps(out), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
