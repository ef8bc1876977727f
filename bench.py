#!/usr/bin/env python
"""bench.py -- pixel-evals/s of the fused -logL + gradient hot path (BASELINE.json `metric`) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload c3h|c5|c3|c2] [--batch B]

A step = one pass of the hot path over one batch: cs_build_sed_tables (a1) + cs_spectral_like_grad (a2 + a3,
value and gradient) for every batch entry.  The default workload "c3h" is the shape the metric is quoted on
("nside=64 with batch >= 1024", BASELINE.json north_star): nside 64, K = (500, 50, 100), 1024 entries each with its
own noise realisation, so that the data stream (6.04 GB per step) is larger than L2 and has to come from HBM.
Inputs are seeded and synthetic (gen/); see DESIGN.md "Input recipe".

Prints ONE JSON line (rank 0).  Keys beyond the base contract: `roofline`, `cpu_baseline`, `e2e`, `clocks`,
`gpu_launches`, `parity` (GPU vs oracle on the cpu_baseline sample), `extras`.
"""
import argparse
import json
import os
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
        desc = f"C3: nside 64 clustering scan, {B} configurations sharing one data set (L2-resident)"
    elif name == "c4":
        w = gen.make_config(3, batch=batch or None)
        desc = f"C4: nside 64, 3 latitude regions, 64 configurations x 100 noise realisations ({w.batch} entries, 100 data sets)"
    elif name == "c2":
        w = gen.make_config(1)
        desc = "C2: nside 64, K=(500,50,100), one entry"
    else:
        raise SystemExit(f"unknown workload {name}")
    if rank:
        w.realizations = tuple(r + rank * w.ndata for r in w.realizations)
    w.bytes_per_pixel_eval = BYTES_PER_PIXEL_EVAL
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
                                          "--format=csv,noheader,nounits", "-lms", "100"],
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


def oracle_sample(w, params, budget_s=12.0, min_entries=2, max_entries=64):
    """Times the oracle, as it stands, on the first entries of the workload until `budget_s` is used.
    Returns (pixel-evals/s, threads, entries, per-entry results)."""
    import oracle
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
    return n * w.npix / t_used, oracle.num_threads(), n, res


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


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c3h")
    ap.add_argument("--batch", type=int, default=0)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-extras", action="store_true")
    args = ap.parse_args()
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

    ctx = cs.Context(w.freqs, w.npix)
    ctx.set_clusters(w.maps, w.Kmap, w.cfg_maps, w.region_idx, w.nregion)
    d_dev = d_host.to(dev)
    ctx.set_data(d_dev, w.ninv)
    ctx.set_batch(w.cfg_of, w.data_of)
    p_dev = torch.from_numpy(params).to(dev)
    nll = torch.zeros(w.batch * w.nregion, dtype=torch.float64, device=dev)
    grad = torch.zeros_like(p_dev)
    stream = torch.cuda.current_stream()

    def step():
        ctx.build_sed_tables(p_dev, stream)
        ctx.spectral_like_grad(nll, grad, stream)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    if ctx.check() != 0:
        raise SystemExit("device error bit set during warm-up")

    sampler = ClockSampler(local_rank)
    sampler.start()
    time.sleep(0.25)
    ctx.profile(True)
    l0 = ctx.kernel_launches()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t0 = time.time()
    ev0.record(stream)
    for _ in range(args.steps):
        step()
    ev1.record(stream)
    barrier()
    t1 = time.time()
    ms = ev0.elapsed_time(ev1)
    launches = ctx.kernel_launches() - l0
    k_ms, k_n = ctx.profile_read()
    ctx.profile(False)
    clocks = sampler.stop(t0, t1)

    ms_t = torch.tensor([ms], dtype=torch.float64, device=dev)
    if dist is not None:
        dist.all_reduce(ms_t, op=dist.ReduceOp.MAX)
    ms_max = float(ms_t.item())
    pe_step = float(w.batch) * w.npix                   # pixel-evals per step on this rank
    value = pe_step * world * args.steps / (ms_max * 1e-3)

    # roofline of the dominant kernel (fused per-pixel kernel, gradient mode)
    peak, peak_src = peaks()
    k_avg_ms = k_ms / max(k_n, 1)
    launches_per_step = max(k_n // max(args.steps, 1), 1)
    alg_bytes = BYTES_PER_PIXEL_EVAL * pe_step / launches_per_step
    achieved = alg_bytes / (k_avg_ms * 1e-3) / 1e9 if k_n else 0.0
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": None, "kernel": "k_like_cell<15,GRAD> (fused per-pixel kernel, cell form)", "kernel_ms": k_avg_ms, "kernel_share_of_step": k_ms / ms if ms else None,
                "peak_source": peak_src, "frac_of_8TBps_nominal": achieved / 8000.0,
                "algorithmic_bytes_per_launch": alg_bytes}
    # dram__bytes_read.sum + dram__bytes_write.sum of one launch, from the committed ncu --set full capture
    # (profiles/r01_v4i_k_like_cell.md); only quoted when the capture was taken on this workload and batch
    traffic_file = os.path.join(ROOT, "profiles", "r01_v4i_traffic.csv")
    if os.path.exists(traffic_file):
        try:
            import csv
            with open(traffic_file) as fh:
                for row in csv.DictReader(fh):
                    if row["workload"] == args.workload and int(row["batch"]) == w.batch:
                        roofline["traffic"] = int(row["dram_bytes_per_launch"])
        except Exception:
            pass

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f32 (fp64 tables and reductions)", "data": "synthetic",
           "config": {"workload": desc, "nside": w.nside, "npix": w.npix, "batch_per_gpu": w.batch, "nfreq": w.nfreq,
                      "l2": "inputs larger than L2 (no flush)" if d_dev.numel() * 4 > 2 * 126e6 else "inputs fit in L2: L2-resident by design of this workload",
                      "step": "cs_build_sed_tables + cs_spectral_like_grad(value+grad)", "datagen_s": round(t_gen, 1)},
           "roofline": roofline, "clocks": clocks, "gpu_launches": int(launches)}

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
        ctx.set_data(d_dev, w.ninv)
        del d_pin

    if rank == 0 and world == 1:
        # ---- parity sample + CPU baseline: the oracle on the first entries of the same workload
        if not args.no_cpu:
            nll_h = nll.cpu().numpy().reshape(w.batch, w.nregion)
            grad_h = grad.cpu().numpy()
            val, cores, n, res = oracle_sample(w, params)
            off = w.param_offsets()
            e_nll, e_g = 0.0, 0.0
            for e, r in enumerate(res):
                e_nll = max(e_nll, float(np.max(np.abs(nll_h[e] - r["nll"]) / np.abs(r["nll"]))))
                dg = np.abs(grad_h[off[e]:off[e + 1]] - r["grad"])
                e_g = max(e_g, float(np.max(dg / (1e-4 * r["absg"] + 1e-6 * r["gscale"]))))
            out["cpu_baseline"] = {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle",
                                   "sample": f"first {n} entries x {w.npix} pixels of the same workload"}
            out["parity"] = {"entries": n, "max_rel_err_nll": e_nll, "max_grad_err_over_T2_bound": e_g,
                             "pass": bool(e_nll <= 1e-5 and e_g <= 1.0)}
        # ---- extras: component maps throughput on a subset
        if not args.no_extras:
            nsel = min(w.batch, 64)
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
            l0 = c2.kernel_launches()
            c2.build_sed_tables(p2, stream)
            n1 = torch.zeros(1, dtype=torch.float64, device=dev)
            g1 = torch.zeros_like(p2)
            e0.record(stream)
            for _ in range(20):
                c2.build_sed_tables(p2, stream)
                c2.spectral_like_grad(n1, g1, stream)
            e1.record(stream)
            torch.cuda.synchronize()
            out["extras"].update({"c2_optimize_200_iters_ms": 1e3 * min(times), "c2_final_nll": float(nf.item()),
                                  "c2_like_grad_call_us": 1e3 * e0.elapsed_time(e1) / 20})
            c2.close()
    if rank == 0:
        print(json.dumps(out), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
