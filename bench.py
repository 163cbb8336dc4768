#!/usr/bin/env python
"""bench.py -- dual-axis attention fwd+bwd ms/layer on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config base] [--impl ours|reference]

A "step" is one pass of the whole hot path: feature fwd, item fwd, item bwd,
feature bwd through the C ABI of libtabattn on one layer of seeded synthetic input (for the
12-layer Ragged config: all 12 layers, reported per layer).  One JSON line is printed by rank 0.
``--impl reference`` times the fp64 CPU oracle (oracle/) on a bounded sample of the same
workload instead; it is the only other place this file executes anything under oracle/
(besides the cpu_baseline leg at N=1).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from workloads import get_config, draw_structure, make_call_inputs  # noqa: E402

METRIC = "dual-axis attn fwd+bwd ms/layer"
UNIT = "ms/layer"
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}


# ---- algorithmic work (SURVEY.md §8(d) "Algorithmic work per unit") ----------
def algorithmic_work(cfg, n_train, col_valid):
    """flops / bytes the method must do per layer, from the seeded structure draw."""
    B, R, C, H, dh, d = cfg.B, cfg.R, cfg.C, cfg.H, cfg.dh, cfg.d
    cv = np.full(B, C) if col_valid is None else col_valid.sum(axis=1).astype(np.int64)
    nt = n_train.astype(np.int64)
    w = {}
    # feature: per valid cell fwd 8d + 4H bytes, bwd 16d + 4H; per invalid cell zero-fill 2d fwd, 6d bwd
    w["feature_fwd_bytes"] = int((cv * R * (8 * d + 4 * H) + (C - cv) * R * 2 * d).sum())
    w["feature_bwd_bytes"] = int((cv * R * (16 * d + 4 * H) + (C - cv) * R * 6 * d).sum())
    w["feature_fwd_flops"] = int((4 * cv * cv * R * d).sum())
    w["feature_bwd_flops"] = int((10 * cv * cv * R * d).sum())
    # item: per valid (b,c): flops 4/10 * R * n * d; bytes fwd (2R+2n)*2d + 4RH, bwd (3R+2n)*2d + 4RH + 3R*2d
    w["item_fwd_flops"] = int((cv * 4 * R * nt * d).sum())
    w["item_bwd_flops"] = int((cv * 10 * R * nt * d).sum())
    w["item_fwd_bytes"] = int((cv * ((2 * R + 2 * nt) * 2 * d + 4 * R * H) + (C - cv) * R * 2 * d).sum())
    w["item_bwd_bytes"] = int((cv * ((3 * R + 2 * nt) * 2 * d + 4 * R * H + 3 * R * 2 * d)
                               + (C - cv) * R * 6 * d).sum())
    return w


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return {"hbm_gbs": float(d["hbm_gbs"]), "bf16_tflops": float(d["bf16_tflops"]),
                    "bf16_tflops_sustained": float(d.get("bf16_tflops_sustained", d["bf16_tflops"])),
                    "source": "measured"}
        except Exception:
            pass
    return dict(FALLBACK_PEAKS, source="fallback")


# ---- clocks during the timed region (B200_PROFILING.md "clocks line") ------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.06)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


# ---- the oracle on a bounded sample (cpu_baseline leg and --impl reference) ------------------------
def oracle_sample_ms_per_layer(cfg, budget_s=12.0):
    """Time the fp64 oracle, as it stands, on a bounded seeded sample of one layer of ``cfg`` and
    extrapolate to ms/layer by algorithmic flops.  Returns (ms_per_layer, cores, sample_text)."""
    from oracle import ref
    n_train, col_valid = draw_structure(cfg)
    work = algorithmic_work(cfg, n_train, col_valid)
    rng = np.random.default_rng(1234 + cfg.seed)
    # sample: n_rows whole feature sequences and n_cols whole item sequences drawn from a sub-table copy
    # of the config (same R, C, H, dh, n_train, mask rule; B clipped so host generation stays small)
    sub = cfg.scaled(B=min(cfg.B, 4), projected=False)
    nt_s, cv_s = n_train[:sub.B], (col_valid[:sub.B] if col_valid is not None else None)
    feat = make_call_inputs(sub, "feature")
    item = make_call_inputs(sub, "item")
    cvn = np.full(sub.B, sub.C) if cv_s is None else cv_s.sum(axis=1)
    # calibrate with a small probe, then size the sample for ~budget_s
    def run_feature(rows):
        t = time.perf_counter()
        ref.feature_fwd(feat["Q"], feat["K"], feat["V"], cv_s, rows=rows)
        ref.feature_bwd(feat["Q"], feat["K"], feat["V"], feat["dO"], cv_s, rows=rows)
        fl = sum(14 * int(cvn[b]) ** 2 * sub.d for b, _ in rows)
        return time.perf_counter() - t, fl

    def run_item(cols):
        t = time.perf_counter()
        ref.item_fwd(item["Q"], item["K"], item["V"], nt_s, cv_s, cols=cols)
        ref.item_bwd(item["Q"], item["K"], item["V"], item["dO"], nt_s, cv_s, cols=cols)
        fl = sum(14 * sub.R * int(nt_s[b]) * sub.d for b, _ in cols)
        return time.perf_counter() - t, fl

    valid_cols = [(b, c) for b in range(sub.B) for c in range(sub.C) if cv_s is None or cv_s[b, c]]
    all_rows = [(b, r) for b in range(sub.B) for r in range(sub.R)]
    threads = ref.num_threads()
    probe_c = [valid_cols[i] for i in rng.choice(len(valid_cols), size=min(threads, len(valid_cols)), replace=False)]
    tc, fc = run_item(probe_c)
    n_cols = int(max(threads, min(len(valid_cols), (0.7 * budget_s / max(tc, 1e-6)) * len(probe_c))))
    n_cols = min(len(valid_cols), (n_cols // threads) * threads or threads)
    cols = [valid_cols[i] for i in rng.choice(len(valid_cols), size=n_cols, replace=False)]
    t_item, f_item = run_item(cols)
    probe_r = [all_rows[i] for i in rng.choice(len(all_rows), size=min(64 * threads, len(all_rows)), replace=False)]
    tr, fr = run_feature(probe_r)
    n_rows = int(min(len(all_rows), max(len(probe_r), (0.3 * budget_s / max(tr, 1e-6)) * len(probe_r))))
    rows = [all_rows[i] for i in rng.choice(len(all_rows), size=n_rows, replace=False)]
    t_feat, f_feat = run_feature(rows)
    tot_item = work["item_fwd_flops"] + work["item_bwd_flops"]
    tot_feat = work["feature_fwd_flops"] + work["feature_bwd_flops"]
    ms = 1e3 * (t_item * tot_item / max(f_item, 1) + t_feat * tot_feat / max(f_feat, 1))
    sample = ("%d whole item sequences (b,c: all heads, all %d rows) + %d whole feature rows of config '%s', "
              "fp64 oracle fwd+bwd, %.1f s measured, extrapolated to one layer by algorithmic flops "
              "(item x%.0f, feature x%.0f)" % (n_cols, sub.R, n_rows, cfg.name, t_item + t_feat,
                                               tot_item / max(f_item, 1), tot_feat / max(f_feat, 1)))
    return ms, threads, sample, (t_item + t_feat)


# ---- the reference arm: the oracle, as it stands, on the host cores ---------------------------------
def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cfg = get_config(args.config)
    vals, walls = [], []
    sample = cores = None
    budget = max(2.0, min(12.0, 100.0 / max(1, args.steps + args.warmup)))
    for i in range(args.warmup + args.steps):
        ms, cores, sample, wall = oracle_sample_ms_per_layer(cfg, budget_s=budget)
        if i >= args.warmup:
            vals.append(ms)
            walls.append(wall)
    v = float(np.mean(vals))
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": v * cfg.layers, "higher_is_better": False,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg.name, "B": cfg.B, "R": cfg.R, "C": cfg.C, "H": cfg.H, "dh": cfg.dh,
                       "layers": cfg.layers, "note": "fp64 CPU oracle on a bounded sample, extrapolated"},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ---- multi-rank host logic (replicas only): max over ranks, whole-job value -------------
def max_over_ranks(ms, world, device=None):
    """MAX of a per-rank device time over all ranks (identity when world == 1)."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(ms_per_step, layers, world):
    """ms/layer of the whole job: every rank runs one replica of the step, so N ranks finish N layers'
    worth of work per `layers` layer-times (time-like metric: lower is better)."""
    return ms_per_step / layers / world


# ---- our arm ----------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_2606_03681_b200 as tab

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; libtabattn has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)
    cfg = get_config(args.config)
    n_train_h, col_valid_h = draw_structure(cfg)
    n_train = torch.from_numpy(n_train_h).to(dev)
    col_valid = torch.from_numpy(col_valid_h).to(dev) if col_valid_h is not None else None
    work = algorithmic_work(cfg, n_train_h, col_valid_h)

    # inputs: resident in HBM before the timed region.  Every layer has its own Q,K,V,dO per axis
    # (replicas only across ranks: each rank runs the same seeded workload on its own GPU).
    x_cache = {}
    layers = []
    for l in range(cfg.layers):
        layers.append({ax: make_call_inputs(cfg, ax, l, device=dev, x_cache=x_cache) for ax in ("feature", "item")})
    x_cache.clear()
    buf = tab.LayerBuffers(cfg.B, cfg.R, cfg.C, cfg.H, cfg.dh, device=dev)
    stream = torch.cuda.current_stream()

    def step(events=None):
        # forward calls in layer order, then backward calls in reverse order would need per-layer O/LSE
        # buffers; per layer the four calls run back to back (reading c17: chained = enqueued back to back)
        for li, L in enumerate(layers):
            f, it = L["feature"], L["item"]
            if events is not None:
                events[li][0].record(stream)
            tab.tabattn_feature_fwd(f["Q"], f["K"], f["V"], col_valid, O=buf.O_f, LSE=buf.LSE_f, ws=buf.ws)
            if events is not None:
                events[li][1].record(stream)
            tab.tabattn_item_fwd(it["Q"], it["K"], it["V"], n_train, col_valid, n_train_host=n_train_h,
                                 O=buf.O_i, LSE=buf.LSE_i, ws=buf.ws)
            if events is not None:
                events[li][2].record(stream)
            tab.tabattn_item_bwd(it["Q"], it["K"], it["V"], buf.O_i, it["dO"], buf.LSE_i, n_train, col_valid,
                                 n_train_host=n_train_h, dQ=buf.grads_i[0], dK=buf.grads_i[1], dV=buf.grads_i[2],
                                 ws=buf.ws)
            if events is not None:
                events[li][3].record(stream)
            tab.tabattn_feature_bwd(f["Q"], f["K"], f["V"], buf.O_f, f["dO"], buf.LSE_f, col_valid,
                                    dQ=buf.grads_f[0], dK=buf.grads_f[1], dV=buf.grads_f[2], ws=buf.ws)
            if events is not None:
                events[li][4].record(stream)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    ev = [[[torch.cuda.Event(enable_timing=True) for _ in range(5)] for _ in layers] for _ in range(args.steps)]
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.12)
    barrier()
    launches0 = tab.launch_count()
    t0.record(stream)
    for k in range(args.steps):
        step(ev[k])
    t1.record(stream)
    barrier()
    launches = tab.launch_count() - launches0
    clocks = sampler.stop() if rank == 0 else None
    total_ms = max_over_ranks(t0.elapsed_time(t1), world, dev)
    ms_per_step = total_ms / args.steps
    # per-call device times (mean over steps and layers), from events on the launching stream
    names = ["feature_fwd", "item_fwd", "item_bwd", "feature_bwd"]
    call_ms = {n: float(np.mean([ev[k][li][i].elapsed_time(ev[k][li][i + 1])
                                 for k in range(args.steps) for li in range(len(layers))]))
               for i, n in enumerate(names)}

    # ---- end to end from pinned host buffers (layer 0), H2D + 4 calls + D2H every step ----------------
    e2e = None
    if not args.no_e2e:
        L0 = layers[0]
        host = {ax: {k: torch.empty(v.shape, dtype=v.dtype, pin_memory=True).copy_(v) for k, v in L0[ax].items()}
                for ax in ("feature", "item")}
        stage = {ax: {k: torch.empty_like(v) for k, v in L0[ax].items()} for ax in ("feature", "item")}
        out_host = [torch.empty(L0["feature"]["Q"].shape, dtype=torch.bfloat16, pin_memory=True) for _ in range(8)]
        e_steps = max(1, min(args.steps, 5))
        for _ in range(2):
            h2d, d2h = tab.layer_fwd_bwd_host(host["feature"], host["item"], stage["feature"], stage["item"],
                                              out_host, n_train, col_valid, buf, n_train_h)
        barrier()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for _ in range(e_steps):
            h2d, d2h = tab.layer_fwd_bwd_host(host["feature"], host["item"], stage["feature"], stage["item"],
                                              out_host, n_train, col_valid, buf, n_train_h)
        b.record(stream)
        barrier()
        et = max_over_ranks(a.elapsed_time(b) / e_steps, world, dev)
        e2e = {"value": job_value(et, 1, world), "unit": UNIT, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(d2h), "note": "one layer per step from pinned host buffers, pipelined over up to 16 table groups (H2D, kernels, D2H on three streams)"}
        del host, stage, out_host

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    peaks = load_peaks()
    # dominant call of the step and its roofline
    dom = max(call_ms, key=call_ms.get)
    if dom.startswith("item"):
        flops = work[dom + "_flops"]
        ach = flops / (call_ms[dom] * 1e-3) / 1e12
        peak = peaks["bf16_tflops_sustained"]
        roof = {"bound": "tensor", "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak,
                "traffic": None, "kernel": "tabattn_" + dom, "peak_source": peaks["source"] + " (sustained bf16)",
                "algorithmic_flops_per_launch": flops}
    else:
        nbytes = work[dom + "_bytes"]
        ach = nbytes / (call_ms[dom] * 1e-3) / 1e9
        peak = peaks["hbm_gbs"]
        roof = {"bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                "traffic": None, "kernel": "tabattn_" + dom, "peak_source": peaks["source"],
                "algorithmic_bytes_per_launch": nbytes}
    traffic_file = os.path.join(ROOT, "profiles", "r01_traffic.csv")   # ncu --set full DRAM bytes per call
    if os.path.exists(traffic_file):
        for row in open(traffic_file).read().splitlines()[1:]:
            f = row.split(",")
            if len(f) == 3 and f[0] == cfg.name and f[1] == dom:
                roof["traffic"] = int(f[2])
    calls = {}
    for n in names:
        ms = call_ms[n]
        calls[n] = {"ms": ms, "TFLOP/s": work[n + "_flops"] / (ms * 1e-3) / 1e12,
                    "GB/s": work[n + "_bytes"] / (ms * 1e-3) / 1e9,
                    "frac_tensor": work[n + "_flops"] / (ms * 1e-3) / 1e12 / peaks["bf16_tflops_sustained"],
                    "frac_hbm": work[n + "_bytes"] / (ms * 1e-3) / 1e9 / peaks["hbm_gbs"]}

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        ms_cpu, cores, sample, _ = oracle_sample_ms_per_layer(cfg, budget_s=args.cpu_budget)
        cpu = {"value": ms_cpu, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}

    value = job_value(ms_per_step, cfg.layers, world)
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": False, "scaling": "weak",
            "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
            "config": {"workload": cfg.name, "B": cfg.B, "R": cfg.R, "C": cfg.C, "H": cfg.H, "dh": cfg.dh,
                       "layers": cfg.layers, "n_train": [int(n_train_h.min()), int(n_train_h.max())],
                       "masked": col_valid_h is not None, "parallelism": "replicas x%d" % world,
                       "l2": "inputs larger than L2 (%.0f MB read per step); no flush"
                             % ((work["feature_fwd_bytes"] + work["item_fwd_bytes"]) / 1e6)},
            "roofline": roof, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches),
            "clocks": clocks, "calls": calls,
            "context": {"paper_l40s_baseline_min": 74.32, "paper_l40s_record_min": 0.92,
                        "note": "full-pretraining wallclock on 1x L40S (PAPER.md:L43, L51); context, not the target"}}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", default="base")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-budget", type=float, default=12.0)
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
