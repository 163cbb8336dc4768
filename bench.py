#!/usr/bin/env python
"""bench.py -- dual-axis attention fwd+bwd ms/layer on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config long_item] [--impl ours|reference]

A "step" is one pass of the whole hot path over one batch of seeded synthetic
input, enqueued as a training step would (reading c17): the forward calls (feature fwd, item fwd)
of every layer of the batch in layer order, then the backward calls (item bwd, feature bwd) in
reverse order, through the C ABI of libtabattn.  The batch holds `layers_per_step` layers: the
config's own layer count (12 for Ragged, 1 otherwise) times a repeat factor chosen so that the K
timed steps last at least --min-region seconds (a sustained-clock number); `value` is ms per
layer.  The default config is long_item, the one SURVEY.md §8(d) grades the tensor-core bar on;
the other timed configs (base, feature_heavy, ragged) are measured in the same run under
`configs`.  One JSON line is printed by rank 0.
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
NOMINAL_PEAKS = {"hbm_gbs": 8000.0, "bf16_tflops": 2250.0}     # BASELINE.json north_star's figures
SECONDARY = ("base", "feature_heavy", "ragged")               # timed beside the headline config


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
                                          "--format=csv,noheader,nounits", "-lms", "100"],
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
def oracle_sample_ms_per_layer(cfg, budget_s=12.0, nthreads=0):
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
        ref.feature_fwd(feat["Q"], feat["K"], feat["V"], cv_s, rows=rows, nthreads=nthreads)
        ref.feature_bwd(feat["Q"], feat["K"], feat["V"], feat["dO"], cv_s, rows=rows, nthreads=nthreads)
        fl = sum(14 * int(cvn[b]) ** 2 * sub.d for b, _ in rows)
        return time.perf_counter() - t, fl

    def run_item(cols):
        t = time.perf_counter()
        ref.item_fwd(item["Q"], item["K"], item["V"], nt_s, cv_s, cols=cols, nthreads=nthreads)
        ref.item_bwd(item["Q"], item["K"], item["V"], item["dO"], nt_s, cv_s, cols=cols, nthreads=nthreads)
        fl = sum(14 * sub.R * int(nt_s[b]) * sub.d for b, _ in cols)
        return time.perf_counter() - t, fl

    valid_cols = [(b, c) for b in range(sub.B) for c in range(sub.C) if cv_s is None or cv_s[b, c]]
    all_rows = [(b, r) for b in range(sub.B) for r in range(sub.R)]
    threads = nthreads if nthreads > 0 else ref.num_threads()
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
CALLS = ("feature_fwd", "item_fwd", "item_bwd", "feature_bwd")


def pick_tensor_peak(peaks, region_s):
    """Guide rule (B200_PROFILING.md): the burst bf16 figure for a kernel timed alone, the sustained one for
    a kernel timed inside a long step.  A timed region of >= 1 s is 'long'."""
    if region_s >= 1.0:
        return peaks["bf16_tflops_sustained"], "sustained"
    return peaks["bf16_tflops"], "burst"


def call_table(call_ms, work, peaks, region_s):
    tpeak, tkind = pick_tensor_peak(peaks, region_s)
    out = {}
    for n in CALLS:
        ms = call_ms[n]
        tf = work[n + "_flops"] / (ms * 1e-3) / 1e12
        gb = work[n + "_bytes"] / (ms * 1e-3) / 1e9
        out[n] = {"ms": ms, "TFLOP/s": tf, "GB/s": gb,
                  "frac_tensor": tf / tpeak, "frac_tensor_kind": tkind,
                  "frac_tensor_sustained": tf / peaks["bf16_tflops_sustained"],
                  "frac_tensor_burst": tf / peaks["bf16_tflops"],
                  "frac_tensor_nominal": tf / NOMINAL_PEAKS["bf16_tflops"],
                  "frac_hbm": gb / peaks["hbm_gbs"], "frac_hbm_nominal": gb / NOMINAL_PEAKS["hbm_gbs"]}
    return out


class Workload:
    """One config resident in HBM: per-layer inputs, per-layer forward outputs (the backward of layer l
    reads its own O/LSE, reading c17), shared gradient buffers and workspace."""

    def __init__(self, torch, tab, cfg, dev):
        self.torch, self.tab, self.cfg = torch, tab, cfg
        self.n_train_h, self.col_valid_h = draw_structure(cfg)
        self.n_train = torch.from_numpy(self.n_train_h).to(dev)
        self.col_valid = torch.from_numpy(self.col_valid_h).to(dev) if self.col_valid_h is not None else None
        self.work = algorithmic_work(cfg, self.n_train_h, self.col_valid_h)
        x_cache = {}
        self.layers = [{ax: make_call_inputs(cfg, ax, l, device=dev, x_cache=x_cache) for ax in ("feature", "item")}
                       for l in range(cfg.layers)]
        x_cache.clear()
        shp = (cfg.B, cfg.R, cfg.C, cfg.H, cfg.dh)
        bf = dict(dtype=torch.bfloat16, device=dev)
        f32 = dict(dtype=torch.float32, device=dev)
        self.fwd = [{"O_f": torch.empty(shp, **bf), "O_i": torch.empty(shp, **bf),
                     "LSE_f": torch.empty((cfg.B, cfg.R, cfg.H, cfg.C), **f32),
                     "LSE_i": torch.empty((cfg.B, cfg.C, cfg.H, cfg.R), **f32)} for _ in range(cfg.layers)]
        self.buf = tab.LayerBuffers(cfg.B, cfg.R, cfg.C, cfg.H, cfg.dh, device=dev)   # gradients + workspace
        self.stream = torch.cuda.current_stream()
        self.reps = 1

    @property
    def calls_per_step(self):
        return 4 * self.cfg.layers * self.reps

    def names_in_order(self):
        one = ["feature_fwd", "item_fwd"] * self.cfg.layers + ["item_bwd", "feature_bwd"] * self.cfg.layers
        return one * self.reps

    def step(self, events=None):
        tab, buf, nt, cv, nth = self.tab, self.buf, self.n_train, self.col_valid, self.n_train_h
        i = 0

        def rec():
            nonlocal i
            if events is not None:
                events[i].record(self.stream)
                i += 1
        rec()
        for _ in range(self.reps):
            for L, F in zip(self.layers, self.fwd):
                f, it = L["feature"], L["item"]
                tab.tabattn_feature_fwd(f["Q"], f["K"], f["V"], cv, O=F["O_f"], LSE=F["LSE_f"], ws=buf.ws)
                rec()
                tab.tabattn_item_fwd(it["Q"], it["K"], it["V"], nt, cv, n_train_host=nth, O=F["O_i"],
                                     LSE=F["LSE_i"], ws=buf.ws)
                rec()
            for L, F in zip(reversed(self.layers), reversed(self.fwd)):
                f, it = L["feature"], L["item"]
                tab.tabattn_item_bwd(it["Q"], it["K"], it["V"], F["O_i"], it["dO"], F["LSE_i"], nt, cv,
                                     n_train_host=nth, dQ=buf.grads_i[0], dK=buf.grads_i[1], dV=buf.grads_i[2],
                                     ws=buf.ws)
                rec()
                tab.tabattn_feature_bwd(f["Q"], f["K"], f["V"], F["O_f"], f["dO"], F["LSE_f"], cv,
                                        dQ=buf.grads_f[0], dK=buf.grads_f[1], dV=buf.grads_f[2], ws=buf.ws)
                rec()


def time_workload(torch, dist, tab, wl, steps, warmup, min_region_s, world, rank, local, dev):
    """W warm-up steps, then exactly K timed steps bracketed by barrier + synchronize; device time from
    CUDA events on the launching stream, max over ranks.  Returns the measurement dict."""
    cfg = wl.cfg

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # calibration (untimed): size the step so that K steps last >= min_region_s
    wl.reps = 1
    wl.step()
    barrier()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(wl.stream)
    wl.step()
    b.record(wl.stream)
    barrier()
    est = max_over_ranks(a.elapsed_time(b), world, dev)
    wl.reps = int(max(1, min(256, -(-min_region_s * 1e3 // max(steps * est, 1e-3)))))
    for _ in range(warmup):
        wl.step()
    barrier()
    n_ev = wl.calls_per_step + 1
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(n_ev)] for _ in range(steps)]
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    barrier()
    launches0 = tab.launch_count()
    t0.record(wl.stream)
    for k in range(steps):
        wl.step(ev[k])
    t1.record(wl.stream)
    barrier()
    launches = tab.launch_count() - launches0
    clocks = sampler.stop() if rank == 0 else None
    total_ms = max_over_ranks(t0.elapsed_time(t1), world, dev)
    names = wl.names_in_order()
    acc = {n: [] for n in CALLS}
    for k in range(steps):
        for i, n in enumerate(names):
            acc[n].append(ev[k][i].elapsed_time(ev[k][i + 1]))
    call_ms = {n: float(np.mean(v)) for n, v in acc.items()}
    layers_per_step = cfg.layers * wl.reps
    return {"total_ms": total_ms, "ms_per_step": total_ms / steps, "layers_per_step": layers_per_step,
            "ms_per_layer": total_ms / steps / layers_per_step, "region_s": total_ms * 1e-3,
            "call_ms": call_ms, "launches": int(launches), "clocks": clocks}


# ---- the rows SURVEY.md §8(f) marks "next": evaluation path, sub-blocks, Newton-Schulz ------------------------------
def _timeit(torch, stream, fn, iters, warmup=3):
    for _ in range(warmup):
        fn()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    a.record(stream)
    for _ in range(iters):
        fn()
    b.record(stream)
    torch.cuda.synchronize()
    return a.elapsed_time(b) / iters


def time_next_rows(torch, tab, dev, peaks, iters=20):
    """Device times of the §8(f) rows on seeded synthetic inputs resident in HBM (inputs larger than L2 except
    Newton-Schulz, which is launch-bound and says so).  Algorithmic work per DESIGN.md §5.2."""
    out = {}
    stream = torch.cuda.current_stream()
    g = torch.Generator(device=dev)
    g.manual_seed(1234)
    bf = torch.bfloat16

    def rnd(*shape, scale=1.0):
        return (torch.randn(*shape, generator=g, device=dev, dtype=torch.float32) * scale).to(bf)

    # (f)-2 evaluation path: PAPER.md:L65 table (24 thinking + 800 train + 200 test rows, 100 features + target),
    # record width (256, 4 heads); five folds batched.  Whole block (all rows) and last block (test rows only).
    B, R, C, H, dh, n = 5, 1024, 101, 4, 64, 824
    d = H * dh
    Q, K, V = (rnd(B, R, C, H, dh) for _ in range(3))
    O = torch.empty_like(Q)
    nt = torch.full((B,), n, dtype=torch.int32, device=dev)
    ev = {}
    for name, r0, r1 in (("all_rows", 0, R), ("test_rows", n, R)):
        tf = _timeit(torch, stream, lambda: tab.tabattn_feature_fwd_infer(Q, K, V, r0, r1, O=O), iters)
        ti = _timeit(torch, stream, lambda: tab.tabattn_item_fwd_infer(Q, K, V, nt, r0, r1, O=O), iters)
        rows = r1 - r0
        fb = B * rows * C * 8 * d                       # Q, K, V in, O out (no LSE)
        ifl = 4 * B * C * rows * n * d
        ib = B * C * (2 * rows + 2 * n) * 2 * d
        ev[name] = {"feature_fwd_infer": {"ms": tf, "GB/s": fb / tf / 1e6, "frac_hbm": fb / tf / 1e6 / peaks["hbm_gbs"]},
                    "item_fwd_infer": {"ms": ti, "TFLOP/s": ifl / ti / 1e9, "GB/s": ib / ti / 1e6,
                                       "frac_tensor_burst": ifl / ti / 1e9 / peaks["bf16_tflops"]}}
    out["eval_1000x100"] = {"shape": {"B": B, "R": R, "C": C, "H": H, "dh": dh, "n_train": n}, **ev}
    del Q, K, V, O
    torch.cuda.empty_cache()

    # (f)-1 / (f)-3 sub-blocks on the long_item table shape (cells = 8 x 4096 x 21, e = 256, hidden = 768)
    cfg = get_config("long_item")
    B, R, C, H, dh = cfg.B, cfg.R, cfg.C, cfg.H, cfg.dh
    e, hid, cells, alpha = H * dh, 768, cfg.B * cfg.R * cfg.C, 0.95
    x, dy = rnd(B, R, C, e), rnd(B, R, C, e)
    gain = (1 + 0.1 * torch.randn(e, generator=g, device=dev)).to(bf)
    Wqkv, Wo = rnd(3 * e, e, scale=e ** -0.5), rnd(e, e, scale=e ** -0.5)
    W1, W2 = rnd(hid, e, scale=e ** -0.5), rnd(e, hid, scale=hid ** -0.5)
    nt = torch.full((B,), cfg.n_train, dtype=torch.int32, device=dev)
    blocks = {}
    for axis, nm in ((0, "feature"), (1, "item")):
        y, sv = tab.tabattn_attn_block_fwd(axis, x, gain, Wqkv, Wo, H, nt, None, alpha)
        wsf = torch.empty(int(tab.lib().tabattn_attn_block_workspace_bytes(
            __import__("ctypes").byref(tab.make_shape(x.view(B, R, C, H, dh), nt)[0]), axis, 1)), dtype=torch.uint8, device=dev)
        tfw = _timeit(torch, stream, lambda: tab.tabattn_attn_block_fwd(axis, x, gain, Wqkv, Wo, H, nt, None, alpha,
                                                                        saved=sv, y=y), iters)
        tbw = _timeit(torch, stream, lambda: tab.tabattn_attn_block_bwd(axis, x, gain, Wqkv, Wo, H, sv, dy, nt, None,
                                                                        alpha, ws=wsf), iters)
        proj_f, proj_b = 8 * cells * e * e, 16 * cells * e * e       # QKV + out projections: 4 e^2 MACs / cell fwd
        att_f = 4 * cells * (C if axis == 0 else cfg.n_train) * e
        att_b = 10 * cells * (C if axis == 0 else cfg.n_train) * e
        blocks["attn_block_" + nm] = {"fwd_ms": tfw, "bwd_ms": tbw,
                                      "fwd_TFLOP/s": (proj_f + att_f) / tfw / 1e9,
                                      "bwd_TFLOP/s": (proj_b + att_b) / tbw / 1e9}
        del sv, wsf, y
    y, sv = tab.tabattn_mlp_fwd(x, gain, W1, W2, alpha)
    wsm = torch.empty(int(tab.lib().tabattn_mlp_workspace_bytes(cells, e, hid)), dtype=torch.uint8, device=dev)
    tfw = _timeit(torch, stream, lambda: tab.tabattn_mlp_fwd(x, gain, W1, W2, alpha, saved=sv, y=y), iters)
    tbw = _timeit(torch, stream, lambda: tab.tabattn_mlp_bwd(x, gain, W1, W2, sv, dy, alpha, ws=wsm), iters)
    ff, fbw = 4 * cells * e * hid, 8 * cells * e * hid
    bytes_f, bytes_b = cells * (4 * e + 2 * hid), cells * (6 * e + 2 * hid)   # x, y, saved u | x, dy, u, dx
    blocks["mlp_block"] = {"fwd_ms": tfw, "bwd_ms": tbw, "fwd_TFLOP/s": ff / tfw / 1e9, "bwd_TFLOP/s": fbw / tbw / 1e9,
                           "fwd_frac_tensor_burst": ff / tfw / 1e9 / peaks["bf16_tflops"],
                           "bwd_frac_tensor_burst": fbw / tbw / 1e9 / peaks["bf16_tflops"],
                           "fwd_frac_hbm": bytes_f / tfw / 1e6 / peaks["hbm_gbs"],
                           "bwd_frac_hbm": bytes_b / tbw / 1e6 / peaks["hbm_gbs"]}
    out["blocks_long_item_shape"] = {"cells": cells, "e": e, "hidden": hid, **blocks}
    del x, dy, y, sv, wsm
    torch.cuda.empty_cache()

    # (f)-4 batched Newton-Schulz over the QKV matrices of the record model: 5 blocks x 2 attentions x 3
    nb, m = 30, 256
    G = rnd(nb, m, m, scale=0.02)
    X = torch.empty_like(G)
    wsn = torch.empty(int(tab.lib().tabattn_newton_schulz_workspace_bytes(nb, m, m)), dtype=torch.uint8, device=dev)
    tns = _timeit(torch, stream, lambda: tab.tabattn_newton_schulz(G, 5, X=X, ws=wsn), iters)
    fl = nb * 5 * 6 * m ** 3
    # the same call captured in a CUDA graph (it allocates nothing): what the 16 launches cost without the host
    side = torch.cuda.Stream()
    side.wait_stream(stream)
    with torch.cuda.stream(side):
        gr = torch.cuda.CUDAGraph()
        with torch.cuda.graph(gr, stream=side):
            tab.tabattn_newton_schulz(G, 5, X=X, ws=wsn)
    stream.wait_stream(side)
    tng = _timeit(torch, stream, gr.replay, iters)
    out["newton_schulz"] = {"nb": nb, "m": m, "n": m, "steps": 5, "ms": tns, "TFLOP/s": fl / tns / 1e9,
                            "graph_ms": tng, "graph_TFLOP/s": fl / tng / 1e9,
                            "launches": 16, "note": "30 matrices of 256x256 (3.9 MB): L2-resident and launch-bound"}
    out["tiny_layer"] = time_tiny_layer(torch, tab, dev, iters=50 * iters)
    return out


def time_tiny_layer(torch, tab, dev, iters=1000):
    """configs[0] (Tiny, 2 x 64 x 6 cells) is launch-bound: one layer through the four ctypes calls against the same
    four calls captured in a CUDA graph (tab.LayerGraph) and replayed.  Not a throughput claim: host overhead."""
    from workloads import get_config, draw_structure, make_call_inputs
    cfg = get_config("tiny")
    nt_h, cv_h = draw_structure(cfg)
    nt = torch.from_numpy(nt_h).to(dev)
    cv = torch.from_numpy(cv_h).to(dev) if cv_h is not None else None
    feat = make_call_inputs(cfg, "feature", 0, device=dev)
    item = make_call_inputs(cfg, "item", 0, device=dev)
    buf = tab.LayerBuffers(cfg.B, cfg.R, cfg.C, cfg.H, cfg.dh, device=dev)
    stream = torch.cuda.current_stream()
    direct = _timeit(torch, stream, lambda: tab.layer_fwd_bwd(feat, item, nt, cv, buf, n_train_host=nt_h), iters, 20)
    graph = tab.LayerGraph(feat, item, nt, cv, buf, n_train_host=nt_h)
    replay = _timeit(torch, stream, graph.replay, iters, 20)
    return {"workload": "tiny", "direct_us_per_layer": direct * 1e3, "graph_us_per_layer": replay * 1e3,
            "kernels_per_replay": graph.kernels_per_replay,
            "note": "launch-bound: the direct figure is the host cost of four ctypes calls, the graph figure one replay"}


def static_traffic(cfg_name, call):
    """DRAM bytes (read + write) of one C-ABI call from the committed ncu --set full capture
    (profiles/r02_traffic.csv; falls back to round 1's).  A static capture, not measured in this run."""
    for fn in ("r02_traffic.csv", "r01_traffic.csv"):
        path = os.path.join(ROOT, "profiles", fn)
        if not os.path.exists(path):
            continue
        for row in open(path).read().splitlines()[1:]:
            f = row.split(",")
            if len(f) >= 3 and f[0] == cfg_name and f[1] == call:
                return int(f[2]), "profiles/" + fn + " (static ncu --set full capture, per call)"
    return None, None


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
    peaks = load_peaks()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    if args.only_next_rows:
        # profiling helper: only the SURVEY.md §8(f) rows, few iterations (ncu captures of the GEMM / norm kernels)
        print(json.dumps({"next_rows": time_next_rows(torch, tab, dev, peaks, iters=args.steps)}))
        return 0

    # ---- headline config: inputs resident in HBM before the timed region (replicas only across ranks:
    # each rank runs the same seeded workload on its own GPU)
    cfg = get_config(args.config)
    if args.layers > 0:
        cfg = cfg.scaled(layers=min(cfg.layers, args.layers))   # profiling runs: fewer layers resident
    wl = Workload(torch, tab, cfg, dev)
    m = time_workload(torch, dist, tab, wl, args.steps, args.warmup, args.min_region, world, rank, local, dev)
    work, call_ms = wl.work, m["call_ms"]

    # ---- end to end from pinned host buffers (layer 0), H2D + 4 calls + D2H every step ----------------
    e2e = None
    if not args.no_e2e:
        L0 = wl.layers[0]
        host = {ax: {k: torch.empty(v.shape, dtype=v.dtype, pin_memory=True).copy_(v) for k, v in L0[ax].items()}
                for ax in ("feature", "item")}
        stage = {ax: {k: torch.empty_like(v) for k, v in L0[ax].items()} for ax in ("feature", "item")}
        out_host = [torch.empty(L0["feature"]["Q"].shape, dtype=torch.bfloat16, pin_memory=True) for _ in range(8)]
        e_steps = max(1, min(args.steps, 5))
        for _ in range(2):
            h2d, d2h = tab.layer_fwd_bwd_host(host["feature"], host["item"], stage["feature"], stage["item"],
                                              out_host, wl.n_train, wl.col_valid, wl.buf, wl.n_train_h)
        barrier()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(wl.stream)
        for _ in range(e_steps):
            h2d, d2h = tab.layer_fwd_bwd_host(host["feature"], host["item"], stage["feature"], stage["item"],
                                              out_host, wl.n_train, wl.col_valid, wl.buf, wl.n_train_h)
        b.record(wl.stream)
        barrier()
        et = max_over_ranks(a.elapsed_time(b) / e_steps, world, dev)
        e2e = {"value": job_value(et, 1, world), "unit": UNIT, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(d2h), "steps": e_steps,
               "note": "one layer per step through layer_fwd_bwd_host (the public API) from pinned host buffers, "
                       "pipelined over up to 16 table groups (H2D, kernels, D2H on three streams); PCIe-bound"}
        del host, stage, out_host
    n_train_h, col_valid_h = wl.n_train_h, wl.col_valid_h
    del wl
    torch.cuda.empty_cache()

    # ---- the other timed configs, same protocol, same run (single GPU only) ----------------------------
    others = {}
    if world == 1 and not args.no_extra:
        for name in SECONDARY:
            if name == cfg.name:
                continue
            c2 = get_config(name)
            w2 = Workload(torch, tab, c2, dev)
            m2 = time_workload(torch, dist, tab, w2, args.steps, args.warmup, args.min_region, world, rank, local, dev)
            others[name] = {"ms_per_layer": m2["ms_per_layer"], "ms_per_step": m2["ms_per_step"], "steps": args.steps,
                            "layers_per_step": m2["layers_per_step"], "timed_region_s": m2["region_s"],
                            "gpu_launches": m2["launches"], "clocks": m2["clocks"],
                            "calls": call_table(m2["call_ms"], w2.work, peaks, m2["region_s"])}
            del w2
            torch.cuda.empty_cache()

    next_rows = None
    if world == 1 and not args.no_extra:
        next_rows = time_next_rows(torch, tab, dev, peaks)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant call of the headline step -----------
    dom = max(call_ms, key=call_ms.get)
    region_s = m["region_s"]
    if dom.startswith("item"):
        flops = work[dom + "_flops"]
        ach = flops / (call_ms[dom] * 1e-3) / 1e12
        peak, kind = pick_tensor_peak(peaks, region_s)
        roof = {"bound": "tensor", "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak,
                "peak_kind": "%s bf16 %s (timed region %.2f s)" % (peaks["source"], kind, region_s),
                "frac_vs": {"measured_sustained": ach / peaks["bf16_tflops_sustained"],
                            "measured_burst": ach / peaks["bf16_tflops"],
                            "nominal_2.25PF": ach / NOMINAL_PEAKS["bf16_tflops"]},
                "kernel": "tabattn_" + dom, "algorithmic_flops_per_launch": flops}
    else:
        nbytes = work[dom + "_bytes"]
        ach = nbytes / (call_ms[dom] * 1e-3) / 1e9
        peak = peaks["hbm_gbs"]
        roof = {"bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                "peak_kind": "%s copy bandwidth" % peaks["source"],
                "frac_vs": {"measured_copy": ach / peak, "nominal_8TBs": ach / NOMINAL_PEAKS["hbm_gbs"]},
                "kernel": "tabattn_" + dom, "algorithmic_bytes_per_launch": nbytes}
    roof["traffic"], roof["traffic_source"] = static_traffic(cfg.name, dom)

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        ms_cpu, cores, sample, _ = oracle_sample_ms_per_layer(cfg, budget_s=args.cpu_budget)
        cpu = {"value": ms_cpu, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}
        ms_1, _, sample_1, _ = oracle_sample_ms_per_layer(cfg, budget_s=args.cpu_budget, nthreads=1)
        cpu["one_core"] = {"value": ms_1, "unit": UNIT, "cores": 1, "sample": sample_1}

    value = job_value(m["ms_per_step"], m["layers_per_step"], world)
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": m["ms_per_step"], "higher_is_better": False, "scaling": "weak",
            "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
            "config": {"workload": cfg.name, "B": cfg.B, "R": cfg.R, "C": cfg.C, "H": cfg.H, "dh": cfg.dh,
                       "layers": cfg.layers, "layers_per_step": m["layers_per_step"],
                       "timed_region_s": region_s,
                       "n_train": [int(n_train_h.min()), int(n_train_h.max())],
                       "masked": col_valid_h is not None, "parallelism": "replicas x%d" % world,
                       "order": "forward calls of all layers of the step in layer order, then backward calls in "
                                "reverse (reading c17); the step repeats the config's layers until K steps last "
                                ">= %.1f s" % args.min_region,
                       "l2": "inputs larger than L2 (%.0f MB read per layer); no flush"
                             % ((work["feature_fwd_bytes"] + work["item_fwd_bytes"]) / 1e6)},
            "roofline": roof, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": m["launches"],
            "clocks": m["clocks"], "calls": call_table(call_ms, work, peaks, region_s), "configs": others,
            "next_rows": next_rows,
            "peaks": {k: peaks[k] for k in ("hbm_gbs", "bf16_tflops", "bf16_tflops_sustained", "source")},
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
    ap.add_argument("--config", default="long_item")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--min-region", type=float, default=3.0, help="seconds the K timed steps must last at least")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="skip the secondary configs")
    ap.add_argument("--cpu-budget", type=float, default=10.0)
    ap.add_argument("--only-next-rows", action="store_true",
                    help="time only the SURVEY §8(f) rows (evaluation path, sub-blocks, Newton-Schulz)")
    ap.add_argument("--layers", type=int, default=0,
                    help="keep only the first L layers of the config resident (ncu captures of ragged)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
