#!/usr/bin/env python
"""bench.py -- the one measurement entry point: MoE-layer decode step time and achieved HBM bandwidth.

  python bench.py [--config 2|3|4|5|prefill|route|mxfp4|fit|gemv] [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
  python bench.py --timeline T:U[,U...]          in-kernel timeline of the fused step (markdown; -DELDR_TRACE build)

A "step" is ONE layer-step = one eldr_moe_decode_layer call: gate GEMV -> softmax top-k + signature accumulation ->
permutation / union compaction -> grouped SwiGLU FFN over the ACTIVE experts -> weighted combine.  Every config
prints ONE JSON line with the same schema.  `value` = algorithmic bytes of the timed steps / device time (CUDA
events, max over ranks); algorithmic bytes per step = (|U| + n_shared) * 3*H*I*2 + activations (x, Wg, out,
ids/weights)  [SURVEY.md 8(d), DESIGN.md 6].  Seeded synthetic inputs (paper_2607_00466_b200/synth.py) stand in for
the paper's models and prompts.

  --config 2 (default; BASELINE.json configs[1], the configuration the metric is quoted on): Qwen3-30B-A3B-shaped
             layer (H=2048, E=128, top-8, I=768, bf16), T=64, gate biased so |U| = 16, 32, 64, 96, 128; K steps per
             union size; union-scaling fit t = a + b*|U|.  L2 defeated by 4 rotating weight copies.
  --config 3 same layer, |U| = 32, T = 1, 8, 32, 128, 256; batch flatness (max-min)/median over T = 8..256.
  --config 4 48-layer stack of such layers (58 GB resident), T = 128, clustered hiddens, cluster-aligned gates:
             single-cluster vs mixed batches; per-layer time, 48-layer stack time, realised unions.
  --config 5 27 layers x (64 routed top-6 + 2 shared experts), I = 1408, T = 256; plus the prefill-shaped signature
             accumulation (32 requests, prompts 512-4096, 16-token KV blocks).
  --config prefill / route / mxfp4 / fit: the SURVEY.md 8(f) rows (prefill-shaped layer, routing decision, MXFP4 experts,
             offline fit -- the last one is host code and needs no GPU).
N > 1: independent replicas, one per GPU (the path does not shard: SURVEY.md 8(e)), launched by torchrun.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

UNIONS = (16, 32, 64, 96, 128)
C3_BATCHES = (1, 8, 32, 128, 256)
N_COPIES = 4
METRIC = "moe_layer_decode_algorithmic_hbm_bandwidth_over_union_sweep"
NOMINAL_HBM_GBS = 8000.0


def algorithmic_bytes(shape, T, n_active, expert_bytes=None):
    H, I, E, k = shape.hidden, shape.inter, shape.n_experts, shape.top_k
    per_expert = 3 * H * I * 2 if expert_bytes is None else expert_bytes
    return (n_active + shape.n_shared) * per_expert + T * H * 2 + E * H * 4 + T * H * 2 + T * k * 8


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            j = json.load(f)
        return j, "measured"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}, "fallback"


class ClockSampler(threading.Thread):
    """Samples SM clock + throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.samples, self.reasons, self.max_mhz = index, False, [], set(), None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "sw_thermal_slowdown": 0x20,
                 "hw_thermal_slowdown": 0x40, "hw_power_brake": 0x80}
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for n, bit in names.items():
                    if r & bit:
                        self.reasons.add(n)
            except Exception:
                pass
            time.sleep(0.005)

    def summary(self):
        s = sorted(self.samples)
        return {"sm_mhz": (s[len(s) // 2] if s else None), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s)}


def ncu_traffic(unions):
    """dram__bytes_read.sum + dram__bytes_write.sum of moe_fused_kernel per launch, READ FROM THE COMMITTED SUMMARY of
    one `ncu --set full` capture per union size (profiles/r2_fused_full.csv, else r1; command in the .md beside it) --
    it is not measured in this run.  Averaged over the sweep's union sizes like `achieved`; None if a size is missing."""
    for name in ("r2_fused_full.csv", "r1_fused_full.csv"):
        path = os.path.join(ROOT, "profiles", name)
        try:
            import csv
            rows = {int(float(r["union"])): float(r["dram__bytes_read.sum"]) + float(r["dram__bytes_write.sum"])
                    for r in csv.DictReader(open(path))}
            per = {u: rows[u] for u in unions}
            return round(sum(per.values()) / len(per)), {str(u): round(v) for u, v in per.items()}, "profiles/" + name
        except Exception:
            continue
    return None, None, None


# ------------------------------------------------------------------------------------------------ workloads
class Case:
    """One input batch and the layer(s) it runs through.  `layers` is a list of dicts with gate_w, w13, w2,
    shared_w13, shared_w2, layer (signature row); step i runs layers[i % len(layers)]."""

    def __init__(self, label, shape, T, x_bits, bias, layers, maps=True, **extra):
        import torch
        from paper_2607_00466_b200 import api, synth
        self.label, self.shape, self.T, self.layers, self.extra = label, shape, T, layers, extra
        self.x_bits, self.bias_np = x_bits, bias
        self.x = api.bf16_from_bits(x_bits)
        self.h_x = api.bf16_from_bits(x_bits, device=None).pin_memory()
        self.bias = torch.from_numpy(bias).cuda() if bias is not None else None
        req, blk = synth.decode_maps(T)
        self.req = torch.from_numpy(req).cuda() if maps else None
        self.blk = torch.from_numpy(blk).cuda() if maps else None
        self.h_req = torch.from_numpy(req).pin_memory() if maps else None
        self.h_blk = torch.from_numpy(blk).pin_memory() if maps else None
        self.n_active = [None] * len(layers)


def device_weights(shape, n_layers, seed):
    """n_layers weight sets drawn ON the device (seeded torch generator, N(0,0.02) -> bf16): the stacks hold 58 / 31 GB.
    They are compared with nothing but their own byte counts (parity of the same shapes: tests/test_gpu_parity.py)."""
    import torch
    g = torch.Generator(device="cuda")
    g.manual_seed(seed)
    H, I, E, ns = shape.hidden, shape.inter, shape.n_experts, shape.n_shared

    def draw(*dims):
        t = torch.empty(dims, dtype=torch.bfloat16, device="cuda")
        for e in range(dims[0]):                       # expert by expert: the fp32 temporary stays small
            t[e] = (torch.randn(dims[1:], generator=g, device="cuda", dtype=torch.float32) * 0.02).to(torch.bfloat16)
        return t
    return [(draw(E, 2 * I, H), draw(E, H, I), draw(ns, 2 * I, H) if ns else None, draw(ns, H, I) if ns else None)
            for _ in range(n_layers)]


def make_cases(config):
    """-> (shape, cases, host_weights_of_layer0, description).  layer 0 always comes from synth (host bits), so the CPU
    oracle can be timed -- and the GPU spot-checked -- on exactly the benchmarked inputs."""
    import torch
    from paper_2607_00466_b200 import api, synth
    if config in ("2", "3"):
        shape = synth.SHAPE_QWEN
        lw = synth.make_layer_weights(shape, synth.WEIGHT_SEED)
        gate = torch.from_numpy(lw.gate_w).cuda()
        w13, w2 = api.bf16_from_bits(lw.w13), api.bf16_from_bits(lw.w2)
        layers = [dict(gate_w=gate, w13=w13, w2=w2, shared_w13=None, shared_w2=None, layer=0)]
        layers += [dict(gate_w=gate, w13=w13.clone(), w2=w2.clone(), shared_w13=None, shared_w2=None, layer=0)
                   for _ in range(N_COPIES - 1)]
        points = [(64, u) for u in UNIONS] if config == "2" else [(T, 32) for T in C3_BATCHES]
        cases = []
        for T, u in points:
            seed = synth.accepted_union_seed(T, u)
            xb, bias = synth.union_case(shape, T, u, seed)
            cases.append(Case("T=%d,u=%d" % (T, u), shape, T, xb, bias, layers, seed=seed, u=u))
        what = ("configs[1]: Qwen3-30B-A3B-shaped MoE layer H=2048 E=128 top-8 I=768, T=64 decode tokens, gate-biased union "
                "sweep |U|=16,32,64,96,128; K steps per union size" if config == "2" else
                "configs[2]: same layer, gate-biased union 32 (8 at T=1), batch sweep T=1,8,32,128,256; K steps per batch size")
        return shape, cases, lw, dict(workload=what, l2="rotating %d weight copies (>=450 MB streamed between reuses; L2 ~126 MB)" % N_COPIES)
    if config == "4":
        shape, L, T = synth.SHAPE_QWEN48, 48, 128
        lw = synth.make_layer_weights(shape, 4, layer=0)
        cent = synth.c4_centroids(shape.hidden, 4)
        lw.gate_w = synth.c4_gate(shape, cent, 4, 0, alpha=0.2)
        dev = device_weights(shape, L - 1, 44)
        layers = [dict(gate_w=torch.from_numpy(lw.gate_w).cuda(), w13=api.bf16_from_bits(lw.w13), w2=api.bf16_from_bits(lw.w2),
                       shared_w13=None, shared_w2=None, layer=0)]
        for l in range(1, L):
            layers.append(dict(gate_w=torch.from_numpy(synth.c4_gate(shape, cent, 4, l, alpha=0.2)).cuda(), w13=dev[l - 1][0],
                               w2=dev[l - 1][1], shared_w13=None, shared_w2=None, layer=l))
        cases = []
        for mode in ("single", "mixed"):
            for b in range(4):
                cl = synth.c4_cluster_assignment(T, mode, step=b, seed=4)
                cases.append(Case("%s,batch=%d" % (mode, b), shape, T, synth.c4_hidden(T, cent, cl, seed=40 + b), None, layers, mode=mode))
        return shape, cases, lw, dict(workload="configs[3]: 48-layer stack of Qwen3-30B-A3B-shaped MoE layers (attention omitted; every layer "
                                      "gets the batch hiddens), T=128, 8 cluster centroids sigma=0.3, gate rows aligned (alpha=0.2); 4 single-"
                                      "cluster and 4 mixed batches; a step = one layer-step, K steps rotate through the 48 layers",
                                      l2="48 distinct layers (58 GB resident)")
    if config == "5":
        shape, L, T = synth.SHAPE_C5, 27, 256
        lw = synth.make_layer_weights(shape, 5, layer=0)
        dev = device_weights(shape, L - 1, 55)
        layers = [dict(gate_w=torch.from_numpy(lw.gate_w).cuda(), w13=api.bf16_from_bits(lw.w13), w2=api.bf16_from_bits(lw.w2),
                       shared_w13=api.bf16_from_bits(lw.shared_w13), shared_w2=api.bf16_from_bits(lw.shared_w2), layer=0)]
        for l in range(1, L):
            layers.append(dict(gate_w=torch.from_numpy(synth.make_gate_w(shape, 5, l)).cuda(), w13=dev[l - 1][0], w2=dev[l - 1][1],
                               shared_w13=dev[l - 1][2], shared_w2=dev[l - 1][3], layer=l))
        cases = [Case("T=256", shape, T, synth.make_hidden(T, shape.hidden, 5), None, layers)]
        return shape, cases, lw, dict(workload="configs[4]: 27 layers x (64 routed top-6 + 2 always-on shared experts), H=2048 I=1408, T=256 "
                                      "decode tokens; a step = one layer-step, K steps rotate through the 27 layers; + prefill-shaped "
                                      "signature accumulation (32 requests, prompts 512-4096, 16-token KV blocks)",
                                      l2="27 distinct layers (31 GB resident)")
    raise SystemExit("unknown --config %s" % config)


def oracle_sample(shape, case, lw, n_sample):
    """The fp64 oracle, as it stands, on the first n_sample tokens of `case` through layer 0 -> seconds (OpenMP threads as set)."""
    from oracle import oracle
    x = np.ascontiguousarray(case.x_bits[:n_sample])
    t0 = time.perf_counter()
    ora = oracle.moe_decode_layer(shape, x, lw.gate_w, case.bias_np, lw.w13, lw.w2, lw.shared_w13, lw.shared_w2)
    return time.perf_counter() - t0, ora


def run_reference(args, rank):
    """--impl reference: the fp64 CPU oracle as it stands, on the box's host cores, same metric and config.  Each step =
    the oracle's whole layer on a bounded sample (the first 4 tokens of a batch), cycling through the config's cases;
    time scaled by T/4 to the full batch (stated in `sample`)."""
    if rank != 0:
        return
    from oracle import oracle
    from paper_2607_00466_b200 import synth
    config = args.config
    if config in ("2", "3"):
        shape = synth.SHAPE_QWEN
        lw = synth.make_layer_weights(shape, synth.WEIGHT_SEED)
        pts = [(64, u) for u in UNIONS] if config == "2" else [(T, 32) for T in C3_BATCHES]
        cases = []
        for T, u in pts:
            xb, bias = synth.union_case(shape, T, u, synth.accepted_union_seed(T, u))
            cases.append((T, min(u, T * shape.top_k), xb, bias))
    elif config == "4":
        shape = synth.SHAPE_QWEN48
        lw = synth.make_layer_weights(shape, 4, layer=0)
        cent = synth.c4_centroids(shape.hidden, 4)
        lw.gate_w = synth.c4_gate(shape, cent, 4, 0, alpha=0.2)
        cases = []
        for mode, u in (("single", 13), ("mixed", 91)):
            cl = synth.c4_cluster_assignment(128, mode, step=0, seed=4)
            cases.append((128, u, synth.c4_hidden(128, cent, cl, seed=40), None))
    else:
        shape = synth.SHAPE_C5
        lw = synth.make_layer_weights(shape, 5, layer=0)
        cases = [(256, 64, synth.make_hidden(256, shape.hidden, 5), None)]
    n_sample = 4
    tot_t, tot_b = 0.0, 0.0
    for i in range(args.warmup + args.steps):
        T, u, xb, bias = cases[i % len(cases)]
        ns_ = min(n_sample, T)
        t0 = time.perf_counter()
        oracle.moe_decode_layer(shape, np.ascontiguousarray(xb[:ns_]), lw.gate_w, bias, lw.w13, lw.w2, lw.shared_w13, lw.shared_w2)
        dt = (time.perf_counter() - t0) * (T / ns_)
        if i >= args.warmup:
            tot_t += dt
            tot_b += algorithmic_bytes(shape, T, u)
    val = tot_b / tot_t / 1e9
    sample = "first %d tokens of each batch per step, cycling the config's %d cases; time x T/%d" % (n_sample, len(cases), n_sample)
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": "GB/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": tot_t / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "BASELINE.json configs[%d] (oracle on a %d-token sample per step, scaled)" % (int(config) - 1, n_sample)},
            "cpu_baseline": {"value": val, "unit": "GB/s", "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------ the GPU arm
def run_ours(args, rank, local_rank, world):
    import torch
    import torch.distributed as dist
    from paper_2607_00466_b200 import api, replicas, synth

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    api.load()
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    config, K, W = args.config, args.steps, args.warmup
    shape, cases, lw0, cfg_desc = make_cases(config)
    if args.unions and config == "2":
        keep = {int(u) for u in args.unions.split(",")}
        cases = [c for c in cases if c.extra["u"] in keep]
    max_T = max(c.T for c in cases)
    E, k, L = shape.n_experts, shape.top_k, shape.n_layers
    workspace = torch.empty(api.eldr_moe_workspace_bytes_host(shape, max_T), dtype=torch.uint8, device="cuda")
    out = torch.empty((max_T, shape.hidden), dtype=torch.bfloat16, device="cuda")
    ids = torch.empty((max_T, k), dtype=torch.int32, device="cuda")
    wts = torch.empty((max_T, k), dtype=torch.float32, device="cuda")
    active = torch.empty((E,), dtype=torch.int32, device="cuda")
    n_active = torch.zeros((1,), dtype=torch.int32, device="cuda")
    sig_req = torch.zeros((max_T, L, E), dtype=torch.int32, device="cuda")
    sig_blk = torch.zeros((max_T, L, E), dtype=torch.int8, device="cuda")
    step_no = [0]

    def step(c, li=None):
        i = step_no[0] if li is None else li
        step_no[0] += 1
        ly = c.layers[i % len(c.layers)]
        api.eldr_moe_decode_layer(shape, ly["layer"], c.x, ly["gate_w"], c.bias, ly["w13"], ly["w2"], ly["shared_w13"],
                                  ly["shared_w2"], out[:c.T], ids[:c.T], wts[:c.T], 0, active, n_active, c.req, c.blk,
                                  sig_req, sig_blk, workspace)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ------------------------------------------------------------------ warm-up, realised unions per (case, layer)
    launches = set()
    for c in cases:
        distinct = len(c.layers) if config in ("4", "5") else 1
        for li in range(distinct):
            step(c, li)
            torch.cuda.synchronize()
            c.n_active[li] = int(n_active.item())
            launches.add(api.eldr_moe_last_launch_count())
        for li in range(distinct, len(c.layers)):
            c.n_active[li] = c.n_active[0]
        c.bytes_of_layer = [algorithmic_bytes(shape, c.T, na) for na in c.n_active]
        # Gate C invariants on the GPU outputs of the last warm-up step (no oracle)
        gi, gw = ids[:c.T].cpu().numpy(), wts[:c.T].cpu().numpy()
        assert np.all(np.abs(gw.sum(1) - 1.0) <= 1e-5) and gi.min() >= 0 and gi.max() < E
        assert all(len(set(r.tolist())) == k for r in gi) and bool(torch.isfinite(out[:c.T].float()).all())
    launches_per_step = max(launches)
    for c in cases:
        for _ in range(W):
            step(c)
    sig_blk.zero_()

    # ------------------------------------------------------------------ timed region (device time)
    sampler = ClockSampler(local_rank)
    sampler.start()
    # One event pair per case around its K back-to-back steps (an event between every two steps adds idle time).
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in cases]
    barrier()
    t_wall0 = time.perf_counter()
    for ci, c in enumerate(cases):
        step_no[0] = 0
        for _ in range(W):                      # untimed: each case's K timed steps directly follow its own warm-up
            step(c)
        step_no[0] = 0
        ev[ci][0].record()
        for i in range(K):
            step(c)
            if (i + 1) % 100 == 0:
                sig_blk.zero_()                 # keep the int8 block cells below their bound (they saturate at 127)
        ev[ci][1].record()
    barrier()
    t_wall = time.perf_counter() - t_wall0
    sampler.stop_flag = True
    sampler.join()
    total_ms, total_bytes, rows = 0.0, 0.0, []
    for ci, c in enumerate(cases):
        ms = ev[ci][0].elapsed_time(ev[ci][1])
        total_ms += ms
        c.us = ms * 1e3 / K
        c.bytes = sum(c.bytes_of_layer[i % len(c.layers)] for i in range(K))
        total_bytes += c.bytes
        na = [c.n_active[i % len(c.layers)] for i in range(K)]
        rows.append({"case": c.label, "T": c.T, "union": round(float(np.mean(na)), 1), "union_min": int(min(na)), "union_max": int(max(na)),
                     "us_per_step": round(c.us, 2), "algorithmic_MB": round(c.bytes / K / 1e6, 1),
                     "GBps": round(c.bytes / K / c.us / 1e3, 1), "tokens_per_s": round(c.T / c.us * 1e6, 0)})
    total_ms = replicas.max_over_ranks(total_ms, dist if world > 1 else None, "cuda")
    value = replicas.job_throughput_gbs(total_bytes, world, total_ms)
    peaks, peak_kind = measured_peaks()
    peak = float(peaks["hbm_gbs"])
    for r in rows:
        r["frac_of_%s_%.0f" % (peak_kind, peak)] = round(r["GBps"] / peak, 3)
        r["frac_of_nominal_8000"] = round(r["GBps"] / NOMINAL_HBM_GBS, 3)
    n_steps = K * len(cases)

    # ------------------------------------------------------------------ derived checks
    derived = {}
    if config == "2" and len(cases) >= 2:
        xs, ys = np.array([r["union"] for r in rows], float), np.array([r["us_per_step"] for r in rows], float)
        b, a = np.polyfit(xs, ys, 1)
        derived["union_scaling_fit"] = {"fixed_us": round(float(a), 2), "us_per_expert": round(float(b), 3),
                                        "marginal_TBps": round(shape.expert_bytes / float(b) / 1e6, 2),
                                        "latency_ratio_max_over_min_union": round(float(ys[-1] / ys[0]), 2),
                                        "paper_context": "MI300X: 4.7x MoE-layer latency growth 16->128 active experts at batch 64 (PAPER.md:83)"}
    if config == "3":
        ts = [r["us_per_step"] for r in rows if r["T"] >= 8]
        derived["batch_flatness"] = {"(max-min)/median over T=8..256": round((max(ts) - min(ts)) / float(np.median(ts)), 3),
                                     "roofline_allows": 0.007, "paper_context": "batch size at a fixed expert count barely moves it (PAPER.md:83)"}
    if config == "4":
        for mode in ("single", "mixed"):
            rs = [r for r in rows if r["case"].startswith(mode)]
            derived[mode] = {"mean_union": round(float(np.mean([r["union"] for r in rs])), 1),
                             "us_per_layer": round(float(np.mean([r["us_per_step"] for r in rs])), 2),
                             "stack_ms_48_layers": round(float(np.mean([r["us_per_step"] for r in rs])) * 48 / 1e3, 3),
                             "frac_of_peak": round(float(np.mean([r["GBps"] for r in rs])) / peak, 3)}
        derived["speedup_single_over_mixed"] = round(derived["mixed"]["us_per_layer"] / derived["single"]["us_per_layer"], 2)
        derived["fewer_experts_single_vs_mixed"] = round(1 - derived["single"]["mean_union"] / derived["mixed"]["mean_union"], 3)
        derived["paper_context"] = "same-domain batches activate 17-21% fewer experts (PAPER.md:119); sigma=0.3 clusters are far more separable"
    if config == "5":
        derived["stack_ms_27_layers"] = round(rows[0]["us_per_step"] * 27 / 1e3, 3)

    # ------------------------------------------------------------------ per-launch pass (roofline of the top kernel)
    # CUDA events recorded by the library on the launching stream around each of its kernels (PDL off while
    # profiling).  On the default path the step IS one kernel (moe_fused_kernel); on the staged path the
    # dominant kernel is the w1/w3 streaming kernel.
    api.eldr_moe_profile_enable(True)
    kern = {n: 0.0 for n in api.PROFILE_SLOTS}
    kbytes, n_prof = 0.0, 0
    fused = launches_per_step == 1
    for c in cases:
        step_no[0] = 0
        for i in range(min(K, 2 * len(c.layers) if config in ("4", "5") else K)):
            step(c)
            for n, v in api.eldr_moe_profile_read().items():
                kern[n] += v
            n_prof += 1
            li = i % len(c.layers)
            if fused:
                kbytes += c.bytes_of_layer[li]
            else:
                kbytes += (c.n_active[li] + shape.n_shared) * 2 * shape.hidden * shape.inter * 2 + c.T * (k + shape.n_shared) * shape.hidden * 2
    api.eldr_moe_profile_enable(False)
    top = "gate" if fused else "ffn13"          # slot 0 spans the single fused launch
    top_ms = kern[top] / n_prof
    top_gbs = kbytes / n_prof / (top_ms * 1e-3) / 1e9
    traffic = ncu_traffic([int(r["union"]) for r in rows]) if (fused and config == "2") else (None, None, None)
    roofline = {"bound": "hbm",
                "kernel": "moe_fused_kernel (whole step: gate, top-k+signature, routing, w1/w3, w2, combine)" if fused
                else "ffn_umma_kernel<0> (w1/w3 weight streaming + SiLU*mul)",
                "achieved": round(top_gbs, 1), "peak": peak,
                "peak_kind": (peak_kind + " HBM copy rate (MEASURED_PEAKS.json)") if peak_kind == "measured"
                else "fallback 6.65 TB/s (B200_PROFILING.md)",
                "unit": "GB/s", "frac": round(top_gbs / peak, 3),
                "traffic": traffic[0], "traffic_per_union": traffic[1],
                "traffic_source": ("read from the committed ncu summary %s, not measured in this run" % traffic[2]) if traffic[2] else None,
                "algorithmic_bytes_per_launch": round(kbytes / n_prof), "avg_launch_us": round(top_ms * 1e3, 2),
                "kernel_share_of_step": {n: round(v / max(sum(kern.values()), 1e-9), 3) for n, v in kern.items()},
                "kernel_us": {n: round(v / n_prof * 1e3, 2) for n, v in kern.items()}}
    if fused:   # one launch per step: profile slot 0 ("gate") spans the whole persistent kernel -- name it so
        for key in ("kernel_share_of_step", "kernel_us"):
            roofline[key] = {"moe_fused_kernel": roofline[key]["gate"]}

    # ------------------------------------------------------------------ end to end through the host-buffer entry point
    h_out = torch.empty((max_T, shape.hidden), dtype=torch.bfloat16).pin_memory()
    h_ids = torch.empty((max_T, k), dtype=torch.int32).pin_memory()
    h_w = torch.empty((max_T, k), dtype=torch.float32).pin_memory()
    h_na = torch.zeros((1,), dtype=torch.int32).pin_memory()

    def step_host(c):
        ly = c.layers[step_no[0] % len(c.layers)]
        step_no[0] += 1
        api.eldr_moe_decode_layer_host(shape, ly["layer"], c.h_x, ly["gate_w"], c.bias, ly["w13"], ly["w2"], ly["shared_w13"],
                                       ly["shared_w2"], h_out[:c.T], h_ids[:c.T], h_w[:c.T], h_na, c.h_req, c.h_blk, sig_req,
                                       sig_blk, workspace)
    Ke = min(K, 50) if config in ("4", "5") else K
    for c in cases:
        for _ in range(3):
            step_host(c)
    barrier()
    sig_blk.zero_()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    e2e_bytes, h2d, d2h = 0.0, 0, 0
    for c in cases:
        step_no[0] = 0
        for i in range(Ke):
            step_host(c)
            e2e_bytes += c.bytes_of_layer[i % len(c.layers)]
            h2d += c.T * shape.hidden * 2 + 2 * c.T * 4
            d2h += c.T * shape.hidden * 2 + c.T * k * 8 + 4
            if (i + 1) % 100 == 0:
                sig_blk.zero_()
    e1.record()
    barrier()
    e2e_ms = replicas.max_over_ranks(e0.elapsed_time(e1), dist if world > 1 else None, "cuda")
    n_e2e = Ke * len(cases)
    e2e = {"value": round(replicas.job_throughput_gbs(e2e_bytes, world, e2e_ms), 1), "unit": "GB/s",
           "h2d_bytes_per_step": h2d // n_e2e, "d2h_bytes_per_step": d2h // n_e2e, "ms_per_step": round(e2e_ms / n_e2e, 4)}

    # ------------------------------------------------------------------ config 5: prefill-shaped signature accumulation
    extra = {}
    if config == "5" and rank == 0:
        extra["signature_accumulate_prefill_shaped"] = signature_row(api, synth, shape)

    # ------------------------------------------------------------------ CPU oracle timed beside it (rank 0, N=1 only)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle import oracle
        c = cases[len(cases) // 2]
        n_full = c.T if config in ("2", "3") and c.T <= 64 else 16           # bounded sample: ~10-30 s of CPU work in all
        dt, ora = oracle_sample(shape, c, lw0, n_full)
        step(c, 0)                                 # parity spot check of the benchmarked inputs against the oracle
        torch.cuda.synchronize()
        o = out[:n_full].float().cpu().numpy().astype(np.float64)
        rms = np.sqrt((ora["out"] ** 2).mean(axis=1, keepdims=True))
        rel = np.abs(o - ora["out"]) / np.maximum(np.abs(ora["out"]), rms)
        clean = ora["margin"] > 1e-5
        threads = oracle.num_threads()
        oracle.set_threads(1)
        n_one = min(4, c.T)
        dt1, _ = oracle_sample(shape, c, lw0, n_one)
        oracle.set_threads(threads)
        cbytes = c.bytes_of_layer[0]
        cpu = {"value": round(cbytes / (dt * c.T / n_full) / 1e9, 4), "unit": "GB/s", "cores": threads, "kind": "oracle",
               "sample": "the first %d of %d tokens of case %s through layer 0 (fp64, OpenMP over tokens), time x %d/%d"
                         % (n_full, c.T, c.label, c.T, n_full),
               "us_per_step": round(dt * c.T / n_full * 1e6, 0),
               "single_thread": {"value": round(cbytes / (dt1 * c.T / n_one) / 1e9, 5), "unit": "GB/s", "cores": 1,
                                 "sample": "the first %d tokens, time x %d/%d" % (n_one, c.T, n_one),
                                 "us_per_step": round(dt1 * c.T / n_one * 1e6, 0)},
               "parity_vs_gpu": {"max_rel": float(rel[clean].max()), "mean_rel": float(rel[clean].mean()),
                                 "near_tie_tokens": int((~clean).sum()),
                                 "ids_equal_on_clean_tokens": bool(np.array_equal(np.sort(ora["ids"][clean], 1),
                                                                                  np.sort(ids[:n_full].cpu().numpy()[clean], 1)))}}

    if rank == 0:
        line = {"metric": METRIC, "value": round(value, 1), "unit": "GB/s", "n_gpus": world, "steps": K, "warmup": W,
                "ms_per_step": round(total_ms / n_steps, 5), "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
                "config": dict(cfg_desc, parallelism="replicas x%d" % world, accumulate="fp32", gate="fp32",
                               launch="cooperative (all CTAs co-resident)" if fused else "staged kernels"),
                "frac_of_peak": round(value / world / peak, 3), "peak_GBps": peak, "peak_kind": peak_kind,
                "frac_of_nominal_8TBps": round(value / world / NOMINAL_HBM_GBS, 3),
                "sweep": rows, "derived": derived, "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e,
                "gpu_launches": launches_per_step * n_steps, "launches_per_step": launches_per_step,
                "clocks": sampler.summary(), "wall_s_timed_region": round(t_wall, 3)}
        line.update(extra)
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def signature_row(api, synth, shape):
    """Prefill-shaped signature accumulation of config 5 (Table 1's 0.48 ms scatter is the context)."""
    import torch
    L = shape.n_layers
    wl = synth.make_signature_workload(shape.n_experts, shape.top_k, seed=5)
    n_tok = int(wl.topk_ids.shape[0])
    sreq = torch.zeros((wl.n_requests, L, shape.n_experts), dtype=torch.int32, device="cuda")
    sblk = torch.zeros((wl.n_blocks, L, shape.n_experts), dtype=torch.int8, device="cuda")
    t_req, t_blk = torch.from_numpy(wl.token_req).cuda(), torch.from_numpy(wl.token_block).cuda()
    ids_all = torch.from_numpy(np.stack([np.ascontiguousarray((wl.topk_ids + layer) % shape.n_experts) for layer in range(L)])).cuda()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def accumulate():
        if hasattr(api, "eldr_signature_accumulate_layers"):
            api.eldr_signature_accumulate_layers(shape, ids_all, t_req, t_blk, sreq, sblk)
        else:
            for layer in range(L):
                api.eldr_signature_accumulate(shape, layer, ids_all[layer], t_req, t_blk, sreq, sblk)
    accumulate()
    torch.cuda.synchronize()
    recorded = int((wl.token_req >= 0).sum())
    assert int(sreq.sum().item()) == recorded * shape.top_k * L, "signature counts do not sum to tokens x layers x k"
    ts = []
    for _ in range(7):
        sreq.zero_(); sblk.zero_()
        e0.record()
        accumulate()
        e1.record()
        torch.cuda.synchronize()
        ts.append(e0.elapsed_time(e1) * 1e3)
    us = float(np.median(ts))
    traffic = n_tok * L * (shape.top_k * 4 + 8)
    return {"tokens": n_tok, "requests": wl.n_requests, "kv_blocks": wl.n_blocks, "layers": L, "us_all_layers": round(us, 1),
            "launches": 1 if hasattr(api, "eldr_signature_accumulate_layers") else L,
            "G_increments_per_s": round(2 * recorded * shape.top_k * L / us / 1e3, 1),
            "id_map_traffic_GBps": round(traffic / us / 1e3, 1), "counts_sum_exact": True,
            "paper_context": "separate scatter kernel: 0.48 ms per prefill on MI300X (PAPER.md Table 1)"}


# ------------------------------------------------------------------------------------------------ 8(f) rows
def run_route(args):
    """eldr_route_decide at the prefill -> decode handoff (48 layers x 128 experts)."""
    import torch
    from paper_2607_00466_b200 import api, synth
    api.load()
    L, E = 48, 128
    shape = synth.MoEShape(hidden=2048, inter=768, n_experts=E, top_k=8, n_layers=L)
    rows = []
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for R, Kw in ((1, 8), (32, 8), (256, 8), (256, 64)):
        w = synth.make_route_workload(R, L, E, Kw, 8, seed=9, prompt_len=(512, 1024))
        idf = torch.from_numpy(np.log((w.n_calib + 1.0) / (w.df + 1.0)).astype(np.float32)).cuda()   # an input table
        d = [torch.from_numpy(a).cuda() for a in (w.counts, w.layer_mask, w.centroids)]
        loads0 = torch.from_numpy(w.loads).cuda()
        worker = torch.zeros(R, dtype=torch.int32, device="cuda")
        sims = torch.zeros((R, Kw), device="cuda")
        ts = []
        for i in range(8):
            loads = loads0.clone()
            torch.cuda.synchronize()
            e0.record()
            for _ in range(20):
                api.eldr_route_decide(shape, d[0], idf, d[1], d[2], loads, 0.1, worker, sims)
            e1.record()
            torch.cuda.synchronize()
            if i >= 2:
                ts.append(e0.elapsed_time(e1) * 1e3 / 20)
        assert int(loads.sum().item()) == int(loads0.sum().item()) + 20 * R
        kept = int(w.layer_mask.sum())
        nbytes = R * kept * E * 8 + R * Kw * kept * E * 4
        us = float(np.median(ts))
        rows.append({"requests": R, "workers": Kw, "kept_layers": kept, "us_per_call": round(us, 1),
                     "MB_read": round(nbytes / 1e6, 2), "GBps": round(nbytes / us / 1e3, 1)})
    print(json.dumps({"metric": "route_decide_latency", "unit": "us", "value": rows[1]["us_per_call"], "higher_is_better": False,
                      "config": {"workload": "SURVEY.md 8(f) row 1: signature -> routing decision, L=48 E=128, tau=0.1"}, "rows": rows,
                      "paper_context": "proxy-side Route (tau-JSQ) 0.15 ms per request (PAPER.md Table 1)"}), flush=True)


def run_prefill(args):
    """the same layer call with prefill-shaped T (tensor-pipe bound)."""
    import torch
    from paper_2607_00466_b200 import api, synth
    api.load()
    shape = synth.SHAPE_QWEN
    H, I, E, k = shape.hidden, shape.inter, shape.n_experts, shape.top_k
    lw = synth.make_layer_weights(shape, synth.WEIGHT_SEED)
    peaks, kind = measured_peaks()
    sustained = float(peaks.get("bf16_tflops_sustained", peaks["bf16_tflops"]))
    Ts = [int(t) for t in args.prefill_T.split(",")]
    dl = api.DecodeLayer(shape, lw, max_T=max(Ts))
    rows = []
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for T in Ts:
        x = api.bf16_from_bits(synth.make_hidden(T, H, 1000 + T))
        for _ in range(3):
            dl.run(x, None)
        n = max(3, min(args.steps, 20))
        e0.record()
        for _ in range(n):
            dl.run(x, None)
        e1.record()
        torch.cuda.synchronize()
        us = e0.elapsed_time(e1) * 1e3 / n
        api.eldr_moe_profile_enable(True)
        dl.run(x, None)
        prof = api.eldr_moe_profile_read()
        api.eldr_moe_profile_enable(False)
        flop = T * k * 6.0 * H * I + 2.0 * T * H * E
        rows.append({"T": T, "union": int(dl.n_active.item()), "ms_per_step": round(us / 1e3, 4), "tokens_per_s": round(T / us * 1e6),
                     "TFLOPs": round(flop / us / 1e6, 1), "frac_of_%s_bf16_sustained_%.0f" % (kind, sustained): round(flop / us / 1e6 / sustained, 3),
                     "kernel_us": {n_: round(v * 1e3, 1) for n_, v in prof.items()}})
    print(json.dumps({"metric": "prefill_shaped_layer_tflops", "unit": "TFLOP/s", "value": rows[-1]["TFLOPs"], "higher_is_better": True,
                      "dtype": "bf16", "config": {"workload": "SURVEY.md 8(f) row 2: Qwen3-30B-A3B-shaped layer, prefill-shaped T, x ~ N(0,1), no bias"},
                      "roofline": {"bound": "tensor", "achieved": rows[-1]["TFLOPs"], "peak": sustained, "unit": "TFLOP/s",
                                   "frac": round(rows[-1]["TFLOPs"] / sustained, 3), "traffic": None}, "rows": rows}), flush=True)


def run_mxfp4(args):
    """GPT-OSS-120B-shaped experts (128 experts, top-4, mxfp4; hidden = intermediate
    = 2880), T = 64, gate-biased union sweep.  Algorithmic bytes per step = |U| * 3*H*I*(1/2 + 1/32) + activations."""
    import torch
    from paper_2607_00466_b200 import api, synth
    api.load()
    shape = synth.MoEShape(hidden=2880, inter=2880, n_experts=128, top_k=4, n_layers=1)
    H, I, E, k, T = shape.hidden, shape.inter, shape.n_experts, shape.top_k, 64
    K, W = args.steps, args.warmup
    per_expert = 3 * H * I // 2 + 3 * H * I // 32
    gate_w = synth.make_gate_w(shape, 7)
    g = torch.Generator(device="cuda")
    g.manual_seed(7)

    def rand_u8(shape_, lo, hi):           # raw bytes drawn on the device (1.7 GB per copy); parity of the same shapes: tests/test_gpu_mxfp4.py
        return torch.randint(lo, hi, shape_, generator=g, device="cuda", dtype=torch.uint8)
    copies = [dict(c13=rand_u8((E, 2 * I, H // 2), 0, 256), s13=rand_u8((E, 2 * I, H // 32), 118, 123),
                   c2=rand_u8((E, H, I // 2), 0, 256), s2=rand_u8((E, H, I // 32), 118, 123)) for _ in range(N_COPIES)]
    d_gate = torch.from_numpy(gate_w).cuda()
    ws = torch.empty(api.eldr_moe_workspace_bytes(shape, T), dtype=torch.uint8, device="cuda")
    out = torch.empty((T, H), dtype=torch.bfloat16, device="cuda")
    ids = torch.empty((T, k), dtype=torch.int32, device="cuda")
    wts = torch.empty((T, k), dtype=torch.float32, device="cuda")
    active = torch.empty((E,), dtype=torch.int32, device="cuda")
    n_active = torch.zeros((1,), dtype=torch.int32, device="cuda")
    n = [0]

    def step(x, b):
        c = copies[n[0] % N_COPIES]
        n[0] += 1
        api.eldr_moe_decode_layer_mxfp4(shape, 0, x, d_gate, b, c["c13"], c["s13"], c["c2"], c["s2"], out, ids, wts, 0,
                                        active, n_active, None, None, None, None, ws)
    peaks, kind = measured_peaks()
    peak = float(peaks["hbm_gbs"])
    rows, tot_b, tot_ms = [], 0.0, 0.0
    kern = {n_: 0.0 for n_ in api.PROFILE_SLOTS}
    kb13, n_prof = 0.0, 0
    sampler = ClockSampler(0)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for u in UNIONS:
        xb, bias = synth.union_case(shape, T, u, 1000)
        x, b = api.bf16_from_bits(xb), torch.from_numpy(bias).cuda()
        for _ in range(W):
            step(x, b)
        torch.cuda.synchronize()
        na = int(n_active.item())
        e0.record()
        for _ in range(K):
            step(x, b)
        e1.record()
        torch.cuda.synchronize()
        us = e0.elapsed_time(e1) * 1e3 / K
        nbytes = algorithmic_bytes(shape, T, na, per_expert)
        rows.append({"case": "T=64,u=%d" % u, "T": T, "union": na, "us_per_step": round(us, 2), "algorithmic_MB": round(nbytes / 1e6, 1),
                     "GBps": round(nbytes / us / 1e3, 1), "frac_of_%s_%.0f" % (kind, peak): round(nbytes / us / 1e3 / peak, 3)})
        tot_b += nbytes * K
        tot_ms += us * K / 1e3
        api.eldr_moe_profile_enable(True)
        for _ in range(min(K, 20)):
            step(x, b)
            for n_, v in api.eldr_moe_profile_read().items():
                kern[n_] += v
            kb13 += na * (2 * H * I // 2 + 2 * H * I // 32) + T * k * H * 2
            n_prof += 1
        api.eldr_moe_profile_enable(False)
    sampler.stop_flag = True
    sampler.join()
    top_ms = kern["ffn13"] / n_prof
    top_gbs = kb13 / n_prof / (top_ms * 1e-3) / 1e9
    value = tot_b / tot_ms / 1e6
    cpu = None
    if not args.no_cpu_baseline:
        from oracle import mxfp4, oracle
        small = synth.MoEShape(hidden=H, inter=I, n_experts=16, top_k=k, n_layers=1)
        c13, s13 = synth.make_mxfp4_tensor(16 * 2 * I, H, 99, "w13")
        c2, s2 = synth.make_mxfp4_tensor(16 * H, I, 99, "w2")
        xs = synth.make_hidden(4, H, 100)
        t0 = time.perf_counter()
        w13b = mxfp4.mxfp4_to_bf16_bits(c13.reshape(16, 2 * I, H // 2), s13.reshape(16, 2 * I, H // 32))
        w2b = mxfp4.mxfp4_to_bf16_bits(c2.reshape(16, H, I // 2), s2.reshape(16, H, I // 32))
        t_dec = time.perf_counter() - t0
        t0 = time.perf_counter()
        oracle.moe_decode_layer(small, xs, synth.make_gate_w(small, 99), None, w13b, w2b)
        dt = (time.perf_counter() - t0) * (T / 4)
        mid = rows[len(rows) // 2]
        cpu = {"value": round(mid["algorithmic_MB"] * 1e6 / dt / 1e9, 4), "unit": "GB/s", "cores": oracle.num_threads(), "kind": "oracle",
               "sample": "oracle layer on 4 tokens of a 16-expert layer of the same H, I, k (decoded weights; decode of 16 experts took "
                         "%.1f s and is not counted), time x 64/4, against the bytes of the |U|=%d row" % (t_dec, mid["union"]),
               "us_per_step": round(dt * 1e6)}
    print(json.dumps({"metric": METRIC, "value": round(value, 1), "unit": "GB/s", "n_gpus": 1, "steps": K, "warmup": W,
                      "ms_per_step": round(tot_ms / (K * len(rows)), 5), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                      "dtype": "mxfp4 weights (E2M1 + E8M0 per 32) x bf16 activations, fp32 accumulate", "data": "synthetic",
                      "config": {"workload": "SURVEY.md 8(f) row 3: GPT-OSS-120B-shaped MoE layer H=I=2880 E=128 top-4, MXFP4 experts, T=64, gate-biased "
                                             "union sweep (realised unions reported; no rejection sampling)",
                                 "l2": "rotating %d weight copies (1.7 GB each)" % N_COPIES},
                      "frac_of_peak": round(value / peak, 3), "peak_GBps": peak, "peak_kind": kind, "sweep": rows,
                      "roofline": {"bound": "hbm", "kernel": "ffn_mx_kernel<0> (w1/w3: packed-code streaming + register decode -> TMEM A operand + tcgen05)",
                                   "achieved": round(top_gbs, 1), "peak": peak, "unit": "GB/s", "frac": round(top_gbs / peak, 3), "traffic": None,
                                   "avg_launch_us": round(top_ms * 1e3, 2), "algorithmic_bytes_per_launch": round(kb13 / n_prof),
                                   "kernel_us": {n_: round(v / n_prof * 1e3, 2) for n_, v in kern.items()}},
                      "cpu_baseline": cpu, "e2e": None, "gpu_launches": 5 * K * len(rows), "launches_per_step": 5,
                      "clocks": sampler.summary()}), flush=True)


def run_gemv(args):
    """north_star: "Tensor cores ... only where tokens-per-expert fill a tile, with a CUDA-core GEMV path otherwise".  The
    comparison that decides the default: FFN kernel times (CUDA events around each launch of the staged step) of the
    tcgen05 swap-AB kernels and of the CUDA-core GEMV kernels (ELDR_OPT_FFN_PATH) at 1..8 tokens per expert, Qwen3-shaped
    layer, plus the fused step.  Forced routing: T tokens share one set of experts so that m = T exactly."""
    import torch
    from paper_2607_00466_b200 import api, synth
    api.load()
    shape = synth.SHAPE_QWEN
    lw = synth.make_layer_weights(shape, synth.WEIGHT_SEED)
    dl = api.DecodeLayer(shape, lw, max_T=128)
    copies = [(dl.w13, dl.w2)] + [(dl.w13.clone(), dl.w2.clone()) for _ in range(N_COPIES - 1)]
    rows = []
    for m, n_exp in ((1, 8), (1, 32), (2, 32), (4, 32), (8, 32), (8, 128)):
        # m tokens per expert on n_exp experts: T = m * n_exp / k tokens, token t takes experts (t // m) * k .. + k - 1
        k = shape.top_k
        T = m * n_exp // k
        ids = np.stack([((t // m) * k + np.arange(k)) % shape.n_experts for t in range(T)]).astype(np.int32)
        x = api.bf16_from_bits(synth.make_hidden(T, shape.hidden, 300 + T))
        row = {"tokens_per_expert": m, "experts": n_exp, "T": T}
        for name, step_path, ffn in (("tcgen05_staged", api.STEP_STAGED, api.FFN_TCGEN05), ("gemv_staged", api.STEP_STAGED, api.FFN_GEMV),
                                     ("fused", api.STEP_FUSED, api.FFN_TCGEN05)):
            api.eldr_moe_set_option(api.OPT_STEP_PATH, step_path)
            api.eldr_moe_set_option(api.OPT_FFN_PATH, ffn)
            n = [0]

            def step():
                dl.w13, dl.w2 = copies[n[0] % N_COPIES]
                n[0] += 1
                dl.ids[:T].copy_(torch.from_numpy(ids))
                dl.w[:T].fill_(1.0 / k)
                dl.run(x, None, force_routing=1)
            for _ in range(5):
                step()
            outs = dl.out[:T].clone()
            api.eldr_moe_profile_enable(True)
            acc = {}
            for _ in range(args.steps):
                step()
                for kk, v in api.eldr_moe_profile_read().items():
                    acc[kk] = acc.get(kk, 0.0) + v * 1e3 / args.steps
            api.eldr_moe_profile_enable(False)
            assert int(dl.n_active.item()) == n_exp
            if name == "fused":
                row["fused_step_us"] = round(acc["gate"], 2)
            else:
                row[name + "_w13_us"], row[name + "_w2_us"] = round(acc["ffn13"], 2), round(acc["ffn2"], 2)
                row[name + "_w13_GBps"] = round(n_exp * 2 * shape.hidden * shape.inter * 2 / acc["ffn13"] / 1e3)
            row.setdefault("_ref", outs)
            assert (outs.float() - row["_ref"].float()).abs().max().item() <= 2e-2 * row["_ref"].float().abs().max().item() + 1e-6
        row.pop("_ref")
        rows.append(row)
    api.eldr_moe_set_option(api.OPT_STEP_PATH, api.STEP_AUTO)
    api.eldr_moe_set_option(api.OPT_FFN_PATH, api.FFN_TCGEN05)
    print(json.dumps({"metric": "ffn_kernel_us_gemv_vs_tcgen05", "unit": "us", "value": rows[0]["gemv_staged_w13_us"], "higher_is_better": False,
                      "config": {"workload": "Qwen3-30B-A3B-shaped layer, forced routing, m tokens per expert on n experts; per-launch CUDA events"},
                      "rows": rows}), flush=True)


def run_fit(args):
    """the offline fit at the paper's scale ("under 10 s on CPU"; 1,000 calibration
    requests per cell): IDF -> greedy layer mask -> Eq. 2 signatures -> Hungarian-balanced K-means (K = 8).
    Host code (the paper's is too); the oracle's K-means step (scipy Hungarian on duplicated slots) is timed beside it."""
    from paper_2607_00466_b200 import api
    api.load()
    N, L, E, K, P = 1000, 48, 128, 8, 2000
    g = np.random.default_rng(33)
    informative = g.permutation(L)[: L // 2]
    proto = np.full((8, L, E), 0.05)
    for d in range(8):
        for l in informative:
            proto[d, l, g.permutation(E)[:4]] += 3.0
    proto[:, :, 0] += 2.0
    dom = g.integers(0, 8, size=N)
    counts = np.empty((N, L, E), np.int32)
    dec = np.empty((N, L, E))
    for r in range(N):
        p = proto[dom[r]] / proto[dom[r]].sum(axis=1, keepdims=True)
        for l in range(L):
            counts[r, l] = g.multinomial(64, p[l] if l in informative else np.full(E, 1.0 / E))
        dec[r] = np.clip(p * 4 + 0.05 * g.random((L, E)), 0, 1)
    pairs = g.integers(0, N, size=(P, 2)).astype(np.int32)
    init = g.permutation(N)[:K].astype(np.int32)
    t = {}
    t0 = time.perf_counter(); idf = api.eldr_fit_idf(counts); t["idf_s"] = time.perf_counter() - t0
    t0 = time.perf_counter(); order, cum, ns, mask = api.eldr_fit_layer_mask(counts, idf, dec, pairs); t["layer_mask_s"] = time.perf_counter() - t0
    x = (counts * idf[None])[:, np.nonzero(mask)[0], :].reshape(N, -1)
    sig = x / np.linalg.norm(x, axis=1, keepdims=True)
    t0 = time.perf_counter(); cent, assign, steps, total = api.eldr_fit_kmeans_balanced(sig, K, init, 50); t["kmeans_s"] = time.perf_counter() - t0
    sizes = np.bincount(assign, minlength=K).tolist()
    purity = float(np.mean([np.bincount(dom[assign == k], minlength=8).max() / max(1, (assign == k).sum()) for k in range(K)]))
    cpu = None
    if not args.no_cpu_baseline:
        from oracle import fit as ofit
        t0 = time.perf_counter(); o_cent, o_assign, o_steps, o_total = ofit.kmeans_balanced(sig, K, init, 50); dt = time.perf_counter() - t0
        cpu = {"value": round(dt, 3), "unit": "s", "cores": 1, "kind": "oracle", "sample": "the balanced K-means step only (same signatures, same seeds)",
               "assignment_equal": bool(np.array_equal(assign, o_assign)), "steps": o_steps, "total_cost_diff": abs(total - o_total)}
    print(json.dumps({"metric": "offline_fit_seconds", "value": round(sum(t.values()), 3), "unit": "s", "higher_is_better": False, "dtype": "f64",
                      "data": "synthetic", "config": {"workload": "SURVEY.md 8(f) row 4: 1000 calibration requests, L=48, E=128, K=8 workers, 2000 pairs (host code)"},
                      "stages_s": {k_: round(v, 4) for k_, v in t.items()}, "kept_layers": int(ns), "rho_at_peak": round(float(cum[ns - 1]), 4),
                      "rho_all_layers": round(float(cum[-1]), 4), "kmeans_steps": steps, "cluster_sizes": sizes, "cluster_purity": round(purity, 3),
                      "cpu_baseline": cpu, "paper_context": "balanced K-means re-fit under 10 s on CPU (PAPER.md:163)"}), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="2", choices=["2", "3", "4", "5", "prefill", "route", "mxfp4", "fit", "gemv"])
    ap.add_argument("--unions", default="", help="config 2: subset of the union sizes, e.g. 16,128")
    ap.add_argument("--prefill-T", default="2048,4096,8192,16384")
    ap.add_argument("--timeline", default="", help="T:U[,U...]  e.g. 64:16,128, or c5 (the config-5 layer, fused path) -- print the fused kernel's in-kernel timeline (markdown)")
    ap.add_argument("--steady", action="store_true", help="--timeline: trace the last of 12 back-to-back steps instead of an isolated one")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.timeline:
        from paper_2607_00466_b200 import timeline
        if args.timeline == "c5":
            timeline.run(256, [], steady=args.steady, config5=True)
        else:
            T, us = args.timeline.split(":")
            timeline.run(int(T), [int(u) for u in us.split(",")], steady=args.steady)
        return
    if args.impl == "reference":
        if args.config not in ("2", "3", "4", "5"):
            print(json.dumps({"impl": "reference", "unavailable": "the oracle arm covers configs 2-5 only"}))
            return
        run_reference(args, rank)
        return
    if args.config == "route":
        return run_route(args)
    if args.config == "prefill":
        return run_prefill(args)
    if args.config == "mxfp4":
        return run_mxfp4(args)
    if args.config == "fit":
        return run_fit(args)
    if args.config == "gemv":
        return run_gemv(args)
    run_ours(args, rank, local_rank, world)


if __name__ == "__main__":
    main()
