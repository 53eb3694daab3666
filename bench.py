#!/usr/bin/env python
"""bench.py -- MoE-layer decode step: time and achieved HBM bandwidth vs the active-expert union.

Workload (BASELINE.json configs[1], the configuration the metric is quoted on): a Qwen3-30B-A3B-shaped MoE
layer (H=2048, E=128, top-8, I=768, bf16 weights ~N(0,0.02), fp32 gate), batch T=64 decode tokens, gate
biased per batch so the active-expert union |U| is swept over 16, 32, 64, 96, 128.  Seeded synthetic inputs
(paper_2607_00466_b200/synth.py) stand in for the paper's models and prompts.

A "step" is one eldr_moe_decode_layer call: gate GEMV -> softmax top-k + signature accumulation ->
permutation / union compaction -> grouped SwiGLU FFN over the ACTIVE experts -> weighted combine.
The timed region runs K steps at each of the five union sizes (5K steps).  `value` = algorithmic bytes of
those steps / device time (CUDA events, max over ranks), algorithmic bytes per step =
(|U| + n_shared) * 3*H*I*2 + activations (x, Wg, out, ids/weights)  [SURVEY.md 8(d), DESIGN.md].
L2 is defeated by rotating through 4 distinct copies of the layer's weights (>= 450 MB streamed between two
uses of the same copy; B200 L2 is ~126 MB).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
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
T_BATCH = 64
N_COPIES = 4
METRIC = "moe_layer_decode_algorithmic_hbm_bandwidth_over_union_sweep"
NOMINAL_HBM_GBS = 8000.0


def algorithmic_bytes(shape, T, n_active):
    H, I, E, k = shape.hidden, shape.inter, shape.n_experts, shape.top_k
    weights = (n_active + shape.n_shared) * 3 * H * I * 2
    act = T * H * 2 + E * H * 4 + T * H * 2 + T * k * 8
    return weights + act


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured"
    return 6650.0, "fallback"


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
    """dram__bytes_read.sum + dram__bytes_write.sum of moe_fused_kernel per launch, from the committed summary of
    one `ncu --set full` capture per union size (profiles/r1_fused_full.csv; command in profiles/r1_fused_full.md).
    Averaged over the sweep's union sizes like `achieved`; None if a size is missing."""
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "profiles", "r1_fused_full.csv")
    try:
        import csv
        rows = {int(float(r["union"])): float(r["dram__bytes_read.sum"]) + float(r["dram__bytes_write.sum"])
                for r in csv.DictReader(open(path))}
        per = {u: rows[u] for u in unions}
        return round(sum(per.values()) / len(per)), {str(u): round(v) for u, v in per.items()}
    except Exception:
        return None, None


def run_reference(args, rank, world):
    """--impl reference: the fp64 CPU oracle as it stands, on the box's host cores, same metric and config.
    Each step = the oracle's whole layer on a bounded sample (the first 4 of the 64 tokens of the batch) at one
    union size, cycling through the sweep; time is scaled by 64/4 to a full batch (stated in `sample`)."""
    if rank != 0:
        return
    from oracle import oracle
    from paper_2607_00466_b200 import synth
    shape = synth.SHAPE_QWEN
    lw = synth.make_layer_weights(shape, synth.WEIGHT_SEED)
    n_sample = 4
    cases = []
    for u in UNIONS:
        x, bias = synth.union_case(shape, T_BATCH, u, synth.accepted_union_seed(T_BATCH, u))
        cases.append((u, np.ascontiguousarray(x[:n_sample]), bias))
    tot_t, tot_b = 0.0, 0.0
    for i in range(args.warmup + args.steps):
        u, x, bias = cases[i % len(cases)]
        t0 = time.perf_counter()
        oracle.moe_decode_layer(shape, x, lw.gate_w, bias, lw.w13, lw.w2)
        dt = (time.perf_counter() - t0) * (T_BATCH / n_sample)
        if i >= args.warmup:
            tot_t += dt
            tot_b += algorithmic_bytes(shape, T_BATCH, u)
    val = tot_b / tot_t / 1e9
    cores = oracle.num_threads()
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": "GB/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": tot_t / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": "configs[1]: Qwen3-30B-A3B-shaped MoE layer, T=64, union sweep 16..128 "
                                   "(oracle on a 4-token sample per step, scaled x16)"},
            "cpu_baseline": {"value": val, "unit": "GB/s", "cores": cores, "kind": "oracle",
                             "sample": "first 4 of 64 tokens per step, cycling |U| in 16,32,64,96,128; time x16"},
            "e2e": {"value": val, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--unions", default=",".join(str(u) for u in UNIONS))
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return

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

    unions = tuple(int(u) for u in args.unions.split(","))
    shape = synth.SHAPE_QWEN
    T, K, W = T_BATCH, args.steps, args.warmup
    lw = synth.make_layer_weights(shape, synth.WEIGHT_SEED)
    base = api.DecodeLayer(shape, lw, max_T=T)
    copies = [(base.w13, base.w2)] + [(base.w13.clone(), base.w2.clone()) for _ in range(N_COPIES - 1)]
    cases = []
    for u in unions:
        xb, bias = synth.union_case(shape, T, u, synth.accepted_union_seed(T, u))
        req, blk = synth.decode_maps(T)
        cases.append(dict(u=u, x=api.bf16_from_bits(xb), bias=torch.from_numpy(bias).cuda(),
                          h_x=api.bf16_from_bits(xb, device=None).pin_memory(), xb=xb, bias_np=bias,
                          req=torch.from_numpy(req).cuda(), blk=torch.from_numpy(blk).cuda(),
                          h_req=torch.from_numpy(req).pin_memory(), h_blk=torch.from_numpy(blk).pin_memory()))
    sig_req = torch.zeros((T, 1, shape.n_experts), dtype=torch.int32, device="cuda")
    sig_blk = torch.zeros((T, 1, shape.n_experts), dtype=torch.int8, device="cuda")
    step_no = [0]

    def step(c):
        w13, w2 = copies[step_no[0] % N_COPIES]
        step_no[0] += 1
        if step_no[0] % 100 == 0:
            sig_blk.zero_()                     # int8 block cells would overflow after 127 steps on one block
        api.eldr_moe_decode_layer(shape, 0, c["x"], base.gate_w, c["bias"], w13, w2, None, None, base.out[:T],
                                  base.ids[:T], base.w[:T], 0, base.active, base.n_active, c["req"], c["blk"],
                                  sig_req, sig_blk, base.workspace)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ------------------------------------------------------------------ warm-up, realised unions
    for c in cases:
        for _ in range(W):
            step(c)
        torch.cuda.synchronize()
        c["n_active"] = int(base.n_active.item())
        c["bytes"] = algorithmic_bytes(shape, T, c["n_active"])
    launches_per_step = api.eldr_moe_last_launch_count()

    # ------------------------------------------------------------------ timed region (device time)
    sampler = ClockSampler(local_rank)
    sampler.start()
    # One event pair per union size around its K back-to-back steps (an event between every two steps would break
    # the programmatic overlap of consecutive launches and add ~9 us to each step: measured).
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in cases]
    barrier()
    t_wall0 = time.perf_counter()
    for ci, c in enumerate(cases):
        for _ in range(W):                      # untimed: each union size's K timed steps directly follow its own
            step(c)                             # warm-up steps (no idle gap in which the GPU drops its clocks)
        ev[ci][0].record()
        for i in range(K):
            step(c)
        ev[ci][1].record()
    barrier()
    t_wall = time.perf_counter() - t_wall0
    sampler.stop_flag = True
    sampler.join()
    # spread of single steps: a separate, untimed pass with an event after every step (isolated launches)
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(K + 1)] for _ in cases]
    for ci, c in enumerate(cases):
        evs[ci][0].record()
        for i in range(K):
            step(c)
            evs[ci][i + 1].record()
    torch.cuda.synchronize()
    total_ms = 0.0
    sweep = []
    for ci, c in enumerate(cases):
        per = np.array([evs[ci][i].elapsed_time(evs[ci][i + 1]) for i in range(K)]) * 1e3   # us
        tot = ev[ci][0].elapsed_time(ev[ci][1])
        total_ms += tot
        c["us"] = tot * 1e3 / K
        sweep.append({"union": c["n_active"], "us_per_step": round(c["us"], 2),
                      "isolated_us_p10": round(float(np.percentile(per, 10)), 2),
                      "isolated_us_median": round(float(np.median(per)), 2),
                      "isolated_us_p90": round(float(np.percentile(per, 90)), 2),
                      "algorithmic_MB": round(c["bytes"] / 1e6, 1), "GBps": round(c["bytes"] / c["us"] / 1e3, 1),
                      "tokens_per_s": round(T / c["us"] * 1e6, 0)})
    total_ms = replicas.max_over_ranks(total_ms, dist if world > 1 else None, "cuda")
    total_bytes = sum(c["bytes"] for c in cases) * K
    value = replicas.job_throughput_gbs(total_bytes, world, total_ms)
    peak, peak_kind = measured_peaks()
    for s in sweep:
        s["frac_of_%s_%.0f" % (peak_kind, peak)] = round(s["GBps"] / peak, 3)
        s["frac_of_nominal_8000"] = round(s["GBps"] / NOMINAL_HBM_GBS, 3)

    # ------------------------------------------------------------------ per-kernel pass (roofline of the top kernel)
    # CUDA events recorded by the library on the launching stream around each of its kernels (PDL off while
    # profiling).  On the default path the step IS one kernel (moe_fused_kernel); on the staged path the
    # dominant kernel is the w1/w3 streaming kernel.
    api.eldr_moe_profile_enable(True)
    kern = {n: 0.0 for n in api.PROFILE_SLOTS}
    kbytes = 0.0
    fused = launches_per_step == 1
    for c in cases:
        for _ in range(K):
            step(c)
            for n, v in api.eldr_moe_profile_read().items():
                kern[n] += v
            if fused:
                kbytes += c["bytes"]
            else:
                kbytes += c["n_active"] * 2 * shape.hidden * shape.inter * 2 + T * shape.top_k * shape.hidden * 2
    api.eldr_moe_profile_enable(False)
    n_steps = K * len(cases)
    top = "gate" if fused else "ffn13"          # slot 0 spans the single fused launch
    top_ms = kern[top] / n_steps
    top_gbs = kbytes / n_steps / (top_ms * 1e-3) / 1e9
    roofline = {"bound": "hbm",
                "kernel": "moe_fused_kernel (whole step: gate, top-k+signature, routing, w1/w3, w2, combine)" if fused
                else "ffn_umma_kernel<0> (w1/w3 weight streaming + SiLU*mul)",
                "achieved": round(top_gbs, 1), "peak": peak,
                "peak_kind": (peak_kind + " HBM copy rate (MEASURED_PEAKS.json)") if peak_kind == "measured"
                else "fallback 6.65 TB/s (B200_PROFILING.md)",
                "unit": "GB/s", "frac": round(top_gbs / peak, 3),
                "traffic": ncu_traffic([c["n_active"] for c in cases])[0] if fused else None,
                "traffic_per_union": ncu_traffic([c["n_active"] for c in cases])[1] if fused else None,
                "algorithmic_bytes_per_launch": round(kbytes / n_steps), "avg_launch_us": round(top_ms * 1e3, 2),
                "kernel_share_of_step": {n: round(v / max(sum(kern.values()), 1e-9), 3) for n, v in kern.items()},
                "kernel_us": {n: round(v / n_steps * 1e3, 2) for n, v in kern.items()}}
    if fused:   # one launch per step: profile slot 0 ("gate") spans the whole persistent kernel -- name it so
        for key in ("kernel_share_of_step", "kernel_us"):
            roofline[key] = {"moe_fused_kernel": roofline[key]["gate"]}

    # ------------------------------------------------------------------ end to end through the host-buffer entry point
    h_out = torch.empty((T, shape.hidden), dtype=torch.bfloat16).pin_memory()
    h_ids = torch.empty((T, shape.top_k), dtype=torch.int32).pin_memory()
    h_w = torch.empty((T, shape.top_k), dtype=torch.float32).pin_memory()
    h_na = torch.zeros((1,), dtype=torch.int32).pin_memory()

    def step_host(c):
        w13, w2 = copies[step_no[0] % N_COPIES]
        step_no[0] += 1
        if step_no[0] % 100 == 0:
            sig_blk.zero_()
        api.eldr_moe_decode_layer_host(shape, 0, c["h_x"], base.gate_w, c["bias"], w13, w2, None, None, h_out, h_ids,
                                       h_w, h_na, c["h_req"], c["h_blk"], sig_req, sig_blk, base.workspace)
    for c in cases:
        for _ in range(3):
            step_host(c)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for c in cases:
        for _ in range(K):
            step_host(c)
    e1.record()
    barrier()
    e2e_ms = e0.elapsed_time(e1)
    e2e_ms = replicas.max_over_ranks(e2e_ms, dist if world > 1 else None, "cuda")
    e2e = {"value": round(replicas.job_throughput_gbs(total_bytes, world, e2e_ms), 1), "unit": "GB/s",
           "h2d_bytes_per_step": T * shape.hidden * 2 + 2 * T * 4,
           "d2h_bytes_per_step": T * shape.hidden * 2 + T * shape.top_k * 8 + 4,
           "ms_per_step": round(e2e_ms / n_steps, 4)}

    # ------------------------------------------------------------------ CPU oracle timed beside it (rank 0, N=1 only)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle import oracle
        c = cases[len(cases) // 2]
        t0 = time.perf_counter()
        ora = oracle.moe_decode_layer(shape, c["xb"], lw.gate_w, c["bias_np"], lw.w13, lw.w2)
        dt = time.perf_counter() - t0
        got = base  # parity spot check of the benchmarked configuration against the oracle
        step(c)
        torch.cuda.synchronize()
        o = base.out[:T].float().cpu().numpy().astype(np.float64)
        rms = np.sqrt((ora["out"] ** 2).mean(axis=1, keepdims=True))
        rel = np.abs(o - ora["out"]) / np.maximum(np.abs(ora["out"]), rms)
        cpu = {"value": round(c["bytes"] / dt / 1e9, 4), "unit": "GB/s", "cores": oracle.num_threads(),
               "kind": "oracle", "sample": "one full layer-step at |U|=%d, T=64 (fp64, OpenMP over tokens)" % c["n_active"],
               "us_per_step": round(dt * 1e6, 0),
               "parity_vs_gpu": {"max_rel": float(rel.max()), "mean_rel": float(rel.mean()),
                                 "ids_equal": bool(np.array_equal(np.sort(ora["ids"], 1),
                                                                  np.sort(base.ids[:T].cpu().numpy(), 1)))}}

    if rank == 0:
        line = {"metric": METRIC, "value": round(value, 1), "unit": "GB/s", "n_gpus": world, "steps": K, "warmup": W,
                "ms_per_step": round(total_ms / n_steps, 5), "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
                "config": {"workload": "configs[1]: Qwen3-30B-A3B-shaped MoE layer H=2048 E=128 top-8 I=768, T=64 decode "
                                       "tokens, gate-biased union sweep |U|=16,32,64,96,128; K steps per union size",
                           "l2": "rotating %d weight copies (>=450 MB streamed between reuses; L2 ~126 MB)" % N_COPIES,
                           "parallelism": "replicas x%d" % world, "accumulate": "fp32", "gate": "fp32"},
                "frac_of_peak": round(value / world / peak, 3), "peak_GBps": peak, "peak_kind": peak_kind,
                "frac_of_nominal_8TBps": round(value / world / NOMINAL_HBM_GBS, 3),
                "sweep": sweep, "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e,
                "gpu_launches": launches_per_step * n_steps, "launches_per_step": launches_per_step,
                "clocks": sampler.summary(), "wall_s_timed_region": round(t_wall, 3),
                "paper_context": "MI300X: 4.7x MoE-layer latency growth 16->128 active experts at batch 64 (PAPER.md:83); "
                                 "here %.2fx" % (sweep[-1]["us_per_step"] / sweep[0]["us_per_step"])}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
