"""In-kernel timeline of the fused decode step (`python bench.py --timeline T:U[,U...] [--steady]`).

A profiling aid, not part of the measured path: it builds a SECOND copy of the library with -DELDR_TRACE
(`libeldr_moe_trace.so`; the normal build carries no trace code), runs a few steps of the Qwen3-30B-A3B-shaped layer at
the requested union sizes and prints, per stamp, the min / median / max over the 148 CTAs of the time since the first
CTA started (`%globaltimer`, microseconds).  Reading %globaltimer and storing it costs the stamping thread ~0.7 us, so
stamped intervals on the serial prelude are inflated by that much each and the whole kernel by a few microseconds; the
point is WHERE the time goes, not the total.
"""
from __future__ import annotations

import ctypes as C
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

ROW0 = [(0, "kernel start (after barrier init / TMEM alloc)"), (5, "weights producer: first TMA stage issued"),
        (6, "MMA issuer: first stage landed"), (11, "weights producer: phase A (w1/w3) fully issued"),
        (13, "MMA issuer: phase A fully issued"), (2, "epilogue: accumulator of the LAST phase-A piece ready"),
        (4, "epilogue: last phase-A piece written (h)"), (15, "last h-tile flag raised"),
        (14, "activations producer: first phase-B (w2) expert ready"), (7, "weights producer: done"),
        (8, "all FFN roles done"), (10, "combine done (warp 0)"), (9, "combine done (all warps)")]
ROW1 = [(8, "kernel entry (before barrier init / TMEM alloc)"), (12, "prelude: own gate tiles done"), (13, "prelude: own top-k groups done (owners only)"),
        (14, "prelude: tagged ids of all tokens seen"), (4, "route_a: masks zeroed (+ forced ids loaded)"),
        (5, "route_a: membership bitmasks built"), (6, "route_a: per-expert counts and prefixes"),
        (7, "route_a: scan, work list, pass table (warp 0)"), (15, "prelude: routing tables built (route_a)")]


def run(T: int, unions, steady: bool = False, config5: bool = False):
    """unions: the config-2/3 union sizes to trace at batch T (Qwen3-30B-A3B-shaped layer); config5 = True traces the
    config-5 layer instead (64 routed top-6 + 2 shared experts, I = 1408, T = 256, fused path forced; `unions` ignored)."""
    import torch
    from paper_2607_00466_b200 import build as b
    from paper_2607_00466_b200 import api, synth
    lib = api.load(path=b.build(trace=True))
    shape = synth.SHAPE_C5 if config5 else synth.SHAPE_QWEN
    lw = synth.make_layer_weights(shape, 5 if config5 else synth.WEIGHT_SEED)
    if config5:
        T, unions = 256, [shape.n_experts]
        api.eldr_moe_set_option(api.OPT_STEP_PATH, api.STEP_FUSED)
    dl = api.DecodeLayer(shape, lw, max_T=T)
    copies = [(dl.w13, dl.w2)] + [(dl.w13.clone(), dl.w2.clone()) for _ in range(3)]
    cmd = "python bench.py --timeline %s%s" % ("c5" if config5 else "%d:%s" % (T, ",".join(str(u) for u in unions)), " --steady" if steady else "")
    print("# In-kernel timeline of `moe_fused_kernel` (`%s`)\n" % cmd)
    print("%s; -DELDR_TRACE build; microseconds since the first CTA passed its prologue; min / median / max over the CTAs that "
          "hit the stamp.  %s (4 rotating weight copies).\n" %
          (torch.cuda.get_device_name(0), "The last of 12 back-to-back steps is the one traced" if steady else
           "The sixth step of each case, alone on the device, is the one traced"))
    for u in unions:
        if config5:
            x, bias_t = api.bf16_from_bits(synth.make_hidden(T, shape.hidden, 5)), None
        else:
            try:
                seed = synth.accepted_union_seed(T, u)
            except KeyError:
                seed = 1000
            xb, bias = synth.union_case(shape, T, u, seed)
            x, bias_t = api.bf16_from_bits(xb), torch.from_numpy(bias).cuda()
        for it in range(12 if steady else 6):
            if it == 5 and not steady:
                torch.cuda.synchronize()
                lib.eldr_debug_clear_trace()
            dl.w13, dl.w2 = copies[it % 4]
            dl.run(x, bias_t)
        torch.cuda.synchronize()
        buf = (C.c_ulonglong * (4096 * 16))()
        lib.eldr_debug_read_trace(buf)
        tr = np.frombuffer(buf, dtype=np.uint64).reshape(4096, 16).astype(np.int64)
        n_cta = int((tr[:1024, 0] > 0).sum())
        r0, r1, r2 = tr[:n_cta], tr[2048:2048 + n_cta], tr[1024:1024 + n_cta]
        t0 = r0[:, 0].min()
        print("## T = %d, realised |U| = %d (%d CTAs)\n\n| stamp | CTAs | min | median | max |\n|---|---|---|---|---|" %
              (T, int(dl.n_active.item()), n_cta))
        for rows, table in ((r1, ROW1), (r0, ROW0)):
            for col, name in table:
                v = rows[:, col]
                v = v[v > 0]
                if len(v):
                    print("| %s | %d | %.2f | %.2f | %.2f |" % (name, len(v), (v.min() - t0) / 1e3,
                                                               (np.median(v) - t0) / 1e3, (v.max() - t0) / 1e3))
        if not steady:
            print("\n| per sub-phase (0: w1/w3 whole rounds, 1: w1/w3 remainder (or the whole phase as stream-K), 2: w2 whole rounds, 3: w2 remainder (or stream-K)) | min | median | max |\n|---|---|---|---|")
            for base, name, is_time in ((0, "weights producer: sub-phase %d fully issued", True), (4, "epilogue: sub-phase %d finished", True),
                                        (8, "activations producer: waited for h flags in sub-phase %d (us)", False),
                                        (12, "epilogue warp 0: waited for partners' parked partials in sub-phase %d (us)", False)):
                for sp in range(4):
                    v = r2[:, base + sp]
                    if is_time:
                        v = v[v > 0]
                        if len(v):
                            print("| %s | %.2f | %.2f | %.2f |" % (name % sp, (v.min() - t0) / 1e3, (np.median(v) - t0) / 1e3, (v.max() - t0) / 1e3))
                    else:
                        print("| %s | %.2f | %.2f | %.2f |" % (name % sp, v.min() / 1e3, np.median(v) / 1e3, v.max() / 1e3))
        stall = r0[:, 12] / 1e3
        print("\nActivations producer waited for h flags: median %.2f us, max %.2f us per CTA.\n" %
              (float(np.median(stall)), float(stall.max())), flush=True)
