"""In-kernel timeline of the fused decode step (diagnostic; not part of the measured path).

Builds a SECOND copy of the library with -DELDR_TRACE (`libeldr_moe_trace.so`; the normal build carries no trace
code), runs a few steps of the Qwen3-30B-A3B-shaped layer at the requested union sizes and prints, per stamp, the
min / median / max over the 148 CTAs of the time since the first CTA started (`%globaltimer`, microseconds).
Reading %globaltimer and storing it costs the stamping thread ~0.7 us (measured: two stamps with nothing between
them are 0.77 us apart), so stamped intervals on the serial prelude are inflated by that much each and the whole
kernel by a few microseconds; the point is WHERE the time goes, not the total.

  python -m paper_2607_00466_b200.trace [--T 64] [--unions 16,128] > profiles/<name>.md
"""
from __future__ import annotations

import argparse
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


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--T", type=int, default=64)
    ap.add_argument("--unions", default="16,128")
    ap.add_argument("--steady", action="store_true", help="trace the last of 12 back-to-back steps (no sync before it)")
    ap.add_argument("--opt", action="append", default=[], help="KEY=VALUE for eldr_moe_set_option (repeatable)")
    args = ap.parse_args()
    os.environ["ELDR_EXTRA_NVCC_FLAGS"] = (os.environ.get("ELDR_EXTRA_NVCC_FLAGS", "") + " -DELDR_TRACE").strip()
    import torch
    from paper_2607_00466_b200 import build as b
    b.LIB = b.LIB.replace("libeldr_moe.so", "libeldr_moe_trace.so")
    b.build(force=True)
    from paper_2607_00466_b200 import api, synth
    lib = api.load()
    for kv in args.opt:
        api.eldr_moe_set_option(*[int(v) for v in kv.split("=")])
    shape, T = synth.SHAPE_QWEN, args.T
    lw = synth.make_layer_weights(shape, synth.WEIGHT_SEED)
    dl = api.DecodeLayer(shape, lw, max_T=T)
    copies = [(dl.w13, dl.w2)] + [(dl.w13.clone(), dl.w2.clone()) for _ in range(3)]
    print("# In-kernel timeline of `moe_fused_kernel` (`python -m paper_2607_00466_b200.trace --T %d --unions %s`)\n" %
          (T, args.unions))
    print("%s; -DELDR_TRACE build; microseconds since the first CTA started; min / median / max over the CTAs that "
          "hit the stamp.  The sixth step of each case is the one traced (4 rotating weight copies).\n" %
          torch.cuda.get_device_name(0))
    for u in [int(v) for v in args.unions.split(",")]:
        try:
            seed = synth.accepted_union_seed(T, u)
        except KeyError:
            seed = 1000
        xb, bias = synth.union_case(shape, T, u, seed)
        x, bias_t = api.bf16_from_bits(xb), torch.from_numpy(bias).cuda()
        for it in range(12 if args.steady else 6):
            if it == 5 and not args.steady:
                torch.cuda.synchronize()
                lib.eldr_debug_clear_trace()
            dl.w13, dl.w2 = copies[it % 4]
            dl.run(x, bias_t)
        torch.cuda.synchronize()
        buf = (C.c_ulonglong * (4096 * 16))()
        lib.eldr_debug_read_trace(buf)
        tr = np.frombuffer(buf, dtype=np.uint64).reshape(4096, 16).astype(np.int64)
        n_cta = int((tr[:2048, 0] > 0).sum())
        r0, r1 = tr[:n_cta], tr[2048:2048 + n_cta]
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
        r2 = tr[1024:1024 + n_cta]
        print("\n| per sub-phase (0..3) | min | median | max |\n|---|---|---|---|")
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
        for col, name in ((0, "weights producer: waited for free ring slots, phase A (us @1.965 GHz)"), (1, "weights producer: waited for free ring slots, phase B (us @1.965 GHz)"),
                          (10, "weights producer: TMA issue, phase A (us @1.965 GHz)"), (11, "weights producer: TMA issue, phase B (us @1.965 GHz)")):
            v = r1[:, col] / 1965.0
            print("| %s | %.2f | %.2f | %.2f |" % (name, v.min(), np.median(v), v.max()))
        stall = r0[:, 12] / 1e3
        print("\nActivations producer waited for h flags: median %.2f us, max %.2f us per CTA.\n" %
              (float(np.median(stall)), float(stall.max())), flush=True)


if __name__ == "__main__":
    main()
