"""%globaltimer timeline of one replayed layer step, from the tracing build of the library.

    python -m paper_2607_04181_b200.timeline [--replicas R] [--replays N]

Builds libcocoscale_trace.so if needed (the product sources with -DCC_TRACE: every kernel records, per trace
point, the earliest and latest timer value over its CTAs), captures cc_forward of the cfg2 layer in a CUDA graph,
replays it and prints, per kernel, the points' (min .. max over CTAs) in microseconds relative to the first
kernel's entry (median over the replays), and the duration of the stream-K fixup passes.  A measurement aid:
the timer reads cost about a microsecond per step, so step times come from bench.py, not from here.
Plumbing only (torch: device memory and graph capture)."""
from __future__ import annotations

import argparse
import os

os.environ["COCOSCALE_TRACE"] = "1"          # before the binding is imported: load the tracing build

import numpy as np
import torch

from . import binding as B
from . import inputs as I
from .harness import DeviceStep, Session

KERNELS = ((0, "prologue", 3), (2, "gemm_qkv", 6), (1, "attention", 3), (3, "gemm_o", 6), (4, "gemm_gate_up", 6), (5, "gemm_down", 6))


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--replicas", type=int, default=1)
    ap.add_argument("--replays", type=int, default=7)
    ap.add_argument("--batch", type=int, default=0, help="decode rows (default: the cfg2 batch, 64)")
    args = ap.parse_args()
    shape = I.CFG2
    batch = args.batch or shape.batch
    w = I.make_weights(shape, 1002)
    st = I.make_step_inputs(shape, 2002, 3002, batch=batch)
    S = Session(shape, w, max_batch=batch, n_slots=3)
    S.scale(args.replicas)
    step = DeviceStep(st, I.even_split(batch, args.replicas))
    for _ in range(3):
        S.forward(step)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        S.forward(step, torch.cuda.current_stream())
    for _ in range(5):
        g.replay()
    rel, raw = [], None
    for _ in range(args.replays):
        for _ in range(3):
            g.replay()
        B.cc_debug_trace(S.ctx, reset=True)
        g.replay()
        raw = B.cc_debug_trace(S.ctx, reset=True).astype(np.float64)
        rel.append((raw - raw[0, 0, 0]) / 1e3)
    t = np.median(np.stack(rel), axis=0)
    print(f"cfg2 layer, batch {batch}, R={args.replicas}, graph replay with PDL; us relative to the prologue's entry, median of {args.replays} "
          f"replays; each point: min..max over the CTAs")
    for k, name, npt in KERNELS:
        print(f"{name:13s}", " | ".join(f"{t[k, pt, 0]:7.2f}..{t[k, pt, 1]:7.2f}" for pt in range(npt)))
    print("GEMM points: entry | dependency wait done (producer) | producer issued its last copy | mainloop drained, partials "
          "stored | first fixup wait done | end")
    print("prologue: entry | dependency wait done | end (row blocks and the two table blocks);  attention: entry | dependency wait done (consumers) | consumers saw "
          "the end marker")
    for kind, name in enumerate(("gemm_qkv", "gemm_o", "gemm_gate_up", "gemm_down")):
        d, a = raw[8 + kind], raw[12 + kind]
        line = []
        for slot, what in ((0, "first"), (1, "second")):
            n = a[slot, 1]
            if n > 0:
                line.append(f"{what} pass {d[slot, 0] / 1e3:.2f}..{d[slot, 1] / 1e3:.2f} us (mean {a[2 + slot, 1] / n / 1e3:.2f}) in {n:.0f} CTAs")
        print(f"{name:13s} stream-K fixup (last replay): " + "; ".join(line))
    assert B.cc_poll_device_error(S.ctx) == 0
    S.close()


if __name__ == "__main__":
    main()
