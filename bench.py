#!/usr/bin/env python
"""bench.py -- replicated decode-layer throughput on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--replicas R] [--impl reference]

A "step" is one pass of the whole hot path (cc_forward: grouping, RMSNorm, QKV GEMM, RoPE + KV
append, paged GQA decode attention, O GEMM, RMSNorm, gate/up GEMM + SwiGLU, down GEMM, residual)
over one decode batch of BASELINE.json configs[1]: the Llama-3-8B-shaped layer, batch 64, contexts
U{512..2048} in shuffled 16-token pages, the batch split evenly over R replicas of the layer
(default R = 2).  Inputs are seeded and synthetic (inputs.py) and resident in HBM before the timed
region; each step streams R x 436 MB of weights + ~335 MB of KV, far more than the 126 MB L2, so
consecutive steps cannot hit in cache.  Prints ONE JSON line.

N > 1 (torchrun): the path does not shard -- "replicas only": every rank runs its own independent
batch on its own GPU, no data-path collective; value = all ranks' tokens / max-over-ranks time.

--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample of the same
workload; it is a deliberately slow baseline, not the target.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "replicated decode-layer tokens/s"
UNIT = "tokens/s"
CPU_BASELINE_ROWS = 64      # cpu_baseline leg and --impl reference alike: the whole batch per step ...
CPU_BASELINE_STEPS = 4      # ... cpu_baseline: four steps (about 10 s of CPU work on 16 cores)
REF_BUDGET_STEPS = 60       # --impl reference: up to this many (steps + warmup) run on the whole batch (~2 s each);
                            # longer runs shrink the rows per step so the arm still ends within a few minutes
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel come from this file, which
# `python -m paper_2607_04181_b200.ncu_summary` writes from an `ncu --set full` export (with the commit it was taken at)
NCU_TRAFFIC_FILE = os.path.join(ROOT, "profiles", "ncu_traffic.json")
FALLBACK_HBM_GBS = 6650.0   # /opt/skills/guides/B200_PROFILING.md, used only if MEASURED_PEAKS.json is absent


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--replicas", type=int, default=2, choices=[1, 2, 3, 4])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--batch", type=int, default=0,
                    help="decode batch of the cfg2 layer benchmark (default: the config's 64); larger batches are for the "
                         "tensor-pipe evidence of the GEMMs (DESIGN.md section 9), not the headline")
    ap.add_argument("--prefill-rows", type=int, default=64,
                    help="cfg5: prompt tokens carried by every step of model A as extra rows (half as many for B); 0 = decode only")
    ap.add_argument("--copy-sweep", action="store_true", help="also sweep the chunk size of the replica copy (replica_copy.chunk_sweep)")
    ap.add_argument("--workload", default="cfg2", choices=["cfg2", "cfg3", "cfg4", "cfg5"],
                    help="cfg2 (default): the headline layer benchmark; cfg3: BASELINE.json configs[2], the 32-layer "
                         "decode graph with layers 10-12 flipped to 2 replicas and back (latency series, not the headline); "
                         "cfg5: configs[4], the co-located serving loop (decode only)")
    ap.add_argument("--horizon", type=float, default=120.0, help="cfg5: seconds of synthetic arrivals")
    ap.add_argument("--layers", type=int, default=1, help="cfg4: layers of the mixed-step graph (configs[3] names 40; default one hot layer)")
    return ap.parse_args()


def ncu_traffic(kernel: str, replicas: int):
    """(bytes per launch, source) of `kernel` at `replicas` from profiles/ncu_traffic.json, or (None, None)."""
    try:
        with open(NCU_TRAFFIC_FILE) as f:
            t = json.load(f)
        e = t["kernels"][kernel][f"R{replicas}"]
        return int(e["dram_bytes_read"]) + int(e["dram_bytes_write"]), f"ncu --set full, {e['summary']} (commit {t['commit']})"
    except Exception:
        return None, None


def measured_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, read+write copy)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


# ---------------------------------------------------------------------------------------------
# clocks during the timed region (NVML, polled from a thread)
# ---------------------------------------------------------------------------------------------
_REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
            0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x10: "sync_boost"}


class ClockSampler:
    def __init__(self, torch_device_index: int):
        self.samples, self.reasons, self.max_mhz, self.ok = [], set(), None, False
        self._stop = threading.Event()
        try:
            import pynvml
            import torch
            pynvml.nvmlInit()
            try:
                uuid = str(torch.cuda.get_device_properties(torch_device_index).uuid)
                self.h = pynvml.nvmlDeviceGetHandleByUUID(("GPU-" + uuid) if not uuid.startswith("GPU-") else uuid)
            except Exception:
                self.h = pynvml.nvmlDeviceGetHandleByIndex(torch_device_index)
            self.nv = pynvml
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.ok = False
        self.t = threading.Thread(target=self._run, daemon=True)

    def _run(self):
        while not self._stop.is_set():
            try:
                self.samples.append(float(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM)))
                try:
                    bits = int(self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    bits = int(self.nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for b, name in _REASONS.items():
                    if bits & b:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.004)

    def start(self):
        if self.ok:
            self.t.start()

    def stop(self):
        self._stop.set()
        if self.ok:
            self.t.join(timeout=2)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ---------------------------------------------------------------------------------------------
# algorithmic bytes; bookkeeping only
# ---------------------------------------------------------------------------------------------
def stage_bytes(shape, seq_lens, n_groups: int) -> dict:
    d, F, QD, KD = shape.hidden, shape.ffn, shape.q_dim, shape.kv_dim
    B = int((seq_lens > 0).sum())
    tok = int(seq_lens[seq_lens > 0].sum())                     # tokens attended, including the new one
    return {
        "gemm_qkv": n_groups * (QD + 2 * KD) * d * 2 + B * d * 2,
        "attention": tok * 2 * KD * 2 + B * QD * 4,
        "gemm_o": n_groups * d * QD * 2 + B * QD * 2,
        "gemm_gate_up": n_groups * 2 * F * d * 2 + B * d * 2,
        "gemm_down": n_groups * d * F * 2 + B * F * 2,
    }


# ---------------------------------------------------------------------------------------------
# the reference arm: the CPU oracle on a bounded sample
# ---------------------------------------------------------------------------------------------
def time_oracle(shape, w, st, rows: int, steps: int, warmup: int):
    import oracle
    sub = slice(0, rows)
    assign = np.zeros(rows, np.int32)

    def one():
        oracle.layer_forward(shape, w, st.hidden[sub], st.k_pool, st.v_pool, st.block_table[sub], st.seq_lens[sub],
                             assign, 1)
    for _ in range(warmup):
        one()
    t0 = time.perf_counter()
    for _ in range(steps):
        one()
    dt = time.perf_counter() - t0
    return rows * steps / dt, dt / steps, oracle.num_threads()


def cpu_baseline_extras(shape, w, st, cores: int) -> dict:
    """BASELINE.md section 4's other CPU figures, each on a bounded sample: the oracle on ONE thread, the oracle on
    cfg1 (the tiny layer), and a host memcpy beside the replica copy (oracle.replica_copy is memcpy)."""
    import oracle
    from paper_2607_04181_b200 import inputs as I
    out = {}
    oracle.set_num_threads(1)
    try:
        tps1, s1, _ = time_oracle(shape, w, st, 2, 1, 0)
        out["one_thread"] = {"value": tps1, "unit": UNIT, "cores": 1, "sample": f"2 rows of the cfg2 batch, one layer step of {s1:.1f} s"}
    finally:
        oracle.set_num_threads(cores)
    w1 = I.make_weights(I.CFG1, 1001)
    st1 = I.make_step_inputs(I.CFG1, 2001, 3001)
    a1 = I.even_split(I.CFG1.batch, 2)
    n1 = 20
    t0 = time.perf_counter()
    for _ in range(n1):
        oracle.layer_forward(I.CFG1, w1, st1.hidden, st1.k_pool, st1.v_pool, st1.block_table, st1.seq_lens, a1, 2)
    out["cfg1"] = {"value": I.CFG1.batch * n1 / (time.perf_counter() - t0), "unit": UNIT, "cores": cores,
                   "sample": f"{n1} steps of configs[0] (tiny layer, batch 4, 2 replicas)"}
    buf = np.ones(256 << 20, np.uint8)
    oracle.replica_copy(buf)
    t0 = time.perf_counter()
    for _ in range(3):
        oracle.replica_copy(buf)
    dt = (time.perf_counter() - t0) / 3
    out["host_memcpy"] = {"GBps_payload": buf.nbytes / dt / 1e9, "GBps_read_plus_write": 2 * buf.nbytes / dt / 1e9,
                          "sample": "oracle.replica_copy (memcpy, one thread) of 256 MiB, mean of 3"}
    return out


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from paper_2607_04181_b200 import inputs as I
    shape = I.CFG2
    w = I.make_weights(shape, 1002)
    st = I.make_step_inputs(shape, 2002, 3002)
    # the same sample as the default arm's cpu_baseline (all 64 rows of the batch per step) at the driver's K and W;
    # a much longer run computes fewer rows per step so that it still ends within a few minutes, and says so
    n_runs = max(1, args.steps + args.warmup)
    rows = CPU_BASELINE_ROWS if n_runs <= REF_BUDGET_STEPS else max(1, CPU_BASELINE_ROWS * REF_BUDGET_STEPS // n_runs)
    tps, s_per_step, cores = time_oracle(shape, w, st, rows, args.steps, args.warmup)
    sample = (f"{'all ' if rows == shape.batch else ''}{rows} of the {shape.batch} rows of the cfg2 decode batch per step (full contexts, full layer), "
              f"oracle/cc_oracle.c as it stands, OpenMP over {cores} threads")
    line = {
        "impl": "reference", "metric": METRIC, "value": tps, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": s_per_step * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": "cfg2: Llama-3-8B-shaped decoder layer, decode batch 64, contexts U{512..2048}, "
                               "16-token pages, shuffled block tables", "sample": sample},
        "cpu_baseline": {"value": tps, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": tps, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ---------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist

    from paper_2607_04181_b200 import binding as B
    from paper_2607_04181_b200 import inputs as I
    from paper_2607_04181_b200 import multirank as M
    from paper_2607_04181_b200.harness import CapturedGraph, DeviceStep, Session

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the library has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    shape, R, K, W = I.CFG2, args.replicas, args.steps, max(args.warmup, 3)
    if args.batch:
        shape = shape.with_batch(args.batch)
    batch = shape.batch
    w = I.make_weights(shape, 1002)
    st = I.make_step_inputs(shape, 2002 + 10 * rank, 3002 + 10 * rank)     # every rank its own batch
    assign = I.even_split(batch, R)
    S = Session(shape, w, max_batch=batch, n_slots=3, device_index=local)
    S.scale(R)
    step = DeviceStep(st, assign, device=f"cuda:{local}")
    stream = torch.cuda.current_stream()
    for _ in range(3):
        S.forward(step)
    torch.cuda.synchronize()
    graph = CapturedGraph(lambda s: S.forward(step, s))     # counts instantiations, keeps the cudaGraphExec_t
    n_graphs = CapturedGraph.instantiations
    n_launch = B.cc_forward_launch_count(S.layer)
    gemm_grids = B.cc_layer_gemm_grids(S.layer)          # CTAs and cluster sizes of QKV / O / gate-up / down

    # ---- device-resident timed region: K graph replays ------------------------------------------
    for _ in range(W):
        graph.replay()
    sampler = ClockSampler(local)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    sampler.start()
    ev0.record()
    for _ in range(K):
        graph.replay()
    ev1.record()
    barrier()
    ms_total = ev0.elapsed_time(ev1)
    # the timed region is short (K x ~0.2 ms): keep the same load running for ~1 s so that the NVML
    # poll sees clocks and throttle reasons under this load (not part of any reported time)
    t_end = time.perf_counter() + max(0.0, 1.0 - ms_total / 1e3)
    while time.perf_counter() < t_end:
        for _ in range(50):
            graph.replay()
        torch.cuda.synchronize()
    clocks = sampler.stop()
    value, ms_step = M.job_throughput(batch, K, ms_total, f"cuda:{local}")     # all ranks' tokens / slowest rank's time
    assert B.cc_poll_device_error(S.ctx) == 0

    # ---- per-kernel roofline: the same step launched kernel by kernel with events between ---------
    peak, peak_src = measured_peak()
    n_prof = min(K, 50)
    stage_ms = np.zeros(n_launch, dtype=np.float64)
    for _ in range(3):
        B.cc_forward_profiled(S.layer, step.hidden, step.k_pool, step.v_pool, step.block_table, step.n_pages,
                              step.seq_lens, step.assign, batch, stream)
    for _ in range(n_prof):
        stage_ms += B.cc_forward_profiled(S.layer, step.hidden, step.k_pool, step.v_pool, step.block_table,
                                          step.n_pages, step.seq_lens, step.assign, batch, stream)
    stage_ms /= n_prof
    sb = stage_bytes(shape, st.seq_lens, R)
    # tensor work of the GEMMs: `planes` operand planes (1 = fp16, 2 = bf16 hi + lo), 2 flops per multiply-add
    planes = 1 if B.cc_layer_operand_format(S.layer) == B.CC_OPERAND_F16 else 2
    rows = int((st.seq_lens > 0).sum())
    gemm_flops = {"gemm_qkv": (shape.q_dim + 2 * shape.kv_dim) * shape.hidden, "gemm_o": shape.hidden * shape.q_dim,
                  "gemm_gate_up": 2 * shape.ffn * shape.hidden, "gemm_down": shape.hidden * shape.ffn}
    stages = {}
    for i, name in enumerate(B.STAGE_NAMES):
        e = {"ms": round(float(stage_ms[i]), 5)}
        if name in gemm_flops:
            e["tensor_TFLOPs_issued"] = round(planes * 2.0 * rows * gemm_flops[name] / (stage_ms[i] * 1e-3) / 1e12, 1)
        if name in sb:
            e["bytes"] = sb[name]
            e["GBps"] = round(sb[name] / (stage_ms[i] * 1e-3) / 1e9, 1)
            e["frac"] = round(e["GBps"] / peak, 4)
        stages[name] = e
    dom = max(sb, key=sb.get)
    dom_ms = float(stage_ms[B.STAGE_NAMES.index(dom)])
    achieved = sb[dom] / (dom_ms * 1e-3) / 1e9
    traffic, traffic_src = ncu_traffic(dom, R) if batch == I.CFG2.batch else (None, None)
    roofline = {"bound": "hbm", "kernel": dom, "achieved": round(achieved, 1), "peak": peak, "unit": "GB/s",
                "frac": round(achieved / peak, 4),
                "traffic": traffic, "traffic_source": traffic_src,
                "peak_source": peak_src,
                "kernel_ms": round(dom_ms, 5), "algorithmic_bytes": sb[dom],
                "how": f"mean of {n_prof} launches, CUDA events around the kernel on its stream (cc_forward_profiled)"}
    alg_bytes = I.forward_algorithmic_bytes(shape, st.seq_lens, R)
    step_gbps = alg_bytes / (ms_step * 1e-3) / 1e9

    # ---- other replica counts (outside the timed region; context for the headline) -------------------
    by_r = {}
    for r in (1, 2, 4):
        S.scale(r)
        step.set_assign(I.even_split(batch, r))
        n_r = min(K, 50)
        for _ in range(min(K, 5)):
            graph.replay()
        a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(n_r):
            graph.replay()
        b_.record()
        torch.cuda.synchronize()
        ms = a.elapsed_time(b_) / n_r
        ab = I.forward_algorithmic_bytes(shape, st.seq_lens, r)
        by_r[str(r)] = {"tokens_per_s": round(batch / (ms * 1e-3), 1), "ms_per_step": round(ms, 5),
                        "algorithmic_GBps": round(ab / (ms * 1e-3) / 1e9, 1),
                        "frac_of_peak": round(ab / (ms * 1e-3) / 1e9 / peak, 4)}
    S.scale(R)
    step.set_assign(assign)
    torch.cuda.synchronize()

    # ---- end to end through the C ABI with HOST buffers (pinned): H2D + step + D2H inside the timing ----
    h_hidden = torch.from_numpy(st.hidden.view(np.int16).copy()).pin_memory()
    h_bt = torch.from_numpy(st.block_table.copy()).pin_memory()
    h_sl = torch.from_numpy(st.seq_lens.copy()).pin_memory()
    h_ra = torch.from_numpy(assign.copy()).pin_memory()
    def host_step(fn):
        fn(S.layer, h_hidden, step.k_pool, step.v_pool, step.n_pages, h_bt, h_sl, h_ra, batch, stream)
    for _ in range(W):
        host_step(B.cc_forward_host)
    barrier()
    t0 = time.perf_counter()
    for _ in range(K):
        host_step(B.cc_forward_host)                 # returns after the step's result is in the host buffer
    torch.cuda.synchronize()
    e2e_sync_s = M.max_over_ranks(time.perf_counter() - t0, f"cuda:{local}")
    # the same K steps enqueue-only (cc_forward_host_async): the host marshals step i + 1 while step i runs; one
    # synchronisation at the end, inside the timed region -- every step still moves its inputs and its result over PCIe
    for _ in range(W):
        host_step(B.cc_forward_host_async)
    barrier()
    t0 = time.perf_counter()
    for _ in range(K):
        host_step(B.cc_forward_host_async)
    torch.cuda.synchronize()
    e2e_s = M.max_over_ranks(time.perf_counter() - t0, f"cuda:{local}")
    h2d = h_hidden.numel() * 2 + h_bt.numel() * 4 + h_sl.numel() * 4 + h_ra.numel() * 4
    e2e = {"value": world * batch * K / e2e_s, "unit": UNIT, "h2d_bytes_per_step": int(h2d),
           "d2h_bytes_per_step": int(h_hidden.numel() * 2), "ms_per_step": e2e_s / K * 1e3,
           "ms_per_step_synchronised_every_step": e2e_sync_s / K * 1e3,
           "api": "cc_forward_host_async x K + one stream synchronisation (pinned host hidden/block_table/seq_lens/replica_assign in, "
                  "hidden out; KV pools and weights are device-resident state); cc_forward_host synchronises every step",
           "transfers": "the three tables in one copy-engine transfer; the hidden rows are read over PCIe by the first kernel and the "
                        "result rows stored to the pinned buffer by the last epilogue (same bytes, no separate copies)"}

    # ---- replica creation: cc_scale_layer (chunked copy on the side stream) -> cc_commit (visible) ----
    copy_ms = []
    S.scale(1)
    torch.cuda.synchronize()
    for _ in range(8):
        a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        B.cc_scale_layer(S.layer, 2)
        B.cc_commit(S.layer, stream)              # stream waits for the copy, then the table flip
        b_.record()
        torch.cuda.synchronize()
        copy_ms.append(a.elapsed_time(b_))
        S.scale(1)
        torch.cuda.synchronize()
    cms = float(np.median(copy_ms[2:]))
    blob = S.blob_bytes
    copy_sweep = None
    if args.copy_sweep:                           # chunk size of the side-stream copy (cc_ctx_set_copy_chunk); default 32 MiB
        copy_sweep = {}
        for mib in (4, 8, 16, 32, 64, 128, 512):
            B.cc_ctx_set_copy_chunk(S.ctx, mib << 20)
            ts = []
            for _ in range(8):
                a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record()
                B.cc_scale_layer(S.layer, 2)
                B.cc_commit(S.layer, stream)
                b_.record()
                torch.cuda.synchronize()
                ts.append(a.elapsed_time(b_))
                S.scale(1)
                torch.cuda.synchronize()
            t = float(np.median(ts[2:]))
            copy_sweep[f"{mib}MiB"] = {"ms_call_to_visible": round(t, 4), "GBps_read_plus_write": round(2 * blob / (t * 1e-3) / 1e9, 1)}
        B.cc_ctx_set_copy_chunk(S.ctx, 32 << 20)
    replica_copy = {"blob_bytes": blob, "ms_call_to_visible": round(cms, 4),
                    "GBps_read_plus_write": round(2 * blob / (cms * 1e-3) / 1e9, 1),
                    "GBps_payload": round(blob / (cms * 1e-3) / 1e9, 1),
                    "frac_of_copy_peak": round(2 * blob / (cms * 1e-3) / 1e9 / peak, 4),
                    # measured: graphs instantiated since the step's graph was captured, and whether the
                    # cudaGraphExec_t replayed after the scale-ups / scale-downs above is still the one captured
                    "graph_recaptures": CapturedGraph.instantiations - n_graphs,
                    "same_cuda_graph_exec": bool(graph.same_exec()), "graph_replays": graph.replays}
    if copy_sweep is not None:
        replica_copy["chunk_sweep"] = copy_sweep

    # ---- replica creation WHILE decoding (the one-GPU analogue of PAPER.md:385's "< 3 % fluctuation"): the copy
    # runs on the side stream under a train of graph replays; what does it cost the steps, and the copy? --------
    S.scale(1)
    step.set_assign(I.even_split(batch, 1))
    torch.cuda.synchronize()
    n_train = 8

    def train(with_copy: bool):
        a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        if with_copy:
            B.cc_scale_layer(S.layer, 2)          # returns at once; chunks run on the side stream
        for _ in range(n_train):
            graph.replay()
        b_.record()
        if with_copy:
            B.cc_commit(S.layer, stream)
        torch.cuda.synchronize()
        if with_copy:
            S.scale(1)
            torch.cuda.synchronize()
        return a.elapsed_time(b_)
    for _ in range(2):
        train(False), train(True)
    t_plain = float(np.median([train(False) for _ in range(5)]))
    t_copy = float(np.median([train(True) for _ in range(5)]))
    copy_during_decode = {"steps_in_train": n_train, "replicas_while_decoding": 1,
                          "ms_train_plain": round(t_plain, 4), "ms_train_with_copy": round(t_copy, 4),
                          "step_inflation": round(t_copy / t_plain - 1.0, 4),
                          "what": "8 graph replays at R=1; a 436 MB replica is copied on the side stream meanwhile"}
    S.scale(R)
    step.set_assign(assign)
    torch.cuda.synchronize()

    # ---- a read-only streaming figure for context (torch reduction over 4 GiB; measurement aid, not the product):
    # the driver's peak is a copy (read + write); decode only reads ---------------------------------------------
    big = torch.empty(1 << 30, dtype=torch.float32, device=f"cuda:{local}").fill_(1.0)
    for _ in range(2):
        big.sum()
    a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(5):
        big.sum()
    b_.record()
    torch.cuda.synchronize()
    read_only_gbps = 5 * big.numel() * 4 / (a.elapsed_time(b_) * 1e-3) / 1e9
    del big

    # ---- KV partition per replica (NEXT-1): plan on the host, migrate pages on the device -------------
    kv_migration = None
    try:
        new_bt, src, dst = B.cc_kv_plan_migration(st.block_table, st.seq_lens, I.even_split(batch, 2), st.n_pages, 2)
        page_bytes = shape.n_kv_heads * shape.page * shape.head_dim * 2
        d_src, d_dst = torch.from_numpy(src).to(f"cuda:{local}"), torch.from_numpy(dst).to(f"cuda:{local}")
        mig_ms = []
        for _ in range(6):
            a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            B.cc_kv_migrate(S.ctx, step.k_pool, step.v_pool, page_bytes, d_src, d_dst, len(src), stream)
            b_.record()
            torch.cuda.synchronize()
            mig_ms.append(a.elapsed_time(b_))
        mms = float(np.median(mig_ms[2:]))
        moved = 2 * len(src) * page_bytes                          # K and V
        kv_migration = {"pages_moved": int(len(src)), "bytes_moved": int(moved), "ms": round(mms, 4),
                        "GBps_read_plus_write": round(2 * moved / (mms * 1e-3) / 1e9, 1),
                        "frac_of_copy_peak": round(2 * moved / (mms * 1e-3) / 1e9 / peak, 4),
                        "what": "batch split 32 + 32 over two page partitions; every page outside its replica's partition moved"}
        # the same move list, chunked on a side stream under a train of decode steps: what do the
        # steps pay, what does the copy pay?  (pre-copy protocol: harness.KvLiveMigration, tests/test_kv_migration.py)
        side, ev, n_mt, chunk = torch.cuda.Stream(), torch.cuda.Event(), 4, 4096

        def mtrain(with_mig: bool):
            a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            if with_mig:
                side.wait_stream(stream)
                for c0 in range(0, len(src), chunk):
                    n = min(chunk, len(src) - c0)
                    B.cc_kv_migrate(S.ctx, step.k_pool, step.v_pool, page_bytes, d_src[c0:c0 + n], d_dst[c0:c0 + n], n, side)
                ev.record(side)
            for _ in range(n_mt):
                graph.replay()
            if with_mig:
                stream.wait_event(ev)
            b_.record()
            torch.cuda.synchronize()
            return a.elapsed_time(b_)
        for _ in range(2):
            mtrain(False), mtrain(True)
        tp = float(np.median([mtrain(False) for _ in range(5)]))
        tm = float(np.median([mtrain(True) for _ in range(5)]))
        kv_migration["overlapped"] = {"steps_in_train": n_mt, "chunk_pages": chunk, "ms_train_plain": round(tp, 4),
                                      "ms_train_with_migration": round(tm, 4), "step_inflation": round(tm / tp - 1.0, 4),
                                      "ms_if_serialised": round(tp + mms, 4),
                                      "ms_bandwidth_bound": round(tp + 2 * moved / (peak * 1e9) * 1e3, 4)}
    except B.CcError as e:
        kv_migration = {"error": str(e)}

    # ---- the oracle on this box's host cores, bounded sample (rank 0, N = 1) --------------------------
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        tps, s_per_step, cores = time_oracle(shape, w, st, min(CPU_BASELINE_ROWS, batch), CPU_BASELINE_STEPS, 0)
        cpu = {"value": tps, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"all {min(CPU_BASELINE_ROWS, batch)} rows of the same cfg2 batch, {CPU_BASELINE_STEPS} full layer steps of "
                         f"{s_per_step:.1f} s each, oracle/cc_oracle.c (OpenMP)"}
        cpu.update(cpu_baseline_extras(shape, w, st, cores))
    S.close()

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "bf16", "data": "synthetic",
            "operand_format": "fp16 weight images x one fp16 activation plane, fp32 accumulation" if planes == 1 else
                              "bf16 weight images x two bf16 activation planes (hi + lo), fp32 accumulation",
            "config": {"workload": "cfg2 (BASELINE.json configs[1]): Llama-3-8B-shaped decoder layer, hidden 4096, "
                                   f"32 q / 8 kv heads x 128, FFN 14336, decode batch {batch}, contexts U{{512..2048}}, "
                                   "16-token pages, shuffled block tables",
                       "replicas": R, "batch_split": np.bincount(assign, minlength=R).tolist(),
                       "launch": "one CUDA graph of cc_forward, replayed; PDL between its kernels",
                       "gemm_grids": dict(zip(("ctas", "cluster_size"), gemm_grids)),
                       "l2": "inputs larger than L2: each step streams R x 436 MB weights + 335 MB KV (L2 = 126 MB)",
                       "parallelism": "replicas only (one independent batch per GPU)" if world > 1 else "single GPU"},
            "clocks": clocks,
            "e2e": e2e,
            "gpu_launches": n_launch * K,
            "roofline": roofline,
            "step_roofline": {"algorithmic_bytes": alg_bytes, "achieved_GBps": round(step_gbps, 1),
                              "frac_of_measured_peak": round(step_gbps / peak, 4),
                              "frac_of_8TBps": round(step_gbps / 8000.0, 4),
                              "frac_of_8p18TBps_theoretical": round(step_gbps / 8184.0, 4),
                              "read_only_stream_GBps_torch_sum": round(read_only_gbps, 1),
                              "frac_of_read_only_stream": round(step_gbps / read_only_gbps, 4)},
            "stages": stages,
            "by_replicas": by_r,
            "replica_copy": replica_copy,
            "kv_migration": kv_migration,
            "copy_during_decode": copy_during_decode,
            "cpu_baseline": cpu,
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


# ---------------------------------------------------------------------------------------------
# cfg3 (BASELINE.json configs[2]): whole-model decode graph with mid-run layer flips
# ---------------------------------------------------------------------------------------------
def run_cfg3(args):
    import torch

    from paper_2607_04181_b200 import binding as B
    from paper_2607_04181_b200 import inputs as I
    from paper_2607_04181_b200.harness import CapturedGraph, ModelSession

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the library has no CPU fallback")
    dev = "cuda:0"
    torch.cuda.set_device(0)
    shape = I.CFG2
    n_layers, batch, hot = 32, 128, (10, 11, 12)
    steps = max(args.steps, 30)
    up, down = steps // 3, 2 * steps // 3
    rng = np.random.default_rng(3003)
    ctx = np.clip(np.rint(np.exp(rng.normal(np.log(1024.0), 0.8, batch))), 16, 8192).astype(np.int64)   # lognormal, median 1024
    seq0 = (ctx + 1).astype(np.int32)
    page = shape.page
    need = (seq0.astype(np.int64) + steps + page - 1) // page
    width = int(need.max())
    n_pages = int(need.sum())
    ids = rng.permutation(n_pages).astype(np.int32)                    # shuffled pages, block tables pre-extended
    bt = np.full((batch, width), -1, np.int32)
    off = 0
    for b in range(batch):
        bt[b, :need[b]] = ids[off:off + need[b]]
        off += int(need[b])
    gen = torch.Generator(device=dev).manual_seed(1003)

    def randn(*shp, std=1.0, mean=0.0):
        return (torch.randn(*shp, generator=gen, device=dev, dtype=torch.float32) * std + mean).to(torch.bfloat16)

    d, F, QD, KD = shape.hidden, shape.ffn, shape.q_dim, shape.kv_dim
    def layer_weights():
        return {"g1": randn(d, std=0.02, mean=1.0), "wq": randn(QD, d, std=0.02), "wk": randn(KD, d, std=0.02),
                "wv": randn(KD, d, std=0.02), "wo": randn(d, QD, std=0.02), "g2": randn(d, std=0.02, mean=1.0),
                "wgate": randn(F, d, std=0.02), "wup": randn(F, d, std=0.02), "wdown": randn(d, F, std=0.02)}
    S = ModelSession(shape, [], max_batch=batch, n_slots=len(hot), max_blocks=width, max_position=width * page)
    for _ in range(n_layers):          # one at a time: only one unpacked copy of a layer's weights is alive
        S.add_layer(layer_weights())
    S.donate()
    pool_shape = (n_pages, shape.n_kv_heads, page, shape.head_dim)
    kp = [randn(*pool_shape) for _ in range(n_layers)]
    vp = [randn(*pool_shape) for _ in range(n_layers)]
    hidden = randn(batch, d)
    btd = torch.from_numpy(bt).to(dev)
    sl = torch.from_numpy(seq0.copy()).to(dev)
    assigns = [torch.zeros(batch, dtype=torch.int32, device=dev) for _ in range(n_layers)]
    split = torch.from_numpy(I.even_split(batch, 2)).to(dev)
    stream = torch.cuda.current_stream()
    S.forward_all(hidden, kp, vp, btd, n_pages, sl, assigns, batch)     # warm-up outside capture
    torch.cuda.synchronize()
    def whole_step(s):
        S.forward_all(hidden, kp, vp, btd, n_pages, sl, assigns, batch, s)
        hidden.mul_(0).add_(1.0)         # keep the synthetic hidden state bounded over hundreds of steps (not part of the method)
        sl.add_(1)
    n_graphs = CapturedGraph.instantiations
    graph = CapturedGraph(whole_step)
    exec_handle = graph.exec_handle      # the cudaGraphExec_t
    for _ in range(3):
        graph.replay()
    sl.copy_(torch.from_numpy(seq0))
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    flip_ms = {}
    sampler = ClockSampler(0)
    sampler.start()
    for t in range(steps):
        ev[t][0].record()
        if t == up:
            for l in hot:
                B.cc_scale_layer(S.layers[l], 2)                    # chunked copies on the side stream
            for l in hot:
                B.cc_commit(S.layers[l], stream)                    # stream waits for the copies, then the table flip
                assigns[l].copy_(split)
        if t == down:
            for l in hot:
                assigns[l].zero_()
                B.cc_scale_layer(S.layers[l], 1)
                B.cc_commit(S.layers[l], stream)
        graph.replay()
        ev[t][1].record()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    captures = CapturedGraph.instantiations - n_graphs
    assert B.cc_poll_device_error(S.ctx) == 0 and graph.exec_handle == exec_handle and graph.same_exec() and captures == 1
    ms = np.array([a.elapsed_time(b) for a, b in ev])
    flip_ms = {"scale_up_step_ms": float(ms[up]), "scale_down_step_ms": float(ms[down])}
    # end to end: per step the input rows come from pinned host memory, the result rows go back to it and the host
    # waits for them (it would sample the next tokens from them); host clock around the loop, contexts start over
    e2e_steps = min(steps, 100)
    h_in = torch.empty((batch, d), dtype=torch.bfloat16).pin_memory()
    h_in.copy_(hidden.cpu())
    h_out = torch.empty((batch, d), dtype=torch.bfloat16).pin_memory()
    sl.copy_(torch.from_numpy(seq0))
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        hidden.copy_(h_in, non_blocking=True)
        graph.replay()
        h_out.copy_(hidden, non_blocking=True)
        stream.synchronize()
    e2e_ms = (time.perf_counter() - t0) * 1e3 / e2e_steps
    assert B.cc_poll_device_error(S.ctx) == 0
    def summ(x):
        return {"mean_ms": round(float(x.mean()), 4), "p50_ms": round(float(np.percentile(x, 50)), 4),
                "p99_ms": round(float(np.percentile(x, 99)), 4), "max_ms": round(float(x.max()), 4)}
    before, during, after = ms[:up], ms[up + 1:down], ms[down + 1:]
    kv_tok = float((seq0.astype(np.float64) + steps / 2).sum())
    bytes_step = n_layers * S.blob_bytes + kv_tok * 2 * KD * 2 * n_layers
    peak, peak_src = measured_peak()
    mean_ms = float(np.concatenate([before, during, after]).mean())
    line = {
        "metric": "32-layer decode step (cfg3): tokens/s and per-step latency across replica flips", "value": batch / (mean_ms * 1e-3),
        "unit": UNIT, "n_gpus": 1, "steps": steps, "warmup": 3, "ms_per_step": mean_ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
        "config": {"workload": "cfg3 (BASELINE.json configs[2]): 32 Llama-3-8B-shaped layers, decode batch 128, contexts lognormal "
                               "(median 1024, sigma 0.8, capped 8192), one CUDA graph for the whole step, seq_lens incremented "
                               f"inside it; layers {list(hot)} scaled to 2 replicas at step {up} and back to 1 at step {down}",
                   "graph_captures": captures, "same_cuda_graph_exec": bool(graph.same_exec()), "graph_replays": graph.replays,
                   "note": "hidden is reset to a constant inside the graph every step to keep the synthetic state bounded"},
        "clocks": clocks,
        "latency": {"before": summ(before), "while_2_replicas": summ(during), "after": summ(after), **flip_ms},
        "replica_creation": {"layers": len(hot), "bytes_each": S.blob_bytes,
                             "extra_ms_of_the_flip_step": round(float(ms[up] - before.mean()), 4)},
        "step_roofline": {"algorithmic_bytes_mid_run": int(bytes_step), "achieved_GBps": round(bytes_step / (mean_ms * 1e-3) / 1e9, 1),
                          "frac_of_measured_peak": round(bytes_step / (mean_ms * 1e-3) / 1e9 / peak, 4), "peak_source": peak_src},
        "gpu_launches": int(B.cc_forward_launch_count(S.layers[0])) * n_layers * steps,
        "e2e": {"value": batch / (e2e_ms * 1e-3), "unit": UNIT, "ms_per_step": e2e_ms, "steps": e2e_steps,
                "h2d_bytes_per_step": int(h_in.numel() * 2), "d2h_bytes_per_step": int(h_out.numel() * 2),
                "how": "per step: the hidden rows copied from pinned host memory, one replay of the 32-layer graph, the result rows "
                       "copied back, one stream synchronisation; host clock; all layers at 1 replica"},
    }
    print(json.dumps(line), flush=True)
    S.close()
    return 0


# ---------------------------------------------------------------------------------------------
# cfg5 (BASELINE.json configs[4]): skewed co-located serving, decode only (no prefill kernel yet: NEXT-2)
# ---------------------------------------------------------------------------------------------
def run_cfg4(args):
    """BASELINE.json configs[3]: the 14B-class shape, a mixed step of two 2048-token prompt chunks and 256 decode rows
    (contexts U{256..4096}) = 4352 rows in ONE cc_forward per layer through the large-M path: k_big_group, CTA-pair
    tcgen05 GEMMs with fused epilogues, chunk-prefill attention on tcgen05 for the prompts, the page-range decode
    attention for the decode rows.  --layers L runs L layers in one graph, the top 25 % by a
    seeded synthetic per-layer load at R = 2 (prompt r on replica r % 2, decode rows split evenly), the rest at R = 1;
    the default is one hot layer.  The GEMMs are tensor-bound here: their roofline is the measured bf16 GEMM peak."""
    import torch

    from paper_2607_04181_b200 import binding as B
    from paper_2607_04181_b200 import inputs as I
    from paper_2607_04181_b200.harness import CapturedGraph, ModelSession

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the library has no CPU fallback")
    dev = "cuda:0"
    torch.cuda.set_device(0)
    shape = I.CFG4_LAYER
    n_layers = max(1, args.layers)
    page, n_dec, prompt, n_prompts = shape.page, 256, 2048, 2
    rows = n_prompts * prompt + n_dec
    rng = np.random.default_rng(3004)
    dec_ctx = rng.integers(256, 4097, n_dec)                                  # decode contexts U{256..4096}
    width = (4096 + 1 + page - 1) // page
    need = np.concatenate([[prompt // page] * n_prompts, (dec_ctx + 1 + page - 1) // page]).astype(np.int64)
    n_pages = int(need.sum())
    ids = rng.permutation(n_pages).astype(np.int32)
    req_bt = np.full((n_prompts + n_dec, width), -1, np.int32)
    off = 0
    for i, n in enumerate(need):
        req_bt[i, :n] = ids[off:off + n]
        off += int(n)
    # rows: prompt 0 (tokens 0..2047 at seq_len t + 1, sharing its request's block-table row), prompt 1, the decode rows
    bt = np.concatenate([np.repeat(req_bt[r:r + 1], prompt, 0) for r in range(n_prompts)] + [req_bt[n_prompts:]]).astype(np.int32)
    seq = np.concatenate([np.arange(1, prompt + 1)] * n_prompts + [dec_ctx + 1]).astype(np.int32)
    hot_assign = np.concatenate([np.full(prompt, r % 2) for r in range(n_prompts)] + [I.even_split(n_dec, 2)]).astype(np.int32)
    load = np.random.default_rng(3104).lognormal(0.0, 1.0, n_layers)
    hot = sorted(np.argsort(-load)[:max(1, n_layers // 4)].tolist())          # top 25 % by synthetic load (one layer: that layer)
    gen = torch.Generator(device=dev).manual_seed(1004)

    def randn(*shp, std=1.0, mean=0.0):
        return (torch.randn(*shp, generator=gen, device=dev, dtype=torch.float32) * std + mean).to(torch.bfloat16)
    d, F, QD, KD = shape.hidden, shape.ffn, shape.q_dim, shape.kv_dim
    S = ModelSession(shape, [], max_batch=rows, n_slots=len(hot), max_blocks=width, max_position=width * page)
    for _ in range(n_layers):
        S.add_layer({"g1": randn(d, std=0.02, mean=1.0), "wq": randn(QD, d, std=0.02), "wk": randn(KD, d, std=0.02),
                     "wv": randn(KD, d, std=0.02), "wo": randn(d, QD, std=0.02), "g2": randn(d, std=0.02, mean=1.0),
                     "wgate": randn(F, d, std=0.02), "wup": randn(F, d, std=0.02), "wdown": randn(d, F, std=0.02)})
    S.donate()
    for l in hot:
        S.scale(l, 2)
    pool_shape = (n_pages, shape.n_kv_heads, page, shape.head_dim)
    # one KV pool per layer while that fits beside the weights; many layers share a few pools round-robin (every layer
    # still streams its own 2.3 GB of decode KV from HBM each step -- far more than L2 -- and appends its rows)
    n_pools = min(n_layers, 8)
    pools = [(randn(*pool_shape), randn(*pool_shape)) for _ in range(n_pools)]
    hidden0 = randn(rows, d)
    hidden = hidden0.clone()
    d_bt, d_seq = torch.from_numpy(bt).to(dev), torch.from_numpy(seq).to(dev)
    d_hot, d_cold = torch.from_numpy(hot_assign).to(dev), torch.zeros(rows, dtype=torch.int32, device=dev)
    stream = torch.cuda.current_stream()

    def mixed_step(st):
        hidden.copy_(hidden0)                                                 # a fresh batch every step (the layers update it in place)
        for l in range(n_layers):
            kp, vp = pools[l % n_pools]
            B.cc_forward(S.layers[l], hidden, kp, vp, d_bt, n_pages, d_seq, d_hot if l in hot else d_cold, rows, st)
    mixed_step(stream)
    torch.cuda.synchronize()
    assert B.cc_poll_device_error(S.ctx) == 0
    graph = CapturedGraph(mixed_step)
    K, W = max(args.steps // 10, 10), max(args.warmup // 4, 3)
    for _ in range(W):
        graph.replay()
    sampler = ClockSampler(0)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(K):
        graph.replay()
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / K
    t_end = time.perf_counter() + 1.0
    while time.perf_counter() < t_end:
        graph.replay()
        torch.cuda.synchronize()
    clocks = sampler.stop()
    # per-kernel times of one hot layer's step (kernel by kernel, events between)
    kp, vp = pools[hot[0] % n_pools]
    stage = None
    for rep in range(4):
        t = B.cc_forward_profiled(S.layers[hot[0]], hidden, kp, vp, d_bt, n_pages, d_seq, d_hot, rows, stream).astype(np.float64)
        stage = t if stage is None else np.minimum(stage, t)
    names = B.BIG_STAGE_NAMES
    planes = 1 if B.cc_layer_operand_format(S.layers[0]) == B.CC_OPERAND_F16 else 2
    n_w = {"gemm_qkv": d * (QD + 2 * KD), "gemm_o": QD * d, "gemm_gate_up": 2 * d * F, "gemm_down": d * F}
    # tensor work issued per projection: the large-step plane policy is {x: 2, o: 1, y: 1, a: 1} for fp16 layers (cc_api.cu)
    pl = {"gemm_qkv": 2, "gemm_o": planes, "gemm_gate_up": planes, "gemm_down": planes}
    peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))) if os.path.exists(os.path.join(ROOT, "MEASURED_PEAKS.json")) else {}
    sust = peaks.get("bf16_tflops_sustained")
    gemm = {}
    for n in n_w:
        t_ms = float(stage[names.index(n)])
        gemm[n] = {"ms": round(t_ms, 4), "useful_TFLOPs": round(2.0 * rows * n_w[n] / (t_ms * 1e-3) / 1e12, 1),
                   "issued_TFLOPs": round(pl[n] * 2.0 * rows * n_w[n] / (t_ms * 1e-3) / 1e12, 1), "planes": pl[n]}
    gemm_ms = sum(float(stage[names.index(n)]) for n in n_w)
    useful = 2.0 * rows * sum(n_w.values()) / (gemm_ms * 1e-3) / 1e12
    issued = sum(pl[n] * 2.0 * rows * n_w[n] for n in n_w) / (gemm_ms * 1e-3) / 1e12
    # attention work: prompts (causal, 4 * n^2 / 2 * Hq * Dh flop each; x 2 for the hi + lo planes of q and p) and decode KV bytes
    pf_flop = n_prompts * 4.0 * (prompt * (prompt + 1) / 2) * QD
    pf_ms, dec_ms = float(stage[names.index("attention_prefill")]), float(stage[names.index("attention_decode")])
    dec_bytes = int((dec_ctx + 1).sum()) * 2 * KD * 2
    hbm, _ = measured_peak()
    S.close()
    line = {
        "metric": "mixed prefill + decode step (cfg4): tokens/s", "value": rows / (ms * 1e-3), "unit": UNIT,
        "n_gpus": 1, "steps": K, "warmup": W, "ms_per_step": ms, "ms_per_layer": ms / n_layers, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
        "operand_format": "fp16 weight images; activation planes per projection below" if planes == 1 else "bf16 x two planes",
        "config": {"workload": f"cfg4 (BASELINE.json configs[3]): {n_layers} layer(s) of hidden 5120, 40 q / 8 kv heads x 128, FFN 17408; "
                               "mixed step = 2 x 2048 prompt tokens (chunk prefill from position 0) + 256 decode rows (contexts U{256..4096}) "
                               "= 4352 rows in one cc_forward per layer (large-M path), one CUDA graph",
                   "layers": n_layers, "hot_layers_at_R2": hot, "kv_pools": n_pools,
                   "l2": "each layer streams 0.66-1.3 GB of weights and 2.3 GB of decode KV per step (L2 = 126 MB)"},
        "clocks": clocks, "gpu_launches": K * n_layers * len(names),
        "roofline": {"bound": "tensor", "kernel": "the four large-M GEMMs of one layer step", "achieved": round(useful, 1),
                     "achieved_issued": round(issued, 1), "peak": sust, "unit": "TFLOP/s",
                     "frac": round(useful / sust, 4) if sust else None, "frac_issued": round(issued / sust, 4) if sust else None,
                     "peak_source": "MEASURED_PEAKS.json bf16_tflops_sustained (cuBLAS bf16, seconds-long loop)", "traffic": None,
                     "how": "useful = 2 * rows * weights flop; issued counts the second activation plane of the QKV projection"},
        "gemm": gemm,
        "attention": {"prefill_ms": round(pf_ms, 4), "prefill_useful_TFLOPs": round(pf_flop / (pf_ms * 1e-3) / 1e12, 1),
                      "prefill_issued_TFLOPs": round(2 * pf_flop / (pf_ms * 1e-3) / 1e12, 1),
                      "decode_ms": round(dec_ms, 4), "decode_kv_bytes": dec_bytes,
                      "decode_GBps": round(dec_bytes / (dec_ms * 1e-3) / 1e9, 1), "decode_frac_of_hbm_peak": round(dec_bytes / (dec_ms * 1e-3) / 1e9 / hbm, 4)},
        "stages_ms": {n: round(float(x), 4) for n, x in zip(names, stage)},
        "sum_of_stages_ms": round(float(stage.sum()), 4),
    }
    print(json.dumps(line), flush=True)
    return 0


def run_cfg5(args):
    import torch

    from paper_2607_04181_b200 import inputs as I
    from paper_2607_04181_b200 import serving as S

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the library has no CPU fallback")
    torch.cuda.set_device(0)
    rng = np.random.default_rng(3005)
    load = rng.lognormal(0.0, 1.0, 32)                               # synthetic per-layer load: the top 25 % are "hot"
    hot = tuple(sorted(np.argsort(-load)[:8].tolist()))
    arrivals = S.make_arrivals(seed=3005, horizon_s=args.horizon, base_rps=7.0, burst_x=5.0, burst_len_s=10.0, burst_every_s=60.0,
                               frac_a=0.75, prompt_mean=512, out_mean=256, sigma=1.0, max_prompt=4096, max_out=1024)
    shape_a = I.CFG2
    shape_b = I.MODEL_B_LAYER
    A = S.ModelRunner("A", shape_a, 32, 128, 12000, 5120, seed=1005, n_slots=0, hot_layers=hot, prefill_rows=args.prefill_rows)
    Bm = S.ModelRunner("B", shape_b, 28, 64, 6000, 5120, seed=1006, n_slots=0, prefill_rows=args.prefill_rows // 2)
    sampler = ClockSampler(0)
    sampler.start()
    t0 = time.perf_counter()
    out, _ = S.simulate(A, Bm, arrivals, burst_hi=48, burst_lo=16)
    wall = time.perf_counter() - t0
    clocks = sampler.stop()
    A.close()
    Bm.close()
    line = {
        "metric": "co-located serving (cfg5): model A tokens/s and per-token latency", "value": out["A"]["tokens_per_s_while_stepping"],
        "unit": UNIT, "n_gpus": 1, "steps": out["steps"], "warmup": 0,
        "ms_per_step": 1e3 * out["clock_s"] / max(1, out["steps"]), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
        "config": {"workload": "cfg5 (BASELINE.json configs[4]): model A = 32 Llama-3-8B-shaped layers (75 % of the requests), model B = 28 "
                               "layers of hidden 1536 / 12 q / 2 kv heads x 128 / FFN 8960; Poisson arrivals 7 req/s with 5x bursts of 10 s every "
                               f"60 s over {args.horizon:.0f} s, prompts lognormal (mean 512), outputs lognormal (mean 256); "
                               + (f"mixed steps: up to {args.prefill_rows} (A) / {args.prefill_rows // 2} (B) prompt tokens per step run as rows of "
                                  "the decode path (causal chunked prefill through the decode kernels; the large-M prefill kernels are not built); "
                                  if args.prefill_rows else "decode only: prompts count as cached KV; ") +
                               "A's 8 hot layers get a second replica in memory lent from B's KV reserve "
                               "while A's backlog is >= 48 requests",
                   "hot_layers": list(hot), "requests": len(arrivals)},
        "clocks": clocks, "serving": out, "wall_s": round(wall, 1),
    }
    print(json.dumps(line), flush=True)
    return 0


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.workload == "cfg5":
        return run_cfg5(args)
    if args.workload == "cfg3":
        return run_cfg3(args)
    if args.workload == "cfg4":
        return run_cfg4(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
