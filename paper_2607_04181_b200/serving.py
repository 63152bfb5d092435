"""Minimal co-located serving loop (BASELINE.json configs[4]): two models on one GPU,
continuous batching of decode steps, a paged-KV allocator per model, and layer-wise scaling of the hot model's
hot layers into memory reclaimed from the cold model's KV budget.

Prefill: with prefill_rows = 0 a request's prompt counts as already cached KV (pages are allocated, their contents
are whatever the pool holds) and only decode steps run.  With prefill_rows = P every step is a MIXED step: beside the
decode rows it carries up to P tokens of the oldest admitted prompt as rows that share the request's block-table row
at consecutive seq_lens -- causal chunked prefill through the decode kernels (tests/test_prefill_chunk.py; the
efficient prefill kernels are NEXT-2) -- and a request starts decoding when its prompt is done, so the first token's
latency includes its prefill.  Time is the sum of the measured
device times of the steps (CUDA events); arrivals are a seeded synthetic process on that clock.  Parity: unpinned
by the paper; the tests check conservation (every request finishes with its token count, no page is lost or
shared) and that the steps go through the same cc_forward graphs as everything else.

No arithmetic of the method lives here: torch is device memory, streams, graphs and events.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np
import torch

from . import binding as B
from . import inputs as I
from .harness import CapturedGraph, ModelSession


@dataclass
class Request:
    rid: int
    model: str
    arrival: float          # seconds on the simulated clock
    prompt: int             # prompt tokens (treated as cached when the runner has no prefill rows)
    out_len: int            # tokens to generate
    prefilled: int = 0      # prompt tokens whose KV has been computed
    pages: list = field(default_factory=list)
    slot: int = -1
    generated: int = 0
    admitted: float = -1.0
    last_token_at: float = -1.0
    finished: float = -1.0


def make_arrivals(seed: int, horizon_s: float, base_rps: float, burst_x: float, burst_len_s: float, burst_every_s: float,
                  frac_a: float, prompt_mean: float, out_mean: float, sigma: float = 1.0, max_prompt: int = 4096,
                  max_out: int = 1024):
    """Poisson arrivals with rate base_rps, multiplied by burst_x during [k*burst_every, k*burst_every + burst_len);
    lognormal prompt / output lengths with the given means (mu = ln(mean) - sigma^2 / 2)."""
    rng = np.random.default_rng(seed)
    t, out, rid = 0.0, [], 0
    while True:
        rate = base_rps * (burst_x if (t % burst_every_s) < burst_len_s else 1.0)
        t += rng.exponential(1.0 / rate)
        if t >= horizon_s:
            break
        model = "A" if rng.random() < frac_a else "B"
        prompt = int(np.clip(np.rint(rng.lognormal(np.log(prompt_mean) - sigma * sigma / 2, sigma)), 1, max_prompt))
        olen = int(np.clip(np.rint(rng.lognormal(np.log(out_mean) - sigma * sigma / 2, sigma)), 1, max_out))
        out.append(Request(rid, model, t, prompt, olen))
        rid += 1
    return out


class PagePool:
    """Lowest-free-page-first allocator over [0, limit) of a pool of n_pages (limit < n_pages while the tail is lent)."""

    def __init__(self, n_pages: int):
        self.n_pages, self.limit = n_pages, n_pages
        self.free = np.ones(n_pages, dtype=bool)

    def alloc(self, n: int):
        idx = np.nonzero(self.free[:self.limit])[0]
        if len(idx) < n:
            return None
        take = idx[:n]
        self.free[take] = False
        return take.tolist()

    def release(self, pages) -> None:
        assert not self.free[pages].any()
        self.free[pages] = True

    def used(self) -> int:
        return int((~self.free).sum())

    def high_water(self) -> int:
        u = np.nonzero(~self.free)[0]
        return int(u[-1]) + 1 if len(u) else 0


class ModelRunner:
    """One model: L layers of one shape in one CUDA graph, a page pool shared by its layers (the same page ids in
    every layer's K/V pool), request slots = rows of the decode batch."""

    def __init__(self, name: str, shape: I.LayerShape, n_layers: int, max_batch: int, n_pages: int, max_tokens: int,
                 seed: int, n_slots: int, hot_layers=(), device: str = "cuda:0", prefill_rows: int = 0):
        self.n_decode, self.P = max_batch, prefill_rows            # rows [0, n_decode): request slots; then the prompt chunk
        max_batch = max_batch + prefill_rows                       # rows of the captured step
        self.name, self.shape, self.L, self.max_batch, self.dev = name, shape, n_layers, max_batch, device
        self.width = (max_tokens + shape.page - 1) // shape.page
        gen = torch.Generator(device=device).manual_seed(seed)

        def randn(*shp, std=1.0, mean=0.0):
            return (torch.randn(*shp, generator=gen, device=device, dtype=torch.float32) * std + mean).to(torch.bfloat16)
        d, F, QD, KD = shape.hidden, shape.ffn, shape.q_dim, shape.kv_dim
        self.M = ModelSession(shape, [], max_batch=max_batch, n_slots=n_slots, max_blocks=self.width,
                              max_position=self.width * shape.page)
        for _ in range(n_layers):
            self.M.add_layer({"g1": randn(d, std=0.02, mean=1.0), "wq": randn(QD, d, std=0.02), "wk": randn(KD, d, std=0.02),
                              "wv": randn(KD, d, std=0.02), "wo": randn(d, QD, std=0.02), "g2": randn(d, std=0.02, mean=1.0),
                              "wgate": randn(F, d, std=0.02), "wup": randn(F, d, std=0.02), "wdown": randn(d, F, std=0.02)})
        self.M.donate()
        pool_shape = (n_pages, shape.n_kv_heads, shape.page, shape.head_dim)
        self.kp = [randn(*pool_shape) for _ in range(n_layers)]
        self.vp = [randn(*pool_shape) for _ in range(n_layers)]
        self.pool = PagePool(n_pages)
        self.n_pages = n_pages
        self.hidden_src = randn(max_batch, d)
        self.hidden = self.hidden_src.clone()
        self.bt_host = torch.full((max_batch, self.width), -1, dtype=torch.int32).pin_memory()
        self.sl_host = torch.zeros(max_batch, dtype=torch.int32).pin_memory()
        self.bt = self.bt_host.to(device)
        self.sl = self.sl_host.to(device)
        self.assigns = [torch.zeros(max_batch, dtype=torch.int32, device=device) for _ in range(n_layers)]
        self.hot = tuple(hot_layers)
        self.replicas = 1
        self.slots = [None] * self.n_decode
        self.prefilling = []            # admitted requests whose prompt is not done yet, oldest first
        self.prompt_tokens = 0
        self._decoded = []              # slots that decoded a token in the last step
        self.graph = None
        self.captures = 0
        self.scale_events = []          # (clock, n_replicas, ms, GB/s read+write)

    def capture(self) -> None:
        M = self.M
        M.forward_all(self.hidden, self.kp, self.vp, self.bt, self.n_pages, self.sl, self.assigns, self.max_batch)
        torch.cuda.synchronize()
        def whole_step(s):
            self.hidden.copy_(self.hidden_src)            # the synthetic "embedding" of the step (keeps the state bounded)
            M.forward_all(self.hidden, self.kp, self.vp, self.bt, self.n_pages, self.sl, self.assigns, self.max_batch, s)
        before = CapturedGraph.instantiations
        self.graph = CapturedGraph(whole_step)            # replay() refuses any other cudaGraphExec_t
        self.captures += CapturedGraph.instantiations - before

    # ---- requests ----------------------------------------------------------------------------------------------
    def active(self):
        return [r for r in self.slots if r is not None]

    def try_admit(self, r: Request, now: float) -> bool:
        if None not in self.slots:
            return False
        need = (r.prompt + r.out_len + self.shape.page - 1) // self.shape.page     # reserve the whole request: no stalls later
        if need > self.width:
            need = self.width
            r.out_len = max(1, self.width * self.shape.page - r.prompt)
        pages = self.pool.alloc(need)
        if pages is None:
            return False
        r.pages, r.slot, r.admitted, r.last_token_at = pages, self.slots.index(None), now, now
        self.slots[r.slot] = r
        self.bt_host[r.slot].fill_(-1)
        self.bt_host[r.slot, :need] = torch.tensor(pages, dtype=torch.int32)
        if self.P > 0:
            r.prefilled = 0
            self.prefilling.append(r)
        else:
            r.prefilled = r.prompt
        return True

    def step(self) -> float:
        """One step: a decode token for every request whose prompt is done and, with prefill rows, the next chunk of the
        oldest unfinished prompt; returns the device time in seconds."""
        self._decoded = []
        for b, r in enumerate(self.slots):
            live = r is not None and r.prefilled >= r.prompt
            self.sl_host[b] = r.prompt + r.generated + 1 if live else 0
            if live:
                self._decoded.append(b)
        chunk = 0
        if self.P > 0:
            self.sl_host[self.n_decode:] = 0
            if self.prefilling:
                r = self.prefilling[0]
                chunk = min(self.P, r.prompt - r.prefilled)
                rows = slice(self.n_decode, self.n_decode + chunk)
                self.bt_host[rows] = self.bt_host[r.slot]                          # the chunk's rows share the request's pages
                self.sl_host[rows] = torch.arange(r.prefilled + 1, r.prefilled + chunk + 1, dtype=torch.int32)
        self.bt.copy_(self.bt_host, non_blocking=True)
        self.sl.copy_(self.sl_host, non_blocking=True)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        self.graph.replay()
        e1.record()
        e1.synchronize()
        if chunk:
            r = self.prefilling[0]
            r.prefilled += chunk
            self.prompt_tokens += chunk
            if r.prefilled >= r.prompt:
                self.prefilling.pop(0)                                             # decodes from the next step on
        return e0.elapsed_time(e1) * 1e-3

    def finish_tokens(self, now: float, lat_out: list, done_out: list) -> None:
        for b in self._decoded:
            r = self.slots[b]
            r.generated += 1
            lat_out.append(now - r.last_token_at)
            r.last_token_at = now
            if r.generated >= r.out_len:
                r.finished = now
                self.pool.release(r.pages)
                self.slots[b] = None
                done_out.append(r)

    # ---- layer-wise scaling of the hot layers (no recapture) --------------------------------------
    def scale_hot(self, n: int, now: float) -> None:
        if n == self.replicas:
            return
        stream = torch.cuda.current_stream()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for l in self.hot:
            B.cc_scale_layer(self.M.layers[l], n)
        for l in self.hot:
            B.cc_commit(self.M.layers[l], stream)
        e1.record()
        e1.synchronize()
        split = torch.arange(self.max_batch, dtype=torch.int32, device=self.dev) % n
        split[self.n_decode:] = n - 1        # the rows of a prompt chunk are ONE request: one replica (
                                             # rows of one request on two replicas raise CC_DEVERR_SPLIT_REQUEST)
        for l in self.hot:
            self.assigns[l].copy_(split)
        ms = e0.elapsed_time(e1)
        grown = max(0, n - self.replicas) * len(self.hot)
        gbps = 2 * grown * self.M.blob_bytes / (ms * 1e-3) / 1e9 if grown else 0.0
        self.scale_events.append((now, n, ms, gbps))
        self.replicas = n

    def close(self) -> None:
        self.graph = None
        self.M.close()


def simulate(A: ModelRunner, Bm: ModelRunner, arrivals, burst_hi: int, burst_lo: int, max_steps: int = 1_000_000):
    """Continuous batching of A and B on one GPU.  Policy (a stand-in for the paper's controller, which needs a latency
    model of a multi-device cluster): when A's backlog (waiting + running requests) reaches burst_hi, B's KV reserve is
    lent to A's context and A's hot layers get a second replica; when it falls to burst_lo they are released and the
    memory goes back.  Returns a dict of measurements."""
    dev = A.dev
    slot_bytes = (A.M.blob_bytes + 1023) // 1024 * 1024
    b_reserve = torch.empty(len(A.hot) * slot_bytes + 2048, dtype=torch.uint8, device=dev)   # part of B's KV budget, idle
    lent = False
    for m in (A, Bm):
        m.capture()
    queue = {"A": [], "B": []}
    pending = sorted(arrivals, key=lambda r: r.arrival)
    nxt, now, steps = 0, 0.0, 0
    lat = {"A": [], "B": []}
    done = {"A": [], "B": []}
    step_s = {"A": [], "B": []}
    a_batch_trace = []
    while steps < max_steps:
        while nxt < len(pending) and pending[nxt].arrival <= now:
            queue[pending[nxt].model].append(pending[nxt])
            nxt += 1
        for name, m in (("A", A), ("B", Bm)):
            q = queue[name]
            while q and m.try_admit(q[0], now):
                q.pop(0)
        backlog = len(queue["A"]) + len(A.active())
        if A.hot and not lent and backlog >= burst_hi:
            B.cc_ctx_donate(A.M.ctx, b_reserve, b_reserve.numel())
            A.scale_hot(2, now)
            lent = True
        elif lent and backlog <= burst_lo:
            A.scale_hot(1, now)
            torch.cuda.synchronize()
            B.cc_ctx_reclaim(A.M.ctx, b_reserve)
            lent = False
        ran = False
        for name, m in (("A", A), ("B", Bm)):
            if m.active():
                dt = m.step()
                now += dt
                steps += 1
                step_s[name].append((dt, len(m.active()), m.replicas))
                m.finish_tokens(now, lat[name], done[name])
                ran = True
        a_batch_trace.append(len(A.active()))
        if not ran:
            if nxt >= len(pending):
                break
            now = max(now, pending[nxt].arrival)        # idle: jump to the next arrival
    if lent:
        A.scale_hot(1, now)
        torch.cuda.synchronize()
        B.cc_ctx_reclaim(A.M.ctx, b_reserve)

    def pct(x, p):
        return float(np.percentile(x, p)) if len(x) else None

    out = {"clock": "simulated: the sum of the measured device times of the steps (no host time, no queueing outside a step)",
           "clock_s": now, "steps": steps, "requests": {k: len(v) for k, v in done.items()},
           "unfinished": {k: len(queue[k]) + len(m.active()) for k, m in (("A", A), ("B", Bm))},
           "graph_captures": {"A": A.captures, "B": Bm.captures}}
    for name, m in (("A", A), ("B", Bm)):
        toks = sum(r.generated for r in done[name])
        busy = sum(s[0] for s in step_s[name])
        out[name] = {"tokens": toks, "tokens_per_s_wall": toks / now if now else None,
                     "tokens_per_s_while_stepping": toks / busy if busy else None,
                     "per_layer_step_us_mean": 1e6 * busy / max(1, len(step_s[name])) / m.L,
                     "token_latency_ms_p50": None if not lat[name] else 1e3 * pct(lat[name], 50),
                     "token_latency_ms_p99": None if not lat[name] else 1e3 * pct(lat[name], 99),
                     "mean_batch": float(np.mean([s[1] for s in step_s[name]])) if step_s[name] else 0.0,
                     "prompt_tokens_prefilled": m.prompt_tokens, "prefill_rows": m.P,
                     "pages_in_use_at_end": m.pool.used()}
    by_rep = {}
    for dt, nb, rep in step_s["A"]:
        by_rep.setdefault(rep, []).append(dt / max(nb, 1))
    out["A"]["s_per_token_by_replicas"] = {str(k): float(np.mean(v)) for k, v in by_rep.items()}
    out["A"]["scale_events"] = [{"clock_s": round(t, 4), "replicas": n, "ms": round(ms, 3), "copy_GBps_read_plus_write": round(g, 1)}
                                for t, n, ms, g in A.scale_events]
    out["A"]["max_batch_seen"] = int(max(a_batch_trace)) if a_batch_trace else 0
    return out, done
