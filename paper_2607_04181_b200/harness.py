"""Plumbing shared by tests/, bench.py and __graft_entry__.smoke(): moves the seeded inputs of
`inputs.py` into torch CUDA tensors and drives the C ABI through `binding`.  No arithmetic of the
method lives here -- torch is used for device memory, streams and CUDA graphs only.
"""
from __future__ import annotations

import numpy as np
import torch

from . import binding as B
from . import inputs as I


def _dev_u16(a: np.ndarray, device) -> torch.Tensor:
    """uint16 bf16 bit patterns -> torch bf16 tensor on the device (bit-exact)."""
    t = torch.from_numpy(np.ascontiguousarray(a).view(np.int16))
    return t.to(device).view(torch.bfloat16)


def _host_u16(t: torch.Tensor) -> np.ndarray:
    return t.detach().cpu().contiguous().view(torch.int16).numpy().view(np.uint16).copy()


def make_desc(shape: I.LayerShape, max_batch: int, max_blocks: int | None = None,
              max_position: int | None = None) -> B.cc_layer_desc:
    mb = shape.max_blocks if max_blocks is None else max_blocks
    mp = mb * shape.page if max_position is None else max_position
    return B.cc_layer_desc(shape.hidden, shape.n_q_heads, shape.n_kv_heads, shape.head_dim, shape.ffn,
                           shape.rms_eps, shape.rope_base, shape.page, max_batch, mb, mp)


class CapturedGraph:
    """A CUDA graph captured ONCE, with the evidence for "no recapture" (north_star; the paper re-captures when the
    replica set changes): the `cudaGraphExec_t` handle taken right after instantiation, a class-wide
    count of instantiations (every capture in tests and bench goes through here, so `instantiations` minus the
    number of graphs alive is the number of re-captures), and `replay()` refusing to launch anything but that
    handle.  Plumbing only: torch captures and launches; the kernels inside come from the C ABI."""

    instantiations = 0

    def __init__(self, enqueue):
        """`enqueue(stream)` issues the work to capture (it is called exactly once, under capture)."""
        self.graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(self.graph):
            enqueue(torch.cuda.current_stream())
        CapturedGraph.instantiations += 1
        self.exec_handle = int(self.graph.raw_cuda_graph_exec())    # the cudaGraphExec_t itself
        self.replays = 0

    def same_exec(self) -> bool:
        return int(self.graph.raw_cuda_graph_exec()) == self.exec_handle

    def replay(self) -> None:
        assert self.same_exec(), "the graph was re-instantiated"
        self.graph.replay()
        self.replays += 1


class DeviceStep:
    """One batch of step inputs resident in HBM."""

    def __init__(self, st: I.StepInputs, assign: np.ndarray, device="cuda:0"):
        self.device = device
        self.batch = st.hidden.shape[0]
        self.n_pages = st.n_pages
        self.hidden = _dev_u16(st.hidden, device)
        self.k_pool = _dev_u16(st.k_pool, device)
        self.v_pool = _dev_u16(st.v_pool, device)
        self.block_table = torch.from_numpy(st.block_table).to(device)
        self.seq_lens = torch.from_numpy(st.seq_lens).to(device)
        self.assign = torch.from_numpy(np.ascontiguousarray(assign, dtype=np.int32)).to(device)

    def reset(self, st: I.StepInputs) -> None:
        """Re-upload hidden and the KV pools (both are modified in place by a step)."""
        self.hidden.copy_(_dev_u16(st.hidden, self.device))
        self.k_pool.copy_(_dev_u16(st.k_pool, self.device))
        self.v_pool.copy_(_dev_u16(st.v_pool, self.device))

    def set_assign(self, assign: np.ndarray) -> None:
        self.assign.copy_(torch.from_numpy(np.ascontiguousarray(assign, dtype=np.int32)))

    def out_bits(self) -> np.ndarray:
        return _host_u16(self.hidden)

    def pools_bits(self):
        return _host_u16(self.k_pool), _host_u16(self.v_pool)


class Session:
    """Context + one layer + a donated arena for replica slots."""

    def __init__(self, shape: I.LayerShape, weights: dict, max_batch: int, n_slots: int = I.MAX_REPLICAS - 1,
                 device_index: int = 0, max_blocks: int | None = None, max_position: int | None = None,
                 operand_format: int | None = None):
        self.shape = shape
        self.device = f"cuda:{device_index}"
        torch.cuda.set_device(device_index)
        self.ctx = B.cc_ctx_create(device_index)
        if operand_format is not None:
            B.cc_ctx_set_operand_format(self.ctx, operand_format)
        self.desc = make_desc(shape, max_batch, max_blocks, max_position)
        wdev = {k: _dev_u16(v, self.device) for k, v in weights.items()}
        self.layer = B.cc_create_layer(self.ctx, self.desc, wdev)
        del wdev                                   # the library keeps its own packed copy (slot 0)
        self.blob_bytes = B.cc_layer_blob_bytes(self.layer)
        self.arena = None
        if n_slots > 0:
            slot = (self.blob_bytes + 1023) // 1024 * 1024
            self.arena = torch.empty(n_slots * slot + 2048, dtype=torch.uint8, device=self.device)
            B.cc_ctx_donate(self.ctx, self.arena, self.arena.numel())

    def forward(self, step: DeviceStep, stream=None) -> None:
        B.cc_forward(self.layer, step.hidden, step.k_pool, step.v_pool, step.block_table, step.n_pages,
                     step.seq_lens, step.assign, step.batch, stream)

    def scale(self, n: int, stream=None) -> None:
        """cc_scale_layer + cc_commit on `stream` (default: torch's current stream)."""
        B.cc_scale_layer(self.layer, n)
        B.cc_commit(self.layer, torch.cuda.current_stream() if stream is None else stream)

    def tap(self, which: int, batch: int) -> np.ndarray:
        dims = {B.CC_TAP_X: self.shape.hidden, B.CC_TAP_Q: self.shape.q_dim, B.CC_TAP_O: self.shape.q_dim,
                B.CC_TAP_H1: self.shape.hidden, B.CC_TAP_Y: self.shape.hidden, B.CC_TAP_A: self.shape.ffn}
        return B.cc_debug_tap(self.layer, which, batch, dims[which])

    def close(self) -> None:
        if self.layer is not None:
            torch.cuda.synchronize()
            B.cc_destroy_layer(self.layer)
            self.layer = None
        if self.ctx is not None:
            if self.arena is not None:
                B.cc_ctx_reclaim(self.ctx, self.arena)
            B.cc_ctx_destroy(self.ctx)
            self.ctx = None
        self.arena = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()
        return False


class ModelSession:
    """Context + L layers of one shape (each its own weights) + one donated arena: the plumbing for
    whole-model decode steps (BASELINE.json configs[2]): one CUDA graph holds the cc_forward of every
    layer; replicas of single layers come and go through the device replica table (cc_commit)."""

    def __init__(self, shape: I.LayerShape, weights_dev: list, max_batch: int, n_slots: int, device_index: int = 0,
                 max_blocks: int | None = None, max_position: int | None = None):
        self.shape = shape
        self.device = f"cuda:{device_index}"
        torch.cuda.set_device(device_index)
        self.ctx = B.cc_ctx_create(device_index)
        self.desc = make_desc(shape, max_batch, max_blocks, max_position)
        self.layers = []
        self.blob_bytes = 0
        self.arena = None
        self.n_slots = n_slots
        for w in weights_dev:
            self.add_layer(w)
        if self.layers:
            self.donate()

    def add_layer(self, w: dict) -> None:
        """One more layer from device weight tensors (the library packs its own copy, so `w` may be freed)."""
        self.layers.append(B.cc_create_layer(self.ctx, self.desc, w))
        self.blob_bytes = B.cc_layer_blob_bytes(self.layers[0])

    def donate(self) -> None:
        """Lend the replica arena (n_slots slots of one layer blob each) once the layers exist."""
        if self.n_slots > 0 and self.arena is None:
            slot = (self.blob_bytes + 1023) // 1024 * 1024
            self.arena = torch.empty(self.n_slots * slot + 2048, dtype=torch.uint8, device=self.device)
            B.cc_ctx_donate(self.ctx, self.arena, self.arena.numel())

    def forward_all(self, hidden, k_pools, v_pools, block_table, n_pages, seq_lens, assigns, batch, stream=None) -> None:
        """hidden flows through the layers in place; layer l uses k_pools[l], v_pools[l], assigns[l]."""
        for l, layer in enumerate(self.layers):
            B.cc_forward(layer, hidden, k_pools[l], v_pools[l], block_table, n_pages, seq_lens, assigns[l], batch, stream)

    def scale(self, l: int, n: int, stream=None) -> None:
        B.cc_scale_layer(self.layers[l], n)
        B.cc_commit(self.layers[l], torch.cuda.current_stream() if stream is None else stream)

    def close(self) -> None:
        torch.cuda.synchronize()
        for layer in self.layers:
            B.cc_destroy_layer(layer)
        self.layers = []
        if self.ctx is not None:
            if self.arena is not None:
                B.cc_ctx_reclaim(self.ctx, self.arena)
            B.cc_ctx_destroy(self.ctx)
            self.ctx = None
        self.arena = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()
        return False


class KvLiveMigration:
    """KV redistribution overlapped with decoding, as a pre-copy:

      start()   plans on the table as it is (cc_kv_plan_migration) and enqueues the page copies chunk by chunk
                on a side stream; decode steps keep running on the main stream with the OLD table;
      finish()  makes the main stream wait for that copy, plans what the steps wrote meanwhile
                (cc_kv_plan_catchup: the tail page of then, pages added since), copies those few pages on the
                main stream and overwrites the device block table in place -- the next replay of a captured
                graph reads the new table from the same address.

    One copy block moves one page, so the hardware already interleaves the copy with the decode kernels page by
    page; cutting the list into many launches only adds launch gaps (measured: DESIGN.md 7b), hence the large
    default chunk.  Plumbing only: both plans are the library's, both copies are its kernel.  While a migration runs the page
    allocator of the caller must not hand out `reserved` (the destinations of the first plan)."""

    def __init__(self, ctx, step: DeviceStep, page_bytes: int, n_replicas: int, chunk_pages: int = 4096):
        self.ctx, self.step, self.page_bytes, self.R, self.chunk = ctx, step, page_bytes, n_replicas, max(1, chunk_pages)
        self.done = torch.cuda.Event()
        self.planned_bt = self.seq_planned = self.assign = None
        self.reserved: set[int] = set()
        self.bulk_moves = self.catchup_moves = 0
        self._keep = []

    def _enqueue(self, src: np.ndarray, dst: np.ndarray, stream) -> None:
        if len(src) == 0:
            return
        s = torch.from_numpy(src).to(self.step.device)
        d = torch.from_numpy(dst).to(self.step.device)
        self._keep += [s, d]                       # the lists must outlive the kernels that read them
        for c0 in range(0, len(src), self.chunk):
            n = min(self.chunk, len(src) - c0)
            B.cc_kv_migrate(self.ctx, self.step.k_pool, self.step.v_pool, self.page_bytes, s[c0:c0 + n], d[c0:c0 + n], n, stream)

    def start(self, block_table_host: np.ndarray, seq_lens_host: np.ndarray, assign: np.ndarray, side_stream) -> int:
        self.seq_planned = np.array(seq_lens_host, dtype=np.int32)
        self.assign = np.array(assign, dtype=np.int32)
        self.planned_bt, src, dst = B.cc_kv_plan_migration(block_table_host, self.seq_planned, self.assign, self.step.n_pages, self.R)
        self.reserved = set(dst.tolist())
        self.bulk_moves = len(src)
        side_stream.wait_stream(torch.cuda.current_stream())   # pages written by steps already enqueued are final
        self._enqueue(src, dst, side_stream)
        self.done.record(side_stream)
        return self.bulk_moves

    def finish(self, block_table_now_host: np.ndarray, seq_lens_now_host: np.ndarray, stream=None) -> np.ndarray:
        stream = torch.cuda.current_stream() if stream is None else stream
        stream.wait_event(self.done)
        final_bt, src, dst = B.cc_kv_plan_catchup(block_table_now_host, self.seq_planned, seq_lens_now_host, self.planned_bt,
                                                  self.assign, self.step.n_pages, self.R)
        self.catchup_moves = len(src)
        with torch.cuda.stream(stream):
            self._enqueue(src, dst, stream)
            self.step.block_table.copy_(torch.from_numpy(final_bt))
        self.reserved = set()
        return final_bt
