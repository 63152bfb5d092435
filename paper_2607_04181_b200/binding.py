"""Thin ctypes binding over libcocoscale.so -- same names as include/cocoscale.h, argument
marshalling only (every step of the hot path runs in the CUDA kernels behind the C ABI).

Device pointers may be given as torch CUDA tensors (their data_ptr() is passed), as ints, or as
None (NULL); host buffers as numpy arrays / torch CPU tensors.  Streams are passed as the raw
`cudaStream_t` integer (torch.cuda.Stream.cuda_stream) or None for the legacy default stream.
Every call raises CcError when the library returns a non-zero cc_status.  There is no CPU
fallback: if the library cannot be loaded, importing this module raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

CC_MAX_REPLICAS = 4
CC_PAGE_SIZE = 16
CC_MAX_LAYERS = 128
CC_OK, CC_ERR_INVALID, CC_ERR_NO_SLOT, CC_ERR_CUDA, CC_ERR_BUSY, CC_ERR_STATE = range(6)
STATUS_NAMES = ("CC_OK", "CC_ERR_INVALID", "CC_ERR_NO_SLOT", "CC_ERR_CUDA", "CC_ERR_BUSY", "CC_ERR_STATE")
CC_DEVERR_BAD_REPLICA, CC_DEVERR_BAD_PAGE, CC_DEVERR_BAD_SEQLEN, CC_DEVERR_HANG, CC_DEVERR_SPLIT_REQUEST = 1, 2, 4, 8, 16
CC_DEVERR_TOO_MANY_DECODE = 32
CC_TAP_X, CC_TAP_Q, CC_TAP_O, CC_TAP_H1, CC_TAP_Y, CC_TAP_A = range(6)
CC_OPERAND_AUTO, CC_OPERAND_F16, CC_OPERAND_BF16X2 = range(3)

# every function include/cocoscale.h declares (checked against the header by tests/test_cabi.py)
EXPORTS = (
    "cc_ctx_create", "cc_ctx_destroy", "cc_ctx_donate", "cc_ctx_reclaim", "cc_ctx_set_copy_chunk",
    "cc_ctx_set_pdl", "cc_ctx_set_operand_format", "cc_ctx_set_operand_planes", "cc_layer_operand_format", "cc_poll_device_error", "cc_create_layer", "cc_destroy_layer", "cc_layer_blob_bytes",
    "cc_scale_layer", "cc_commit", "cc_release_replica", "cc_query", "cc_layer_set_kv_partition", "cc_active_replicas", "cc_replica_blob", "cc_forward",
    "cc_forward_host", "cc_forward_host_async", "cc_forward_profiled", "cc_forward_launch_count", "cc_layer_gemm_grids", "cc_replica_copy", "cc_kv_plan_migration", "cc_kv_plan_catchup", "cc_kv_migrate", "cc_debug_tap", "cc_debug_grouping", "cc_debug_trace",
    "cc_slotalloc_create", "cc_slotalloc_destroy", "cc_slotalloc_donate", "cc_slotalloc_reclaim",
    "cc_slotalloc_alloc", "cc_slotalloc_free", "cc_slotalloc_free_bytes", "cc_last_error", "cc_version",
    "cc_static_scratch_bytes", "cc_attention_decode_static",
    "cc_ctl_mem_bytes", "cc_ctl_flops", "cc_ctl_comm_seconds", "cc_ctl_speedup", "cc_ctl_speedup_vec", "cc_ctl_distance",
    "cc_ctl_candidate_count", "cc_ctl_decide", "cc_ctl_place",
)


class CcError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{STATUS_NAMES[status] if 0 <= status < len(STATUS_NAMES) else status}: {message}")
        self.status = status


class cc_layer_desc(C.Structure):
    _fields_ = [("hidden", C.c_int32), ("n_q_heads", C.c_int32), ("n_kv_heads", C.c_int32),
                ("head_dim", C.c_int32), ("ffn", C.c_int32), ("rms_eps", C.c_float), ("rope_base", C.c_float),
                ("page_size", C.c_int32), ("max_batch", C.c_int32), ("max_blocks_per_seq", C.c_int32),
                ("max_position", C.c_int32)]


class cc_layer_weights(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("g1", "wq", "wk", "wv", "wo", "g2", "wgate", "wup", "wdown")]


class cc_kv_pages(C.Structure):
    _fields_ = [("k_pool", C.c_void_p), ("v_pool", C.c_void_p), ("block_table", C.c_void_p), ("n_pages", C.c_int32)]


_TRACE = os.environ.get("COCOSCALE_TRACE", "0") not in ("", "0")   # load the tracing build (timeline.py sets it)


def _load() -> C.CDLL:
    path = _build.LIB_TRACE if _TRACE else _build.LIB
    if _build.needs_build(_TRACE):
        try:
            _build.build(trace=_TRACE)
        except Exception as e:  # no nvcc and no prebuilt library: fail loudly, never fall back
            if not os.path.exists(path):
                raise ImportError(f"libcocoscale.so is missing and could not be built: {e}") from e
    return C.CDLL(path)


_lib = _load()
_lib.cc_last_error.restype = C.c_char_p
_lib.cc_version.restype = C.c_char_p
_lib.cc_slotalloc_create.restype = C.c_void_p
_lib.cc_slotalloc_free_bytes.restype = C.c_uint64
_lib.cc_slotalloc_free_bytes.argtypes = [C.c_void_p]
_lib.cc_slotalloc_destroy.argtypes = [C.c_void_p]
_lib.cc_slotalloc_destroy.restype = None


def library_path() -> str:
    return _build.LIB_TRACE if _TRACE else _build.LIB


def _ptr(x) -> C.c_void_p:
    if x is None:
        return C.c_void_p(0)
    if isinstance(x, int):
        return C.c_void_p(x)
    if hasattr(x, "data_ptr"):
        return C.c_void_p(x.data_ptr())
    if isinstance(x, np.ndarray):
        assert x.flags["C_CONTIGUOUS"]
        return C.c_void_p(x.ctypes.data)
    if isinstance(x, C.c_void_p):
        return x
    raise TypeError(f"cannot pass {type(x)} as a pointer")


def _stream(s) -> C.c_void_p:
    if s is None:
        return C.c_void_p(0)
    if hasattr(s, "cuda_stream"):
        return C.c_void_p(s.cuda_stream)
    return C.c_void_p(int(s))


def _check(status: int) -> None:
    if status != CC_OK:
        raise CcError(status, cc_last_error())


def cc_last_error() -> str:
    return (_lib.cc_last_error() or b"").decode()


def cc_version() -> str:
    return _lib.cc_version().decode()


# ---- context ---------------------------------------------------------------------------------
def cc_ctx_create(device: int = 0) -> C.c_void_p:
    out = C.c_void_p()
    _check(_lib.cc_ctx_create(C.c_int(device), C.byref(out)))
    return out


def cc_ctx_destroy(ctx) -> None:
    _check(_lib.cc_ctx_destroy(ctx))


def cc_ctx_donate(ctx, dev_base, nbytes: int) -> None:
    _check(_lib.cc_ctx_donate(ctx, _ptr(dev_base), C.c_size_t(nbytes)))


def cc_ctx_reclaim(ctx, dev_base) -> None:
    _check(_lib.cc_ctx_reclaim(ctx, _ptr(dev_base)))


def cc_ctx_set_copy_chunk(ctx, chunk_bytes: int) -> None:
    _check(_lib.cc_ctx_set_copy_chunk(ctx, C.c_size_t(chunk_bytes)))


def cc_ctx_set_pdl(ctx, enabled: bool) -> None:
    _check(_lib.cc_ctx_set_pdl(ctx, C.c_int(1 if enabled else 0)))


def cc_ctx_set_operand_format(ctx, fmt: int) -> None:
    _check(_lib.cc_ctx_set_operand_format(ctx, C.c_int(fmt)))


def cc_ctx_set_operand_planes(ctx, rows: int, planes_upto_rows, planes_above) -> None:
    a = (C.c_int * 4)(*[int(x) for x in planes_upto_rows])
    b = (C.c_int * 4)(*[int(x) for x in planes_above])
    _check(_lib.cc_ctx_set_operand_planes(ctx, C.c_int(rows), a, b))


def cc_poll_device_error(ctx) -> int:
    bits = C.c_uint32()
    _check(_lib.cc_poll_device_error(ctx, C.byref(bits)))
    return bits.value


# ---- layer lifecycle ---------------------------------------------------------------------------
def cc_create_layer(ctx, desc: cc_layer_desc, weights: dict) -> C.c_void_p:
    """`weights`: name -> device tensor / pointer for g1 wq wk wv wo g2 wgate wup wdown (bf16)."""
    w = cc_layer_weights(*[_ptr(weights[n[0]]) for n in cc_layer_weights._fields_])
    out = C.c_void_p()
    _check(_lib.cc_create_layer(ctx, C.byref(desc), C.byref(w), C.byref(out)))
    return out


def cc_destroy_layer(layer) -> None:
    _check(_lib.cc_destroy_layer(layer))


def cc_layer_operand_format(layer) -> int:
    f = C.c_int()
    _check(_lib.cc_layer_operand_format(layer, C.byref(f)))
    return f.value


def cc_layer_blob_bytes(layer) -> int:
    n = C.c_size_t()
    _check(_lib.cc_layer_blob_bytes(layer, C.byref(n)))
    return n.value


def cc_scale_layer(layer, n_replicas: int) -> None:
    _check(_lib.cc_scale_layer(layer, C.c_int(n_replicas)))


def cc_layer_set_kv_partition(layer, replica: int, k_pool, v_pool, n_pages: int, stream=None) -> None:
    _check(_lib.cc_layer_set_kv_partition(layer, C.c_int(replica), _ptr(k_pool), _ptr(v_pool), C.c_int32(n_pages), _stream(stream)))


def cc_commit(layer, stream=None) -> None:
    _check(_lib.cc_commit(layer, _stream(stream)))


def cc_release_replica(layer, replica: int) -> None:
    _check(_lib.cc_release_replica(layer, C.c_int(replica)))


def cc_query(layer):
    a, p = C.c_int(), C.c_int()
    _check(_lib.cc_query(layer, C.byref(a), C.byref(p)))
    return a.value, p.value


def cc_active_replicas(layer) -> list:
    """Replica indices that forwards enqueued now may name (not compacted: {0, 2} after releasing 1 of three)."""
    m = C.c_uint32()
    _check(_lib.cc_active_replicas(layer, C.byref(m)))
    return [r for r in range(CC_MAX_REPLICAS) if (m.value >> r) & 1]


def cc_replica_blob(layer, replica: int):
    ptr, n = C.c_void_p(), C.c_size_t()
    _check(_lib.cc_replica_blob(layer, C.c_int(replica), C.byref(ptr), C.byref(n)))
    return ptr.value, n.value


# ---- hot path ----------------------------------------------------------------------------------
def cc_forward(layer, hidden, k_pool, v_pool, block_table, n_pages: int, seq_lens, replica_assign, batch: int,
               stream=None) -> None:
    kv = cc_kv_pages(_ptr(k_pool), _ptr(v_pool), _ptr(block_table), C.c_int32(n_pages))
    _check(_lib.cc_forward(layer, _ptr(hidden), C.byref(kv), _ptr(seq_lens), _ptr(replica_assign), C.c_int(batch),
                           _stream(stream)))


def cc_forward_host(layer, hidden_host, k_pool, v_pool, n_pages: int, block_table_host, seq_lens_host,
                    replica_assign_host, batch: int, stream=None) -> None:
    _check(_lib.cc_forward_host(layer, _ptr(hidden_host), _ptr(k_pool), _ptr(v_pool), C.c_int32(n_pages),
                                _ptr(block_table_host), _ptr(seq_lens_host), _ptr(replica_assign_host),
                                C.c_int(batch), _stream(stream)))


def cc_forward_host_async(layer, hidden_host, k_pool, v_pool, n_pages: int, block_table_host, seq_lens_host,
                          replica_assign_host, batch: int, stream=None) -> None:
    _check(_lib.cc_forward_host_async(layer, _ptr(hidden_host), _ptr(k_pool), _ptr(v_pool), C.c_int32(n_pages),
                                      _ptr(block_table_host), _ptr(seq_lens_host), _ptr(replica_assign_host),
                                      C.c_int(batch), _stream(stream)))


STAGE_NAMES = ("prologue", "gemm_qkv", "attention", "gemm_o", "gemm_gate_up", "gemm_down")
BIG_STAGE_NAMES = ("group", "norm", "gemm_qkv", "attention_decode", "attention_prefill", "gemm_o", "rowstat", "gemm_gate_up",
                   "gemm_down")          # steps of more than 256 rows
CC_MAX_PROFILE_STAGES = 10


def cc_forward_profiled(layer, hidden, k_pool, v_pool, block_table, n_pages: int, seq_lens, replica_assign,
                        batch: int, stream=None) -> np.ndarray:
    kv = cc_kv_pages(_ptr(k_pool), _ptr(v_pool), _ptr(block_table), C.c_int32(n_pages))
    ms = np.zeros(CC_MAX_PROFILE_STAGES, dtype=np.float32)
    _check(_lib.cc_forward_profiled(layer, _ptr(hidden), C.byref(kv), _ptr(seq_lens), _ptr(replica_assign),
                                    C.c_int(batch), _stream(stream), _ptr(ms)))
    return ms[:len(BIG_STAGE_NAMES if batch > 256 else STAGE_NAMES)]


def cc_layer_gemm_grids(layer):
    ctas, cluster = (C.c_int * 4)(), (C.c_int * 4)()
    _check(_lib.cc_layer_gemm_grids(layer, ctas, cluster))
    return list(ctas), list(cluster)


def cc_forward_launch_count(layer) -> int:
    n = C.c_int()
    _check(_lib.cc_forward_launch_count(layer, C.byref(n)))
    return n.value


# ---- the entry point that allocates nothing (include/cocoscale.h) -------------------------------------
_lib.cc_static_scratch_bytes.restype = C.c_size_t


def cc_static_scratch_bytes() -> int:
    return int(_lib.cc_static_scratch_bytes())


def cc_attention_decode_static(q, k_pool, v_pool, block_table, seq_lens, out, batch: int, n_q_heads: int, n_kv_heads: int,
                               head_dim: int, max_blocks: int, n_pages: int, stream=None) -> None:
    """Device pointers / torch CUDA tensors in, `out` written on the device; needs no context or layer."""
    _check(_lib.cc_attention_decode_static(_ptr(q), _ptr(k_pool), _ptr(v_pool), _ptr(block_table), _ptr(seq_lens), _ptr(out),
                                           C.c_int(batch), C.c_int(n_q_heads), C.c_int(n_kv_heads), C.c_int(head_dim),
                                           C.c_int(max_blocks), C.c_int(n_pages), _stream(stream)))


def cc_replica_copy(ctx, dst, src, nbytes: int, chunk_bytes: int = 0, stream=None) -> None:
    _check(_lib.cc_replica_copy(ctx, _ptr(dst), _ptr(src), C.c_size_t(nbytes), C.c_size_t(chunk_bytes),
                                _stream(stream)))


# ---- KV partition per replica ----------------------------------------------------------------------
def cc_kv_plan_migration(block_table: np.ndarray, seq_lens: np.ndarray, assign: np.ndarray, n_pages: int, n_replicas: int):
    """-> (new_block_table, src_pages, dst_pages); host arrays, argument marshalling only."""
    bt = np.ascontiguousarray(block_table, dtype=np.int32)
    sl = np.ascontiguousarray(seq_lens, dtype=np.int32)
    ra = np.ascontiguousarray(assign, dtype=np.int32)
    batch, width = bt.shape
    new_bt = np.empty_like(bt)
    src = np.empty(batch * width, dtype=np.int32)
    dst = np.empty(batch * width, dtype=np.int32)
    n = C.c_int(0)
    _check(_lib.cc_kv_plan_migration(_ptr(bt), _ptr(sl), _ptr(ra), C.c_int(batch), C.c_int(width), C.c_int(n_pages),
                                     C.c_int(n_replicas), _ptr(new_bt), _ptr(src), _ptr(dst), C.byref(n)))
    return new_bt, src[:n.value].copy(), dst[:n.value].copy()


def cc_kv_plan_catchup(block_table_now: np.ndarray, seq_lens_planned: np.ndarray, seq_lens_now: np.ndarray,
                       planned_block_table: np.ndarray, assign: np.ndarray, n_pages: int, n_replicas: int):
    """-> (final_block_table, src_pages, dst_pages); host arrays, argument marshalling only."""
    bt = np.ascontiguousarray(block_table_now, dtype=np.int32)
    s0 = np.ascontiguousarray(seq_lens_planned, dtype=np.int32)
    s1 = np.ascontiguousarray(seq_lens_now, dtype=np.int32)
    pb = np.ascontiguousarray(planned_block_table, dtype=np.int32)
    ra = np.ascontiguousarray(assign, dtype=np.int32)
    batch, width = bt.shape
    assert pb.shape == bt.shape
    final_bt = np.empty_like(bt)
    src = np.empty(batch * width, dtype=np.int32)
    dst = np.empty(batch * width, dtype=np.int32)
    n = C.c_int(0)
    _check(_lib.cc_kv_plan_catchup(_ptr(bt), _ptr(s0), _ptr(s1), _ptr(pb), _ptr(ra), C.c_int(batch), C.c_int(width),
                                   C.c_int(n_pages), C.c_int(n_replicas), _ptr(final_bt), _ptr(src), _ptr(dst), C.byref(n)))
    return final_bt, src[:n.value].copy(), dst[:n.value].copy()


def cc_kv_migrate(ctx, k_pool, v_pool, page_bytes: int, src_pages, dst_pages, n_moves: int, stream=None) -> None:
    _check(_lib.cc_kv_migrate(ctx, _ptr(k_pool), _ptr(v_pool), C.c_size_t(page_bytes), _ptr(src_pages), _ptr(dst_pages),
                              C.c_int(n_moves), _stream(stream)))


# ---- cost / speed-up model and scaling decision (host only) --------------------------------------------
class cc_ctl_params(C.Structure):
    _fields_ = [("L", C.c_int32), ("P_max", C.c_int32), ("slo", C.c_double), ("delta", C.c_double),
                ("beta", C.c_double * (CC_MAX_REPLICAS + 1)), ("cost_per_device", C.c_double),
                ("cost_per_layer_copy", C.c_double)]


CC_CTL_NONE, CC_CTL_UPDATED, CC_CTL_INSTANCE_SCALE = range(3)
for _n, _res, _args in (
        ("cc_ctl_mem_bytes", C.c_double, [C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double]),
        ("cc_ctl_flops", C.c_double, [C.c_int, C.c_int, C.c_int, C.c_int, C.c_int]),
        ("cc_ctl_comm_seconds", C.c_double, [C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double]),
        ("cc_ctl_speedup", C.c_double, [C.c_int, C.c_int, C.c_int, C.c_double]),
        ("cc_ctl_speedup_vec", C.c_double, [C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_int, C.c_double, C.c_double]),
        ("cc_ctl_distance", C.c_int, [C.c_int, C.c_int, C.c_int, C.c_int]),
        ("cc_ctl_candidate_count", C.c_int, [C.c_int, C.c_int])):
    getattr(_lib, _n).restype = _res
    getattr(_lib, _n).argtypes = _args
cc_ctl_mem_bytes, cc_ctl_flops, cc_ctl_comm_seconds = _lib.cc_ctl_mem_bytes, _lib.cc_ctl_flops, _lib.cc_ctl_comm_seconds
cc_ctl_speedup, cc_ctl_distance, cc_ctl_candidate_count = _lib.cc_ctl_speedup, _lib.cc_ctl_distance, _lib.cc_ctl_candidate_count


def cc_ctl_speedup_vec(v, bs: int, t_comp_s: float, d_hidden: int, kappa: float, bandwidth: float) -> float:
    a = np.ascontiguousarray(v, dtype=np.int32)
    return _lib.cc_ctl_speedup_vec(_ptr(a), len(a), bs, t_comp_s, d_hidden, kappa, bandwidth)


def cc_ctl_decide(params: "cc_ctl_params", N_cur: int, P_cur: int, latency: float, cold_capacity: float):
    """-> (action, N_new, P_new, cold_capacity_after)"""
    cold, n, p_, act = C.c_double(cold_capacity), C.c_int(0), C.c_int(0), C.c_int(0)
    _check(_lib.cc_ctl_decide(C.byref(params), C.c_int(N_cur), C.c_int(P_cur), C.c_double(latency), C.byref(cold),
                              C.byref(n), C.byref(p_), C.byref(act)))
    return act.value, n.value, p_.value, cold.value


class cc_ctl_instance(C.Structure):
    _fields_ = [("L", C.c_int32), ("bs", C.c_int32), ("l", C.c_int32), ("d_hidden", C.c_int32), ("kappa", C.c_double),
                ("load", C.c_double), ("capacity", C.c_double)]


class cc_ctl_device(C.Structure):
    _fields_ = [("load", C.c_double), ("free_mem_bytes", C.c_double)]


class cc_ctl_placement(C.Structure):
    _fields_ = [("instance", C.c_int32), ("N", C.c_int32), ("P", C.c_int32), ("devices", C.c_int32 * (CC_MAX_REPLICAS - 1)),
                ("speedup", C.c_double)]


def cc_ctl_place(params: "cc_ctl_params", instances: list, devices: list, tau_idle: float) -> list:
    """Algorithm 1.  instances: cc_ctl_instance, devices: cc_ctl_device -> [(instance, N, P, [devices], speedup)]"""
    ia = (cc_ctl_instance * max(len(instances), 1))(*instances)
    da = (cc_ctl_device * max(len(devices), 1))(*devices)
    out = (cc_ctl_placement * max(len(instances), 1))()
    n = C.c_int(0)
    _check(_lib.cc_ctl_place(C.byref(params), ia, C.c_int(len(instances)), da, C.c_int(len(devices)), C.c_double(tau_idle),
                             out, C.byref(n)))
    return [(o.instance, o.N, o.P, [d for d in o.devices if d >= 0], o.speedup) for o in out[:n.value]]


# ---- timeline of a tracing build -----------------------------------------------------------------
def cc_debug_trace(ctx, reset: bool = True):
    """-> uint64 [16][8][2] (kernel, point, min / max of %globaltimer); CcError(CC_ERR_STATE) in a product build."""
    out = np.zeros((16, 8, 2), dtype=np.uint64)
    _check(_lib.cc_debug_trace(ctx, _ptr(out), C.c_int(1 if reset else 0)))
    return out


# ---- stage taps (tests) ------------------------------------------------------------------------
def cc_debug_tap(layer, which: int, batch: int, dim: int) -> np.ndarray:
    out = np.zeros((batch, dim), dtype=np.float32)
    _check(_lib.cc_debug_tap(layer, C.c_int(which), _ptr(out), C.c_int(batch)))
    return out


def cc_debug_grouping(layer, max_batch: int):
    perm = np.full(max_batch + 80, -1, dtype=np.int32)
    counts = np.zeros(CC_MAX_REPLICAS, dtype=np.int32)
    n_pos = C.c_int32()
    _check(_lib.cc_debug_grouping(layer, _ptr(perm), _ptr(counts), C.byref(n_pos)))
    return perm[:n_pos.value].copy(), counts, n_pos.value


# ---- host-only slot allocator --------------------------------------------------------------------
def cc_slotalloc_create() -> C.c_void_p:
    return C.c_void_p(_lib.cc_slotalloc_create())


def cc_slotalloc_destroy(a) -> None:
    _lib.cc_slotalloc_destroy(a)


def cc_slotalloc_donate(a, base: int, nbytes: int) -> int:
    return _lib.cc_slotalloc_donate(a, C.c_uint64(base), C.c_uint64(nbytes))


def cc_slotalloc_reclaim(a, base: int) -> int:
    return _lib.cc_slotalloc_reclaim(a, C.c_uint64(base))


def cc_slotalloc_alloc(a, nbytes: int):
    addr = C.c_uint64()
    st = _lib.cc_slotalloc_alloc(a, C.c_uint64(nbytes), C.byref(addr))
    return st, (addr.value if st == CC_OK else None)


def cc_slotalloc_free(a, addr: int) -> int:
    return _lib.cc_slotalloc_free(a, C.c_uint64(addr))


def cc_slotalloc_free_bytes(a) -> int:
    return int(_lib.cc_slotalloc_free_bytes(a))
