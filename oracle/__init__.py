"""oracle/ -- TEST INFRASTRUCTURE, NOT PRODUCT (see oracle/cc_oracle.c header).

ctypes loader for the plain-C CPU oracle plus a pure-Python integer simulation of the host-side
structures (slot allocator, replica state machine).  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this package.  It imports nothing
from the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libcc_oracle.so")
_SRC = os.path.join(_HERE, "cc_oracle.c")


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp -shared; rebuilt when the source is newer than the library."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
               "-ffp-contract=off", "-o", _SO, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _SO


class _Desc(C.Structure):
    _fields_ = [("hidden", C.c_int32), ("n_q_heads", C.c_int32), ("n_kv_heads", C.c_int32),
                ("head_dim", C.c_int32), ("ffn", C.c_int32), ("page", C.c_int32),
                ("rms_eps", C.c_float), ("rope_base", C.c_float)]


class _Weights(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("g1", "wq", "wk", "wv", "wo", "g2", "wgate", "wup", "wdown")]


_TAP_NAMES = ("x", "q", "k_new", "v_new", "o", "h1", "y", "a", "out")


class _Taps(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in _TAP_NAMES]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_bf16_to_f32.restype = C.c_float
        _lib.orc_bf16_to_f32.argtypes = [C.c_uint16]
        _lib.orc_f32_to_bf16.restype = C.c_uint16
        _lib.orc_f32_to_bf16.argtypes = [C.c_float]
        _lib.orc_silu.restype = C.c_float
        _lib.orc_silu.argtypes = [C.c_float]
        _lib.orc_num_threads.restype = C.c_int
        _lib.orc_set_num_threads.argtypes = [C.c_int]
        _lib.orc_rmsnorm.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_float, C.c_void_p]
        _lib.orc_matmul_wt.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p]
        _lib.orc_rope.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_float]
        _lib.orc_attention_decode.restype = C.c_int
        _lib.orc_attention_decode.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int,
                                              C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_void_p]
        _lib.orc_replica_copy.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t]
        _lib.orc_layer_forward.restype = C.c_int
        _lib.orc_layer_forward.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                           C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p,
                                           C.c_int, C.c_int, C.c_void_p]
        _lib.orc_group_rows.restype = C.c_int
        _lib.orc_group_rows.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p]
    return _lib


def _p(a: np.ndarray):
    assert a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(C.c_void_p)


def _f32(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float32)


def _u16(a) -> np.ndarray:
    a = np.ascontiguousarray(a)
    assert a.dtype == np.uint16
    return a


def num_threads() -> int:
    return int(lib().orc_num_threads())


def set_num_threads(n: int) -> None:
    lib().orc_set_num_threads(int(n))


def bf16_to_f32(u: int) -> float:
    return float(lib().orc_bf16_to_f32(int(u)))


def f32_to_bf16(f: float) -> int:
    return int(lib().orc_f32_to_bf16(float(np.float32(f))))


def silu(z: float) -> float:
    return float(lib().orc_silu(float(np.float32(z))))


def rmsnorm(h, g_bf16, eps: float) -> np.ndarray:
    h = _f32(h)
    rows, d = h.shape
    g = _u16(g_bf16)
    x = np.empty_like(h)
    lib().orc_rmsnorm(_p(h), _p(g), rows, d, C.c_float(eps), _p(x))
    return x


def matmul_wt(X, W_bf16) -> np.ndarray:
    X = _f32(X)
    W = _u16(W_bf16)
    M, K = X.shape
    N, K2 = W.shape
    assert K == K2
    Y = np.empty((M, N), dtype=np.float32)
    lib().orc_matmul_wt(_p(X), _p(W), M, K, N, _p(Y))
    return Y


def rope(u, n_heads: int, head_dim: int, pos: int, base: float) -> np.ndarray:
    v = _f32(u).copy().reshape(n_heads * head_dim)
    lib().orc_rope(_p(v), n_heads, head_dim, int(pos), C.c_float(base))
    return v.reshape(np.shape(u))


def attention_decode(q, k_pool, v_pool, bt_row, s: int, Hq: int, Hkv: int, Dh: int, page: int,
                     return_weights: bool = False):
    q = _f32(q).reshape(Hq * Dh)
    k_pool, v_pool = _u16(k_pool), _u16(v_pool)
    bt_row = np.ascontiguousarray(bt_row, dtype=np.int32)
    o = np.empty(Hq * Dh, dtype=np.float32)
    w = np.empty((Hq, max(s, 1)), dtype=np.float32) if return_weights else None
    rc = lib().orc_attention_decode(_p(q), _p(k_pool), _p(v_pool), _p(bt_row), int(s), Hq, Hkv, Dh, page,
                                    _p(o), _p(w) if w is not None else None)
    if rc:
        raise RuntimeError(f"orc_attention_decode rc={rc}")
    o = o.reshape(Hq, Dh)
    return (o, w[:, :s]) if return_weights else o


def replica_copy(src: np.ndarray) -> np.ndarray:
    src = np.ascontiguousarray(src)
    dst = np.empty_like(src)
    lib().orc_replica_copy(_p(dst), _p(src), src.nbytes)
    return dst


def group_rows(replica_assign, seq_lens, R: int):
    ra = np.ascontiguousarray(replica_assign, dtype=np.int32)
    sl = np.ascontiguousarray(seq_lens, dtype=np.int32)
    B = ra.shape[0]
    perm = np.full(B, -1, dtype=np.int32)
    counts = np.zeros(R, dtype=np.int32)
    n = lib().orc_group_rows(_p(ra), _p(sl), B, R, _p(perm), _p(counts))
    return perm[:n].copy(), counts


def layer_forward(shape, weights: dict, hidden, k_pool, v_pool, block_table, seq_lens, replica_assign,
                  n_replicas: int, taps: bool = False):
    """Runs the replicated layer.  `shape` needs .hidden .n_q_heads .n_kv_heads .head_dim .ffn .page
    .rms_eps .rope_base.  Returns dict(out=bf16 bits [B,d], k_pool=, v_pool= (copies, with the new
    token appended), taps={name: fp32 array} if requested).  Inputs are not modified."""
    D = _Desc(shape.hidden, shape.n_q_heads, shape.n_kv_heads, shape.head_dim, shape.ffn, shape.page,
              shape.rms_eps, shape.rope_base)
    keep = {f[0]: _u16(weights[f[0]]) for f in _Weights._fields_}
    W = _Weights(*[keep[f[0]].ctypes.data for f in _Weights._fields_])
    hidden = _u16(hidden)
    B, d = hidden.shape
    kp, vp = _u16(k_pool).copy(), _u16(v_pool).copy()
    bt = np.ascontiguousarray(block_table, dtype=np.int32)
    sl = np.ascontiguousarray(seq_lens, dtype=np.int32)
    ra = np.ascontiguousarray(replica_assign, dtype=np.int32)
    out = np.empty_like(hidden)
    tap_arrays, T = {}, None
    if taps:
        QD, KD = shape.n_q_heads * shape.head_dim, shape.n_kv_heads * shape.head_dim
        dims = {"x": d, "q": QD, "k_new": KD, "v_new": KD, "o": QD, "h1": d, "y": d, "a": shape.ffn, "out": d}
        tap_arrays = {n: np.zeros((B, dims[n]), dtype=np.float32) for n in _TAP_NAMES}
        T = _Taps(*[tap_arrays[n].ctypes.data for n in _TAP_NAMES])
    rc = lib().orc_layer_forward(C.byref(D), C.byref(W), _p(hidden), _p(out), _p(kp), _p(vp), _p(bt),
                                 bt.shape[1], _p(sl), _p(ra), B, int(n_replicas),
                                 C.byref(T) if T is not None else None)
    if rc:
        raise RuntimeError(f"orc_layer_forward rc={rc}")
    return {"out": out, "k_pool": kp, "v_pool": vp, "taps": tap_arrays}
