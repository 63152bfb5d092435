"""Seeded synthetic inputs for the replicated-decoder-layer hot path.

This module is shared by the CPU oracle's tests and by the CUDA path's tests/bench.  It holds
NONE of the method's arithmetic: only shapes, seeded random draws, dtype conversion
(fp32 <-> bf16 bit patterns, round-to-nearest-even) and integer bookkeeping for the paged KV
cache (which page holds which token range).  Neither `oracle/` nor the CUDA library imports it;
callers hand its arrays to both.

Recipe (SURVEY.md section 8(c) readings 5, 9, 10, 12-15; BASELINE.json configs):
  * projection weights ~ N(0, 0.02) (std), norm gains = 1 + N(0, 0.02), all rounded to bf16
  * hidden ~ N(0, 1) bf16;  the WHOLE KV pool ~ N(0, 1) bf16 (optionally NaN outside [0, s))
  * context length c ~ U{lo..hi} tokens already cached, seq_lens = c + 1 (the token being decoded
    is included), pages of 16 tokens, page ids a seeded permutation (no request is contiguous),
    block-table padding = -1
  * replica_assign: even split, replica r gets rows [r*B/R, (r+1)*B/R), remainder to the lowest
    replicas ("15 -> 7 and 8" becomes 8 + 7 under this rule; PAPER.md:203 ceil/floor)
The paper's own workloads (Alibaba/Azure traces, LongBench, Alpaca, Qwen3 weights; PAPER.md:129,
401) are not available; these inputs stand in for them and take only their shapes.
"""
from __future__ import annotations

from dataclasses import dataclass, replace
import numpy as np

PAGE = 16
MAX_REPLICAS = 4  # P_max = 4


@dataclass(frozen=True)
class LayerShape:
    name: str
    hidden: int
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    ffn: int
    rms_eps: float
    rope_base: float
    batch: int
    ctx_lo: int
    ctx_hi: int
    page: int = PAGE

    @property
    def q_dim(self) -> int:
        return self.n_q_heads * self.head_dim

    @property
    def kv_dim(self) -> int:
        return self.n_kv_heads * self.head_dim

    @property
    def max_blocks(self) -> int:
        # block table width: enough pages for seq_len = ctx_hi + 1
        return (self.ctx_hi + 1 + self.page - 1) // self.page

    @property
    def n_params(self) -> int:
        d, F = self.hidden, self.ffn
        return d * (self.q_dim + 2 * self.kv_dim) + self.q_dim * d + 3 * d * F

    def with_batch(self, batch: int) -> "LayerShape":
        return replace(self, batch=batch)


# BASELINE.json configs[0], configs[1]; cfg4/modelB are layer shapes used by parity/size tests.
CFG1 = LayerShape("cfg1", 256, 4, 2, 64, 688, 1e-6, 10000.0, 4, 16, 64)
CFG2 = LayerShape("cfg2", 4096, 32, 8, 128, 14336, 1e-5, 500000.0, 64, 512, 2048)
CFG4_LAYER = LayerShape("cfg4", 5120, 40, 8, 128, 17408, 1e-5, 500000.0, 256, 256, 4096)
MODEL_B_LAYER = LayerShape("modelB", 1536, 12, 2, 128, 8960, 1e-6, 10000.0, 64, 256, 1024)
CONFIGS = {c.name: c for c in (CFG1, CFG2, CFG4_LAYER, MODEL_B_LAYER)}

WEIGHT_NAMES = ("g1", "wq", "wk", "wv", "wo", "g2", "wgate", "wup", "wdown")


# ---------------------------------------------------------------------------------------------
# dtype conversion (bit-level; no arithmetic of the method)
# ---------------------------------------------------------------------------------------------
def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """fp32 -> bf16 bit pattern (uint16), round-to-nearest-even, NaN kept quiet."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    w = x.view(np.uint32)
    nan = (w & np.uint32(0x7FFFFFFF)) > np.uint32(0x7F800000)
    lsb = (w >> np.uint32(16)) & np.uint32(1)
    r = ((w + np.uint32(0x7FFF) + lsb) >> np.uint32(16)).astype(np.uint16)
    if nan.any():
        r = np.where(nan, ((w >> np.uint32(16)) | np.uint32(0x40)).astype(np.uint16), r)
    return r


def bf16_bits_to_f32(u: np.ndarray) -> np.ndarray:
    u = np.ascontiguousarray(u, dtype=np.uint16)
    return (u.astype(np.uint32) << np.uint32(16)).view(np.float32)


def _rng(seed: int, stream: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[seed, stream]))


def _normal_bf16(rng: np.random.Generator, shape, mean: float, std: float) -> np.ndarray:
    n = int(np.prod(shape))
    out = np.empty(n, dtype=np.uint16)
    step = 1 << 24
    for i in range(0, n, step):  # chunked so cfg2-sized tensors never hold an fp64 temp
        m = min(step, n - i)
        v = rng.standard_normal(m, dtype=np.float32)
        v *= np.float32(std)
        v += np.float32(mean)
        out[i:i + m] = f32_to_bf16_bits(v)
    return out.reshape(shape)


# ---------------------------------------------------------------------------------------------
# tensors
# ---------------------------------------------------------------------------------------------
def make_weights(shape: LayerShape, seed: int) -> dict:
    """bf16 bit patterns, [out, in] row-major. Reading #9: std 0.02; gains 1 + N(0, 0.02)."""
    d, F = shape.hidden, shape.ffn
    dims = {
        "g1": (d,), "wq": (shape.q_dim, d), "wk": (shape.kv_dim, d), "wv": (shape.kv_dim, d),
        "wo": (d, shape.q_dim), "g2": (d,), "wgate": (F, d), "wup": (F, d), "wdown": (d, F),
    }
    w = {}
    for i, name in enumerate(WEIGHT_NAMES):
        mean = 1.0 if name in ("g1", "g2") else 0.0
        w[name] = _normal_bf16(_rng(seed, i), dims[name], mean, 0.02)
    return w


@dataclass
class StepInputs:
    hidden: np.ndarray        # uint16 [B, d]          bf16 bits
    k_pool: np.ndarray        # uint16 [n_pages, Hkv, page, Dh]
    v_pool: np.ndarray        # uint16 [n_pages, Hkv, page, Dh]
    block_table: np.ndarray   # int32  [B, max_blocks], pad = -1
    seq_lens: np.ndarray      # int32  [B]  tokens attended INCLUDING the one being decoded
    n_pages: int

    def clone(self) -> "StepInputs":
        return StepInputs(self.hidden.copy(), self.k_pool.copy(), self.v_pool.copy(),
                          self.block_table.copy(), self.seq_lens.copy(), self.n_pages)


def draw_contexts(shape: LayerShape, seed: int, batch: int | None = None) -> np.ndarray:
    B = shape.batch if batch is None else batch
    return _rng(seed, 100).integers(shape.ctx_lo, shape.ctx_hi + 1, size=B).astype(np.int32)


def make_step_inputs(shape: LayerShape, seed_act: int, seed_len: int, *, batch: int | None = None,
                     contexts: np.ndarray | None = None, n_pages: int | None = None,
                     poison_unused: bool = False, max_blocks: int | None = None) -> StepInputs:
    B = shape.batch if batch is None else batch
    page = shape.page
    ctx = draw_contexts(shape, seed_len, B) if contexts is None else np.asarray(contexts, np.int32)
    assert ctx.shape == (B,)
    seq = (ctx + 1).astype(np.int32)
    mb = shape.max_blocks if max_blocks is None else max_blocks
    need = (seq + page - 1) // page
    assert int(need.max(initial=0)) <= mb
    total = int(need.sum())
    if n_pages is None:
        n_pages = max(B * mb, total)          # worst-case pool (cfg2: 64*129 = 8256 pages)
    assert n_pages >= total
    ids = _rng(seed_len, 101).permutation(n_pages).astype(np.int32)
    bt = np.full((B, mb), -1, dtype=np.int32)
    # interleave requests page by page so that no request's pages are contiguous ids either
    cursor = 0
    for j in range(int(need.max(initial=0))):
        for b in range(B):
            if j < need[b]:
                bt[b, j] = ids[cursor]
                cursor += 1
    pool_shape = (n_pages, shape.n_kv_heads, page, shape.head_dim)
    k_pool = _normal_bf16(_rng(seed_act, 1), pool_shape, 0.0, 1.0)
    v_pool = _normal_bf16(_rng(seed_act, 2), pool_shape, 0.0, 1.0)
    hidden = _normal_bf16(_rng(seed_act, 0), (B, shape.hidden), 0.0, 1.0)
    if poison_unused:
        poison_unused_kv(k_pool, v_pool, bt, seq, page)
    return StepInputs(hidden, k_pool, v_pool, bt, seq, n_pages)


def poison_unused_kv(k_pool, v_pool, block_table, seq_lens, page: int = PAGE) -> None:
    """NaN every KV slot that no request may read: token index >= seq_len - 1 is excluded from the
    poison only for the slot the step itself writes (position seq_len - 1 is written, then read)."""
    nan = np.uint16(0x7FC0)
    used = np.zeros(k_pool.shape[0] * page, dtype=bool)        # [page*slot]
    for b in range(block_table.shape[0]):
        s = int(seq_lens[b])
        for t in range(max(s - 1, 0)):                         # tokens 0..s-2 are cached input
            used[int(block_table[b, t // page]) * page + t % page] = True
    mask = ~used.reshape(k_pool.shape[0], page)
    for pool in (k_pool, v_pool):
        view = pool.transpose(0, 2, 1, 3)                      # [n_pages, page, Hkv, Dh]
        view[mask] = nan


def even_split(batch: int, n_replicas: int) -> np.ndarray:
    """Reading #15: contiguous ranges; the first (batch % R) replicas take ceil(batch/R) rows."""
    base, rem = divmod(batch, n_replicas)
    out = np.empty(batch, dtype=np.int32)
    pos = 0
    for r in range(n_replicas):
        cnt = base + (1 if r < rem else 0)
        out[pos:pos + cnt] = r
        pos += cnt
    return out


# ---------------------------------------------------------------------------------------------
# algorithmic byte accounting -- bookkeeping only
# ---------------------------------------------------------------------------------------------
def layer_weight_bytes(shape: LayerShape) -> int:
    return 2 * (shape.n_params + 2 * shape.hidden)


def forward_algorithmic_bytes(shape: LayerShape, seq_lens: np.ndarray, n_replicas: int) -> int:
    """R*W_layer + sum_b c_b*(2*Hkv*Dh*2) + B*(2*Hkv*Dh*2) [append] + 2*B*d*2 [hidden in/out]."""
    B = int((np.asarray(seq_lens) > 0).sum())
    ctx = int(np.maximum(np.asarray(seq_lens, np.int64) - 1, 0).sum())
    per_tok = 2 * shape.kv_dim * 2
    return n_replicas * layer_weight_bytes(shape) + ctx * per_tok + B * per_tok + 2 * B * shape.hidden * 2
