"""oracle/hostsim.py -- TEST INFRASTRUCTURE: brute-force integer simulation of the host-side
structures of the hot path.  Written independently of the C++
allocator: it keeps only the set of live allocations and searches candidate addresses, whereas
the library keeps an address-ordered free list with coalescing.

Rule being simulated: donated ranges are trimmed to
ALIGN-byte boundaries; an allocation of `size` bytes (rounded up to ALIGN) goes to the LOWEST
address, over all donated ranges, at which it fits without overlapping a live allocation;
a range can be reclaimed only while it holds no live allocation.  This is the single-GPU
analogue of the paper's free_mem / Delta_res bookkeeping.
"""
from __future__ import annotations

ALIGN = 1024


def _up(x: int, a: int = ALIGN) -> int:
    return (x + a - 1) // a * a


class SlotAllocSim:
    def __init__(self):
        self.ranges = {}   # base(as donated) -> (lo, hi) trimmed
        self.live = {}     # addr -> size (rounded)

    def donate(self, base: int, nbytes: int) -> bool:
        lo, hi = _up(base), (base + nbytes) // ALIGN * ALIGN
        if hi <= lo or base in self.ranges:
            return False
        for (l, h) in self.ranges.values():
            if lo < h and l < hi:
                return False
        self.ranges[base] = (lo, hi)
        return True

    def reclaim(self, base: int) -> str:
        if base not in self.ranges:
            return "invalid"
        lo, hi = self.ranges[base]
        if any(lo <= a < hi for a in self.live):
            return "busy"
        del self.ranges[base]
        return "ok"

    def alloc(self, nbytes: int):
        size = _up(max(nbytes, 1))
        best = None
        for (lo, hi) in self.ranges.values():
            cands = [lo] + [a + s for a, s in self.live.items() if lo <= a < hi]
            for c in sorted(cands):
                if c + size > hi:
                    continue
                if all(not (c < a + s and a < c + size) for a, s in self.live.items()):
                    if best is None or c < best:
                        best = c
                    break
        if best is None:
            return None
        self.live[best] = size
        return best

    def free(self, addr: int) -> bool:
        return self.live.pop(addr, None) is not None

    def free_bytes(self) -> int:
        tot = sum(h - l for l, h in self.ranges.values())
        return tot - sum(self.live.values())


def split_counts(bs: int, v: int):
    """the heaviest device processes ceil(bs/v) tokens, the others floor(bs/v)."""
    return -(-bs // v), bs // v


# ---------------------------------------------------------------------------------------------
# KV partition per replica.  Independent statement of
# the planner's rule, written with sets and searches instead of the library's cursor walk.
# ---------------------------------------------------------------------------------------------
def plan_kv_migration(block_table, seq_lens, assign, n_pages: int, n_replicas: int, page: int = 16):
    """Rule: partition r = pages [r*psz, (r+1)*psz), psz = n_pages // n_replicas.  Rows in increasing order,
    their pages in increasing order: a page outside the partition of its row's replica moves to the lowest
    page of that partition that was referenced by no live row before the call and was not taken by an
    earlier move.  Returns (new_block_table, moves) with moves = [(src, dst), ...], or None when a
    partition runs out of free pages."""
    import numpy as np
    bt = np.array(block_table, dtype=np.int64)
    psz = n_pages // n_replicas
    referenced = set()
    for b in range(bt.shape[0]):
        if seq_lens[b] > 0:
            for j in range(-(-int(seq_lens[b]) // page)):
                referenced.add(int(bt[b, j]))
    taken = set()
    moves = []
    new_bt = bt.copy()
    for b in range(bt.shape[0]):
        if seq_lens[b] <= 0:
            continue
        r = int(assign[b])
        part = range(r * psz, (r + 1) * psz)
        for j in range(-(-int(seq_lens[b]) // page)):
            pg = int(bt[b, j])
            if pg in part:
                continue
            free = [q for q in part if q not in referenced and q not in taken]
            if not free:
                return None
            q = min(free)
            taken.add(q)
            moves.append((pg, q))
            new_bt[b, j] = q
    return new_bt.astype(np.int32), moves


def plan_kv_catchup(block_table_now, seq_planned, seq_now, planned_block_table, assign, n_pages: int, n_replicas: int,
                    page: int = 16):
    """Second half of a pre-copy migration (decoding continues while the cache is moved chunk by
    chunk).  Token t of a row lives in page t // page of its row, and a decode step of length s only writes
    token s - 1: after a plan made with seq_planned, only tokens >= seq_planned - 1 can have been
    written.  Pages holding such a token -- wherever the row holds them NOW -- are (re)planned by
    plan_kv_migration's rule, the others stay where the first plan put them.  Returns (final_block_table, moves) or None when a partition is full."""
    import numpy as np
    now = np.array(block_table_now, dtype=np.int64)
    planned = np.array(planned_block_table, dtype=np.int64)
    mixed = now.copy()
    for b in range(now.shape[0]):
        if seq_now[b] <= 0:
            continue
        assert seq_now[b] >= seq_planned[b]
        for j in range(-(-int(seq_now[b]) // page)):
            written_since = (j + 1) * page > int(seq_planned[b]) - 1            # holds a token position >= seq_planned - 1
            if not written_since:
                mixed[b, j] = planned[b, j]
    return plan_kv_migration(mixed, seq_now, assign, n_pages, n_replicas, page)


def apply_kv_migration(k_pool, v_pool, moves):
    """Byte copy of whole pages (all kv heads) in both pools, in move order."""
    for s, d in moves:
        k_pool[d] = k_pool[s]
        v_pool[d] = v_pool[s]
