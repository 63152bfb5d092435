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
