"""CPU tests of the C-ABI boundary (-m "not gpu"): the library builds and loads without a GPU,
exports every function include/cocoscale.h declares, fails loudly without a device (no CPU
fallback), and its host-only slot allocator agrees with the oracle-side brute-force simulation."""
import ctypes
import os
import re

import numpy as np
import pytest

from oracle import hostsim
from paper_2607_04181_b200 import binding as B

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "cocoscale.h")


def declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(cc_[a-z0-9_]+)\s*\(", src)))


def test_header_and_library_export_the_same_functions():
    decl = declared_functions()
    assert len(decl) >= 25
    lib = ctypes.CDLL(B.library_path())
    for name in decl:
        assert hasattr(lib, name), f"{name} is declared in cocoscale.h but not exported"
    assert sorted(B.EXPORTS) == decl
    for name in decl:                                   # the binding has a function of the same name for each
        assert callable(getattr(B, name)), name
    assert "sm_100a" in B.cc_version()


def test_struct_layouts_match_the_header():
    assert ctypes.sizeof(B.cc_layer_desc) == 11 * 4
    assert ctypes.sizeof(B.cc_layer_weights) == 9 * 8
    assert ctypes.sizeof(B.cc_kv_pages) == 32
    assert B.cc_layer_desc.rms_eps.offset == 20 and B.cc_layer_desc.page_size.offset == 28


def test_struct_layouts_match_what_the_c_compiler_sees(tmp_path):
    """sizeof and every field offset of the structs that cross the boundary, as gcc lays them out from
    include/cocoscale.h, against the ctypes mirrors in binding.py."""
    import os
    import subprocess
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    structs = {"cc_layer_desc": B.cc_layer_desc, "cc_layer_weights": B.cc_layer_weights, "cc_kv_pages": B.cc_kv_pages,
               "cc_ctl_params": B.cc_ctl_params, "cc_ctl_instance": B.cc_ctl_instance, "cc_ctl_device": B.cc_ctl_device,
               "cc_ctl_placement": B.cc_ctl_placement}
    lines = ['#include <stdio.h>', '#include <stddef.h>', '#include "include/cocoscale.h"', 'int main(void) {']
    for name, st in structs.items():
        lines.append(f'  printf("{name} %zu\\n", sizeof({name}));')
        for field, _ in st._fields_:
            lines.append(f'  printf("{name}.{field} %zu\\n", offsetof({name}, {field}));')
    lines += ['  return 0;', '}']
    src, exe = tmp_path / "layout.c", tmp_path / "layout"
    src.write_text("\n".join(lines))
    subprocess.run(["gcc", "-std=c99", "-I", root, str(src), "-o", str(exe)], check=True)
    seen = dict(l.split() for l in subprocess.run([str(exe)], check=True, stdout=subprocess.PIPE, text=True).stdout.splitlines())
    for name, st in structs.items():
        assert int(seen[name]) == ctypes.sizeof(st), name
        for field, _ in st._fields_:
            assert int(seen[f"{name}.{field}"]) == getattr(st, field).offset, f"{name}.{field}"


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(B.CcError) as e:
        B.cc_ctx_create(0)
    assert e.value.status == B.CC_ERR_CUDA
    assert "no CPU fallback" in str(e.value)


def test_slot_allocator_scripted_scenarios():
    a = B.cc_slotalloc_create()
    try:
        assert B.cc_slotalloc_donate(a, 0x10000, 10 * 4096) == B.CC_OK
        assert B.cc_slotalloc_donate(a, 0x10000, 4096) == B.CC_ERR_INVALID       # same base
        assert B.cc_slotalloc_donate(a, 0x11000, 4096) == B.CC_ERR_INVALID       # overlaps
        got = [B.cc_slotalloc_alloc(a, 4096)[1] for _ in range(3)]
        assert got == [0x10000, 0x11000, 0x12000]                                # lowest free first
        assert B.cc_slotalloc_free(a, got[1]) == B.CC_OK
        assert B.cc_slotalloc_alloc(a, 4096) == (B.CC_OK, got[1])                # the freed middle slot is reused
        assert B.cc_slotalloc_reclaim(a, 0x10000) == B.CC_ERR_BUSY
        assert B.cc_slotalloc_alloc(a, 8 * 4096)[0] == B.CC_ERR_NO_SLOT          # 7 pages left
        assert B.cc_slotalloc_free_bytes(a) == 7 * 4096
        for x in got:
            assert B.cc_slotalloc_free(a, x) == B.CC_OK
        assert B.cc_slotalloc_free(a, got[0]) == B.CC_ERR_INVALID                # double free
        assert B.cc_slotalloc_reclaim(a, 0x10000) == B.CC_OK
        assert B.cc_slotalloc_reclaim(a, 0x10000) == B.CC_ERR_INVALID
        assert B.cc_slotalloc_alloc(a, 16)[0] == B.CC_ERR_NO_SLOT
        # unaligned donation is trimmed to 1024-byte boundaries
        assert B.cc_slotalloc_donate(a, 1000, 5000) == B.CC_OK
        assert B.cc_slotalloc_free_bytes(a) == 4096
        assert B.cc_slotalloc_alloc(a, 1)[1] == 1024
    finally:
        B.cc_slotalloc_destroy(a)


def test_slot_allocator_matches_bruteforce_simulation():
    rng = np.random.default_rng(7)
    for trial in range(20):
        a, sim = B.cc_slotalloc_create(), hostsim.SlotAllocSim()
        live, bases = [], []
        try:
            for step in range(300):
                op = rng.integers(0, 10)
                if op == 0 or not bases:
                    base = int(rng.integers(0, 1 << 22)) * int(rng.choice([1, 16, 1024]))
                    n = int(rng.integers(1, 64)) * int(rng.choice([1000, 1024, 4096]))
                    ok = sim.donate(base, n)
                    assert (B.cc_slotalloc_donate(a, base, n) == B.CC_OK) == ok
                    if ok:
                        bases.append(base)
                elif op == 1:
                    base = bases[int(rng.integers(len(bases)))]
                    want = sim.reclaim(base)
                    st = B.cc_slotalloc_reclaim(a, base)
                    assert st == {"ok": B.CC_OK, "busy": B.CC_ERR_BUSY, "invalid": B.CC_ERR_INVALID}[want]
                    if want == "ok":
                        bases.remove(base)
                elif op < 7:
                    n = int(rng.integers(1, 24)) * int(rng.choice([512, 1024, 3000]))
                    want = sim.alloc(n)
                    st, addr = B.cc_slotalloc_alloc(a, n)
                    assert addr == want and (st == B.CC_OK) == (want is not None)
                    if want is not None:
                        live.append(want)
                elif live:
                    x = live.pop(int(rng.integers(len(live))))
                    assert sim.free(x) and B.cc_slotalloc_free(a, x) == B.CC_OK
                assert B.cc_slotalloc_free_bytes(a) == sim.free_bytes()
        finally:
            B.cc_slotalloc_destroy(a)
