"""The tracing build (python -m paper_2607_04181_b200.build --trace): the product library refuses cc_debug_trace,
the tracing library produces a timeline whose points are ordered the way the kernels are chained."""
import os
import re
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_product_build_has_no_trace_points():
    from paper_2607_04181_b200 import binding as B
    ctx = B.cc_ctx_create(0)
    try:
        with pytest.raises(B.CcError) as e:
            B.cc_debug_trace(ctx)
        assert e.value.status == B.CC_ERR_STATE
    finally:
        B.cc_ctx_destroy(ctx)


def test_timeline_of_the_tracing_build():
    r = subprocess.run([sys.executable, "-m", "paper_2607_04181_b200.timeline", "--replays", "3", "--replicas", "2"], cwd=ROOT,
                       stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True, timeout=900)
    assert r.returncode == 0, r.stdout[-2000:]
    rows = {}
    for line in r.stdout.splitlines():
        m = re.match(r"^(prologue|gemm_qkv|attention|gemm_o|gemm_gate_up|gemm_down)\s+(.*\.\..*)$", line)
        if m and "|" in m.group(2):
            rows[m.group(1)] = [tuple(float(x) for x in p.split("..")) for p in m.group(2).split("|")]
    assert set(rows) == {"prologue", "gemm_qkv", "attention", "gemm_o", "gemm_gate_up", "gemm_down"}
    for name, pts in rows.items():
        assert all(lo <= hi for lo, hi in pts), name
        assert all(a[1] <= b[1] + 1e-6 for a, b in zip(pts, pts[1:])), name          # the latest CTA passes the points in order
    # the chain: a kernel's dependency wait ends only after its predecessor's last CTA has ended
    chain = ["prologue", "gemm_qkv", "attention", "gemm_o", "gemm_gate_up", "gemm_down"]
    for a, b in zip(chain, chain[1:]):
        assert rows[b][1][0] >= rows[a][-1][1] - 0.5, (a, b, rows[a][-1], rows[b][1])
    assert 150.0 < rows["gemm_down"][-1][1] < 400.0                                   # a cfg2 step at R=2 takes ~240 us
    assert "stream-K fixup" in r.stdout
