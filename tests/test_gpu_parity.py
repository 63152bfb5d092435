"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Tolerance from BASELINE.json north_star: |gpu - ref| <= 1e-2 + 2e-2 |ref|
per element (bf16), checked on the layer output, on the appended K/V, and on every stage tap
(the final-output check alone could hide an attention bug)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2607_04181_b200 import inputs as I

pytestmark = [pytest.mark.gpu, pytest.mark.usefixtures("operand_format")]   # both GEMM operand formats

ATOL, RTOL = 1e-2, 2e-2


def within(gpu, ref, what):
    gpu = np.asarray(gpu, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    assert gpu.shape == ref.shape, what
    assert np.isfinite(gpu).all(), f"{what}: non-finite GPU values"
    err = np.abs(gpu - ref)
    bound = ATOL + RTOL * np.abs(ref)
    bad = err > bound
    assert not bad.any(), (f"{what}: {int(bad.sum())}/{bad.size} elements outside tolerance; worst |err|="
                           f"{err.max():.4g} at {np.unravel_index(err.argmax(), err.shape)}, ref rms={np.sqrt((ref**2).mean()):.4g}")
    return float(np.sqrt((err ** 2).mean()) / max(np.sqrt((ref ** 2).mean()), 1e-30))


def run_case(shape, batch, n_replicas, assign=None, contexts=None, poison=False, seeds=(1001, 2001, 3001), taps=True,
             seq_override=None):
    from paper_2607_04181_b200 import binding as B
    from paper_2607_04181_b200.harness import DeviceStep, Session

    w = I.make_weights(shape, seeds[0])
    st = I.make_step_inputs(shape, seeds[1], seeds[2], batch=batch, contexts=contexts, poison_unused=poison)
    if seq_override is not None:
        st.seq_lens[:] = seq_override
    if assign is None:
        assign = I.even_split(batch, n_replicas)
    ref = oracle.layer_forward(shape, w, st.hidden, st.k_pool, st.v_pool, st.block_table, st.seq_lens, assign,
                               n_replicas, taps=taps)
    with Session(shape, w, max_batch=batch) as S:
        if n_replicas > 1:
            S.scale(n_replicas)
        step = DeviceStep(st, assign)
        S.forward(step)
        torch.cuda.synchronize()
        assert B.cc_poll_device_error(S.ctx) == 0
        out = step.out_bits()
        kp, vp = step.pools_bits()
        gtaps = {}
        if taps:
            for name, which in (("x", B.CC_TAP_X), ("q", B.CC_TAP_Q), ("o", B.CC_TAP_O), ("h1", B.CC_TAP_H1),
                                ("y", B.CC_TAP_Y), ("a", B.CC_TAP_A)):
                gtaps[name] = S.tap(which, batch)
        perm, counts, n_pos = B.cc_debug_grouping(S.layer, batch)
    return st, ref, out, kp, vp, gtaps, (perm, counts, n_pos), assign


def check_against_oracle(shape, st, ref, out, kp, vp, gtaps, assign, n_replicas):
    live = st.seq_lens > 0
    rel = {}
    for name in ("x", "q", "o", "h1", "y", "a"):
        if name in gtaps:
            rel[name] = within(gtaps[name][live], ref["taps"][name][live], f"tap {name}")
    # appended K/V: every pool slot except the ones this step wrote must be bit-identical to the
    # input; the written ones match the oracle's within tolerance (bf16 of an fp32 sum)
    rk, rv = ref["k_pool"], ref["v_pool"]
    written = np.zeros(st.k_pool.shape[:1] + st.k_pool.shape[2:3], dtype=bool)       # [page, slot]
    for b in np.nonzero(live)[0]:
        p = int(st.seq_lens[b]) - 1
        written[int(st.block_table[b, p // shape.page]), p % shape.page] = True
    wmask = np.broadcast_to(written[:, None, :, None], st.k_pool.shape)
    assert np.array_equal(kp[~wmask], st.k_pool[~wmask]) and np.array_equal(vp[~wmask], st.v_pool[~wmask])
    rel["k_new"] = within(I.bf16_bits_to_f32(kp[wmask]), I.bf16_bits_to_f32(rk[wmask]), "appended K")
    rel["v_new"] = within(I.bf16_bits_to_f32(vp[wmask]), I.bf16_bits_to_f32(rv[wmask]), "appended V")
    rel["out"] = within(I.bf16_bits_to_f32(out), I.bf16_bits_to_f32(ref["out"]), "layer output")
    # padding rows pass through untouched
    assert np.array_equal(out[~live], st.hidden[~live])
    return rel


def check_grouping(grouping, assign, seq_lens, n_replicas):
    perm, counts, n_pos = grouping
    operm, ocounts = oracle.group_rows(assign, seq_lens, n_replicas)
    assert np.array_equal(counts[:n_replicas], ocounts) and not counts[n_replicas:].any()
    assert np.array_equal(perm[perm >= 0], operm)                         # stable partition, exact
    off = 0
    for r in range(n_replicas):                                           # groups start at multiples of 16
        assert np.array_equal(perm[off:off + counts[r]], operm[ocounts[:r].sum():ocounts[:r + 1].sum()])
        off += (counts[r] + 15) // 16 * 16
    assert n_pos == off


@pytest.mark.parametrize("R", [1, 2])
def test_cfg1_parity_with_taps(R):
    shape = I.CFG1
    st, ref, out, kp, vp, gtaps, grouping, assign = run_case(shape, shape.batch, R)
    rel = check_against_oracle(shape, st, ref, out, kp, vp, gtaps, assign, R)
    check_grouping(grouping, assign, st.seq_lens, R)
    print("cfg1 R=%d normalised rms error per stage:" % R, {k: round(v, 5) for k, v in rel.items()})
    assert max(rel.values()) < 1e-2


def test_cfg1_ragged_batch_and_page_boundaries():
    # contexts straddling page boundaries (15,16,17 cached tokens), a padding row, uneven 3-replica split
    shape = I.CFG1
    ctx = np.array([15, 16, 17, 0, 31, 32, 64, 1, 47], dtype=np.int32)
    B_ = ctx.shape[0]
    assign = np.array([0, 2, 1, 1, 0, 2, 2, 0, 1], dtype=np.int32)
    seq = ctx + 1
    seq[3] = 0                                                            # padding row
    st, ref, out, kp, vp, gtaps, grouping, assign = run_case(shape, B_, 3, assign=assign, contexts=ctx, seq_override=seq)
    check_against_oracle(shape, st, ref, out, kp, vp, gtaps, assign, 3)
    check_grouping(grouping, assign, st.seq_lens, 3)


def test_cfg1_nan_poison_outside_context_never_read():
    shape = I.CFG1
    st, ref, out, kp, vp, gtaps, _, assign = run_case(shape, shape.batch, 1, poison=True)
    assert np.isnan(I.bf16_bits_to_f32(st.k_pool)).any()
    assert np.isfinite(I.bf16_bits_to_f32(out)).all()
    check_against_oracle(shape, st, ref, out, kp, vp, gtaps, assign, 1)


def test_context_of_length_one_returns_v():
    # s = 1: attention over the single (just appended) token returns its V for every q head of the group
    shape = I.CFG1
    st, ref, out, kp, vp, gtaps, _, assign = run_case(shape, 4, 1, contexts=np.zeros(4, np.int32))
    G = shape.n_q_heads // shape.n_kv_heads
    for b in range(4):
        page = int(st.block_table[b, 0])
        v = I.bf16_bits_to_f32(vp[page, :, 0, :])                          # [Hkv, Dh] as stored (bf16)
        o = gtaps["o"][b].reshape(shape.n_q_heads, shape.head_dim)
        for hq in range(shape.n_q_heads):
            assert np.array_equal(I.f32_to_bf16_bits(o[hq]), I.f32_to_bf16_bits(v[hq // G]))
    check_against_oracle(shape, st, ref, out, kp, vp, gtaps, assign, 1)


def test_midsize_shape_spans_tiles_and_chunks():
    # several GEMM tiles / k-blocks per CTA range, > 1 attention chunk per row, ragged group sizes
    shape = I.LayerShape("mid", 512, 8, 2, 128, 1408, 1e-5, 500000.0, 21, 200, 700)
    assign = (np.arange(21) * 7 % 4).astype(np.int32)
    st, ref, out, kp, vp, gtaps, grouping, assign = run_case(shape, 21, 4, assign=assign, seeds=(1007, 2007, 3007))
    rel = check_against_oracle(shape, st, ref, out, kp, vp, gtaps, assign, 4)
    check_grouping(grouping, assign, st.seq_lens, 4)
    print("mid R=4 normalised rms error per stage:", {k: round(v, 5) for k, v in rel.items()})
