"""Mixed prefill + decode steps of MORE than 256 rows (BASELINE.json configs[3]): the large-M
path -- k_big_group, the CTA-pair tcgen05 GEMMs (cc_big_gemm.cu) and the causal chunk-prefill attention kernel over
the paged cache (cc_prefill.cu) beside the decode attention kernel for the rows outside the chunks -- against the
oracle, element by element: every stage tap, the output, the appended K/V.  The oracle needs nothing new: a prompt
chunk is rows of one step that share their request's block-table row at consecutive seq_lens, each row appends
before it attends, so row t sees exactly the positions <= t (tests/test_prefill_chunk.py pins that on the oracle:
chunk step == one token at a time bitwise, and causality).  Every cache slot a chunk is going to write holds NaN
beforehand, so a read of a position not yet appended cannot hide inside the tolerance."""
import numpy as np
import pytest

import oracle
from paper_2607_04181_b200 import inputs as I
from tests.test_gpu_parity import check_grouping, within

pytestmark = pytest.mark.gpu


def mixed_step(shape, seed, chunks, dec_ctx, replicas, interleave=True):
    """`chunks`: [(cached tokens, chunk length)], `dec_ctx`: cached tokens of the decode rows.  Rows: a few decode
    rows, then chunk 0, more decode rows, chunk 1, ... (a chunk's rows are consecutive, as the large path needs).
    Chunk c lives on replica c % R; decode rows alternate."""
    n_req, n_dec = len(chunks), len(dec_ctx)
    ctx = np.array([c + n - 1 for c, n in chunks] + list(dec_ctx), np.int32)
    base = I.make_step_inputs(shape, 2500 + seed, 3500 + seed, batch=n_req + n_dec, n_pages=int(((ctx + 1 + shape.page) // shape.page).sum()) + 8,
                              contexts=ctx)
    rng = np.random.default_rng(4500 + seed)
    k_pool, v_pool = base.k_pool.copy(), base.v_pool.copy()
    bt, seq, ra = [], [], []
    dec_left = list(range(n_dec))
    per_gap = (n_dec + n_req) // (n_req + 1) if interleave else 0

    def add_dec(k):
        for _ in range(k):
            if dec_left:
                j = dec_left.pop(0)
                bt.append(base.block_table[n_req + j]); seq.append(int(dec_ctx[j]) + 1); ra.append(j % replicas)
    for r, (cached, n) in enumerate(chunks):
        add_dec(per_gap)
        for t in range(cached, cached + n):
            bt.append(base.block_table[r]); seq.append(t + 1); ra.append(r % replicas)
            pg = int(base.block_table[r, t // shape.page])
            k_pool[pg, :, t % shape.page, :] = 0x7FC0
            v_pool[pg, :, t % shape.page, :] = 0x7FC0
    add_dec(len(dec_left))
    hidden = I._normal_bf16(rng, (len(seq), shape.hidden), 0.0, 1.0)
    st = I.StepInputs(hidden, k_pool, v_pool, np.stack(bt).astype(np.int32), np.array(seq, np.int32), base.n_pages)
    return st, np.array(ra, np.int32)


def run_gpu(shape, w, st, assign, R, taps=True, max_batch=None):
    import torch
    from paper_2607_04181_b200 import binding as B
    from paper_2607_04181_b200.harness import DeviceStep, Session

    batch = st.hidden.shape[0]
    with Session(shape, w, max_batch=max_batch or batch, max_blocks=st.block_table.shape[1],
                 max_position=st.block_table.shape[1] * shape.page) as S:
        if R > 1:
            S.scale(R)
        step = DeviceStep(st, assign)
        S.forward(step)
        torch.cuda.synchronize()
        assert B.cc_poll_device_error(S.ctx) == 0
        out, (kp, vp) = step.out_bits(), step.pools_bits()
        g = {}
        if taps:
            g = {n: S.tap(t, batch) for n, t in (("x", B.CC_TAP_X), ("q", B.CC_TAP_Q), ("o", B.CC_TAP_O), ("h1", B.CC_TAP_H1),
                                                 ("y", B.CC_TAP_Y), ("a", B.CC_TAP_A))}
        grouping = B.cc_debug_grouping(S.layer, max_batch or batch)   # the buffer is sized from the LAYER's max_batch
    return out, kp, vp, g, grouping


def check(shape, st, assign, R, ref, out, kp, vp, g, grouping):
    rel = {n: within(g[n], ref["taps"][n], f"tap {n}") for n in g}
    written = ~np.isnan(I.bf16_bits_to_f32(ref["k_pool"]))           # NaN left = slots nobody wrote (and nobody attended)
    rel["k"] = within(I.bf16_bits_to_f32(kp)[written], I.bf16_bits_to_f32(ref["k_pool"])[written], "K cache")
    rel["v"] = within(I.bf16_bits_to_f32(vp)[written], I.bf16_bits_to_f32(ref["v_pool"])[written], "V cache")
    assert np.array_equal(kp[~written], st.k_pool[~written]) and np.array_equal(vp[~written], st.v_pool[~written])
    rel["out"] = within(I.bf16_bits_to_f32(out), I.bf16_bits_to_f32(ref["out"]), "layer output")
    check_grouping(grouping, assign, st.seq_lens, R)
    assert max(rel.values()) < 1e-2, rel
    return rel


MID = I.LayerShape("mixmid", 512, 8, 2, 128, 1408, 1e-5, 500000.0, 8, 0, 600)


def test_two_chunks_and_decode_rows_mid_shape():
    """300 rows: a 150-token chunk behind 37 cached tokens (crosses tile and page boundaries, ragged last query tile and
    kv tile), a 70-token chunk from position 0, 80 decode rows with contexts 0..500; two replicas; GQA group 4."""
    shape = MID
    rng = np.random.default_rng(1)
    st, assign = mixed_step(shape, 1, [(37, 150), (0, 70)], rng.integers(0, 500, 80), 2)
    assert st.hidden.shape[0] == 300
    w = I.make_weights(shape, 1501)
    ref = oracle.layer_forward(shape, w, st.hidden, st.k_pool, st.v_pool, st.block_table, st.seq_lens, assign, 2, taps=True)
    out, kp, vp, g, grouping = run_gpu(shape, w, st, assign, 2)
    rel = check(shape, st, assign, 2, ref, out, kp, vp, g, grouping)
    print("mixed mid R=2 normalised rms error per stage:", {k: round(v, 5) for k, v in rel.items()})
    # one replica gives the same bits
    out1, kp1, vp1, _, _ = run_gpu(shape, w, st, np.zeros_like(assign), 1, taps=False)
    assert np.array_equal(out1, out) and np.array_equal(kp1, kp) and np.array_equal(vp1, vp)


def test_cfg4_shape_chunk_with_gqa_group_5():
    """The 14B-class layer of configs[3] (hidden 5120, 40 q / 8 kv heads: 25 tokens x 5 heads per query tile, three rows
    of every MMA tile unused), one 290-token chunk behind 100 cached tokens + 30 decode rows, three replicas."""
    shape = I.LayerShape("mixcfg4", 5120, 40, 8, 128, 17408, 1e-5, 500000.0, 8, 0, 500)
    rng = np.random.default_rng(2)
    st, assign = mixed_step(shape, 2, [(100, 290)], rng.integers(0, 400, 30), 3)
    w = I.make_weights(shape, 1004)
    ref = oracle.layer_forward(shape, w, st.hidden, st.k_pool, st.v_pool, st.block_table, st.seq_lens, assign, 3, taps=True)
    out, kp, vp, g, grouping = run_gpu(shape, w, st, assign, 3)
    rel = check(shape, st, assign, 3, ref, out, kp, vp, g, grouping)
    print("mixed cfg4-shape R=3 normalised rms error per stage:", {k: round(v, 5) for k, v in rel.items()})


def test_causality_and_repeatability_on_the_large_path():
    """Perturbing chunk token 100 changes the rows of tokens >= 100 of that chunk and nothing else (causal mask on the
    diagonal tiles, no leak between the chunks or into the decode rows); the same step twice gives the same bits."""
    shape = MID
    rng = np.random.default_rng(3)
    st, assign = mixed_step(shape, 3, [(20, 200), (5, 60)], rng.integers(0, 300, 40), 2, interleave=False)
    w = I.make_weights(shape, 1501)
    out, kp, vp, _, _ = run_gpu(shape, w, st, assign, 2, taps=False)
    again, kp2, vp2, _, _ = run_gpu(shape, w, st, assign, 2, taps=False)
    assert np.array_equal(out, again) and np.array_equal(kp, kp2) and np.array_equal(vp, vp2)
    st2 = I.StepInputs(st.hidden.copy(), st.k_pool, st.v_pool, st.block_table, st.seq_lens, st.n_pages)
    st2.hidden[100] ^= 0x0040                                        # rows 0..199 are the first chunk (interleave off)
    pert, _, _, _, _ = run_gpu(shape, w, st2, assign, 2, taps=False)
    same = np.array([np.array_equal(pert[b], out[b]) for b in range(out.shape[0])])
    assert same[:100].all() and same[200:].all()
    assert not same[100:200].any()


def test_prefill_then_decode_equals_the_longer_prefill():
    """prefill(n) on the large path, then one decode step of token n on the small path, against prefill(n + 1) on the
    large path: the last row and the cache agree within the tolerance of the same oracle values (the two paths sum K in a
    different order, so bits may differ), and the oracle itself gives the two bitwise equal."""
    import torch
    from paper_2607_04181_b200 import binding as B
    from paper_2607_04181_b200.harness import DeviceStep, Session

    shape = MID
    n = 280
    st, assign = mixed_step(shape, 4, [(0, n + 1)], [], 1)
    w = I.make_weights(shape, 1501)
    ref = oracle.layer_forward(shape, w, st.hidden, st.k_pool, st.v_pool, st.block_table, st.seq_lens, assign, 1)
    full, kpf, vpf, _, _ = run_gpu(shape, w, st, assign, 1, taps=False)
    batch = n + 1
    with Session(shape, w, max_batch=batch, max_blocks=st.block_table.shape[1], max_position=st.block_table.shape[1] * shape.page) as S:
        step = DeviceStep(st, assign)
        step.seq_lens[n:].zero_()                                    # prefill(n): the last row is padding
        S.forward(step)
        torch.cuda.synchronize()
        head = step.out_bits()[:n].copy()
        one = DeviceStep(I.StepInputs(st.hidden[n:], st.k_pool, st.v_pool, st.block_table[n:], st.seq_lens[n:], st.n_pages), assign[n:])
        one.k_pool, one.v_pool = step.k_pool, step.v_pool            # the cache prefill(n) left behind
        B.cc_forward(S.layer, one.hidden, one.k_pool, one.v_pool, one.block_table, one.n_pages, one.seq_lens, one.assign, 1, None)
        torch.cuda.synchronize()
        assert B.cc_poll_device_error(S.ctx) == 0
        last = one.out_bits()[0]
        kp, vp = step.pools_bits()
    assert np.array_equal(head, full[:n])                            # rows 0..n-1 do not see token n: same path, same bits
    want = I.bf16_bits_to_f32(ref["out"][n])
    within(I.bf16_bits_to_f32(last), want, "decode after prefill")
    within(I.bf16_bits_to_f32(full[n]), want, "last row of the longer prefill")
    written = ~np.isnan(I.bf16_bits_to_f32(ref["k_pool"]))
    within(I.bf16_bits_to_f32(kp)[written], I.bf16_bits_to_f32(kpf)[written], "cache: prefill + decode vs longer prefill")
    within(I.bf16_bits_to_f32(vp)[written], I.bf16_bits_to_f32(vpf)[written], "cache: prefill + decode vs longer prefill")


def test_small_steps_of_a_large_layer_take_the_decode_path_and_keep_their_bits():
    """A layer created for large steps (max_batch 2048) runs a 40-row step through the decode kernels: same bits as the
    same step on a layer created with max_batch 40."""
    shape = MID
    rng = np.random.default_rng(5)
    st, assign = mixed_step(shape, 5, [(10, 25)], rng.integers(0, 300, 15), 2)
    w = I.make_weights(shape, 1501)
    a = run_gpu(shape, w, st, assign, 2, taps=False)
    b = run_gpu(shape, w, st, assign, 2, taps=False, max_batch=2048)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2])


@pytest.mark.parametrize("hkv,g", [(1, 8), (2, 1), (4, 3), (8, 2), (1, 1)])
def test_large_path_head_layouts(hkv, g):
    """The chunk-prefill kernel packs T = 128 // G tokens x G query heads into the 128 rows of its MMA tile and stages one
    kv head per work item: every kv-head count the library takes and GQA groups 1, 2, 3 and 8 (T = 128, 64, 42, 16; G = 3
    leaves two rows of the tile unused), chunk lengths that are not multiples of T, kv lengths that end on and next to the
    64-token kv tile and the 16-token page boundaries, a 2-token chunk."""
    shape = I.LayerShape(f"mixh{hkv}g{g}", 256, hkv * g, hkv, 128, 512, 1e-5, 10000.0, 8, 0, 400)
    rng = np.random.default_rng(40 + hkv * 10 + g)
    chunks = [(0, 64), (63, 130), (1, 2), (128, 191)]            # ends at kv 64, 193, 3, 319
    st, assign = mixed_step(shape, 40 + hkv * 10 + g, chunks, rng.integers(0, 200, 20), 2)
    assert st.hidden.shape[0] > 256
    w = I.make_weights(shape, 1700 + hkv * 10 + g)
    ref = oracle.layer_forward(shape, w, st.hidden, st.k_pool, st.v_pool, st.block_table, st.seq_lens, assign, 2, taps=True)
    out, kp, vp, gt, grouping = run_gpu(shape, w, st, assign, 2)
    check(shape, st, assign, 2, ref, out, kp, vp, gt, grouping)


def test_too_many_decode_rows_are_reported_not_faulted():
    """A large step may hold at most 256 rows outside prompt chunks: 300 lone rows set CC_DEVERR_TOO_MANY_DECODE (the
    surplus rows' attention is skipped), nothing faults, and the first 256 decode rows are still right."""
    import torch
    from paper_2607_04181_b200 import binding as B
    from paper_2607_04181_b200.harness import DeviceStep, Session

    shape = MID
    rng = np.random.default_rng(9)
    st, assign = mixed_step(shape, 9, [], rng.integers(0, 120, 300), 2)
    w = I.make_weights(shape, 1501)
    ref = oracle.layer_forward(shape, w, st.hidden, st.k_pool, st.v_pool, st.block_table, st.seq_lens, assign, 2, taps=True)
    with Session(shape, w, max_batch=300, max_blocks=st.block_table.shape[1], max_position=st.block_table.shape[1] * shape.page) as S:
        S.scale(2)
        step = DeviceStep(st, assign)
        S.forward(step)
        torch.cuda.synchronize()
        assert B.cc_poll_device_error(S.ctx) == B.CC_DEVERR_TOO_MANY_DECODE
        o = S.tap(B.CC_TAP_O, 300)
    within(o[:256], ref["taps"]["o"][:256], "attention output of the first 256 decode rows")


def test_cfg4_full_size_mixed_step_on_sampled_oracle_rows():
    """BASELINE.json configs[3] at FULL size, the step `bench.py --workload cfg4` times: the 14B-class layer, two
    2048-token prompt chunks from position 0 and 256 decode rows with contexts U{256..4096} = 4352 rows in one cc_forward,
    two replicas (prompt r on replica r % 2, decode rows alternate).  The oracle cannot run 4352 rows of this layer in a
    test's time, so: (1) the K/V every row of the step appends -- the oracle's own a1-a4 (rmsnorm, matmul_wt, rope, bf16
    round: oracle/cc_oracle.c orc_sub_batch) over ALL rows -- against the GPU's cache, slot by slot, every other slot
    bit-identical to the input; (2) with those K/V in the cache, oracle.layer_forward on SAMPLED rows one by one: the
    first, second, tile-boundary (G = 5: 25 tokens per query tile; kv tiles of 64), middle and last tokens of both chunks,
    the decode rows with the shortest and the longest context and six more -- layer output and the taps q, o, h1."""
    import torch
    from paper_2607_04181_b200 import binding as B
    from paper_2607_04181_b200.harness import DeviceStep, Session

    shape = I.LayerShape("cfg4full", 5120, 40, 8, 128, 17408, 1e-5, 500000.0, 256, 256, 4096)
    Hkv, Dh, page = shape.n_kv_heads, shape.head_dim, shape.page
    rng = np.random.default_rng(44)
    dec_ctx = rng.integers(256, 4097, 256)
    dec_ctx[0], dec_ctx[1] = 4096, 256
    st, assign = mixed_step(shape, 44, [(0, 2048), (0, 2048)], dec_ctx, 2)
    batch = st.hidden.shape[0]
    assert batch == 4352
    w = I.make_weights(shape, 1004)
    with Session(shape, w, max_batch=batch, max_blocks=st.block_table.shape[1],
                 max_position=st.block_table.shape[1] * page) as S:
        S.scale(2)
        step = DeviceStep(st, assign)
        S.forward(step)
        torch.cuda.synchronize()
        assert B.cc_poll_device_error(S.ctx) == 0
        out, (kp, vp) = step.out_bits(), step.pools_bits()
        gt = {n: S.tap(t, batch) for n, t in (("q", B.CC_TAP_Q), ("o", B.CC_TAP_O), ("h1", B.CC_TAP_H1))}
        del step
    # (1) the appended K/V of all rows
    seq = st.seq_lens.astype(np.int64)
    x = oracle.rmsnorm(I.bf16_bits_to_f32(st.hidden), w["g1"], shape.rms_eps)
    k, v = oracle.matmul_wt(x, w["wk"]), oracle.matmul_wt(x, w["wv"])
    for b in range(batch):
        k[b] = oracle.rope(k[b], Hkv, Dh, int(seq[b]) - 1, shape.rope_base)
    kb = I.f32_to_bf16_bits(k).reshape(batch, Hkv, Dh)
    vb = I.f32_to_bf16_bits(v).reshape(batch, Hkv, Dh)
    pg = st.block_table[np.arange(batch), (seq - 1) // page]
    sl = (seq - 1) % page
    rel_k = within(I.bf16_bits_to_f32(kp[pg, :, sl, :]), I.bf16_bits_to_f32(kb), "appended K of all 4352 rows")
    rel_v = within(I.bf16_bits_to_f32(vp[pg, :, sl, :]), I.bf16_bits_to_f32(vb), "appended V of all 4352 rows")
    for mine, theirs in ((st.k_pool, kp), (st.v_pool, vp)):          # nothing else in the cache changed
        tmp = mine.copy()
        tmp[pg, :, sl, :] = theirs[pg, :, sl, :]
        assert np.array_equal(tmp, theirs)
        del tmp
    # (2) sampled rows through the whole layer
    kin, vin = st.k_pool.copy(), st.v_pool.copy()
    kin[pg, :, sl, :] = kb
    vin[pg, :, sl, :] = vb
    starts = np.nonzero(seq == 1)[0]
    assert len(starts) == 2
    in_chunk = np.zeros(batch, bool)
    sample = []
    for s0 in starts:
        assert np.array_equal(seq[s0:s0 + 2048], np.arange(1, 2049))
        in_chunk[s0:s0 + 2048] = True
        sample += [s0 + t for t in (0, 1, 24, 25, 63, 64, 1023, 2047)]
    dec = np.nonzero(~in_chunk)[0]
    assert len(dec) == 256
    sample += [int(dec[np.argmax(seq[dec])]), int(dec[np.argmin(seq[dec])])] + [int(b) for b in rng.choice(dec, 6, replace=False)]
    sample = np.array(sorted(set(sample)))
    ref = oracle.layer_forward(shape, w, st.hidden[sample], kin, vin, st.block_table[sample], st.seq_lens[sample], assign[sample],
                               2, taps=True)
    rel = {"k": rel_k, "v": rel_v}
    for n in ("q", "o", "h1"):
        rel[n] = within(gt[n][sample], ref["taps"][n], f"tap {n} of the sampled rows")
    rel["out"] = within(I.bf16_bits_to_f32(out[sample]), I.bf16_bits_to_f32(ref["out"]), "layer output of the sampled rows")
    print("cfg4 full size, sampled rows, normalised rms error per stage:", {a: round(b, 5) for a, b in rel.items()})
    assert max(rel.values()) < 1e-2, rel
