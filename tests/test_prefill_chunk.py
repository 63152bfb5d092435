"""Chunked prefill through the decode path (the part that needs no new kernel): the tokens of
a prompt chunk are rows of one step that share their request's block-table row, token t at seq_len = t + 1.  Every
row's K/V is appended before any row attends (PAPER.md:103 appends, then the attention of the step), so row t sees
exactly the positions <= t: causal attention over the paged cache.  Pins: on the oracle one step over the chunk equals
the same tokens decoded one by one BITWISE; on the GPU the chunk step matches the oracle within the tolerance, and its
KV cache equals the one-by-one GPU run bitwise.  (Cost: each row streams its own prefix, so this is the functional
path for short chunks, not the large-M kernels NEXT-2 asks for -- DESIGN.md section 10.)"""
import numpy as np
import pytest

import oracle
from paper_2607_04181_b200 import inputs as I

SHAPE = I.LayerShape("chunk", 512, 8, 2, 128, 1408, 1e-5, 500000.0, 8, 40, 1800)
# (tokens already cached, chunk length): positions 90..126 cross pages 5|6 and 6|7; the long one writes 13 pages behind
# 94 pages of prefix, which the attention kernel streams while the QKV kernel is still appending
CASES = [(90, 37), (1500, 200)]


def _scenario(CACHED, N_CHUNK):
    """6 ordinary decode rows + one request whose N_CHUNK-token chunk starts after CACHED cached tokens."""
    base = I.make_step_inputs(SHAPE, 2401, 3401, batch=7, n_pages=7 * SHAPE.max_blocks,
                              contexts=np.array([41, 300, 77, 128, 255, 64, CACHED + N_CHUNK - 1], np.int32))
    rng = np.random.default_rng(2402)
    B = 6 + N_CHUNK
    hidden = np.empty((B, SHAPE.hidden), np.uint16)
    hidden[:6] = base.hidden[:6]
    hidden[6:] = I._normal_bf16(rng, (N_CHUNK, SHAPE.hidden), 0.0, 1.0)
    bt = np.vstack([base.block_table[:6]] + [base.block_table[6:7]] * N_CHUNK).astype(np.int32)
    seq = np.concatenate([base.seq_lens[:6], CACHED + 1 + np.arange(N_CHUNK)]).astype(np.int32)
    assign = np.concatenate([[0, 1, 0, 1, 0, 1], np.ones(N_CHUNK)]).astype(np.int32)    # a request lives on ONE replica
    # every cache slot the chunk is going to fill holds NaN beforehand: a row that read a position before the row of
    # that position had appended it (the attention kernel streams pages ahead of the QKV kernel's end) shows up as NaN
    k_pool, v_pool = base.k_pool.copy(), base.v_pool.copy()
    for t in range(CACHED, CACHED + N_CHUNK):
        pg = int(base.block_table[6, t // SHAPE.page])
        k_pool[pg, :, t % SHAPE.page, :] = 0x7FC0
        v_pool[pg, :, t % SHAPE.page, :] = 0x7FC0
    return I.StepInputs(hidden, k_pool, v_pool, bt, seq, base.n_pages), assign


def _one_by_one(st, assign):
    """The same tokens as single steps: the decode rows and token 0 of the chunk first, then one chunk token per step."""
    steps = [np.arange(7)] + [np.array([6 + t]) for t in range(1, st.hidden.shape[0] - 6)]
    return [(rows, I.StepInputs(st.hidden[rows], None, None, st.block_table[rows], st.seq_lens[rows], st.n_pages), assign[rows])
            for rows in steps]


@pytest.mark.parametrize("cached,n_chunk", CASES)
def test_oracle_chunk_step_equals_one_token_at_a_time_bitwise(cached, n_chunk):
    w = I.make_weights(SHAPE, 1401)
    st, assign = _scenario(cached, n_chunk)
    N_CHUNK = n_chunk
    chunk = oracle.layer_forward(SHAPE, w, st.hidden, st.k_pool, st.v_pool, st.block_table, st.seq_lens, assign, 2)
    kp, vp = st.k_pool, st.v_pool
    out = np.empty_like(st.hidden)
    for rows, s, a in _one_by_one(st, assign):
        r = oracle.layer_forward(SHAPE, w, s.hidden, kp, vp, s.block_table, s.seq_lens, a, 2)
        out[rows], kp, vp = r["out"], r["k_pool"], r["v_pool"]
    assert np.array_equal(out, chunk["out"])
    assert np.array_equal(kp, chunk["k_pool"]) and np.array_equal(vp, chunk["v_pool"])
    # and causality has teeth: a chunk row's output changes when an EARLIER chunk token's input changes, not a later one's
    h2 = st.hidden.copy()
    h2[6 + 20] ^= 0x0040
    again = oracle.layer_forward(SHAPE, w, h2, st.k_pool, st.v_pool, st.block_table, st.seq_lens, assign, 2)["out"]
    assert np.array_equal(again[:6 + 20], chunk["out"][:6 + 20])              # rows before token 20: untouched
    assert all(not np.array_equal(again[6 + t], chunk["out"][6 + t]) for t in range(20, N_CHUNK))


@pytest.mark.gpu
@pytest.mark.parametrize("cached,n_chunk", CASES)
def test_gpu_chunk_step_matches_oracle_and_the_one_by_one_cache_bitwise(cached, n_chunk):
    import torch
    from paper_2607_04181_b200 import binding as B
    from paper_2607_04181_b200.harness import DeviceStep, Session
    from tests.test_gpu_parity import within

    w = I.make_weights(SHAPE, 1401)
    st, assign = _scenario(cached, n_chunk)
    ref = oracle.layer_forward(SHAPE, w, st.hidden, st.k_pool, st.v_pool, st.block_table, st.seq_lens, assign, 2, taps=True)
    batch = st.hidden.shape[0]
    with Session(SHAPE, w, max_batch=batch) as S:
        S.scale(2)
        step = DeviceStep(st, assign)
        S.forward(step)
        torch.cuda.synchronize()
        assert B.cc_poll_device_error(S.ctx) == 0
        out, (kp, vp) = step.out_bits(), step.pools_bits()
        assert within(I.bf16_bits_to_f32(out), I.bf16_bits_to_f32(ref["out"]), "chunk step output") < 1e-2
        assert within(S.tap(B.CC_TAP_O, batch), ref["taps"]["o"], "chunk step attention output") < 1e-2
        # the same tokens one by one on the GPU: the cache must come out bit for bit the same (per-row GEMM results do not
        # depend on the batch), the outputs within the tolerance of the same oracle values
        step.reset(st)
        seq_out = np.empty_like(out)
        for rows, s, a in _one_by_one(st, assign):
            n = len(rows)
            step.hidden[:n].copy_(torch.from_numpy(s.hidden.view(np.int16)).cuda().view(torch.bfloat16))
            step.block_table[:n].copy_(torch.from_numpy(s.block_table))
            step.seq_lens.zero_()
            step.seq_lens[:n].copy_(torch.from_numpy(s.seq_lens))
            step.assign[:n].copy_(torch.from_numpy(a))
            S.forward(step)
            torch.cuda.synchronize()
            seq_out[rows] = step.out_bits()[:n]
        kp1, vp1 = step.pools_bits()
        assert np.array_equal(kp1, kp) and np.array_equal(vp1, vp)
        assert within(I.bf16_bits_to_f32(seq_out), I.bf16_bits_to_f32(ref["out"]), "one-by-one output") < 1e-2
        assert B.cc_poll_device_error(S.ctx) == 0


def _random_mixed_step(seed):
    """1-3 requests with a prompt chunk each (random cached length and chunk length), 0-9 decode rows, a random small
    layer shape and replica count; the rows of a request name one replica but need not be adjacent or in position
    order; every slot a chunk will write holds NaN beforehand."""
    rng = np.random.default_rng(seed)
    dh, hkv, g = int(rng.choice([64, 128])), int(rng.choice([1, 2, 4, 8])), int(rng.integers(1, 5))
    shape = I.LayerShape(f"mix{seed}", 64 * int(rng.integers(2, 9)), hkv * g, hkv, dh, 8 * int(rng.integers(8, 120)), 1e-5, 10000.0, 8, 0, 900)
    R, n_req, n_dec = int(rng.integers(1, 5)), int(rng.integers(1, 4)), int(rng.integers(0, 10))
    cached, chunk, dec_ctx = rng.integers(0, 700, n_req), rng.integers(1, 70, n_req), rng.integers(0, 800, n_dec)
    base = I.make_step_inputs(shape, 5000 + seed, 6000 + seed, batch=n_req + n_dec, n_pages=(n_req + n_dec) * shape.max_blocks,
                              contexts=np.concatenate([cached + chunk - 1, dec_ctx]).astype(np.int32))
    k_pool, v_pool = base.k_pool.copy(), base.v_pool.copy()
    bt, seq, ra = [], [], []
    for r in range(n_req):
        rep = int(rng.integers(0, R))
        for t in range(int(cached[r]), int(cached[r] + chunk[r])):
            bt.append(base.block_table[r]); seq.append(t + 1); ra.append(rep)
            pg = int(base.block_table[r, t // shape.page])
            k_pool[pg, :, t % shape.page, :] = 0x7FC0
            v_pool[pg, :, t % shape.page, :] = 0x7FC0
    for j in range(n_dec):
        bt.append(base.block_table[n_req + j]); seq.append(int(dec_ctx[j]) + 1); ra.append(int(rng.integers(0, R)))
    order = rng.permutation(len(seq)) if seed % 2 else np.arange(len(seq))
    hidden = I._normal_bf16(rng, (len(seq), shape.hidden), 0.0, 1.0)
    st = I.StepInputs(hidden, k_pool, v_pool, np.stack(bt)[order].astype(np.int32), np.array(seq, np.int32)[order], base.n_pages)
    return shape, R, st, np.array(ra, np.int32)[order]


@pytest.mark.gpu
@pytest.mark.parametrize("seed", range(8))
def test_gpu_random_mixed_prefill_and_decode_steps(seed):
    import torch
    from paper_2607_04181_b200 import binding as B
    from paper_2607_04181_b200.harness import DeviceStep, Session
    from tests.test_gpu_parity import within

    shape, R, st, ra = _random_mixed_step(seed)
    w = I.make_weights(shape, 7000 + seed)
    ref = oracle.layer_forward(shape, w, st.hidden, st.k_pool, st.v_pool, st.block_table, st.seq_lens, ra, R, taps=True)
    batch = st.hidden.shape[0]
    with Session(shape, w, max_batch=batch) as S:
        if R > 1:
            S.scale(R)
        step = DeviceStep(st, ra)
        first = None
        for rep in range(3):
            step.reset(st)
            S.forward(step)
            torch.cuda.synchronize()
            assert B.cc_poll_device_error(S.ctx) == 0
            out, (kp, vp) = step.out_bits(), step.pools_bits()
            assert within(I.bf16_bits_to_f32(out), I.bf16_bits_to_f32(ref["out"]), "mixed step output") < 1e-2
            assert within(S.tap(B.CC_TAP_O, batch), ref["taps"]["o"], "mixed step attention output") < 1e-2
            written = ~np.isnan(I.bf16_bits_to_f32(ref["k_pool"]))            # NaN left = slots nobody wrote (none attended)
            assert within(I.bf16_bits_to_f32(kp)[written], I.bf16_bits_to_f32(ref["k_pool"])[written], "K cache") < 1e-2
            assert within(I.bf16_bits_to_f32(vp)[written], I.bf16_bits_to_f32(ref["v_pool"])[written], "V cache") < 1e-2
            if first is None:
                first = (out, kp, vp)
            else:                                                             # and the same bits every time
                assert np.array_equal(out, first[0]) and np.array_equal(kp, first[1]) and np.array_equal(vp, first[2])
