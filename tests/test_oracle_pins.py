"""Pins for the CPU oracle (-m "not gpu").  Each test ties one oracle function to something other
than itself: a pure-Python brute force, a closed form, an invariant, a library routine, or a value
the paper prints (tests/golden/paper_values.txt).  SURVEY.md 8(c) "What pins each part"."""
import math
import os

import numpy as np
import pytest
import torch

import oracle
from oracle import hostsim
from paper_2607_04181_b200 import inputs as I
from tests import ref_torch

GOLD = os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")


def golden():
    out = {}
    for line in open(GOLD):
        line = line.split("#")[0].strip()
        if "=" in line:
            k, v = line.split("=", 1)
            out[k.strip()] = v.strip()
    return out


def bf(x):
    return I.f32_to_bf16_bits(np.asarray(x, dtype=np.float32))


def unbf(u):
    return I.bf16_bits_to_f32(u)


# ------------------------------------------------------------------ bf16 conversion
def test_bf16_roundtrip_and_rne():
    # exactly representable values survive; ties go to even; matches torch's conversion
    assert oracle.bf16_to_f32(oracle.f32_to_bf16(1.0)) == 1.0
    assert oracle.f32_to_bf16(1.0 + 2 ** -8) == oracle.f32_to_bf16(1.0)          # tie -> even (1.0)
    assert oracle.f32_to_bf16(1.0 + 3 * 2 ** -8) == oracle.f32_to_bf16(1.0 + 2 ** -6)  # tie -> even (up)
    rng = np.random.default_rng(0)
    v = (rng.standard_normal(4096) * 10 ** rng.uniform(-20, 20, 4096)).astype(np.float32)
    t = torch.from_numpy(v).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    mine = np.array([oracle.f32_to_bf16(float(z)) for z in v], dtype=np.uint16)
    assert np.array_equal(mine, t)
    assert np.array_equal(I.f32_to_bf16_bits(v), t)                               # the input generator too
    assert np.array_equal(unbf(t), np.array([oracle.bf16_to_f32(int(z)) for z in t], dtype=np.float32))


# ------------------------------------------------------------------ GEMM (a2, a6, a8, a9)
def test_matmul_vs_python_triple_loop_exact():
    rng = np.random.default_rng(1)
    for (M, K, N) in [(1, 1, 1), (3, 5, 2), (8, 16, 8), (2, 7, 5)]:
        X = rng.standard_normal((M, K)).astype(np.float32)
        W = bf(rng.standard_normal((N, K)))
        Wf = unbf(W)
        want = np.empty((M, N), dtype=np.float32)
        for m in range(M):
            for n in range(N):
                acc = 0.0                                   # python float = fp64
                for k in range(K):
                    acc += float(X[m, k]) * float(Wf[n, k])
                want[m, n] = np.float32(acc)
        got = oracle.matmul_wt(X, W)
        assert np.array_equal(got, want)


def test_matmul_identity_onehot_and_transpose_sensitivity():
    rng = np.random.default_rng(2)
    X = rng.standard_normal((3, 6)).astype(np.float32)
    assert np.array_equal(oracle.matmul_wt(X, bf(np.eye(6))), X)
    # one-hot row n selects column k: Y[:, n] = X[:, sel[n]]  (fails if W were read [in][out])
    sel = [4, 0, 5, 2]
    W = np.zeros((4, 6), dtype=np.float32)
    for n, k in enumerate(sel):
        W[n, k] = 1.0
    assert np.array_equal(oracle.matmul_wt(X, bf(W)), X[:, sel])


def test_matmul_vs_torch_library_cfg1_shapes():
    rng = np.random.default_rng(3)
    X = rng.standard_normal((4, 256)).astype(np.float32)
    W = bf(rng.standard_normal((688, 256)) * 0.02)
    want = (torch.from_numpy(X).double() @ torch.from_numpy(unbf(W)).double().T).numpy()
    got = oracle.matmul_wt(X, W)
    assert np.max(np.abs(got - want)) <= 1e-6 * np.max(np.abs(want)) + 1e-7


# ------------------------------------------------------------------ RMSNorm (a1, a7)
def test_rmsnorm_closed_forms():
    d, eps = 64, 1e-6
    g = bf(1.0 + 0.25 * np.arange(d) / d)
    gf = unbf(g).astype(np.float64)
    for c in (3.0, -0.5, 1e-3):                             # constant row: g*c/sqrt(c^2+eps); 1e-3 exposes eps
        x = oracle.rmsnorm(np.full((1, d), c, np.float32), g, eps)[0]
        want = gf * np.float64(np.float32(c)) / math.sqrt(float(np.float32(c)) ** 2 + eps)
        assert np.allclose(x, want, rtol=2e-7, atol=0)
    z = oracle.rmsnorm(np.zeros((2, d), np.float32), g, eps)
    assert np.all(z == 0) and not np.isnan(z).any()
    rng = np.random.default_rng(4)
    h = rng.standard_normal((5, d)).astype(np.float32)
    x = oracle.rmsnorm(h, g, eps).astype(np.float64)
    ms = (h.astype(np.float64) ** 2).mean(-1)
    assert np.allclose(((x / gf) ** 2).sum(-1), d * ms / (ms + eps), rtol=1e-6)   # invariant
    # eps really is inside the sqrt and added to the MEAN (not the sum)
    tiny = np.full((1, d), 1e-3, np.float32)
    assert abs(oracle.rmsnorm(tiny, bf(np.ones(d)), 1e-6)[0, 0] - 1e-3 / math.sqrt(1e-6 + 1e-6)) < 1e-6


# ------------------------------------------------------------------ RoPE (a3)
def test_rope_closed_forms():
    Dh, H, base = 64, 3, 10000.0
    rng = np.random.default_rng(5)
    u = rng.standard_normal((H, Dh)).astype(np.float32)
    assert np.array_equal(oracle.rope(u, H, Dh, 0, base), u)                       # p = 0 identity
    r = oracle.rope(u, H, Dh, 7, base)
    half = Dh // 2
    n0 = u[:, :half] ** 2 + u[:, half:] ** 2
    n1 = r[:, :half] ** 2 + r[:, half:] ** 2
    assert np.allclose(n0, n1, rtol=1e-5)                                          # pairwise norm kept
    a, b = 5, 11                                                                   # group law
    assert np.allclose(oracle.rope(oracle.rope(u, H, Dh, a, base), H, Dh, b, base),
                       oracle.rope(u, H, Dh, a + b, base), atol=2e-6)
    # hand value at p = 1: pair i=0 rotates by exactly 1 rad, pair i by base^(-2i/Dh)
    x = np.zeros((1, Dh), np.float32)
    x[0, 0], x[0, half] = 2.0, 3.0
    x[0, 5], x[0, half + 5] = 1.0, 0.0
    y = oracle.rope(x, 1, Dh, 1, base)[0]
    assert abs(y[0] - (2 * math.cos(1) - 3 * math.sin(1))) < 1e-6
    assert abs(y[half] - (3 * math.cos(1) + 2 * math.sin(1))) < 1e-6
    th5 = base ** (-2 * 5 / Dh)
    assert abs(y[5] - math.cos(th5)) < 1e-6 and abs(y[half + 5] - math.sin(th5)) < 1e-6


def test_rope_relative_position_property():
    Dh, base = 64, 10000.0
    rng = np.random.default_rng(6)
    q = rng.standard_normal((1, Dh)).astype(np.float32)
    k = rng.standard_normal((1, Dh)).astype(np.float32)
    dots = [float(oracle.rope(q, 1, Dh, m, base)[0].astype(np.float64) @ oracle.rope(k, 1, Dh, n, base)[0].astype(np.float64))
            for (m, n) in [(9, 4), (25, 20), (105, 100)]]
    assert max(dots) - min(dots) < 1e-4


# ------------------------------------------------------------------ attention (a5)
def _pool(rng, n_pages, Hkv, Dh, page=16):
    return bf(rng.standard_normal((n_pages, Hkv, page, Dh)))


def test_attention_softmax_rows_sum_to_one_and_brute_force():
    rng = np.random.default_rng(7)
    Hq, Hkv, Dh, page, s = 4, 2, 8, 16, 37
    kp, vp = _pool(rng, 6, Hkv, Dh), _pool(rng, 6, Hkv, Dh)
    bt = np.array([4, 1, 5, -1], np.int32)
    q = rng.standard_normal((Hq, Dh)).astype(np.float32)
    o, w = oracle.attention_decode(q, kp, vp, bt, s, Hq, Hkv, Dh, page, return_weights=True)
    assert np.allclose(w.sum(-1), 1.0, atol=1e-6)
    kf, vf = unbf(kp).astype(np.float64), unbf(vp).astype(np.float64)
    for hq in range(Hq):                                     # brute force, pure python
        hk = hq // (Hq // Hkv)
        sc = [sum(float(q[hq, i]) * kf[bt[t // page], hk, t % page, i] for i in range(Dh)) / math.sqrt(Dh)
              for t in range(s)]
        mx = max(sc)
        e = [math.exp(z - mx) for z in sc]
        tot = sum(e)
        for i in range(Dh):
            want = sum(e[t] / tot * vf[bt[t // page], hk, t % page, i] for t in range(s))
            assert abs(o[hq, i] - want) < 1e-5


def test_attention_context_of_one_returns_v_and_gqa_map():
    rng = np.random.default_rng(8)
    Hq, Hkv, Dh, page = 6, 2, 8, 16
    kp = _pool(rng, 3, Hkv, Dh)
    vp = _pool(rng, 3, Hkv, Dh)
    bt = np.array([2], np.int32)
    q = rng.standard_normal((Hq, Dh)).astype(np.float32)
    o = oracle.attention_decode(q, kp, vp, bt, 1, Hq, Hkv, Dh, page)
    for hq in range(Hq):                                     # s = 1  =>  o = V[token 0] of head hq/G
        assert np.array_equal(o[hq], unbf(vp)[2, hq // 3, 0])
    # V constant per kv head = head index reveals hq -> hq / G for any s
    vconst = np.empty((3, Hkv, page, Dh), np.float32)
    for hk in range(Hkv):
        vconst[:, hk] = hk + 1
    o = oracle.attention_decode(q, kp, bf(vconst), np.array([0, 1, 2], np.int32), 40, Hq, Hkv, Dh, page)
    for hq in range(Hq):
        assert np.allclose(o[hq], hq // 3 + 1, atol=1e-6)


def test_attention_equal_k_gives_mean_dominant_k_selects():
    rng = np.random.default_rng(9)
    Hq, Hkv, Dh, page, s = 2, 1, 8, 16, 20
    krow = rng.standard_normal(Dh).astype(np.float32)
    kp = bf(np.broadcast_to(krow, (2, Hkv, page, Dh)).copy())
    vp = _pool(rng, 2, Hkv, Dh)
    bt = np.array([1, 0], np.int32)
    q = rng.standard_normal((Hq, Dh)).astype(np.float32)
    o = oracle.attention_decode(q, kp, vp, bt, s, Hq, Hkv, Dh, page)
    vf = unbf(vp).astype(np.float64)
    toks = np.stack([vf[bt[t // page], 0, t % page] for t in range(s)])
    assert np.allclose(o[0], toks.mean(0), atol=1e-6) and np.allclose(o[1], toks.mean(0), atol=1e-6)
    # one key aligned with q and huge: weight -> 1 on that token (t = 17 lives in page bt[1], slot 1)
    kz = np.zeros((2, Hkv, page, Dh), np.float32)
    kz[bt[1], 0, 1] = 100.0 * q[0] / np.linalg.norm(q[0])
    o = oracle.attention_decode(np.stack([q[0], q[0]]), bf(kz), vp, bt, s, Hq, Hkv, Dh, page)
    assert np.allclose(o[0], vf[bt[1], 0, 1], atol=1e-5)


def test_attention_page_reshuffle_is_bitwise_invariant():
    rng = np.random.default_rng(10)
    Hq, Hkv, Dh, page = 4, 2, 16, 16
    kp, vp = _pool(rng, 8, Hkv, Dh), _pool(rng, 8, Hkv, Dh)
    q = rng.standard_normal((Hq, Dh)).astype(np.float32)
    bt = np.array([3, 6, 0, 5], np.int32)
    perm = rng.permutation(8)                                # physical page p moves to perm[p]
    kp2, vp2 = np.empty_like(kp), np.empty_like(vp)
    kp2[perm], vp2[perm] = kp, vp
    for s in (15, 16, 17, 33, 64):                           # page-boundary cases
        a = oracle.attention_decode(q, kp, vp, bt, s, Hq, Hkv, Dh, page)
        b = oracle.attention_decode(q, kp2, vp2, perm[bt].astype(np.int32), s, Hq, Hkv, Dh, page)
        assert np.array_equal(a, b)


def test_attention_rejects_padding_page_inside_context():
    rng = np.random.default_rng(11)
    kp, vp = _pool(rng, 2, 1, 8), _pool(rng, 2, 1, 8)
    with pytest.raises(RuntimeError):
        oracle.attention_decode(np.ones((1, 8), np.float32), kp, vp, np.array([0, -1], np.int32), 20, 1, 1, 8, 16)


# ------------------------------------------------------------------ SwiGLU (a8)
def test_silu_hand_values():
    assert oracle.silu(0.0) == 0.0
    assert abs(oracle.silu(1.0) - 1.0 / (1.0 + math.exp(-1.0))) < 1e-7
    assert abs(oracle.silu(-1.0) + 1.0 / (1.0 + math.exp(1.0))) < 1e-7
    assert abs(oracle.silu(30.0) - 30.0) < 1e-5
    assert abs(oracle.silu(-30.0)) < 1e-10
    assert abs(oracle.silu(2.5) - float(torch.nn.functional.silu(torch.tensor(2.5, dtype=torch.float64)))) < 1e-6


# ------------------------------------------------------------------ whole layer on cfg1
@pytest.fixture(scope="module")
def cfg1():
    shape = I.CFG1
    w = I.make_weights(shape, 1001)
    st = I.make_step_inputs(shape, 2001, 3001)
    return shape, w, st


def test_layer_vs_independent_torch_restatement_cfg1(cfg1):
    shape, w, st = cfg1
    res = oracle.layer_forward(shape, w, st.hidden, st.k_pool, st.v_pool, st.block_table, st.seq_lens,
                               np.zeros(shape.batch, np.int32), 1, taps=True)
    out, taps, kp, vp = ref_torch.layer_step(shape, w, st.hidden, st.k_pool, st.v_pool, st.block_table, st.seq_lens)
    for name, ref in taps.items():
        got, ref = res["taps"][name].astype(np.float64), ref.numpy()
        scale = np.sqrt((ref ** 2).mean())
        assert np.max(np.abs(got - ref)) <= 2e-6 * max(scale, 1.0) + 2e-6 * np.max(np.abs(ref)), name
    assert np.array_equal(res["k_pool"], kp) and np.array_equal(res["v_pool"], vp)   # appended slots, bitwise
    want = torch.from_numpy(taps["out"].numpy()).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    mism = np.count_nonzero(res["out"] != want)
    assert mism <= 2                                          # fp32-vs-fp64 ties at a bf16 rounding boundary


def test_layer_only_touches_the_appended_kv_slots(cfg1):
    shape, w, st = cfg1
    res = oracle.layer_forward(shape, w, st.hidden, st.k_pool, st.v_pool, st.block_table, st.seq_lens,
                               np.zeros(shape.batch, np.int32), 1)
    changed = np.argwhere((res["k_pool"] != st.k_pool).any(axis=(1, 3)))   # [page, slot]
    want = sorted((int(st.block_table[b, (s - 1) // 16]), int((s - 1) % 16)) for b, s in enumerate(st.seq_lens))
    assert sorted(map(tuple, changed.tolist())) == want


def test_replicated_equals_unreplicated_bitwise(cfg1):
    shape, w, st = cfg1
    base = oracle.layer_forward(shape, w, st.hidden, st.k_pool, st.v_pool, st.block_table, st.seq_lens,
                                np.zeros(shape.batch, np.int32), 1)
    for R, assign in [(2, I.even_split(4, 2)), (4, I.even_split(4, 4)), (2, np.array([1, 0, 1, 1], np.int32)),
                      (3, np.array([2, 2, 0, 2], np.int32))]:          # incl. an empty group
        res = oracle.layer_forward(shape, w, st.hidden, st.k_pool, st.v_pool, st.block_table, st.seq_lens, assign, R)
        assert np.array_equal(res["out"], base["out"])
        assert np.array_equal(res["k_pool"], base["k_pool"]) and np.array_equal(res["v_pool"], base["v_pool"])


def test_uneven_split_15_rows_bitwise_and_row_permutation():
    g = golden()
    bs = int(g["split_example_bs"])
    parts = sorted(int(z) for z in g["split_example_parts"].split())
    shape = I.CFG1.with_batch(bs)
    w = I.make_weights(shape, 1001)
    st = I.make_step_inputs(shape, 2011, 3011)
    assign = I.even_split(bs, 2)
    assert sorted(np.bincount(assign).tolist()) == parts                # 15 -> 7 + 8
    assert hostsim.split_counts(bs, 2) == (max(parts), min(parts))      # ceil / floor
    assert hostsim.split_counts(1, int(g["p_max"])) == (1, 0)           # bs = 1: no speed-up
    base = oracle.layer_forward(shape, w, st.hidden, st.k_pool, st.v_pool, st.block_table, st.seq_lens,
                                np.zeros(bs, np.int32), 1)
    rep = oracle.layer_forward(shape, w, st.hidden, st.k_pool, st.v_pool, st.block_table, st.seq_lens, assign, 2)
    assert np.array_equal(base["out"], rep["out"])
    # permuting batch rows permutes outputs bitwise
    p = np.random.default_rng(12).permutation(bs)
    res = oracle.layer_forward(shape, w, st.hidden[p], st.k_pool, st.v_pool, st.block_table[p], st.seq_lens[p],
                               assign, 2)
    assert np.array_equal(res["out"], base["out"][p])


def test_padding_rows_pass_through(cfg1):
    shape, w, st = cfg1
    sl = st.seq_lens.copy()
    sl[1] = 0
    res = oracle.layer_forward(shape, w, st.hidden, st.k_pool, st.v_pool, st.block_table, sl,
                               np.zeros(shape.batch, np.int32), 1)
    base = oracle.layer_forward(shape, w, st.hidden, st.k_pool, st.v_pool, st.block_table, st.seq_lens,
                                np.zeros(shape.batch, np.int32), 1)
    assert np.array_equal(res["out"][1], st.hidden[1])
    assert np.array_equal(res["out"][[0, 2, 3]], base["out"][[0, 2, 3]])


def test_nan_poison_outside_context_is_never_read(cfg1):
    shape, w, _ = cfg1
    clean = I.make_step_inputs(shape, 2001, 3001)
    dirty = I.make_step_inputs(shape, 2001, 3001, poison_unused=True)
    assert np.isnan(unbf(dirty.k_pool)).any()
    a = oracle.layer_forward(shape, w, clean.hidden, clean.k_pool, clean.v_pool, clean.block_table, clean.seq_lens,
                             np.zeros(shape.batch, np.int32), 1)
    b = oracle.layer_forward(shape, w, dirty.hidden, dirty.k_pool, dirty.v_pool, dirty.block_table, dirty.seq_lens,
                             np.zeros(shape.batch, np.int32), 1)
    assert np.array_equal(a["out"], b["out"]) and not np.isnan(unbf(b["out"])).any()


# ------------------------------------------------------------------ integer structures (a0, a11, a12)
def test_group_rows_stable_partition():
    ra = np.array([1, 0, 1, 2, 0, 1, 0], np.int32)
    sl = np.array([5, 5, 0, 5, 5, 5, 5], np.int32)             # row 2 is a padding row
    perm, counts = oracle.group_rows(ra, sl, 4)
    assert perm.tolist() == [1, 4, 6, 0, 5, 3] and counts.tolist() == [3, 2, 1, 0]


def test_replica_copy_is_byte_exact():
    rng = np.random.default_rng(13)
    blob = rng.integers(0, 65536, 100003, dtype=np.uint16)
    assert np.array_equal(oracle.replica_copy(blob), blob)


def test_slot_alloc_sim_lowest_first_and_reuse():
    A = hostsim.SlotAllocSim()
    assert A.donate(0x10000, 10 * 4096)
    a = A.alloc(4096); b = A.alloc(4096); c = A.alloc(4096)
    assert (a, b, c) == (0x10000, 0x11000, 0x12000)
    assert A.free(b)
    assert A.alloc(4096) == b                                  # the freed middle slot is reused first
    assert A.reclaim(0x10000) == "busy"
    for x in (a, b, c):
        A.free(x)
    assert A.reclaim(0x10000) == "ok" and A.alloc(1) is None


# ------------------------------------------------------------------ byte / flop accounting vs Eq. 1-2
def test_param_count_matches_eq1_when_assumptions_hold():
    g = golden()
    assert g["params_per_layer"] == "12*d^2" and g["flops_per_layer"] == "24*bs*l*d^2"
    d = 384                                                    # Hkv = Hq and F = 8d/3  =>  exactly 12 d^2
    shp = I.LayerShape("eq1", d, 6, 6, 64, 8 * d // 3, 1e-6, 1e4, 1, 1, 1)
    assert shp.n_params == 12 * d * d
    assert 2 * shp.n_params * 5 == 24 * 5 * 1 * d * d          # 2 flops / param / token, bs = 5, l = 1
    assert I.layer_weight_bytes(I.CFG2) == 2 * (218_103_808 + 8192)      # 436.2 MB
    assert I.CFG2.max_blocks == 129
