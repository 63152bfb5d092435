"""GPU parity on the other layer shapes the configs name and on the kernel's corner shapes, each against
the oracle with stage taps (tests/test_gpu_parity.py): the 14B-class layer of configs[3], model B of
configs[4], every supported kv-head count (1, 2, 4, 8: the attention kernel stages 8 / Hkv pages per
TMA stage), GQA groups of 5, 6 and 8, head_dim 64 and 128, and the maximum batch of 256 rows over four
uneven replica groups including contexts of zero cached tokens."""
import numpy as np
import pytest

from paper_2607_04181_b200 import inputs as I
from tests.test_gpu_parity import check_against_oracle, check_grouping, run_case

pytestmark = [pytest.mark.gpu, pytest.mark.usefixtures("operand_format")]   # both GEMM operand formats

CASES = {
    # name: (shape, batch, replicas)
    "cfg4_layer": (I.LayerShape("cfg4s", 5120, 40, 8, 128, 17408, 1e-5, 500000.0, 8, 256, 700), 8, 2),   # configs[3]: contexts from 256 up
    "model_b": (I.LayerShape("modelBs", 1536, 12, 2, 128, 8960, 1e-6, 10000.0, 10, 30, 400), 10, 3),
    "hkv4_dh64": (I.LayerShape("hkv4", 512, 8, 4, 64, 1024, 1e-5, 10000.0, 9, 10, 150), 9, 2),
    "hkv1_g8": (I.LayerShape("hkv1", 256, 8, 1, 128, 512, 1e-5, 10000.0, 5, 20, 200), 5, 1),
    # nothing a multiple of 128: hidden 5 x 64, q width 5 x 64, FFN 200 (not a multiple of 64), odd GQA group
    "odd_sizes": (I.LayerShape("odd", 320, 5, 1, 64, 200, 1e-5, 10000.0, 6, 10, 90), 6, 2),
    "hkv8_g1": (I.LayerShape("hkv8", 1024, 8, 8, 128, 2048, 1e-5, 500000.0, 7, 100, 600), 7, 4),
}


@pytest.mark.parametrize("name", list(CASES))
def test_shape_parity(name):
    shape, batch, R = CASES[name]
    rng = np.random.default_rng(7)
    assign = rng.integers(0, R, batch).astype(np.int32)
    st, ref, out, kp, vp, gtaps, grouping, assign = run_case(shape, batch, R, assign=assign, seeds=(1201, 2201, 3201))
    rel = check_against_oracle(shape, st, ref, out, kp, vp, gtaps, assign, R)
    check_grouping(grouping, assign, st.seq_lens, R)
    print(name, "normalised rms error per stage:", {k: round(v, 5) for k, v in rel.items()})
    assert max(rel.values()) < 1e-2


def test_max_batch_256_rows_uneven_groups_and_empty_contexts():
    shape = I.LayerShape("wide", 256, 4, 2, 64, 688, 1e-6, 10000.0, 256, 0, 40)
    rng = np.random.default_rng(11)
    assign = rng.choice(4, size=256, p=[0.55, 0.05, 0.3, 0.1]).astype(np.int32)
    ctx = rng.integers(0, 41, 256).astype(np.int32)
    ctx[:5] = 0                                                    # seq_len 1: attention over the new token only
    st, ref, out, kp, vp, gtaps, grouping, assign = run_case(shape, 256, 4, assign=assign, contexts=ctx,
                                                             seeds=(1202, 2202, 3202))
    rel = check_against_oracle(shape, st, ref, out, kp, vp, gtaps, assign, 4)
    check_grouping(grouping, assign, st.seq_lens, 4)
    assert max(rel.values()) < 1e-2, rel


@pytest.mark.parametrize("seed", range(10))
def test_random_shapes_batches_and_assignments(seed):
    """Seeded random layers inside what cc_create_layer accepts (hidden a multiple of 64, FFN of 8, 1/2/4/8 kv
    heads, GQA groups 1..8, head_dim 64/128), random batch, contexts, replica counts and assignments (some replicas
    left empty, some rows padding): every stage tap, the output and the appended KV against the oracle."""
    rng = np.random.default_rng(9000 + seed)
    dh = int(rng.choice([64, 128]))
    hkv = int(rng.choice([1, 2, 4, 8]))
    g = int(rng.integers(1, 9))
    hidden = 64 * int(rng.integers(2, 17))
    ffn = 8 * int(rng.integers(8, 260))
    batch = int(rng.integers(1, 49))
    R = int(rng.integers(1, 5))
    lo = int(rng.integers(0, 30))
    hi = lo + int(rng.integers(1, 400))
    shape = I.LayerShape(f"rnd{seed}", hidden, hkv * g, hkv, dh, ffn, 1e-5, float(rng.choice([10000.0, 500000.0])), batch, lo, hi)
    assign = rng.integers(0, R, batch).astype(np.int32)
    if R > 1 and seed % 2:
        assign[assign == R - 1] = 0                                   # an active replica that serves no row
    seq = None
    if batch > 3 and seed % 3 == 0:
        ctx = I.draw_contexts(shape, 3300 + seed, batch)
        seq = (ctx + 1).astype(np.int32)
        seq[rng.integers(0, batch, 2)] = 0                            # padding rows
    st, ref, out, kp, vp, gtaps, grouping, assign = run_case(shape, batch, R, assign=assign, seeds=(1300 + seed, 2300 + seed, 3300 + seed),
                                                             seq_override=seq)
    rel = check_against_oracle(shape, st, ref, out, kp, vp, gtaps, assign, R)
    check_grouping(grouping, assign, st.seq_lens, R)
    print(shape, "R", R, {k: round(v, 5) for k, v in rel.items()})
    assert max(rel.values()) < 1e-2, rel
    if R > 1:
        # the same batch through one replica gives the same bits (outputs and appended KV)
        _, _, out1, kp1, vp1, _, _, _ = run_case(shape, batch, 1, assign=np.zeros(batch, np.int32),
                                                 seeds=(1300 + seed, 2300 + seed, 3300 + seed), seq_override=seq, taps=False)
        assert np.array_equal(out1, out) and np.array_equal(kp1, kp) and np.array_equal(vp1, vp)
