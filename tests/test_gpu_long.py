"""GPU parity at the sizes the other configs' bench lines reach: contexts up to the
8 192-token cap of BASELINE.json configs[2] in a batch small enough that the attention kernel cuts the long row
into far more than 32 pieces (the last-finisher merge then walks the pieces in strides, cc_attention.cu), RoPE
table rows up to position 8 192, 1 and 2 kv heads (several pages per TMA stage, inter-warp merge) with many
pieces, and replica groups of 128 and 256 rows at hidden 4096 / 5120 (the three-stage ring and the single
TMEM buffer of cc_gemm.cu).  Every stage tap, the output and the appended K/V against the oracle, with
max(rel) < 1e-2 on top of the per-element tolerance (the small-RMS taps would otherwise pass with 10 % error)."""
import numpy as np
import pytest

from paper_2607_04181_b200 import inputs as I
from tests.test_gpu_parity import check_against_oracle, check_grouping, run_case

pytestmark = [pytest.mark.gpu, pytest.mark.usefixtures("operand_format")]   # both GEMM operand formats

LONG = 8192                                                        # cached tokens of the long row (seq_len 8193)


def _long_case(shape, batch, R, assign, ctx, seeds):
    st, ref, out, kp, vp, gtaps, grouping, assign = run_case(shape, batch, R, assign=assign, contexts=ctx, seeds=seeds)
    rel = check_against_oracle(shape, st, ref, out, kp, vp, gtaps, assign, R)
    check_grouping(grouping, assign, st.seq_lens, R)
    print(shape.name, "normalised rms error per stage:", {k: round(v, 5) for k, v in rel.items()})
    assert max(rel.values()) < 1e-2
    return st, out, kp, vp


def test_one_8192_token_row_among_short_rows_cfg2_layer():
    """(a) 513 pages of one row + 6 pages of three 16-token rows over 148 CTAs: the long row is cut into > 100
    pieces; its position is 8 192 (the last RoPE table row of configs[2])."""
    shape = I.LayerShape("long8k", 4096, 32, 8, 128, 14336, 1e-5, 500000.0, 4, 16, LONG)
    ctx = np.array([16, LONG, 16, 16], np.int32)
    assign = np.array([0, 1, 1, 0], np.int32)
    st, out, kp, vp = _long_case(shape, 4, 2, assign, ctx, (1002, 2402, 3402))
    assert int(st.seq_lens.max()) == LONG + 1 and st.block_table.shape[1] == 513
    # one replica gives the same bits
    _, _, out1, kp1, vp1, _, _, _ = run_case(shape, 4, 1, assign=np.zeros(4, np.int32), contexts=ctx, seeds=(1002, 2402, 3402), taps=False)
    assert np.array_equal(out1, out) and np.array_equal(kp1, kp) and np.array_equal(vp1, vp)


@pytest.mark.parametrize("hkv,g", [(1, 8), (2, 4)])
def test_long_row_with_few_kv_heads(hkv, g):
    """(b) Hkv 1 / 2: 8 / 4 pages per TMA stage, the warps of one kv head are merged through shared memory at the
    end of every piece, and the long row still has > 32 pieces."""
    shape = I.LayerShape(f"long_hkv{hkv}", 512, hkv * g, hkv, 128, 1024, 1e-5, 500000.0, 5, 16, LONG)
    ctx = np.array([40, 3, LONG, 17, 600], np.int32)
    assign = np.array([0, 0, 1, 2, 1], np.int32)
    _long_case(shape, 5, 3, assign, ctx, (1410 + hkv, 2410 + hkv, 3410 + hkv))


def test_dh64_long_row():
    shape = I.LayerShape("long_dh64", 256, 4, 2, 64, 688, 1e-6, 10000.0, 3, 16, 5000)
    ctx = np.array([5000, 1, 31], np.int32)
    _long_case(shape, 3, 1, np.zeros(3, np.int32), ctx, (1420, 2420, 3420))


@pytest.mark.parametrize("rows", [128, 256])
def test_cfg2_layer_with_one_group_of_128_and_256_rows(rows):
    """(c) configs[2]'s batch (128) and the library's maximum (256) in ONE replica group at hidden 4096: UMMA N =
    128 / 256, three ring stages, one TMEM buffer at 256.  Short contexts keep the oracle's step in seconds; all
    rows are compared."""
    shape = I.LayerShape(f"cfg2_b{rows}", 4096, 32, 8, 128, 14336, 1e-5, 500000.0, rows, 1, 96)
    assign = np.zeros(rows, np.int32)
    assign[-3:] = 1                                               # a second, tiny group beside the wide one
    _long_case(shape, rows, 2, assign, None, (1002, 2430 + rows, 3430 + rows))


def test_cfg4_layer_with_256_rows_in_one_group():
    """(d) the 14B-class layer of configs[3] (hidden 5120, FFN 17408, GQA 5) with 256 rows in one group."""
    shape = I.LayerShape("cfg4_b256", 5120, 40, 8, 128, 17408, 1e-5, 500000.0, 256, 1, 64)
    _long_case(shape, 256, 1, np.zeros(256, np.int32), None, (1004, 2440, 3440))
