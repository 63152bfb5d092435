"""The GEMM operand format is a per-layer choice made when the weights are packed (include/cocoscale.h,
cc_ctx_set_operand_format): fp16 weight images + one fp16 activation plane, or bf16 images + two bf16 planes for
weights outside the fp16 range.  Both must meet the same tolerance against the oracle; AUTO must pick fp16 for
ordinary weights and fall back for a layer whose weights do not fit."""
import numpy as np
import pytest
import torch

import oracle
from paper_2607_04181_b200 import inputs as I
from tests.test_gpu_parity import check_against_oracle

pytestmark = pytest.mark.gpu


def _run(shape, w, st, assign, R, fmt):
    from paper_2607_04181_b200 import binding as B
    from paper_2607_04181_b200.harness import DeviceStep, Session

    with Session(shape, w, max_batch=shape.batch, operand_format=fmt) as S:
        got = B.cc_layer_operand_format(S.layer)
        if R > 1:
            S.scale(R)
        step = DeviceStep(st, assign)
        S.forward(step)
        torch.cuda.synchronize()
        assert B.cc_poll_device_error(S.ctx) == 0
        taps = {n: S.tap(t, shape.batch) for n, t in (("x", B.CC_TAP_X), ("q", B.CC_TAP_Q), ("o", B.CC_TAP_O), ("h1", B.CC_TAP_H1),
                                                      ("y", B.CC_TAP_Y), ("a", B.CC_TAP_A))}
        return got, step.out_bits(), step.pools_bits(), taps


def test_auto_picks_fp16_and_falls_back_for_weights_outside_its_range():
    from paper_2607_04181_b200 import binding as B

    shape = I.CFG1
    w = I.make_weights(shape, 1001)
    st = I.make_step_inputs(shape, 2001, 3001)
    assign = I.even_split(shape.batch, 2)
    fmt, out, (kp, vp), taps = _run(shape, w, st, assign, 2, B.CC_OPERAND_AUTO)
    assert fmt == B.CC_OPERAND_F16
    ref = oracle.layer_forward(shape, w, st.hidden, st.k_pool, st.v_pool, st.block_table, st.seq_lens, assign, 2, taps=True)
    check_against_oracle(shape, st, ref, out, kp, vp, taps, assign, 2)

    # one weight of 2^17 (bf16-exact, above fp16's 65504): the layer must come up in bf16 x 2 and still match the oracle
    big = {k: v.copy() for k, v in w.items()}
    big["wup"][3, 5] = I.f32_to_bf16_bits(np.array([131072.0], np.float32))[0]
    fmt, out, (kp, vp), taps = _run(shape, big, st, assign, 2, B.CC_OPERAND_AUTO)
    assert fmt == B.CC_OPERAND_BF16X2
    ref = oracle.layer_forward(shape, big, st.hidden, st.k_pool, st.v_pool, st.block_table, st.seq_lens, assign, 2, taps=True)
    check_against_oracle(shape, st, ref, out, kp, vp, taps, assign, 2)
    with pytest.raises(B.CcError) as e:
        _run(shape, big, st, assign, 2, B.CC_OPERAND_F16)
    assert e.value.status == B.CC_ERR_INVALID


def test_tiny_weights_round_to_the_fp16_subnormal_grid_and_stay_inside_the_tolerance():
    # weights below 2^-17 are not exact in fp16 (absolute error <= 2^-25 each): a whole matrix of them still
    # has to meet the tolerance, and the format must not fall back for them
    from paper_2607_04181_b200 import binding as B

    shape = I.CFG1
    w = I.make_weights(shape, 1001)
    rng = np.random.default_rng(5)
    tiny = (rng.standard_normal(w["wo"].shape) * 3e-6).astype(np.float32)
    w["wo"] = I.f32_to_bf16_bits(tiny)
    st = I.make_step_inputs(shape, 2001, 3001)
    assign = np.zeros(shape.batch, np.int32)
    fmt, out, (kp, vp), taps = _run(shape, w, st, assign, 1, B.CC_OPERAND_AUTO)
    assert fmt == B.CC_OPERAND_F16
    ref = oracle.layer_forward(shape, w, st.hidden, st.k_pool, st.v_pool, st.block_table, st.seq_lens, assign, 1, taps=True)
    check_against_oracle(shape, st, ref, out, kp, vp, taps, assign, 1)
    # the O projection's contribution h1 - h is ~1e-5 here; compare it directly, far below the absolute tolerance
    h = I.bf16_bits_to_f32(st.hidden)
    d_gpu, d_ref = taps["h1"] - h, ref["taps"]["h1"] - h
    assert np.abs(d_gpu - d_ref).max() <= 2e-2 * np.abs(d_ref).max() + 1e-7


def test_operand_saturates_instead_of_overflowing_fp16():
    # hidden of 3e4 per element: h1 * g2 would pass 65504 for gains above 2; the O epilogue stores y' scaled by the input row's 1/rms
    from paper_2607_04181_b200 import binding as B

    shape = I.CFG1
    w = I.make_weights(shape, 1001)
    st = I.make_step_inputs(shape, 2001, 3001)
    st.hidden[:] = I.f32_to_bf16_bits((I.bf16_bits_to_f32(st.hidden) * 3.0e4).astype(np.float32))
    assign = np.zeros(shape.batch, np.int32)
    fmt, out, (kp, vp), taps = _run(shape, w, st, assign, 1, B.CC_OPERAND_F16)
    ref = oracle.layer_forward(shape, w, st.hidden, st.k_pool, st.v_pool, st.block_table, st.seq_lens, assign, 1, taps=True)
    assert np.isfinite(I.bf16_bits_to_f32(out)).all()
    got, want = I.bf16_bits_to_f32(out).astype(np.float64), I.bf16_bits_to_f32(ref["out"]).astype(np.float64)
    assert (np.abs(got - want) <= 1e-2 + 2e-2 * np.abs(want)).all()
    for name in ("y", "a"):
        g, r = taps[name].astype(np.float64), ref["taps"][name].astype(np.float64)
        assert (np.abs(g - r) <= 1e-2 + 2e-2 * np.abs(r)).all(), name
