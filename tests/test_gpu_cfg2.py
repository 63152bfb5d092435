"""GPU parity at BASELINE.json's full size (configs[1], the workload bench.py times): the
Llama-3-8B-shaped layer, decode batch 64, contexts U{512..2048}, shuffled 16-token pages.  The
oracle computes the whole step (about 20 s on 8 cores), so every output element, every appended
K/V value and every stage tap is compared, and the outputs must be bit-identical for 1, 2 and 4
replicas -- in the launch configuration (CUDA graph replay) that bench.py times."""
import numpy as np
import pytest
import torch

import oracle
from paper_2607_04181_b200 import inputs as I
from tests.test_gpu_parity import check_against_oracle, check_grouping

pytestmark = [pytest.mark.gpu, pytest.mark.usefixtures("operand_format")]   # both GEMM operand formats


@pytest.fixture(scope="module")
def cfg2():
    shape = I.CFG2
    w = I.make_weights(shape, 1002)
    st = I.make_step_inputs(shape, 2002, 3002)
    ref = oracle.layer_forward(shape, w, st.hidden, st.k_pool, st.v_pool, st.block_table, st.seq_lens,
                               np.zeros(shape.batch, np.int32), 1, taps=True)
    return shape, w, st, ref


def test_cfg2_full_parity_and_bit_identity_across_replicas(cfg2):
    from paper_2607_04181_b200 import binding as B
    from paper_2607_04181_b200.harness import DeviceStep, Session

    shape, w, st, ref = cfg2
    batch = shape.batch
    with Session(shape, w, max_batch=batch) as S:
        step = DeviceStep(st, np.zeros(batch, np.int32))
        S.forward(step)                                            # warm-up (also first-touch of the workspace)
        torch.cuda.synchronize()
        step.reset(st)
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):
            S.forward(step, torch.cuda.current_stream())
        results = {}
        for R in (1, 2, 4):
            if R > 1:
                S.scale(R)
            assign = I.even_split(batch, R)
            step.reset(st)
            step.set_assign(assign)
            graph.replay()
            torch.cuda.synchronize()
            assert B.cc_poll_device_error(S.ctx) == 0
            out = step.out_bits()
            kp, vp = step.pools_bits()
            results[R] = (out, kp, vp)
            if R == 1:
                gtaps = {n: S.tap(t, batch) for n, t in (("x", B.CC_TAP_X), ("q", B.CC_TAP_Q), ("o", B.CC_TAP_O),
                                                         ("h1", B.CC_TAP_H1), ("y", B.CC_TAP_Y), ("a", B.CC_TAP_A))}
                rel = check_against_oracle(shape, st, ref, out, kp, vp, gtaps, assign, 1)
                print("cfg2 normalised rms error per stage:", {k: round(v, 5) for k, v in rel.items()})
                assert max(rel.values()) < 1e-2
            check_grouping(B.cc_debug_grouping(S.layer, batch), assign, st.seq_lens, R)
        for R in (2, 4):
            assert np.array_equal(results[R][0], results[1][0]), f"R={R} output bits differ from R=1"
            assert np.array_equal(results[R][1], results[1][1]) and np.array_equal(results[R][2], results[1][2])
