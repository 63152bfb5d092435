"""Whole-model decode steps in ONE CUDA graph (BASELINE.json configs[2] at reduced size): four layers, the
graph holds every layer's cc_forward plus the in-graph seq_lens increment; mid-run two layers are scaled
to 2 replicas and later back to 1 by flipping the device replica table (cc_commit) -- never a recapture
(the paper re-captures when the configuration vector changes).  Every step's hidden
state must be bit-identical to a run without any flip, and the first layer of the first
step is checked against the oracle."""
import numpy as np
import pytest
import torch

import oracle
from paper_2607_04181_b200 import inputs as I

pytestmark = pytest.mark.gpu

SHAPE = I.LayerShape("mid4", 512, 8, 2, 64, 1408, 1e-5, 10000.0, 12, 40, 200)
L, STEPS, FLIP_UP, FLIP_DOWN, HOT = 4, 9, 3, 6, (1, 2)


def _run(flips: bool):
    from paper_2607_04181_b200 import binding as B
    from paper_2607_04181_b200.harness import ModelSession, _dev_u16, _host_u16

    batch = SHAPE.batch
    ws = [I.make_weights(SHAPE, 1100 + l) for l in range(L)]
    sts = [I.make_step_inputs(SHAPE, 2100 + l, 3100, batch=batch, n_pages=batch * (SHAPE.max_blocks + 1)) for l in range(L)]
    st0 = sts[0]
    # room for STEPS more tokens: extend the block table with the pool's unused pages
    width = SHAPE.max_blocks + 1
    bt = np.full((batch, width), -1, np.int32)
    bt[:, :st0.block_table.shape[1]] = st0.block_table
    used = set(int(x) for x in st0.block_table.ravel() if x >= 0)
    free = [p for p in range(st0.n_pages) if p not in used]
    for b in range(batch):
        need = (int(st0.seq_lens[b]) + STEPS + SHAPE.page - 1) // SHAPE.page
        for j in range(need):
            if bt[b, j] < 0:
                bt[b, j] = free.pop()
    dev = "cuda:0"
    wdev = [{k: _dev_u16(v, dev) for k, v in w.items()} for w in ws]
    outs = []
    with ModelSession(SHAPE, wdev, max_batch=batch, n_slots=len(HOT), max_blocks=width,
                      max_position=width * SHAPE.page) as M:
        del wdev
        hidden = _dev_u16(st0.hidden, dev)
        kp = [_dev_u16(s.k_pool, dev) for s in sts]
        vp = [_dev_u16(s.v_pool, dev) for s in sts]
        btd = torch.from_numpy(bt).to(dev)
        sl = torch.from_numpy(st0.seq_lens.copy()).to(dev)
        assigns = [torch.zeros(batch, dtype=torch.int32, device=dev) for _ in range(L)]
        M.forward_all(hidden, kp, vp, btd, st0.n_pages, sl, assigns, batch)          # warm-up, then restore
        torch.cuda.synchronize()
        first_layer_kp = _host_u16(kp[0])
        hidden.copy_(_dev_u16(st0.hidden, dev))
        for l in range(L):
            kp[l].copy_(_dev_u16(sts[l].k_pool, dev)); vp[l].copy_(_dev_u16(sts[l].v_pool, dev))
        from paper_2607_04181_b200.harness import CapturedGraph

        def whole_step(s):
            M.forward_all(hidden, kp, vp, btd, st0.n_pages, sl, assigns, batch, s)
            sl.add_(1)                                              # the next token's position, inside the graph
        n_inst = CapturedGraph.instantiations
        graph = CapturedGraph(whole_step)
        exec_handle = graph.exec_handle                             # the cudaGraphExec_t
        split = torch.from_numpy(I.even_split(batch, 2)).to(dev)
        for step in range(STEPS):
            if flips and step == FLIP_UP:
                for l in HOT:
                    M.scale(l, 2)
                    assigns[l].copy_(split)
                assert B.cc_query(M.layers[HOT[0]]) == (2, 0) and graph.same_exec()
            if flips and step == FLIP_DOWN:
                for l in HOT:
                    assigns[l].zero_()
                    M.scale(l, 1)
                assert B.cc_query(M.layers[HOT[0]]) == (1, 0) and graph.same_exec()
            graph.replay()
            torch.cuda.synchronize()
            assert B.cc_poll_device_error(M.ctx) == 0
            outs.append(_host_u16(hidden))
        # one instantiation; the same cudaGraphExec_t was launched before and after every cc_commit
        assert CapturedGraph.instantiations == n_inst + 1 and graph.exec_handle == exec_handle and graph.replays == STEPS
        assert sl.cpu().numpy().tolist() == (st0.seq_lens + STEPS).tolist()
    return ws, sts, outs, first_layer_kp


def test_model_graph_survives_layer_flips_bitwise():
    ws, sts, plain, _ = _run(flips=False)
    _, _, flipped, _ = _run(flips=True)
    for step, (a, b) in enumerate(zip(plain, flipped)):
        assert np.array_equal(a, b), f"hidden after step {step} differs between the flipped and the plain run"
    assert not np.array_equal(plain[0], plain[1])                 # the steps really advance


def test_model_graph_first_step_matches_layerwise_oracle():
    ws, sts, plain, _ = _run(flips=False)
    st0 = sts[0]
    h = st0.hidden
    assign = np.zeros(SHAPE.batch, np.int32)
    bt = st0.block_table
    for l in range(L):                                            # the oracle, layer after layer (fp32 -> bf16 between layers)
        ref = oracle.layer_forward(SHAPE, ws[l], h, sts[l].k_pool, sts[l].v_pool, bt, st0.seq_lens, assign, 1)
        h = ref["out"]
    got, want = I.bf16_bits_to_f32(plain[0]).astype(np.float64), I.bf16_bits_to_f32(h).astype(np.float64)
    err = np.abs(got - want)
    # tolerance of one layer (north_star) times the number of layers the rounding differences pass through
    assert (err <= L * (1e-2 + 2e-2 * np.abs(want))).all(), f"max err {err.max()}"
