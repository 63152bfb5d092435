"""cc_attention_decode_static (include/cocoscale.h): the one entry point that allocates nothing -- paged GQA decode attention
whose split-KV partials live in a file-scope device array (csrc/cc_noalloc.cu) -- against the existing path: the attention
stage of cc_forward (tap "o") on the same q (tap "q") and the same KV pools, within the tolerance of tests/test_gpu_parity.py.
Calls in a row, of different geometry, share the array: each must still match its own existing-path result.

Named test_zz_* so that pytest collects it last: the suite runs with `pytest -x`."""
import numpy as np
import pytest
import torch

from paper_2607_04181_b200 import inputs as I

pytestmark = pytest.mark.gpu

ATOL, RTOL = 1e-2, 2e-2          # BASELINE.json north_star, as in tests/test_gpu_parity.py


def within(gpu, ref, what):
    gpu = np.asarray(gpu, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    assert gpu.shape == ref.shape, what
    assert np.isfinite(gpu).all(), f"{what}: non-finite values"
    err = np.abs(gpu - ref)
    bad = err > ATOL + RTOL * np.abs(ref)
    assert not bad.any(), f"{what}: {int(bad.sum())}/{bad.size} elements outside tolerance; worst |err| = {err.max():.4g}"
    return float(np.sqrt((err ** 2).mean()) / max(np.sqrt((ref ** 2).mean()), 1e-30))


class ExistingPath:
    """One cc_forward step of `shape`; keeps what the attention stage read (q, the pools after the append, the tables) on
    the device and what it produced (tap "o") on the host."""

    def __init__(self, shape, batch, seeds, pad_row=None):
        from paper_2607_04181_b200 import binding as B
        from paper_2607_04181_b200.harness import DeviceStep, Session

        w = I.make_weights(shape, seeds[0])
        st = I.make_step_inputs(shape, seeds[1], seeds[2], batch=batch)
        if pad_row is not None:
            st.seq_lens[pad_row] = 0                                                  # a row that does not run
        self.shape, self.batch, self.live = shape, batch, st.seq_lens > 0
        with Session(shape, w, max_batch=batch, n_slots=0) as S:
            self.step = DeviceStep(st, np.zeros(batch, dtype=np.int32))
            S.forward(self.step)
            torch.cuda.synchronize()
            assert B.cc_poll_device_error(S.ctx) == 0
            self.q = torch.from_numpy(S.tap(B.CC_TAP_Q, batch)).to("cuda:0")          # fp32 [batch][Hq * Dh], post-RoPE
            self.o_ref = S.tap(B.CC_TAP_O, batch)
        self.max_blocks = int(self.step.block_table.shape[1])
        self.out = torch.full((batch, shape.q_dim), float("nan"), dtype=torch.float32, device="cuda:0")

    def call_static(self, stream=None):
        from paper_2607_04181_b200 import binding as B
        s = self.shape
        self.out.fill_(float("nan"))
        B.cc_attention_decode_static(self.q, self.step.k_pool, self.step.v_pool, self.step.block_table, self.step.seq_lens, self.out,
                                     self.batch, s.n_q_heads, s.n_kv_heads, s.head_dim, self.max_blocks, self.step.n_pages, stream)

    def check(self, what):
        got = self.out.cpu().numpy()
        assert np.abs(self.o_ref[self.live]).max() > 1e-3, "the reference attention output is not all zeros"
        return within(got[self.live], self.o_ref[self.live], what), got


def test_static_attention_matches_cc_forward_on_calls_in_a_row():
    from paper_2607_04181_b200 import binding as B

    assert B.cc_static_scratch_bytes() == 8 << 20
    # head_dim 128, 6 query heads per kv head, contexts of 256..1024 positions: three ranges per row;
    # head_dim 64, 2 query heads per kv head, contexts of 16..64 positions, one padding row: one range per row
    a = ExistingPath(I.MODEL_B_LAYER, 24, (1101, 2101, 3101))
    b = ExistingPath(I.CFG1, 4, (1102, 2102, 3102), pad_row=2)
    a.call_static()                                  # the first call on the device also takes the array's address
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    stream = torch.cuda.current_stream()
    a.call_static(stream)                            # two calls in a row on one stream, different geometry,
    b.call_static(stream)                            # sharing the one scratch array
    torch.cuda.synchronize()
    rel_a, out_a1 = a.check("static attention, modelB shape")
    rel_b, out_b1 = b.check("static attention, cfg1 shape, after a call of another geometry")
    assert rel_a < 1e-2 and rel_b < 1e-2, (rel_a, rel_b)
    b.call_static(stream)
    a.call_static(stream)
    torch.cuda.synchronize()
    _, out_a2 = a.check("static attention, modelB shape, second round")
    _, out_b2 = b.check("static attention, cfg1 shape, second round")
    assert np.array_equal(out_a1, out_a2) and np.array_equal(out_b1, out_b2)       # fixed merge order: the same bits
    assert torch.cuda.mem_get_info()[0] >= free0, "the calls took device memory"


def test_static_attention_rejects_what_does_not_fit():
    from paper_2607_04181_b200 import binding as B

    t = torch.zeros(16, dtype=torch.float32, device="cuda:0")
    i = torch.zeros(16, dtype=torch.int32, device="cuda:0")
    with pytest.raises(B.CcError) as e:              # 2048 rows x 64 heads x 130 floats = 68 MB of partials
        B.cc_attention_decode_static(t, t, t, i, i, t, 2048, 64, 8, 128, 4, 1)
    assert e.value.status == B.CC_ERR_INVALID and "CC_STATIC_SCRATCH_BYTES" in str(e.value)
    with pytest.raises(B.CcError) as e:
        B.cc_attention_decode_static(t, t, t, i, i, t, 1, 4, 2, 96, 4, 1)
    assert e.value.status == B.CC_ERR_INVALID and "head_dim" in str(e.value)
