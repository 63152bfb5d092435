"""GPU tests of the replication mechanics: bit-identity across replica counts, the
byte-exact chunked replica copy, one CUDA graph surviving scale-up and
scale-down without recapture (north_star; the paper re-captures), the two-phase
publish / retire state machine and the sticky device error word."""
import numpy as np
import pytest
import torch

import oracle
from paper_2607_04181_b200 import inputs as I

pytestmark = pytest.mark.gpu

MID = I.LayerShape("mid", 512, 8, 2, 128, 1408, 1e-5, 500000.0, 21, 200, 700)


def _binding():
    from paper_2607_04181_b200 import binding as B
    from paper_2607_04181_b200.harness import DeviceStep, Session
    return B, DeviceStep, Session


def _read_device(ptr: int, nbytes: int) -> np.ndarray:
    """Raw device memory -> host bytes (torch has no public raw-pointer tensor; use cudart)."""
    out = np.empty(nbytes, dtype=np.uint8)
    from cuda.bindings import runtime as cudart  # cuda-python, in the image
    (err,) = cudart.cudaMemcpy(out.ctypes.data, ptr, nbytes, cudart.cudaMemcpyKind.cudaMemcpyDeviceToHost)
    assert int(err) == 0, err
    return out


@pytest.mark.parametrize("shape,batch,seeds", [(I.CFG1, 4, (1001, 2001, 3001)), (MID, 21, (1007, 2007, 3007))])
def test_bit_identical_across_replica_counts_and_assignments(shape, batch, seeds):
    B, DeviceStep, Session = _binding()
    w = I.make_weights(shape, seeds[0])
    st = I.make_step_inputs(shape, seeds[1], seeds[2], batch=batch)
    rng = np.random.default_rng(5)
    with Session(shape, w, max_batch=batch) as S:
        step = DeviceStep(st, np.zeros(batch, np.int32))
        S.forward(step)
        torch.cuda.synchronize()
        base_out, (base_k, base_v) = step.out_bits(), step.pools_bits()
        S.scale(4)
        cases = [I.even_split(batch, 2), I.even_split(batch, 4), rng.integers(0, 4, batch).astype(np.int32),
                 np.full(batch, 3, np.int32), (np.arange(batch) % 3).astype(np.int32)]
        for assign in cases:
            step.reset(st)
            step.set_assign(assign)
            S.forward(step)
            torch.cuda.synchronize()
            assert B.cc_poll_device_error(S.ctx) == 0
            k, v = step.pools_bits()
            assert np.array_equal(step.out_bits(), base_out), f"outputs differ for assignment {assign}"
            assert np.array_equal(k, base_k) and np.array_equal(v, base_v)


def test_replica_copy_is_byte_exact_and_stays_inside_its_slot():
    B, DeviceStep, Session = _binding()
    shape = I.CFG1
    w = I.make_weights(shape, 1001)
    with Session(shape, w, max_batch=4) as S:
        S.arena.fill_(0xA5)                                       # guard pattern over the whole donated range
        torch.cuda.synchronize()
        B.cc_ctx_set_copy_chunk(S.ctx, 1 << 20)                   # several chunks per blob (blob ~1.4 MiB)
        S.scale(4)
        torch.cuda.synchronize()
        assert B.cc_query(S.layer) == (4, 0)
        p0, n0 = B.cc_replica_blob(S.layer, 0)
        src = _read_device(p0, n0)
        want = oracle.replica_copy(src)                           # the oracle's definition: memcpy
        arena = S.arena.cpu().numpy()
        base = S.arena.data_ptr()
        covered = np.zeros(arena.shape[0], dtype=bool)
        for r in (1, 2, 3):
            p, n = B.cc_replica_blob(S.layer, r)
            assert n == n0 and p % 1024 == 0
            off = p - base
            assert np.array_equal(arena[off:off + n], want), f"replica {r} differs from slot 0"
            covered[off:off + n] = True
        assert (arena[~covered] == 0xA5).all(), "bytes outside the slots were touched"


@pytest.mark.parametrize("nbytes", [16, 48, 4096, 1 << 20, (1 << 20) + 16, 3 * (1 << 20) + 4080])
def test_copy_kernel_ragged_sizes(nbytes):
    B, _, _ = _binding()
    ctx = B.cc_ctx_create(0)
    try:
        g = torch.Generator(device="cpu").manual_seed(nbytes)
        src = torch.randint(0, 256, (nbytes + 64,), dtype=torch.uint8, generator=g).cuda()
        dst = torch.full((nbytes + 64,), 0x5A, dtype=torch.uint8, device="cuda")
        B.cc_replica_copy(ctx, dst[32:], src[32:], nbytes, 1 << 20, torch.cuda.current_stream())
        torch.cuda.synchronize()
        d, s = dst.cpu().numpy(), src.cpu().numpy()
        assert np.array_equal(d[32:32 + nbytes], oracle.replica_copy(s[32:32 + nbytes]))
        assert (d[:32] == 0x5A).all() and (d[32 + nbytes:] == 0x5A).all()
        with pytest.raises(B.CcError):
            B.cc_replica_copy(ctx, dst[16:], src[32:], 32, 0, None)            # dst not 32-byte aligned
    finally:
        B.cc_ctx_destroy(ctx)


def test_one_graph_survives_scale_up_and_down_without_recapture():
    B, DeviceStep, Session = _binding()
    shape, batch = MID, 21
    w = I.make_weights(shape, 1007)
    st = I.make_step_inputs(shape, 2007, 3007, batch=batch)
    with Session(shape, w, max_batch=batch) as S:
        step = DeviceStep(st, np.zeros(batch, np.int32))
        S.forward(step)                                            # warm-up outside capture
        torch.cuda.synchronize()
        base = step.out_bits()
        from paper_2607_04181_b200.harness import CapturedGraph
        step.reset(st)
        n_inst = CapturedGraph.instantiations
        graph = CapturedGraph(lambda s: S.forward(step, s))
        exec_handle = graph.exec_handle                             # the cudaGraphExec_t, not a Python id
        assert exec_handle != 0

        def replay(assign):
            step.reset(st)
            step.set_assign(assign)
            graph.replay()
            torch.cuda.synchronize()
            assert B.cc_poll_device_error(S.ctx) == 0
            return step.out_bits()

        assert np.array_equal(replay(np.zeros(batch, np.int32)), base)
        # scale up: copy on the side stream, publish on the replay stream; same graph, no recapture
        S.scale(2)
        assert B.cc_query(S.layer) == (2, 0) and graph.same_exec()
        two = I.even_split(batch, 2)
        assert np.array_equal(replay(two), base)
        # prove the replayed graph really reads replica 1's slot through the table: corrupt that slot
        p1, n1 = B.cc_replica_blob(S.layer, 1)
        off = p1 - S.arena.data_ptr()
        saved = S.arena[off:off + n1].clone()
        S.arena[off:off + n1].zero_()
        out = replay(two)
        assert np.array_equal(out[two == 0], base[two == 0])
        assert not np.array_equal(out[two == 1], base[two == 1])
        S.arena[off:off + n1].copy_(saved)
        assert np.array_equal(replay(two), base)
        # scale down: retire the row first, then the slot returns to the allocator
        S.scale(1)
        assert B.cc_query(S.layer) == (1, 0) and graph.same_exec()
        assert np.array_equal(replay(np.zeros(batch, np.int32)), base)
        # a row still naming the retired replica is served by replica 0 and flagged, never a fault
        step.reset(st)
        step.set_assign(two)
        graph.replay()
        torch.cuda.synchronize()
        assert B.cc_poll_device_error(S.ctx) == B.CC_DEVERR_BAD_REPLICA
        assert np.array_equal(step.out_bits(), base)
        # measured, not declared: one instantiation, and every replay above launched that same cudaGraphExec_t
        assert CapturedGraph.instantiations == n_inst + 1 and graph.exec_handle == exec_handle and graph.same_exec()
        assert graph.replays == 6


def test_forward_with_a_non_contiguous_live_set():
    """After releasing replica 1 of three the live indices are {0, 2}: cc_active_replicas reports them,
    a batch split over THOSE indices really uses replica 2's slot, and naming index 1 is flagged and rerouted."""
    B, DeviceStep, Session = _binding()
    shape, batch = MID, 21
    w = I.make_weights(shape, 1007)
    st = I.make_step_inputs(shape, 2007, 3007, batch=batch)
    with Session(shape, w, max_batch=batch) as S:
        step = DeviceStep(st, np.zeros(batch, np.int32))
        S.forward(step)
        torch.cuda.synchronize()
        base = step.out_bits()
        S.scale(3)
        assert B.cc_active_replicas(S.layer) == [0, 1, 2]
        B.cc_release_replica(S.layer, 1)
        assert B.cc_active_replicas(S.layer) == [0, 1, 2]           # nothing changes before the commit
        B.cc_commit(S.layer, torch.cuda.current_stream())
        live = B.cc_active_replicas(S.layer)
        assert live == [0, 2] and B.cc_query(S.layer) == (2, 0)
        assign = np.array(live, np.int32)[I.even_split(batch, len(live))]
        step.reset(st)
        step.set_assign(assign)
        S.forward(step)
        torch.cuda.synchronize()
        assert B.cc_poll_device_error(S.ctx) == 0
        assert np.array_equal(step.out_bits(), base)
        perm, counts, _ = B.cc_debug_grouping(S.layer, batch)
        assert counts[1] == 0 and counts[2] == int((assign == 2).sum()) > 0
        # the rows named to replica 2 do read its slot: zero it and only they change
        p2, n2 = B.cc_replica_blob(S.layer, 2)
        off = p2 - S.arena.data_ptr()
        S.arena[off:off + n2].zero_()
        step.reset(st)
        S.forward(step)
        torch.cuda.synchronize()
        out = step.out_bits()
        assert np.array_equal(out[assign == 0], base[assign == 0]) and not np.array_equal(out[assign == 2], base[assign == 2])
        # the retired index is not a replica any more
        step.reset(st)
        step.set_assign(I.even_split(batch, 2))                     # names index 1
        S.forward(step)
        torch.cuda.synchronize()
        assert B.cc_poll_device_error(S.ctx) == B.CC_DEVERR_BAD_REPLICA
        assert np.array_equal(step.out_bits(), base)


def test_rows_of_one_request_on_different_replicas_are_flagged():
    """Rows that share a first page id are one request (a prompt chunk); naming them to different replicas would put
    one request's KV in two partitions: CC_DEVERR_SPLIT_REQUEST.  The rows still run where named."""
    B, DeviceStep, Session = _binding()
    shape = I.CFG1
    w = I.make_weights(shape, 1001)
    st = I.make_step_inputs(shape, 2001, 3001)
    st.block_table[1] = st.block_table[0]                           # rows 0 and 1: one request, consecutive tokens
    st.seq_lens[0] = 20
    st.seq_lens[1] = 21
    with Session(shape, w, max_batch=4) as S:
        S.scale(2)
        step = DeviceStep(st, np.array([0, 0, 1, 1], np.int32))
        S.forward(step)
        torch.cuda.synchronize()
        assert B.cc_poll_device_error(S.ctx) == 0
        good = step.out_bits()
        step.reset(st)
        step.set_assign(np.array([0, 1, 1, 0], np.int32))
        S.forward(step)
        torch.cuda.synchronize()
        assert B.cc_poll_device_error(S.ctx) == B.CC_DEVERR_SPLIT_REQUEST
        assert np.array_equal(step.out_bits(), good)                # replicas hold the same weights: same bits


def test_all_padding_step_replayed_after_a_live_step():
    """A batch of padding rows only (every seq_len 0) in the same captured graph, right after a live step and before
    another (kernels of an empty step must still retire in launch order under PDL): nothing is written,
    and the next live step is bitwise the first."""
    B, DeviceStep, Session = _binding()
    from paper_2607_04181_b200.harness import CapturedGraph
    shape, batch = MID, 21
    w = I.make_weights(shape, 1007)
    st = I.make_step_inputs(shape, 2007, 3007, batch=batch)
    with Session(shape, w, max_batch=batch) as S:
        step = DeviceStep(st, np.zeros(batch, np.int32))
        S.forward(step)
        torch.cuda.synchronize()
        base, (bk, bv) = step.out_bits(), step.pools_bits()
        step.reset(st)
        graph = CapturedGraph(lambda s: S.forward(step, s))
        live_seq = step.seq_lens.clone()
        for _ in range(3):
            step.reset(st)
            step.seq_lens.copy_(live_seq)
            graph.replay()
            step.seq_lens.zero_()                                   # all rows padding; hidden now holds the live output
            graph.replay()
            torch.cuda.synchronize()
            assert B.cc_poll_device_error(S.ctx) == 0
            k, v = step.pools_bits()
            assert np.array_equal(step.out_bits(), base) and np.array_equal(k, bk) and np.array_equal(v, bv)
        assert graph.same_exec() and graph.replays == 6


def test_two_phase_publish_and_slot_reuse():
    B, DeviceStep, Session = _binding()
    shape = I.CFG1
    w = I.make_weights(shape, 1001)
    with Session(shape, w, max_batch=4, n_slots=2) as S:
        B.cc_scale_layer(S.layer, 3)
        assert B.cc_query(S.layer) == (1, 2)                        # copies enqueued, nothing visible yet
        B.cc_commit(S.layer, torch.cuda.current_stream())
        assert B.cc_query(S.layer) == (3, 0)
        with pytest.raises(B.CcError) as e:
            B.cc_scale_layer(S.layer, 4)                           # only two slots were donated
        assert e.value.status == B.CC_ERR_NO_SLOT
        assert B.cc_query(S.layer) == (3, 0)
        with pytest.raises(B.CcError) as e:
            B.cc_release_replica(S.layer, 0)
        assert e.value.status == B.CC_ERR_STATE
        p1, _ = B.cc_replica_blob(S.layer, 1)
        B.cc_release_replica(S.layer, 1)
        with pytest.raises(B.CcError) as e:
            B.cc_release_replica(S.layer, 1)                       # already retiring
        assert e.value.status == B.CC_ERR_STATE
        with pytest.raises(B.CcError) as e:
            B.cc_ctx_reclaim(S.ctx, S.arena)                       # live slots inside
        assert e.value.status == B.CC_ERR_BUSY
        B.cc_commit(S.layer, torch.cuda.current_stream())
        assert B.cc_query(S.layer) == (2, 0)
        torch.cuda.synchronize()
        S.scale(3)                                                 # the freed (lowest) slot is reused
        q1, _ = B.cc_replica_blob(S.layer, 1)
        assert q1 == p1
        # outputs with the re-created replica are still those of the unreplicated layer
        st = I.make_step_inputs(shape, 2001, 3001)
        step = DeviceStep(st, np.zeros(4, np.int32))
        S.forward(step)
        torch.cuda.synchronize()
        base = step.out_bits()
        step.reset(st)
        step.set_assign(np.array([1, 1, 2, 0], np.int32))
        S.forward(step)
        torch.cuda.synchronize()
        assert np.array_equal(step.out_bits(), base)


def test_device_error_word_and_bad_rows():
    B, DeviceStep, Session = _binding()
    shape = I.CFG1
    w = I.make_weights(shape, 1001)
    st = I.make_step_inputs(shape, 2001, 3001)
    with Session(shape, w, max_batch=4) as S:
        step = DeviceStep(st, np.zeros(4, np.int32))
        S.forward(step)
        torch.cuda.synchronize()
        base = step.out_bits()
        # seq_len beyond what the block table can address: row skipped, flagged
        bad = st.clone()
        bad.seq_lens[2] = shape.max_blocks * shape.page + 5
        step2 = DeviceStep(bad, np.zeros(4, np.int32))
        S.forward(step2)
        torch.cuda.synchronize()
        assert B.cc_poll_device_error(S.ctx) & B.CC_DEVERR_BAD_SEQLEN
        out = step2.out_bits()
        assert np.array_equal(out[2], st.hidden[2])
        assert np.array_equal(out[[0, 1, 3]], base[[0, 1, 3]])
        # a block-table entry of -1 below seq_len: flagged, no fault
        bad = st.clone()
        bad.block_table[1, 0] = -1
        step3 = DeviceStep(bad, np.zeros(4, np.int32))
        S.forward(step3)
        torch.cuda.synchronize()
        assert B.cc_poll_device_error(S.ctx) & B.CC_DEVERR_BAD_PAGE
        assert np.array_equal(step3.out_bits()[[0, 2, 3]], base[[0, 2, 3]])
        assert B.cc_poll_device_error(S.ctx) == 0                  # reading clears


def test_forward_host_matches_forward():
    B, DeviceStep, Session = _binding()
    shape = I.CFG1
    w = I.make_weights(shape, 1001)
    st = I.make_step_inputs(shape, 2001, 3001)
    assign = I.even_split(4, 2)
    with Session(shape, w, max_batch=4) as S:
        S.scale(2)
        step = DeviceStep(st, assign)
        S.forward(step)
        torch.cuda.synchronize()
        want = step.out_bits()
        step.reset(st)
        hidden = torch.from_numpy(st.hidden.view(np.int16).copy()).pin_memory()
        bt = torch.from_numpy(st.block_table.copy()).pin_memory()
        sl = torch.from_numpy(st.seq_lens.copy()).pin_memory()
        ra = torch.from_numpy(assign.copy()).pin_memory()
        B.cc_forward_host(S.layer, hidden, step.k_pool, step.v_pool, step.n_pages, bt, sl, ra, 4,
                          torch.cuda.current_stream())
        assert np.array_equal(hidden.numpy().view(np.uint16), want)
        assert B.cc_forward_launch_count(S.layer) == len(B.STAGE_NAMES)


@pytest.mark.parametrize("pinned", [True, False])
def test_forward_host_direct_and_staged_paths_match_forward(pinned):
    """cc_forward_host with pinned buffers lets the kernels read / write the host memory in place; with pageable
    buffers it stages through copies.  Both: output rows and the KV pools bitwise those of cc_forward; padding
    rows of the host buffer untouched; repeated calls (the staging is reused) stay identical."""
    B, DeviceStep, Session = _binding()
    shape, batch, R = MID, 21, 3
    w = I.make_weights(shape, 1011)
    st = I.make_step_inputs(shape, 2011, 3011, batch=batch)
    st.seq_lens[[3, 17]] = 0                                            # padding rows
    assign = (np.arange(batch) * 7 % R).astype(np.int32)
    with Session(shape, w, max_batch=batch) as S:
        S.scale(R)
        step = DeviceStep(st, assign)
        S.forward(step)
        torch.cuda.synchronize()
        want, (kw, vw) = step.out_bits(), step.pools_bits()
        assert np.array_equal(want[[3, 17]], st.hidden[[3, 17]])
        for rep in range(3):
            step.reset(st)
            bufs = [torch.from_numpy(a.copy()) for a in (st.hidden.view(np.int16), st.block_table, st.seq_lens, assign)]
            if pinned:
                bufs = [t.pin_memory() for t in bufs]
            hidden, bt, sl, ra = bufs
            B.cc_forward_host(S.layer, hidden, step.k_pool, step.v_pool, step.n_pages, bt, sl, ra, batch,
                              torch.cuda.current_stream())
            assert B.cc_poll_device_error(S.ctx) == 0
            assert np.array_equal(hidden.numpy().view(np.uint16), want), f"call {rep}"
            kp, vp = step.pools_bits()
            assert np.array_equal(kp, kw) and np.array_equal(vp, vw)
            assert np.array_equal(bt.numpy(), st.block_table) and np.array_equal(sl.numpy(), st.seq_lens)
        if pinned:
            # the kernel-by-kernel timing call takes the same pinned buffer (tables on the device)
            step.reset(st)
            hidden = torch.from_numpy(st.hidden.view(np.int16).copy()).pin_memory()
            ms = B.cc_forward_profiled(S.layer, hidden, step.k_pool, step.v_pool, step.block_table, step.n_pages,
                                       step.seq_lens, step.assign, batch, torch.cuda.current_stream())
            assert len(ms) == len(B.STAGE_NAMES) and (ms > 0).all()
            assert np.array_equal(hidden.numpy().view(np.uint16), want)


def test_forward_host_async_pipelines_steps_with_different_tables():
    """cc_forward_host_async is enqueue-only: eight steps with DIFFERENT tables (row order and replica assignment
    change from step to step) are enqueued back to back, each from its own pinned hidden buffer, one synchronisation at
    the end.  The pinned table mirror is a ring: every step must have run with the tables it was called with -- each
    result equals cc_forward of that step bit for bit.  Pageable hidden buffers are refused."""
    B, DeviceStep, Session = _binding()
    shape, batch, R = MID, 21, 3
    w = I.make_weights(shape, 1011)
    rng = np.random.default_rng(77)
    steps = []
    for i in range(8):
        st = I.make_step_inputs(shape, 2011, 3011, batch=batch)          # the same cache every step (the steps append the same slots)
        perm = rng.permutation(batch)
        st = I.StepInputs(st.hidden[perm].copy(), st.k_pool, st.v_pool, st.block_table[perm].copy(), st.seq_lens[perm].copy(), st.n_pages)
        steps.append((st, rng.integers(0, R, batch).astype(np.int32)))
    with Session(shape, w, max_batch=batch) as S:
        S.scale(R)
        want = []
        for st, assign in steps:
            step = DeviceStep(st, assign)
            S.forward(step)
            torch.cuda.synchronize()
            want.append(step.out_bits())
        dev = DeviceStep(steps[0][0], steps[0][1])
        stream = torch.cuda.current_stream()
        bufs = []
        for st, assign in steps:
            h = torch.from_numpy(st.hidden.view(np.int16).copy()).pin_memory()
            bt, sl, ra = st.block_table.copy(), st.seq_lens.copy(), assign.copy()
            B.cc_forward_host_async(S.layer, h, dev.k_pool, dev.v_pool, dev.n_pages, bt, sl, ra, batch, stream)
            bt[:] = -7; sl[:] = 0; ra[:] = 9                             # the tables were consumed before the call returned
            bufs.append(h)
        torch.cuda.synchronize()
        assert B.cc_poll_device_error(S.ctx) == 0
        for i, h in enumerate(bufs):
            assert np.array_equal(h.numpy().view(np.uint16), want[i]), f"step {i}"
        pageable = torch.from_numpy(steps[0][0].hidden.view(np.int16).copy())
        with pytest.raises(B.CcError):
            B.cc_forward_host_async(S.layer, pageable, dev.k_pool, dev.v_pool, dev.n_pages, steps[0][0].block_table, steps[0][0].seq_lens,
                                    steps[0][1], batch, stream)


def test_run_to_run_determinism_and_pdl_off_is_bitwise_the_same():
    """The fixups and merges are finished by whichever CTA arrives last: the result must not depend on that.
    Twenty replays from the same inputs, with and without programmatic dependent launch, give one bit pattern
    (PAPER.md:385 asks for bit-wise consistency; a timing-dependent sum order would break it silently)."""
    B, DeviceStep, Session = _binding()
    shape, batch = MID, 21
    w = I.make_weights(shape, 1007)
    st = I.make_step_inputs(shape, 2007, 3007, batch=batch)
    assign = (np.arange(batch) * 5 % 3).astype(np.int32)
    outs = []
    with Session(shape, w, max_batch=batch) as S:
        S.scale(3)
        step = DeviceStep(st, assign)
        for pdl in (1, 0):
            B.cc_ctx_set_pdl(S.ctx, pdl)
            for _ in range(10):
                step.reset(st)
                S.forward(step)
                torch.cuda.synchronize()
                kp, vp = step.pools_bits()
                outs.append((step.out_bits(), kp, vp))
        assert B.cc_poll_device_error(S.ctx) == 0
    for o, kp, vp in outs[1:]:
        assert np.array_equal(o, outs[0][0]) and np.array_equal(kp, outs[0][1]) and np.array_equal(vp, outs[0][2])
