"""KV partition per replica: the library's planner against
the independent host simulation (block tables and move lists must match EXACTLY), its invariants, and --
on the GPU -- that a migrated cache gives bit-identical layer outputs."""
import numpy as np
import pytest

from oracle import hostsim
from paper_2607_04181_b200 import inputs as I


def _scenario(rng, batch, n_pages, width, R):
    seq = rng.integers(0, width * 16 + 1, batch).astype(np.int32)
    seq[rng.random(batch) < 0.15] = 0                                       # padding rows
    need = (seq + 15) // 16
    ids = rng.permutation(n_pages).astype(np.int32)
    bt = np.full((batch, width), -1, np.int32)
    off = 0
    for b in range(batch):
        bt[b, :need[b]] = ids[off:off + need[b]]
        off += int(need[b])
    assign = rng.integers(0, R, batch).astype(np.int32)
    return bt, seq, assign


def test_planner_matches_the_host_simulation_exactly():
    from paper_2607_04181_b200 import binding as B
    rng = np.random.default_rng(5)
    for trial in range(60):
        R = int(rng.integers(1, 5))
        batch, width = int(rng.integers(1, 12)), int(rng.integers(1, 7))
        n_pages = int(batch * width * rng.uniform(1.0, 3.0)) + R
        bt, seq, assign = _scenario(rng, batch, n_pages, width, R)
        want = hostsim.plan_kv_migration(bt, seq, assign, n_pages, R)
        try:
            new_bt, src, dst = B.cc_kv_plan_migration(bt, seq, assign, n_pages, R)
        except B.CcError as e:
            assert e.status == B.CC_ERR_NO_SLOT and want is None
            continue
        assert want is not None
        assert np.array_equal(new_bt, want[0]) and list(zip(src.tolist(), dst.tolist())) == want[1]
        # invariants: every live page sits in its replica's partition, no page is referenced twice, destinations
        # were free before, sources and destinations are disjoint
        psz = n_pages // R
        seen = set()
        for b in range(batch):
            for j in range((int(seq[b]) + 15) // 16 if seq[b] > 0 else 0):
                pg = int(new_bt[b, j])
                assert assign[b] * psz <= pg < (assign[b] + 1) * psz and pg not in seen
                seen.add(pg)
        before = {int(bt[b, j]) for b in range(batch) for j in range((int(seq[b]) + 15) // 16 if seq[b] > 0 else 0)}
        assert not (set(dst.tolist()) & before) and not (set(dst.tolist()) & set(src.tolist()))
        assert len(set(dst.tolist())) == len(dst)


def test_planner_and_catchup_on_a_hand_worked_scenario():
    """Tables written out by hand from the rule, pinning BOTH the host simulation
    and the library to something other than each other.  12 pages, 2 replicas: partition 0 = pages 0..5, partition
    1 = pages 6..11; pages of 16 tokens.

    Plan.  Row 0 (33 tokens, replica 0) holds pages [7, 2, 9]: 7 and 9 lie outside 0..5.  Referenced pages are
    {7, 2, 9, 0, 10, 3} (row 2 is a padding row: its table entry 5 does not count).  7 -> lowest unreferenced page
    of 0..5 = 1; 2 stays; 9 -> 4 (0 referenced, 1 taken, 2, 3 referenced).  Row 1 (16 tokens, replica 1) holds
    [0]: 0 -> 6.  Row 3 (20 tokens, replica 1) holds [10, 3]: 10 stays; 3 -> 8 (6 taken, 7 still referenced as a
    source).

    Catch-up after the rows decoded on with the OLD table: row 0 grew 33 -> 35 tokens, row 1 16 -> 18 (a second
    page, 11, from the caller's allocator), row 3 stayed at 20.  Only tokens >= seq_planned - 1 can have been
    written since: row 0: tokens >= 32 = its page 2 (dirty, still at 9), pages 0 and 1 keep their planned places 1
    and 2; row 1: token 15 is in page 0 (dirty, at 0) and page 1 is new (at 11, inside partition 1 already); row
    3: tokens >= 19 = page 1 (dirty, at 3), page 0 keeps 10.  Re-planning [1, 2, 9], [0, 11], [10, 3]: 9 -> 4
    (0, 1, 2, 3 referenced); 0 -> 6; 11 stays; 3 -> 7 (no longer referenced: row 0's first page now counts as 1)."""
    from paper_2607_04181_b200 import binding as B
    bt = np.array([[7, 2, 9], [0, -1, -1], [5, -1, -1], [10, 3, -1]], np.int32)
    seq = np.array([33, 16, 0, 20], np.int32)
    assign = np.array([0, 1, 0, 1], np.int32)
    want_bt = np.array([[1, 2, 4], [6, -1, -1], [5, -1, -1], [10, 8, -1]], np.int32)
    want_moves = [(7, 1), (9, 4), (0, 6), (3, 8)]
    sim_bt, sim_moves = hostsim.plan_kv_migration(bt, seq, assign, 12, 2)
    assert np.array_equal(sim_bt, want_bt) and sim_moves == want_moves
    new_bt, src, dst = B.cc_kv_plan_migration(bt, seq, assign, 12, 2)
    assert np.array_equal(new_bt, want_bt) and list(zip(src.tolist(), dst.tolist())) == want_moves

    bt_now = np.array([[7, 2, 9], [0, 11, -1], [5, -1, -1], [10, 3, -1]], np.int32)
    seq_now = np.array([35, 18, 0, 20], np.int32)
    want_final = np.array([[1, 2, 4], [6, 11, -1], [5, -1, -1], [10, 7, -1]], np.int32)
    want_catchup = [(9, 4), (0, 6), (3, 7)]
    sim_final, sim_catchup = hostsim.plan_kv_catchup(bt_now, seq, seq_now, want_bt, assign, 12, 2)
    assert np.array_equal(sim_final, want_final) and sim_catchup == want_catchup
    final_bt, src, dst = B.cc_kv_plan_catchup(bt_now, seq, seq_now, want_bt, assign, 12, 2)
    assert np.array_equal(final_bt, want_final) and list(zip(src.tolist(), dst.tolist())) == want_catchup


def test_planner_rejects_bad_tables():
    from paper_2607_04181_b200 import binding as B
    bt = np.array([[0, 1], [1, 2]], np.int32)
    with pytest.raises(B.CcError) as e:
        B.cc_kv_plan_migration(bt, np.array([32, 32], np.int32), np.zeros(2, np.int32), 8, 2)
    assert e.value.status == B.CC_ERR_INVALID                                   # page 1 referenced twice


@pytest.mark.gpu
def test_migrated_cache_gives_bit_identical_outputs():
    import torch
    from paper_2607_04181_b200 import binding as B
    from paper_2607_04181_b200.harness import DeviceStep, Session

    shape = I.LayerShape("mid", 512, 8, 2, 128, 1408, 1e-5, 500000.0, 21, 200, 700)
    batch, R = 21, 2
    w = I.make_weights(shape, 1301)
    st = I.make_step_inputs(shape, 2301, 3301, batch=batch, n_pages=4 * batch * shape.max_blocks)
    assign = I.even_split(batch, R)
    with Session(shape, w, max_batch=batch) as S:
        S.scale(R)
        step = DeviceStep(st, assign)
        S.forward(step)
        torch.cuda.synchronize()
        base = step.out_bits()
        # plan + migrate on the device, swap the table in place (same device address: graph-safe)
        new_bt, src, dst = B.cc_kv_plan_migration(st.block_table, st.seq_lens, assign, st.n_pages, R)
        assert len(src) > 0
        step.reset(st)
        page_bytes = shape.n_kv_heads * shape.page * shape.head_dim * 2
        B.cc_kv_migrate(S.ctx, step.k_pool, step.v_pool, page_bytes, torch.from_numpy(src).cuda(), torch.from_numpy(dst).cuda(),
                        len(src), torch.cuda.current_stream())
        torch.cuda.synchronize()
        kp, vp = step.pools_bits()
        k_ref, v_ref = st.k_pool.copy(), st.v_pool.copy()
        hostsim.apply_kv_migration(k_ref, v_ref, list(zip(src.tolist(), dst.tolist())))
        assert np.array_equal(kp, k_ref) and np.array_equal(vp, v_ref)           # byte-exact page copies, nothing else touched
        step.block_table.copy_(torch.from_numpy(new_bt))
        S.forward(step)
        torch.cuda.synchronize()
        assert B.cc_poll_device_error(S.ctx) == 0
        assert np.array_equal(step.out_bits(), base)
        # the rows' pages now lie in their replica's partition
        psz = st.n_pages // R
        for b in range(batch):
            for j in range((int(st.seq_lens[b]) + 15) // 16):
                assert assign[b] * psz <= new_bt[b, j] < (assign[b] + 1) * psz


def _pages_of(bt, seq):
    return {int(bt[b, j]) for b in range(bt.shape[0]) if seq[b] > 0 for j in range((int(seq[b]) + 15) // 16)}


def _grow(rng, bt, seq, n_pages, reserved, steps, finish_prob=0.0):
    """Rows decode `steps` more tokens with the old table: a new page (any free one that is not reserved, drawn at
    random so that it usually lies outside the row's partition) whenever a token starts a page."""
    bt, seq = bt.copy(), seq.copy()
    free = sorted(set(range(n_pages)) - _pages_of(bt, seq) - set(reserved))
    rng.shuffle(free)
    for _ in range(steps):
        for b in range(len(seq)):
            if seq[b] <= 0 or seq[b] >= bt.shape[1] * 16:
                continue
            seq[b] += 1
            if (seq[b] - 1) % 16 == 0:                                     # the token being decoded opens a page
                bt[b, (seq[b] - 1) // 16] = free.pop()
    for b in range(len(seq)):
        if seq[b] > 0 and rng.random() < finish_prob:
            seq[b] = 0
    return bt, seq


def test_catchup_plan_matches_the_host_simulation_exactly():
    """Pre-copy migration: decode steps go on with the old table while the bulk is copied; the
    catch-up plan covers what they wrote.  Library == independent simulation, plus what must hold whatever the
    rule: untouched pages keep their first-plan place, everything ends in its partition, nothing is shared."""
    from paper_2607_04181_b200 import binding as B
    rng = np.random.default_rng(11)
    done = 0
    for trial in range(80):
        R = int(rng.integers(1, 5))
        batch, width = int(rng.integers(1, 12)), int(rng.integers(2, 8))
        n_pages = int(batch * width * rng.uniform(2.5, 4.0)) + 4 * R
        bt, seq, assign = _scenario(rng, batch, n_pages, width, R)
        first = hostsim.plan_kv_migration(bt, seq, assign, n_pages, R)
        if first is None:
            continue
        planned_bt, moves = first
        bt_now, seq_now = _grow(rng, bt, seq, n_pages, [d for _, d in moves], int(rng.integers(0, 40)), finish_prob=0.1)
        want = hostsim.plan_kv_catchup(bt_now, seq, seq_now, planned_bt, assign, n_pages, R)
        try:
            final_bt, src, dst = B.cc_kv_plan_catchup(bt_now, seq, seq_now, planned_bt, assign, n_pages, R)
        except B.CcError as e:
            assert e.status == B.CC_ERR_NO_SLOT and want is None
            continue
        assert want is not None
        assert np.array_equal(final_bt, want[0]) and list(zip(src.tolist(), dst.tolist())) == want[1]
        psz = n_pages // R
        seen = set()
        for b in range(batch):
            if seq_now[b] <= 0:
                continue
            for j in range((int(seq_now[b]) + 15) // 16):
                pg = int(final_bt[b, j])
                assert assign[b] * psz <= pg < (assign[b] + 1) * psz and pg not in seen
                seen.add(pg)
                if (j + 1) * 16 <= seq[b] - 1:                              # only tokens < seq_planned - 1: never rewritten
                    assert pg == planned_bt[b, j]
        # no page is both read and written by the catch-up copy, and it moves only what the steps touched
        assert not (set(dst.tolist()) & set(src.tolist())) and len(set(dst.tolist())) == len(dst)
        assert len(src) <= sum(1 + (int(seq_now[b]) + 15) // 16 - (int(seq[b]) + 15) // 16 if seq[b] > 0 else (int(seq_now[b]) + 15) // 16
                               for b in range(batch) if seq_now[b] > 0)
        done += 1
    assert done > 40


def test_catchup_rejects_a_row_that_shrank():
    from paper_2607_04181_b200 import binding as B
    bt = np.array([[0, 1, 2]], np.int32)
    with pytest.raises(B.CcError) as e:
        B.cc_kv_plan_catchup(bt, np.array([40], np.int32), np.array([33], np.int32), bt, np.zeros(1, np.int32), 8, 1)
    assert e.value.status == B.CC_ERR_INVALID


@pytest.mark.gpu
def test_migration_overlapped_with_decode_steps_changes_nothing():
    """the cache is redistributed while decoding goes on.  Six decode steps (rows grow, some open
    a page) run while the bulk copy is in flight on a side stream; catch-up + table swap; two more steps.  Every
    step's output and, at the end, every row's cache (gathered through its table) equal the run without migration
    bit for bit; all pages end inside their replica's partition; the graph is never re-captured."""
    import torch
    from paper_2607_04181_b200 import binding as B
    from paper_2607_04181_b200.harness import DeviceStep, KvLiveMigration, Session

    shape = I.LayerShape("mid", 512, 8, 2, 128, 1408, 1e-5, 500000.0, 23, 200, 690)
    batch, R, during, after = 23, 2, 6, 2
    w = I.make_weights(shape, 1302)
    n_pages = 4 * batch * shape.max_blocks
    ctx = I.draw_contexts(shape, 3302, batch)
    ctx[:4] = [207, 208, 223, 224]                  # rows that open a page at the first step, just did, or will later
    st = I.make_step_inputs(shape, 2302, 3302, batch=batch, n_pages=n_pages, contexts=ctx)
    assign = I.even_split(batch, R)
    page_bytes = shape.n_kv_heads * shape.page * shape.head_dim * 2
    rng = np.random.default_rng(7)

    def run(migrate: bool):
        with Session(shape, w, max_batch=batch) as S:
            S.scale(R)
            step = DeviceStep(st, assign)
            h0 = step.hidden.clone()
            bt, seq = st.block_table.copy(), st.seq_lens.copy()
            graph = torch.cuda.CUDAGraph()
            main = torch.cuda.Stream()
            side = torch.cuda.Stream()
            outs = []
            with torch.cuda.stream(main):
                S.forward(step, main)                                       # warm-up (appends position seq - 1)
                main.synchronize()
                with torch.cuda.graph(graph, stream=main):
                    S.forward(step, main)
                mig = KvLiveMigration(S.ctx, step, page_bytes, R, chunk_pages=64)
                free = None
                for i in range(during + after):
                    if migrate and i == 0:
                        assert mig.start(bt, seq, assign, side) > 100
                    if migrate and i == during:
                        final_bt = mig.finish(bt, seq, main)
                        assert mig.catchup_moves > 0
                        bt = final_bt.copy()
                        free = None                                         # old places are free again, new ones taken
                    if free is None:
                        free = sorted(set(range(n_pages)) - _pages_of(bt, seq) - mig.reserved)
                        rng.shuffle(free)
                    # the step decodes one more token per row
                    seq = seq + 1
                    for b in range(batch):
                        if (seq[b] - 1) % 16 == 0:
                            bt[b, (seq[b] - 1) // 16] = free.pop()
                    step.block_table.copy_(torch.from_numpy(bt))
                    step.seq_lens.copy_(torch.from_numpy(seq))
                    step.hidden.copy_(h0)
                    graph.replay()
                    outs.append(step.hidden.clone())
                main.synchronize()
            side.synchronize()
            assert B.cc_poll_device_error(S.ctx) == 0
            kp, vp = step.pools_bits()
            rows = [(kp[bt[b, :(seq[b] + 15) // 16]].copy(), vp[bt[b, :(seq[b] + 15) // 16]].copy()) for b in range(batch)]
            return [o.cpu().view(torch.int16).numpy() for o in outs], rows, bt, seq

    rng = np.random.default_rng(7)
    base_out, base_rows, _, _ = run(False)
    rng = np.random.default_rng(7)
    mig_out, mig_rows, bt, seq = run(True)
    for i, (a, b_) in enumerate(zip(base_out, mig_out)):
        assert np.array_equal(a, b_), f"step {i} differs"
    for b in range(batch):
        n_tok = int(seq[b])
        for (x, y) in zip(base_rows[b], mig_rows[b]):
            # [pages][kv heads][16][head_dim] -> compare the tokens that exist
            xs = x.transpose(1, 0, 2, 3).reshape(shape.n_kv_heads, -1, shape.head_dim)[:, :n_tok]
            ys = y.transpose(1, 0, 2, 3).reshape(shape.n_kv_heads, -1, shape.head_dim)[:, :n_tok]
            assert np.array_equal(xs, ys)
    psz = n_pages // R
    for b in range(batch):
        # pages present at the swap are in the partition (the two later steps may have opened one anywhere)
        for j in range((int(seq[b]) - after + 15) // 16):
            assert assign[b] * psz <= bt[b, j] < (assign[b] + 1) * psz


@pytest.mark.gpu
@pytest.mark.parametrize("big", [False, True])
def test_replica_with_its_own_kv_partition_as_a_separate_allocation(big):
    """cc_layer_set_kv_partition (SURVEY.md 8(c) reading 17): replica 1's requests keep their pages in a
    SEPARATE allocation, page ids relative to it.  The pages of replica 1's rows are moved there (compacted ids, their
    old places in the shared pool poisoned with NaN); outputs must be bitwise those of the one-pool run, the appended
    K/V must land in the partition, and the shared pool must stay untouched where replica 1's rows used to live.  Small
    step (decode kernels) and large step (a prompt chunk through the prefill kernel + decode rows)."""
    import torch
    from paper_2607_04181_b200 import binding as B
    from paper_2607_04181_b200.harness import DeviceStep, Session, _dev_u16, _host_u16

    shape = I.LayerShape("kvpart", 512, 8, 2, 128, 1408, 1e-5, 500000.0, 8, 0, 600)
    page = shape.page
    if big:
        from tests.test_gpu_mixed import mixed_step
        rng = np.random.default_rng(8)
        st, assign = mixed_step(shape, 8, [(30, 180), (0, 90)], rng.integers(0, 400, 50), 2)    # chunk 0 -> replica 0, chunk 1 -> replica 1
    else:
        st = I.make_step_inputs(shape, 2601, 3601, batch=24)
        assign = (np.arange(24) % 2).astype(np.int32)
        assign[5] = 0
    batch = st.hidden.shape[0]
    w = I.make_weights(shape, 1601)
    kw = dict(max_batch=batch, max_blocks=st.block_table.shape[1], max_position=st.block_table.shape[1] * page)
    with Session(shape, w, **kw) as S:
        S.scale(2)
        step = DeviceStep(st, assign)
        S.forward(step)
        torch.cuda.synchronize()
        want, (kw1, vw1) = step.out_bits(), step.pools_bits()
    # move replica 1's pages into their own pools
    rows1 = np.nonzero((assign == 1) & (st.seq_lens > 0))[0]
    remap, bt2 = {}, st.block_table.copy()
    for b in rows1:                                                       # whole rows: the rows of a prompt chunk carry identical copies
        for j in range(st.block_table.shape[1]):
            pg = int(st.block_table[b, j])
            if pg >= 0:
                remap.setdefault(pg, len(remap))
                bt2[b, j] = remap[pg]
    n1 = len(remap)
    old = np.array(list(remap.keys())), np.array(list(remap.values()))
    k1 = np.zeros((n1,) + st.k_pool.shape[1:], np.uint16); v1 = np.zeros_like(k1)
    k1[old[1]], v1[old[1]] = st.k_pool[old[0]], st.v_pool[old[0]]
    k0, v0 = st.k_pool.copy(), st.v_pool.copy()
    k0[old[0]] = 0x7FC0; v0[old[0]] = 0x7FC0                              # nobody may read replica 1's old pages
    st2 = I.StepInputs(st.hidden, k0, v0, bt2, st.seq_lens, st.n_pages)
    with Session(shape, w, **kw) as S:
        S.scale(2)
        d_k1, d_v1 = _dev_u16(k1, S.device), _dev_u16(v1, S.device)
        B.cc_layer_set_kv_partition(S.layer, 1, d_k1, d_v1, n1, torch.cuda.current_stream())
        step = DeviceStep(st2, assign)
        S.forward(step)
        torch.cuda.synchronize()
        assert B.cc_poll_device_error(S.ctx) == 0
        got, (kg0, vg0) = step.out_bits(), step.pools_bits()
        kg1, vg1 = _host_u16(d_k1), _host_u16(d_v1)
        # a page id beyond the partition is refused for replica 1's rows although the shared pool has that page
        bad = bt2.copy(); bad[rows1[0], 0] = n1 + 3
        step.block_table.copy_(torch.from_numpy(bad).to(S.device))
        S.forward(step)
        torch.cuda.synchronize()
        assert B.cc_poll_device_error(S.ctx) & B.CC_DEVERR_BAD_PAGE
    assert np.array_equal(got, want)
    assert np.array_equal(kg1[old[1]], kw1[old[0]]) and np.array_equal(vg1[old[1]], vw1[old[0]])     # partition == what the one-pool run left on those pages
    keep = np.ones(st.k_pool.shape[0], bool); keep[old[0]] = False
    assert np.array_equal(kg0[keep], kw1[keep]) and np.array_equal(vg0[keep], vw1[keep])
    assert np.array_equal(kg0[~keep], k0[~keep]) and np.array_equal(vg0[~keep], v0[~keep])             # still the poison
