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
