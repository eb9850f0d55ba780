"""db_deliver_external_static -- the entry point that allocates no device memory (its scratch, the device copy of the
id list, is a static device array of DB_EXTERNAL_STATIC_MAX ids) -- against the existing db_deliver_external: two
identical handles that own the same half of a network get the same outside spikes, one through each entry point, on
two calls in a row and then over a closed loop.  Ring, state, raster and counters must be equal bit for bit (the bar
of the other parity tests: integer work).  Collected last on purpose (file name)."""
import numpy as np
import pytest

import db_inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def db():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2211_15963_b200 as m
    m.load()
    return m


def _same(db, a, b):
    assert np.array_equal(a.db_read_state(db.FIELD_RING), b.db_read_state(db.FIELD_RING))
    for x, y in zip(a.state(), b.state()):
        assert np.array_equal(x, y)
    ca, cb = a.db_get_counters(), b.db_get_counters()
    for k in ("steps", "spikes", "events", "bg_events", "ring_overflow"):
        assert ca[k] == cb[k], k


@pytest.mark.parametrize("fp16", [False, True])
def test_static_scratch_entry_point_matches_the_allocating_one(db, fp16):
    cfg = db_inputs.config(2, scale=0.004)                       # 20,000 neurons, K = 160 + 40
    cfg["net"].update(n_regions=8, delay_intra_min=3, delay_inter_min=20, weight_fp16=int(fp16))
    t = db_inputs.type_params(bg_weight=0.02)
    t.update(G=[0.5, 0.125, 0.5, 0.5])
    cfg["sim"]["types"] = [t, dict(t)]
    N = cfg["net"]["N"]
    cut = 9 * 1024
    mk = lambda first, count: db.Sim.db_create(cfg["net"], cfg["sim"], seed=db_inputs.GEN_SEED, exec_mode=db.EXEC_KERNELS,
                                               own=(first, count))
    ref, new, other = mk(0, cut), mk(0, cut), mk(cut, N - cut)     # `other` only supplies plausible outside spikes
    rng = np.random.default_rng(3)
    # ---- two calls in a row, the second with a shorter list (the array still holds the tail of the first)
    ring0 = ref.db_read_state(db.FIELD_RING).copy()
    for step, n_ids in ((0, 700), (1, 90)):
        ids = np.sort(rng.choice(np.arange(cut, N), n_ids, replace=False)).astype(np.int32)
        ref.db_deliver_external(step, ids)
        new.db_deliver_external_static(step, ids)
        _same(db, ref, new)
    assert ref.db_get_counters()["events"] > 10_000 and not np.array_equal(ring0, ref.db_read_state(db.FIELD_RING))
    # ---- closed loop: 60 steps, lists exchanged every 3 steps (smallest delay)
    done = 0
    while done < 60:
        for s in (ref, new, other):
            s.db_step(3)
        st, ids = other.db_read_spikes(done, done + 3)
        st_r, ids_r = ref.db_read_spikes(done, done + 3)
        for step in range(done, done + 3):
            ref.db_deliver_external(step, ids[st == step])
            new.db_deliver_external_static(step, ids[st == step])
            other.db_deliver_external(step, ids_r[st_r == step])
        done += 3
    _same(db, ref, new)
    a, b = ref.db_read_spikes(0, 60), new.db_read_spikes(0, 60)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and len(a[1]) > 50
    # ---- limits and argument checks: same answers as the allocating entry point, plus the size limit
    big = np.resize(np.arange(cut, N, dtype=np.int32), db.binding.EXTERNAL_STATIC_MAX + 1)    # every outside neuron ~6 times
    with pytest.raises(db.DbError) as e:
        new.db_deliver_external_static(60, big)
    assert e.value.code == db.binding.DB_EINVAL and "DB_EXTERNAL_STATIC_MAX" in str(e.value)
    new.db_deliver_external_static(60, big[:-1]); ref.db_deliver_external(60, big[:-1])      # exactly the maximum is fine
    _same(db, ref, new)
    with pytest.raises(db.DbError):
        new.db_deliver_external_static(60, np.array([5], np.int32))                          # owned id
    with pytest.raises(db.DbError) as e:
        new.db_deliver_external_static(10, np.array([cut + 1], np.int32))                    # too late
    assert e.value.code == db.binding.DB_ERANGE
    new.db_deliver_external_static(60, np.zeros(0, np.int32))                                # empty list: no-op
    _same(db, ref, new)
    for s in (ref, new, other):
        s.db_destroy()
