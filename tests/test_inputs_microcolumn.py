"""The cortical micro-column workload (Extended Data Table 3) as a synthetic CSR recipe
(db_inputs.microcolumn_csr): the recipe reproduces the table's proportions and the paper's rule for the voxel's mean
in-degree, and the oracle runs it.  Host logic only (no GPU)."""
import numpy as np
import pytest

import db_inputs

VOX, NV, DIN = 2500, 3, 100


@pytest.fixture(scope="module")
def net():
    return db_inputs.microcolumn_csr(NV, VOX, DIN, seed=11)


def _edges(net):
    src = np.repeat(np.arange(net["N"]), np.diff(net["row_ptr"]))
    return src, net["tgt"].astype(np.int64)


def test_table_as_printed():
    T = db_inputs.MC_TABLE3
    assert T.shape == (10, 10)
    # a few cells and the row sums of the printed table
    assert T[0, 9] == 10133 and T[2, 1] == 3554 and T[4, 7] == 1686 and T[9, 8] == 499 and T[5, 0] == 0
    assert T.sum(axis=1).tolist() == [12504, 8526, 7004, 3529, 5642, 3229, 6908, 2966, 6020, 2722]


def test_sizes_and_mean_indegree():
    s = db_inputs.microcolumn_sizes(VOX)
    assert s.sum() == VOX and np.all(s[0::2] == 4 * s[1::2])          # 80 / 20 in every layer
    K = db_inputs.microcolumn_indegrees(VOX, DIN)
    mean = (s * K.sum(axis=1)).sum() / s.sum()
    assert abs(mean - DIN) < 0.5                                        # the voxel's mean in-degree is d_in
    ratio = K[db_inputs.MC_TABLE3 > 200] / db_inputs.MC_TABLE3[db_inputs.MC_TABLE3 > 200]
    assert ratio.max() / ratio.min() < 1.25                             # one scale factor (up to rounding)


def test_csr_structure_follows_the_table(net):
    src, tgt = _edges(net)
    assert net["E"] == len(tgt) and net["row_ptr"][-1] == net["E"]
    s = db_inputs.microcolumn_sizes(VOX)
    pop_of = np.repeat(np.arange(10), s)
    K = db_inputs.microcolumn_indegrees(VOX, DIN)
    sv, tv = src // VOX, tgt // VOX
    sp, tp = pop_of[src % VOX], pop_of[tgt % VOX]
    intra = sv == tv
    # in-degree of every neuron from every population of its own voxel = the scaled table cell, exactly
    pre_pop = [db_inputs.MC_POPS.index(q) for q in db_inputs.MC_PRE[:9]]
    cnt = np.zeros((net["N"], 10), np.int64)
    np.add.at(cnt, (tgt[intra], sp[intra]), 1)
    for p in range(10):
        rows = cnt[np.tile(pop_of == p, NV)]
        for c, q in enumerate(pre_pop):
            assert np.all(rows[:, q] == K[p][c]), (p, q)
        assert np.all(rows[:, 0] == 0)                                  # nobody receives from e1 inside the voxel
    # cortico-cortical share: from excitatory neurons of OTHER voxels, K[p][CC] per neuron
    cc = np.bincount(tgt[~intra], minlength=net["N"])
    assert np.array_equal(cc, np.tile(K[:, 9][pop_of], NV))
    assert np.all(net["ntype"][src[~intra]] == 0)
    # receptors by source type, delays by kind, rows sorted by target
    inh = net["ntype"][src] == 1
    assert np.all((net["rec"] >= 2) == inh)
    assert net["delay"][intra].max() <= 8 and net["delay"][~intra].min() >= 10 and net["delay"].min() >= 1
    assert np.all(net["w"] >= 0) and net["w"][~inh].max() <= 0.008 and net["w"][inh].max() <= 0.032
    same_row = src[1:] == src[:-1]
    assert np.all(tgt[1:][same_row] >= tgt[:-1][same_row])
    assert tp.max() == 9


def test_oracle_runs_the_microcolumn_in_the_papers_rate_range(net):
    import oracle
    t = db_inputs.type_params(bg_weight=0.0072)
    sim = db_inputs.sim_params(types=[t, dict(t)], D=32)
    o = oracle.OracleSim(sim, net, db_inputs.DYN_SEED)
    o.step(1500)
    c = o.counters()
    rate = c["spikes"] / net["N"] / 0.15
    assert 5.0 < rate < 30.0                                            # the paper's operating range
    st, ids = o.spikes()
    assert c["events"] == int(np.diff(net["row_ptr"])[ids].sum())
