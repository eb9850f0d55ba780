"""Pins of the oracle's network generator: invariants the paper fixes (P:L322-331,
P:L414-417: fixed in-degree, no autapses, no multapses, receptor class follows the
source type, 80/20 exc/inh) and the distributions BASELINE.json names.  CPU only."""
import math

import numpy as np
import pytest
from scipy import stats

import db_inputs


def _src_of(net):
    return np.repeat(np.arange(net["N"]), np.diff(net["row_ptr"]))


@pytest.fixture(scope="module")
def net0(oracle_mod):
    spec = db_inputs.config(0)["net"]
    return spec, oracle_mod.generate(spec, db_inputs.GEN_SEED)


def test_config0_degrees_and_simple_graph(net0):
    spec, net = net0
    N, K = spec["N"], spec["K"]
    assert net["E"] == N * K
    src, tgt = _src_of(net), net["tgt"].astype(np.int64)
    assert np.all(np.bincount(tgt, minlength=N) == K)          # fixed in-degree
    assert not np.any(src == tgt)                               # no autapses
    pair = src * N + tgt
    assert len(np.unique(pair)) == len(pair)                    # no multapses
    # rows sorted by target
    same_row = src[1:] == src[:-1]
    assert np.all(tgt[1:][same_row] > tgt[:-1][same_row])
    # out-degree ~ Binomial(N*K draws, 1/N): mean K, variance ~K
    od = np.diff(net["row_ptr"])
    assert abs(od.mean() - K) < 1e-9 and 0.8 * K < od.var() < 1.2 * K


def test_config0_types_receptors_weights_delays(net0):
    spec, net = net0
    N = spec["N"]
    assert net["ntype"][:8000].sum() == 0 and net["ntype"][8000:].sum() == 2000
    src = _src_of(net)
    inh = net["ntype"][src] == 1
    rec = net["rec"]
    assert np.all((rec >= 2) == inh)                            # class follows the source
    for m in (~inh, inh):
        slow = (rec[m] & 1).mean()
        assert abs(slow - 0.2) < 4 * math.sqrt(0.16 / m.sum())  # 80/20 split
    assert abs(inh.mean() - 0.2) < 0.01                         # sources uniform over all neurons
    # weights: exc lognormal(mu=-1, sigma=0.5)*0.01, inh 4x
    lw = np.log(net["w"][~inh].astype(np.float64))
    assert abs(lw.mean() - (math.log(0.01) - 1.0)) < 0.005 and abs(lw.std() - 0.5) < 0.005
    lwi = np.log(net["w"][inh].astype(np.float64))
    assert abs(lwi.mean() - (math.log(0.04) - 1.0)) < 0.01 and abs(lwi.std() - 0.5) < 0.01
    assert stats.kstest((lw - lw.mean()) / lw.std(), "norm").statistic < 0.01
    # delays uniform on 1..20
    d = net["delay"]
    assert d.min() == 1 and d.max() == 20
    cnt = np.bincount(d, minlength=21)[1:]
    chi2 = ((cnt - len(d) / 20) ** 2 / (len(d) / 20)).sum()
    assert chi2 < stats.chi2.ppf(0.9999, 19)
    # attributes are independent of each other
    assert abs(np.corrcoef(d, net["w"])[0, 1]) < 0.01


def test_sources_are_uniform(net0):
    spec, net = net0
    # every neuron is a source equally often: chi-square on out-degrees in 100 bins
    od = np.diff(net["row_ptr"]).reshape(100, -1).sum(1)
    chi2 = ((od - od.mean()) ** 2 / od.mean()).sum()
    assert chi2 < stats.chi2.ppf(0.9999, 99)


def test_generator_is_seeded(oracle_mod):
    spec = db_inputs.config(0, scale=0.05)["net"]
    a = oracle_mod.generate(spec, 1)
    b = oracle_mod.generate(spec, 1)
    c = oracle_mod.generate(spec, 2)
    assert all(np.array_equal(a[k], b[k]) for k in ("row_ptr", "tgt", "w", "delay", "rec"))
    assert not np.array_equal(a["tgt"], c["tgt"])


def test_weight_table_is_the_lognormal_quantile_function(oracle_mod):
    tab = oracle_mod.weight_table(-1.0, 0.5, 0.01)
    q = (np.arange(65536) + 0.5) / 65536
    want = 0.01 * stats.lognorm.ppf(q, s=0.5, scale=math.exp(-1.0))
    assert np.max(np.abs(tab / want - 1)) < 3e-7
    assert np.all(np.diff(tab) >= 0)


def test_fp16_weights(oracle_mod):
    spec = dict(db_inputs.config(0, scale=0.05)["net"], weight_fp16=1)
    net = oracle_mod.generate(spec, 3)
    w = net["w"]
    assert np.array_equal(w, w.astype(np.float16).astype(np.float32))
    ref = oracle_mod.generate(dict(spec, weight_fp16=0), 3)
    assert np.array_equal(ref["w"].astype(np.float16).astype(np.float32), w)


@pytest.fixture(scope="module")
def net_regions(oracle_mod):
    spec = dict(db_inputs.config(2)["net"], N=60_000, n_regions=20, K=50)
    return spec, oracle_mod.generate(spec, db_inputs.GEN_SEED)


def test_regions_structure(oracle_mod, net_regions):
    spec, net = net_regions
    N, R, K = spec["N"], spec["n_regions"], spec["K"]
    rs = net["region_start"]
    sizes = np.diff(rs)
    assert rs[0] == 0 and rs[-1] == N and np.all(sizes > K)
    # lognormal(0, 0.7) sizes, normalised: log-sizes have about that spread
    assert 0.35 < np.log(sizes).std() < 1.1
    assert np.array_equal(sizes, oracle_mod.region_sizes(db_inputs.GEN_SEED, N, R, 0.7))
    for r in range(R):
        nt = net["ntype"][rs[r]:rs[r + 1]]
        ne = int(net["region_nexc"][r])
        assert ne == int(math.floor(0.8 * sizes[r] + 0.5))
        assert nt[:ne].sum() == 0 and nt[ne:].sum() == sizes[r] - ne     # exc first, 80/20
    src, tgt = _src_of(net), net["tgt"].astype(np.int64)
    assert np.all(np.bincount(tgt, minlength=N) == K)
    assert not np.any(src == tgt)
    assert len(np.unique(src * N + tgt)) == len(src)
    rsrc = np.searchsorted(rs, src, side="right") - 1
    rtgt = np.searchsorted(rs, tgt, side="right") - 1
    intra = rsrc == rtgt
    K_intra = int(math.floor(0.8 * K + 0.5))
    assert np.all(np.bincount(tgt[intra], minlength=N) == K_intra)       # 80 % intra-region
    # long-range inputs are excitatory only with delays 20..200 steps; local 1..20
    assert np.all(net["ntype"][src[~intra]] == 0)
    d = net["delay"]
    assert d[~intra].min() == 20 and d[~intra].max() == 200
    assert d[intra].min() == 1 and d[intra].max() == 20
    # the source region follows the row-normalised region matrix
    T = oracle_mod.region_cdf(db_inputs.GEN_SEED, R, 1.0).astype(np.float64)
    cdf = np.concatenate([T / 2.0 ** 32, np.ones((R, 1))], axis=1)
    P = np.diff(np.concatenate([np.zeros((R, 1)), cdf], axis=1), axis=1)
    assert np.allclose(P.sum(1), 1.0) and np.all(np.abs(np.diag(P)) < 1e-9)
    offd = np.log(P[~np.eye(R, dtype=bool)])
    assert 0.8 < offd.std() < 1.2                                        # lognormal(0, 1) entries
    cnt = np.zeros((R, R))
    np.add.at(cnt, (rtgt[~intra], rsrc[~intra]), 1)
    exp = P * cnt.sum(1, keepdims=True)
    m = exp > 5
    chi2 = ((cnt[m] - exp[m]) ** 2 / exp[m]).sum()
    assert chi2 < stats.chi2.ppf(0.9999, m.sum())


def test_outdegree_mode(oracle_mod):
    spec = dict(db_inputs.config(4)["net"], N=4000, outdeg_mean=60.0, outdeg_cap=400)
    net = oracle_mod.generate(spec, 8)
    N = spec["N"]
    od = np.diff(net["row_ptr"])
    assert od.min() >= 1 and od.max() == 400                    # capped
    mu = math.log(60.0) - 0.5
    assert abs(np.log(od[od < 400]).mean() - mu) < 0.08         # lognormal, mean of the law = 60 (R27)
    assert 0.9 < np.log(od).std() < 1.05
    src, tgt = _src_of(net), net["tgt"].astype(np.int64)
    assert not np.any(src == tgt) and len(np.unique(src * N + tgt)) == len(src)
    ind = np.bincount(tgt, minlength=N)                         # targets uniform: in-degree ~ Poisson
    assert abs(ind.var() / ind.mean() - 1) < 0.15
    tab = oracle_mod.outdeg_table(60.0, 1.0, 400)
    q = (np.arange(65536) + 0.5) / 65536
    want = np.clip(np.floor(stats.lognorm.ppf(q, s=1.0, scale=math.exp(mu)) + 0.5), 1, 400)
    assert (tab != want).sum() <= 2                             # rounding ties only


# ---- an independent restatement of the generator's draws ----
def _philox(c, k):
    M0, M1, W0, W1 = 0xD2511F53, 0xCD9E8D57, 0x9E3779B9, 0xBB67AE85
    c = list(c); k = list(k)
    for _ in range(10):
        p0, p1 = M0 * c[0], M1 * c[2]
        c = [(p1 >> 32) ^ c[1] ^ k[0], p1 & 0xFFFFFFFF, (p0 >> 32) ^ c[3] ^ k[1], p0 & 0xFFFFFFFF]
        k = [(k[0] + W0) & 0xFFFFFFFF, (k[1] + W1) & 0xFFFFFFFF]
    return c


def _draw(seed, stream, a, b):
    return _philox([a & 0xFFFFFFFF, (a >> 32) | (stream << 24), b & 0xFFFFFFFF, b >> 32],
                   [seed & 0xFFFFFFFF, seed >> 32])


def test_second_implementation_reproduces_small_network(oracle_mod):
    from test_oracle_pins import _prp_py
    spec = dict(db_inputs.config(0)["net"], N=90, K=11)
    seed = 77
    net = oracle_mod.generate(spec, seed)
    N, K = 90, 11
    n_exc = 72
    wtab = oracle_mod.weight_table(-1.0, 0.5, 0.01)     # pinned above against scipy
    edges = []
    for i in range(N):
        key = _draw(seed, 3, i, 0)
        for k in range(K):
            j = _prp_py(k, N - 1, key)
            j += j >= i
            o = _draw(seed, 4, i, k)
            inh = j >= n_exc
            w = np.float32(wtab[o[0] >> 16]) * (np.float32(4.0) if inh else np.float32(1.0))
            d = 1 + ((o[1] * 20) >> 32)
            rec = (2 if inh else 0) + (1 if o[2] < int(0.2 * 2 ** 32) else 0)
            edges.append((j, i, float(np.float32(w)), d, rec))
    edges.sort()
    assert [e[1] for e in edges] == net["tgt"].tolist()
    assert [e[0] for e in edges] == _src_of(net).tolist()
    assert [e[2] for e in edges] == [float(x) for x in net["w"]]
    assert [e[3] for e in edges] == net["delay"].tolist()
    assert [e[4] for e in edges] == net["rec"].tolist()


def test_owner_edges_match_full_generation(oracle_mod, net_regions):
    spec, net = net_regions
    oe = oracle_mod.OwnerEdges(spec, db_inputs.GEN_SEED)
    src_all = _src_of(net)
    for i in (0, 1, 777, spec["N"] - 1):
        e = oe(i)
        assert np.all(e["tgt"] == i) and len(e["src"]) == spec["K"]
        m = net["tgt"] == i
        order = np.argsort(e["src"], kind="stable")
        assert np.array_equal(src_all[m], e["src"][order])
        assert np.array_equal(net["w"][m], e["w"][order])
        assert np.array_equal(net["delay"][m], e["delay"][order])
        assert np.array_equal(net["rec"][m], e["rec"][order])


def test_impossible_spec_is_rejected(oracle_mod):
    # 200 regions of ~250 neurons cannot supply 160 distinct intra-region sources each
    spec = dict(db_inputs.config(2)["net"], N=50_000)
    with pytest.raises(ValueError):
        oracle_mod.generate(spec, db_inputs.GEN_SEED)
