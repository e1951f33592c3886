"""Pins for the oracle's pairing rule (reading R25; "sPEGG accommodates alternative mating
systems (random, shared preference across individuals, or assortative; monogamy or polygynandry)").
-m "not gpu".

With `monogamy` every mother has one mate per time step: the father's draws are addressed by the
mother instead of by the egg.  Pinned by (1) every clutch having exactly one father while the fathers
of different mothers are uniform and independent, (2) the compound-Poisson closed form: the number of
eggs a male fathers has mean lambda under both rules but variance lambda + lambda^2 under monogamy
(he fathers whole clutches of Poisson(lambda) eggs from Poisson(1) mothers) against lambda under
polygynandry, (3) the weighted (R19), sexed (R21) and assortative (R23) rules acting at the level of
the pair, a new partner every step, (4) monogamy = 0 being the unchanged path bit for bit.  A draw
still addressed by the egg, by the laying instead of the drawn mother (R24), or re-used across steps
fails one of them."""
import math

import numpy as np
from scipy import stats

from helpers import cfg, species
from paper_1603_09255_b200 import workloads


def _cfg(n0, L=16, fec_a=4.0, K=1e12, omega=0.0, seed=25, grid=(1, 1), **extra):
    sp = species(L=L, kind="q10", r=0.5, mu=0.0, fec_a=fec_a, K=K, omega=omega,
                 capacity=max(4096, int(n0 * (fec_a + 1.5))))
    sp["monogamy"] = 1
    sp.update(extra)
    c = cfg(sp, seed=seed, grid=grid)
    c["n0"] = [n0]
    c["init_sd"] = 0.1
    return c


def _step(oracle_mod, c, rows=None, sex=None, ps=None):
    o = oracle_mod.Oracle(c)
    rows = workloads.initial_rows(c, 0) if rows is None else rows
    o.write_state(0, rows, ps, 0)
    if sex is not None:
        o.write_sex(0, sex)
    o.step(1)
    return o, o.debug(0), rows


def test_one_father_per_clutch_and_compound_poisson_variance(oracle_mod):
    n0, lam = 20000, 4.0
    c = _cfg(n0, fec_a=lam)
    o, d, _ = _step(oracle_mod, c)
    mo, fa = d["mother"], d["father"]
    # (1) one father per mother
    first = np.full(n0, -1, np.int64)
    first[mo[::-1]] = fa[::-1]
    assert np.array_equal(fa, first[mo])
    mothers = np.unique(mo)
    pair = first[mothers]
    # fathers of different mothers: uniform over the adults, independent of the mother's index
    cnt = np.bincount(pair % 50, minlength=50)
    assert ((cnt - cnt.mean()) ** 2 / cnt.mean()).sum() < stats.chi2.ppf(1 - 1e-4, 49)
    assert abs(np.corrcoef(mothers, pair)[0, 1]) < 5 / math.sqrt(len(mothers))
    # the father of mother i is the uniform index on word 0 of block 0 of stream PAIR (8), entity i
    for i in mothers[:: max(1, len(mothers) // 40)]:
        x = oracle_mod.draw(c["seed"], 0, 8, int(i), 0, 0)
        assert (int(x[0]) * n0) >> 32 == first[i]
    # (2) eggs fathered per male: mean lambda, variance lambda + lambda^2 (polygynandry: lambda)
    per_male = np.bincount(fa, minlength=n0).astype(np.float64)
    assert abs(per_male.mean() - lam) < 5 * math.sqrt(lam / n0) * 2
    v_mono = per_male.var()
    c0 = _cfg(n0, fec_a=lam)
    c0["species"][0]["monogamy"] = 0
    _, d0, _ = _step(oracle_mod, c0)
    v_poly = np.bincount(d0["father"], minlength=n0).astype(np.float64).var()
    assert abs(v_poly / lam - 1) < 0.06
    assert abs(v_mono / (lam + lam * lam) - 1) < 0.08
    # same eggs, same mothers: only the fathers differ between the two rules
    assert d0["m_t"] == d["m_t"] and np.array_equal(d0["mother"], mo) and not np.array_equal(d0["father"], fa)


def test_pair_level_weights_sexes_assortment_and_new_partner_each_step(oracle_mod):
    # R19 at the level of the pair: classes 0, 1, 2 with v = ln 2 are CHOSEN BY MOTHERS 1 : 2 : 4
    n0 = 3000
    c = _cfg(n0, fec_a=3.0, mate_skew=math.log(2.0))
    rows = np.zeros((n0, 32), np.int16)
    rows[:, 0] = 1024 * (np.arange(n0) % 3)
    rows[:, 16] = 1024 * (np.arange(n0) % 3)
    o, d, _ = _step(oracle_mod, c, rows=rows)
    first = np.full(n0, -1, np.int64)
    first[d["mother"][::-1]] = d["father"][::-1]
    assert np.array_equal(d["father"], first[d["mother"]])
    pair = first[np.unique(d["mother"])]
    cls = np.bincount(pair % 3, minlength=3)
    expect = len(pair) * np.array([1.0, 2.0, 4.0]) / 7.0
    assert ((cls - expect) ** 2 / expect).sum() < stats.chi2.ppf(1 - 1e-4, 2)
    # R21: the one mate is a male; R24 + R25: the pair belongs to the DRAWN mother
    c = _cfg(2000, fec_a=6.0, separate_sexes=1, mother_skew=1.0)
    sex = (np.arange(2000) % 2).astype(np.uint8)
    o, d, _ = _step(oracle_mod, c, sex=sex)
    assert (sex[d["father"]] == 1).all() and (sex[d["mother"]] == 0).all()
    first = np.full(2000, -1, np.int64)
    first[d["mother"][::-1]] = d["father"][::-1]
    assert np.array_equal(d["father"], first[d["mother"]])
    # R23: assortment at the level of the pair (positive father-mother correlation, one father per clutch)
    c = _cfg(6000, L=64, fec_a=3.0, assort=8.0)
    o, d, rows = _step(oracle_mod, c)
    z = rows.astype(np.int64).sum(axis=1) * 2.0 ** -11
    first = np.full(6000, -1, np.int64)
    first[d["mother"][::-1]] = d["father"][::-1]
    assert np.array_equal(d["father"], first[d["mother"]])
    m = np.unique(d["mother"])
    assert np.corrcoef(z[m], z[first[m]])[0, 1] > 0.2
    # a new partner every step: with overlapping generations a staying mother re-pairs
    c = _cfg(3000, fec_a=2.0, K=3000.0, adult_survival=0.9)
    c["species"][0]["capacity"] = 65536
    o = oracle_mod.Oracle(c)
    rows = workloads.initial_rows(c, 0)
    o.write_state(0, rows, None, 0)
    o.step(1)
    d1 = o.debug(0)
    stay = np.where(d1["a_alive"])[0]
    o.step(1)
    d2 = o.debug(0)
    f1 = np.full(3000, -1, np.int64); f1[d1["mother"][::-1]] = d1["father"][::-1]
    n2 = d2["n_t"]
    f2 = np.full(n2, -1, np.int64); f2[d2["mother"][::-1]] = d2["father"][::-1]
    # staying adult number k (old index stay[k]) is adult k of step 2; compare the row of the partner
    both = [(i, k) for k, i in enumerate(stay) if f1[i] >= 0 and f2[k] >= 0]
    assert len(both) > 300
    same = sum(1 for i, k in both if d1["a_alive"][f1[i]] and np.searchsorted(stay, f1[i]) == f2[k])
    assert same < 0.02 * len(both) + 5                    # chance level ~ 1/N, not "always"


def test_monogamy_off_is_the_unchanged_path(oracle_mod):
    a, b = workloads.config(2, scale=0.02), workloads.config(2, scale=0.02)
    b["species"][0]["monogamy"] = 0
    oa, ob = oracle_mod.Oracle(a), oracle_mod.Oracle(b)
    for x, cc in ((oa, a), (ob, b)):
        x.write_state(0, workloads.initial_rows(cc, 0), None, 0)
        x.step(3)
    assert oa.log(0) == ob.log(0) and np.array_equal(oa.read_state(0)[0], ob.read_state(0)[0])
