"""Pins for the oracle's separate sexes (reading R21; eqs. S2-9/S2-10: "For each egg,
the mother and father are drawn at random from mature males and females in the population").
-m "not gpu".

Pinned by the definitions themselves on hand-built populations: only females lay eggs (Poisson mean
lambda each), only males father them (one male: he fathers everything; v_m = 0: uniform over the
males; v_m != 0: R19's weights among the males only), sex at birth is a fair coin independent of
everything else drawn for the newborn, and the sex travels with the individual through the
compaction (patches, overlapping generations).  The two-sex Beverton-Holt balance closes the loop."""
import math

import numpy as np
from scipy import stats

from helpers import cfg, species
from paper_1603_09255_b200 import workloads


def _cfg(n0, v=0.0, L=16, fec_a=4.0, K=1e12, omega=0.0, capacity=None, grid=(1, 1), seed=21, migration=0.0, sA=0.0):
    sp = species(L=L, kind="q10", r=0.5, mu=0.0, fec_a=fec_a, K=K, omega=omega, migration=migration,
                 capacity=capacity or max(4096, int(n0 * (fec_a + 1.5))))
    sp["separate_sexes"] = 1
    sp["mate_skew"] = v
    sp["adult_survival"] = sA
    c = cfg(sp, seed=seed, grid=grid)
    c["n0"] = [n0]
    c["init_sd"] = 0.1
    return c


def _start(oracle_mod, c, sex, rows=None):
    o = oracle_mod.Oracle(c)
    rows = workloads.initial_rows(c, 0) if rows is None else rows
    o.write_state(0, rows, workloads.initial_patch_start(c, 0), 0)
    o.write_sex(0, sex)
    return o, rows


def test_only_females_lay_and_only_males_father(oracle_mod):
    n0 = 6000
    c = _cfg(n0, fec_a=4.0)
    sex = (np.arange(n0) % 3 == 0).astype(np.uint8)          # every third adult is male
    o, rows = _start(oracle_mod, c, sex)
    o.step(1)
    d = o.debug(0)
    f = d["f"].astype(np.float64)
    assert f[sex == 1].sum() == 0
    nf = (sex == 0).sum()
    assert abs(f[sex == 0].mean() - 4.0) < 4.5 * math.sqrt(4.0 / nf)     # Poisson(lambda = R0) per female
    assert (sex[d["mother"]] == 0).all() and (sex[d["father"]] == 1).all()
    # v_m = 0: uniform over the males
    cnt = np.bincount(d["father"], minlength=n0)[sex == 1].astype(np.float64)
    assert ((cnt - cnt.mean()) ** 2 / cnt.mean()).sum() < stats.chi2.ppf(1 - 1e-4, len(cnt) - 1)
    # the running sum steps at males only, by the same amount
    w = np.diff(np.concatenate([[0], d["mate_cum"].astype(np.float64)]))
    assert (w[sex == 0] == 0).all() and len(set(w[sex == 1])) == 1 and w[sex == 1][0] == 123733.0
    # sex at birth: a fair coin, independent of the survival uniform and of the mother
    so = d["sex_off"].astype(np.float64)
    m = d["m_t"]
    assert abs(so.mean() - 0.5) < 4.5 * 0.5 / math.sqrt(m)
    assert abs(np.corrcoef(so, d["u01"])[0, 1]) < 5 / math.sqrt(m)
    assert abs(np.corrcoef(so[1:], so[:-1])[0, 1]) < 5 / math.sqrt(m)
    # the sex travels with the individual: next adults = surviving offspring in order
    assert np.array_equal(o.read_sex(0), d["sex_off"][d["alive"].astype(bool)])


def test_one_male_fathers_everything_and_no_male_falls_back(oracle_mod):
    n0 = 400
    c = _cfg(n0, fec_a=3.0)
    sex = np.zeros(n0, np.uint8)
    sex[137] = 1
    o, _ = _start(oracle_mod, c, sex)
    o.step(1)
    d = o.debug(0)
    assert d["m_t"] > 900 and (d["father"] == 137).all() and d["f"][137] == 0
    # nobody is male: the patch is treated as hermaphroditic (R2's uniform mate)
    o, _ = _start(oracle_mod, c, np.zeros(n0, np.uint8))
    o.step(1)
    d = o.debug(0)
    cnt = np.bincount(d["father"], minlength=n0).astype(np.float64)
    assert ((cnt - cnt.mean()) ** 2 / cnt.mean()).sum() < stats.chi2.ppf(1 - 1e-4, n0 - 1)
    # everybody is male: no eggs, the population ends
    o, _ = _start(oracle_mod, c, np.ones(n0, np.uint8))
    o.step(1)
    assert o.log(0)[0]["m_t"] == 0 and o.n(0) == 0


def test_weighted_among_males_only(oracle_mod):
    """R19's weights, restricted to the males: the fathers' mean is sum_{males} w z / sum_{males} w."""
    n0, v = 20000, 2.0
    c = _cfg(n0, v=v, L=64, fec_a=4.0)
    rng = np.random.default_rng(5)
    sex = rng.integers(0, 2, n0).astype(np.uint8)
    o, rows = _start(oracle_mod, c, sex)
    o.step(1)
    d = o.debug(0)
    z = rows.astype(np.int64).sum(axis=1) * 2.0 ** -11
    w = np.exp(v * (z - z.mean())) * sex
    expect = (w * z).sum() / w.sum()
    Vf = (w * (z - expect) ** 2).sum() / w.sum()
    zf = z[d["father"]]
    assert (sex[d["father"]] == 1).all()
    assert abs(zf.mean() - expect) < 4.5 * math.sqrt(Vf / len(zf))
    assert zf.mean() - z.mean() > 20 * math.sqrt(z.var() / len(zf))


def test_sex_through_patches_and_overlapping_generations(oracle_mod):
    # patches: fathers are males of the mother's patch; next generation ordered by (dest, j)
    n0 = 4000
    c = _cfg(n0, fec_a=3.0, grid=(2, 2), migration=0.2, capacity=32768)
    rng = np.random.default_rng(7)
    sex = rng.integers(0, 2, n0).astype(np.uint8)
    o, _ = _start(oracle_mod, c, sex)
    ps = workloads.initial_patch_start(c, 0)
    o.step(1)
    d = o.debug(0)
    pm = np.searchsorted(ps, d["mother"], side="right") - 1
    pf = np.searchsorted(ps, d["father"], side="right") - 1
    assert np.array_equal(pm, pf) and (sex[d["father"]] == 1).all() and (sex[d["mother"]] == 0).all()
    alive = np.flatnonzero(d["alive"])
    order = alive[np.argsort(d["dest"][alive], kind="stable")]
    assert np.array_equal(o.read_sex(0), d["sex_off"][order])
    # overlapping generations: the staying adults keep their sex, in front of the newborns
    c = _cfg(3000, fec_a=1.0, sA=0.7, capacity=32768)
    sex = rng.integers(0, 2, 3000).astype(np.uint8)
    o, _ = _start(oracle_mod, c, sex)
    o.step(1)
    d = o.debug(0)
    stay = d["a_alive"].astype(bool)
    assert np.array_equal(o.read_sex(0), np.concatenate([sex[stay], d["sex_off"][d["alive"].astype(bool)]]))


def test_two_sex_balance_and_hermaphrodite_default(oracle_mod):
    """Half the adults lay eggs: N' = (N/2) R0 / (1 + N/K)  =>  N* = K (R0/2 - 1)."""
    c = _cfg(2000, fec_a=6.0, K=1000.0, capacity=16384)
    rng = np.random.default_rng(9)
    o, _ = _start(oracle_mod, c, rng.integers(0, 2, 2000).astype(np.uint8))
    o.step(80)
    N = np.array([e["n_t"] for e in o.log(0)[30:]], dtype=np.float64)
    assert abs(N.mean() / 2000.0 - 1) < 0.04
    assert abs(o.read_sex(0).mean() - 0.5) < 0.06
    # separate_sexes = 0 is bit-identical to a configuration without the field
    a, b = workloads.config(1), workloads.config(1)
    b["species"][0]["separate_sexes"] = 0
    outs = []
    for c_ in (a, b):
        o_ = oracle_mod.Oracle(c_)
        o_.write_state(0, workloads.initial_rows(c_, 0), None, 0)
        o_.step(3)
        outs.append(o_)
    assert outs[0].log(0) == outs[1].log(0) and np.array_equal(outs[0].read_state(0)[0], outs[1].read_state(0)[0])
    assert (outs[0].read_sex(0) == 0).all()
