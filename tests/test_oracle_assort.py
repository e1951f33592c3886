"""Pins for the oracle's assortative mating (reading R23; "alternative mating systems
(random, shared preference across individuals, or assortative ...)").  -m "not gpu".

Rejection sampling with a cap of 8 candidates has an exact closed form on a two-class population
built by hand (a truncated geometric), and for a Gaussian trait the father's value regresses on the
mother's with slope 2aV / (1 + 2aV) (product of two Gaussians; the cap of 8 candidates matters
little while acceptance is common).  a = 0 is random mating, bit for bit."""
import math

import numpy as np

from helpers import cfg, species
from paper_1603_09255_b200 import workloads


def _cfg(n0, a, L=16, fec_a=4.0, seed=23, grid=(1, 1)):
    sp = species(L=L, kind="q10", r=0.5, mu=0.0, fec_a=fec_a, K=1e12, omega=0.0, capacity=max(4096, int(n0 * (fec_a + 2))))
    sp["assort"] = a
    c = cfg(sp, seed=seed, grid=grid)
    c["n0"] = [n0]
    c["init_sd"] = 0.1
    return c


def test_two_classes_by_hand(oracle_mod):
    """Half the adults at z = 0, half at z = 1, a = ln 4: a candidate of the mother's class is always
    accepted, one of the other class with probability q = 1/4.  A try ends the search with
    probability s = (1 + q)/2; the father is of the mother's class with probability
    (1/2)(1 - r^8)/(1 - r) + r^7 * 0 ... written out below, r = 1 - s, 8 candidates at most."""
    n0 = 4000
    c = _cfg(n0, math.log(4.0), fec_a=6.0)
    rows = np.zeros((n0, 32), np.int16)
    rows[1::2, 0] = 1024
    rows[1::2, 16] = 1024
    o = oracle_mod.Oracle(c)
    o.write_state(0, rows, None, 0)
    o.step(1)
    d = o.debug(0)
    same = (d["mother"] % 2) == (d["father"] % 2)
    q, r = 0.25, 1 - (1 + 0.25) / 2
    # accepted within the first 7 tries, or whatever the 8th candidate is:
    p_same = sum(r ** t * 0.5 for t in range(7)) + r ** 7 * 0.5
    assert abs(p_same - (0.5 * (1 - r ** 7) / (1 - r) + 0.5 * r ** 7)) < 1e-12
    m = d["m_t"]
    assert m > 20000
    assert abs(same.mean() - p_same) < 4.5 * math.sqrt(p_same * (1 - p_same) / m)
    assert abs(p_same - 0.8) < 0.001                      # = 1/(1+q) up to the r^7 term: not 1/2 (random mating)
    # candidates are uniform: within the mother's class every adult is equally likely to father
    cnt = np.bincount(d["father"][same & (d["mother"] % 2 == 0)], minlength=n0)[0::2].astype(np.float64)
    assert abs(cnt.std() / math.sqrt(cnt.mean()) - 1) < 0.1
    # mothers and everything else drawn for the newborn are those of random mating
    c0 = _cfg(n0, 0.0, fec_a=6.0)
    o0 = oracle_mod.Oracle(c0)
    o0.write_state(0, rows, None, 0)
    o0.step(1)
    d0 = o0.debug(0)
    for k in ("f", "mother", "u01", "dest"):
        assert np.array_equal(d[k], d0[k]), k
    assert abs(((d0["mother"] % 2) == (d0["father"] % 2)).mean() - 0.5) < 4.5 * 0.5 / math.sqrt(m)


def test_regression_of_father_on_mother(oracle_mod):
    n0, a = 30000, 1.0
    c = _cfg(n0, a, L=64, fec_a=3.0)
    rows = workloads.initial_rows(c, 0)
    o = oracle_mod.Oracle(c)
    o.write_state(0, rows, None, 0)
    o.step(1)
    d = o.debug(0)
    z = rows.astype(np.int64).sum(axis=1) * 2.0 ** -11
    V = z.var()
    zm, zf = z[d["mother"]], z[d["father"]]
    slope = np.cov(zm, zf)[0, 1] / zm.var()
    expect = 2 * a * V / (1 + 2 * a * V)
    assert abs(slope - expect) < 0.03, (slope, expect)     # cap of 8 candidates: a little below the unlimited form
    assert slope > 0.25
    # no fecundity or viability selection: the offspring mean stays, the offspring variance grows
    zo = d["zi"].astype(np.float64) * 2.0 ** -11
    assert abs(zo.mean() - z.mean()) < 4.5 * math.sqrt(V / len(zo)) * 1.5


def test_patches_and_zero(oracle_mod):
    n0 = 4000
    c = _cfg(n0, 2.0, grid=(2, 2))
    rows = workloads.initial_rows(c, 0)
    ps = workloads.initial_patch_start(c, 0)
    o = oracle_mod.Oracle(c)
    o.write_state(0, rows, ps, 0)
    o.step(1)
    d = o.debug(0)
    pm = np.searchsorted(ps, d["mother"], side="right") - 1
    pf = np.searchsorted(ps, d["father"], side="right") - 1
    assert np.array_equal(pm, pf)
    a, b = workloads.config(1), workloads.config(1)
    b["species"][0]["assort"] = 0.0
    outs = []
    for c_ in (a, b):
        o_ = oracle_mod.Oracle(c_)
        o_.write_state(0, workloads.initial_rows(c_, 0), None, 0)
        o_.step(3)
        outs.append(o_)
    assert outs[0].log(0) == outs[1].log(0) and np.array_equal(outs[0].read_state(0)[0], outs[1].read_state(0)[0])
