"""Pins for the oracle's individual-level interspecific encounters (reading R20; "for a
given individual of either species we instead simulate a random subset of possible encounters";
eq. S3-2: per-meeting effect e/(1+e), e = exp(-(x - delta)^2)).  -m "not gpu".

Pinned by populations built by hand: (1) one consumer type, one resource type: capture fraction
1 - (1 - v m)^E; (2) two consumer types, E = 1: credits in the ratio of their matching terms and
total (p1 + p2)/2; (3) bookkeeping: every captured newborn is credited once, to a consumer drawn
uniformly; captured newborns are dead whatever the stabilising term says; (4) E = 0 is R14 bit for
bit.  A dropped factor, an e instead of e/(1+e), a credit to the wrong consumer or a second capture
of the same newborn fails one of them."""
import math

import numpy as np
from scipy import stats

from helpers import cfg, species


def _community(n_prey, n_pred, E, v, omega=0.0, L=16, seed=20, fec=4.0):
    prey = species(L=L, kind="q10", r=0.5, mu=0.0, fecundity="bh", fec_a=fec, K=1e12, omega=omega,
                   capacity=int(n_prey * (fec + 2.5)),
                   predation=dict(attack=v, predator=1, encounters=E))
    pred = species(L=L, kind="q10", r=0.5, mu=0.0, fecundity="captures", fec_a=2.0, K=2.5 * n_pred,
                   gaussian=False, capacity=max(4096, 8 * n_pred))
    c = cfg([prey, pred], seed=seed)
    c["n0"] = [n_prey, n_pred]
    return c


def _rows(n, L, zi):
    """n identical-by-class individuals: genetic value zi[k] (integer quanta) split over locus 0 of both haplotypes"""
    rows = np.zeros((n, 2 * L), np.int16)
    zi = np.broadcast_to(np.asarray(zi), (n,))
    rows[:, 0] = zi // 2
    rows[:, L] = zi - zi // 2
    return rows


def _match(x, delta):
    e = math.exp(-(x - delta) ** 2)
    return e / (1.0 + e)


def test_capture_fraction_one_type(oracle_mod):
    """All consumers at x, all newborns at delta: P(captured) = 1 - (1 - v m)^E, m = e/(1+e)."""
    for (x, delta, E, v) in ((0.0, 0.0, 1, 1.0), (0.5, -0.25, 3, 0.8), (1.0, 0.0, 4, 1.6), (0.0, 0.0, 16, 0.1)):
        n_prey, n_pred = 6000, 500
        c = _community(n_prey, n_pred, E, v)
        o = oracle_mod.Oracle(c)
        o.write_state(0, _rows(n_prey, 16, int(delta * 2048)), None, 0)
        o.write_state(1, _rows(n_pred, 16, int(x * 2048)), None, 0)
        o.step(1)
        d, dp = o.debug(0), o.debug(1)
        m = d["m_t"]
        p = 1.0 - (1.0 - v * _match(x, delta)) ** E
        assert m > 20000
        assert abs(d["captured"].mean() - p) < 4.5 * math.sqrt(p * (1 - p) / m), (x, delta, E, v)
        # every captured newborn is credited exactly once and is dead; nobody else dies (omega = inf)
        assert o.log(0)[0]["captures"] == d["captured"].sum() == dp["cap"].sum()
        assert np.array_equal(d["alive"], 1 - d["captured"])
        # the consumers met are uniform over the consumer population
        cnt = dp["cap"].astype(np.float64)
        assert ((cnt - cnt.mean()) ** 2 / cnt.mean()).sum() < stats.chi2.ppf(1 - 1e-4, n_pred - 1)


def test_credit_goes_to_the_consumer_met(oracle_mod):
    """Two consumer types (even rows matched, odd rows 1.5 units off), E = 1: a newborn meets either
    type with probability 1/2, so the types are credited p1/2 and p2/2 per newborn: the matched
    consumers collect m1 / m2 times as many captures -- the selection on the consumer trait."""
    n_prey, n_pred, v = 8000, 400, 1.0
    c = _community(n_prey, n_pred, 1, v)
    o = oracle_mod.Oracle(c)
    o.write_state(0, _rows(n_prey, 16, 0), None, 0)
    o.write_state(1, _rows(n_pred, 16, np.where(np.arange(n_pred) % 2 == 0, 0, 3072)), None, 0)
    o.step(1)
    d, dp = o.debug(0), o.debug(1)
    m = d["m_t"]
    p1, p2 = v * _match(0.0, 0.0), v * _match(1.5, 0.0)
    c1, c2 = dp["cap"][0::2].sum(), dp["cap"][1::2].sum()
    assert abs(c1 - m * p1 / 2) < 4.5 * math.sqrt(m * p1 / 2)
    assert abs(c2 - m * p2 / 2) < 4.5 * math.sqrt(m * p2 / 2)
    assert c1 > 3 * c2                                  # m1/m2 = 0.5/0.0953 = 5.2
    assert abs(d["captured"].mean() - (p1 + p2) / 2) < 4.5 * math.sqrt(0.25 / m)
    # e/(1+e), not e: a matched meeting captures with probability v/2
    assert abs(p1 - 0.5) < 1e-12
    # consumer fecundity follows its captures (R14's table): nobody without a capture reproduces
    f, cap = dp["f"].astype(np.float64), dp["cap"]
    assert f[cap == 0].sum() == 0 and f[cap > 0].sum() > 0


def test_with_stabilising_selection_and_first_capture_stops(oracle_mod):
    """The stabilising term is separate: alive iff not captured and u01 < s; s is the Gaussian term
    alone.  With v m = 1 the first meeting captures: more meetings change nothing."""
    n_prey, n_pred = 5000, 300
    res = []
    for E in (1, 5):
        c = _community(n_prey, n_pred, E, 2.0, omega=1.0)
        o = oracle_mod.Oracle(c)
        o.write_state(0, _rows(n_prey, 16, 1024), None, 0)       # delta = 0.5
        o.write_state(1, _rows(n_pred, 16, 1024), None, 0)       # x = 0.5: m = 1/2, v m = 1
        o.step(1)
        d, dp = o.debug(0), o.debug(1)
        assert d["captured"].all() and not d["alive"].any()
        assert np.allclose(d["s"], math.exp(-0.125), rtol=1e-6)
        assert dp["cap"].sum() == d["m_t"]
        res.append(dp["cap"].copy())
    assert np.array_equal(res[0], res[1])                        # meetings 2..5 never happen
    # half-strength: captured and stabilising deaths are independent
    c = _community(20000, 300, 2, 0.6, omega=1.0)
    o = oracle_mod.Oracle(c)
    o.write_state(0, _rows(20000, 16, 1024), None, 0)
    o.write_state(1, _rows(300, 16, 0), None, 0)
    o.step(1)
    d = o.debug(0)
    capd, ok = d["captured"].astype(bool), d["u01"] < d["s"]
    assert np.array_equal(d["alive"].astype(bool), ~capd & ok)
    pc = 1 - (1 - 0.6 * _match(0.0, 0.5)) ** 2
    assert abs(capd.mean() - pc) < 4.5 * math.sqrt(pc * (1 - pc) / d["m_t"])
    assert abs((capd & ok).mean() - pc * math.exp(-0.125)) < 4.5 * math.sqrt(0.25 / d["m_t"])


def test_zero_encounters_is_the_mean_field_term(oracle_mod):
    from paper_1603_09255_b200 import workloads
    a, b = workloads.config(4, scale=0.003), workloads.config(4, scale=0.003)
    b["species"][0]["predation"]["encounters"] = 0
    outs = []
    for c in (a, b):
        o = oracle_mod.Oracle(c)
        for s in range(2):
            o.write_state(s, workloads.initial_rows(c, s), None, 0)
        o.step(3)
        outs.append(o)
    for s in range(2):
        assert outs[0].log(s) == outs[1].log(s)
        assert np.array_equal(outs[0].read_state(s)[0], outs[1].read_state(s)[0])
    # no consumers: nobody is met
    c = _community(500, 4, 3, 1.0)
    o = oracle_mod.Oracle(c)
    o.write_state(0, _rows(500, 16, 0), None, 0)
    o.step(1)
    assert o.log(0)[0]["captures"] == 0 and o.debug(0)["alive"].all()
