"""Pins for the oracle's mean-field predation term (reading R14, eqs. S3-1 / S3-2 are
what R14 stands in for): s_pred(z) = exp(-a N_C exp(-(z - zbar_C)^2 / 2)), a captured newborn is credited
to a uniformly drawn consumer.  -m "not gpu".

Everything expected here is computed from the INPUT rows and the parameters, never from the oracle's own
debug scalars (zbar_pred, attack_n): populations are built by hand so that the consumers' mean, the
resource's mean, the two phenotype scales and the two population sizes all differ, and a formula that took
any of them from the wrong species lands many standard errors away.  Mutants these tests were written to
kill (each was applied to a copy of oracle/spegg_oracle.cpp and turned this file red):
  M1  zbar_C from the prey's own mean            (sumzi0[si] / N0[si] instead of [pr])
  M2  zbar_C scaled by the prey's pheno_scale    (S.p.pheno_scale instead of sim.sp[pr].p.pheno_scale)
  M3  a * N of the prey instead of a * N_C
  M4  credit to consumer j % N_C                 (instead of the uniform draw)
  M5  credit to consumer 0 / a fixed consumer
"""
import math

import numpy as np
from scipy import stats

from helpers import cfg, species

L = 16
PREY_SCALE, PRED_SCALE = 2.0 ** -11, 2.0 ** -10      # different on purpose (mutant M2)


def _community(n_prey, n_pred, attack, fec=4.0, seed=31, omega=0.0):
    prey = species(L=L, kind="q10", r=0.5, mu=0.0, fecundity="bh", fec_a=fec, K=1e12, omega=omega,
                   capacity=int(n_prey * (fec + 2.5)) + 4096, pheno_scale=PREY_SCALE,
                   predation=dict(attack=attack, predator=1, encounters=0))
    pred = species(L=L, kind="q10", r=0.5, mu=0.0, fecundity="captures", fec_a=2.0, K=2.5 * n_pred,
                   gaussian=False, capacity=max(4096, 8 * n_pred), pheno_scale=PRED_SCALE)
    c = cfg([prey, pred], seed=seed)
    c["n0"] = [n_prey, n_pred]
    return c


def _rows(n, zi):
    """n individuals with integer genetic value zi[k] (EVEN quanta), half on locus 0 of each haplotype: with
    mu = 0 every gamete of such a parent carries zi/2, so a population of one type breeds true."""
    zi = np.broadcast_to(np.asarray(zi, dtype=np.int64), (n,))
    assert np.all(zi % 2 == 0)
    rows = np.zeros((n, 2 * L), np.int16)
    rows[:, 0] = zi // 2
    rows[:, L] = zi // 2
    return rows


def _step(oracle_mod, c, prey_rows, pred_rows):
    o = oracle_mod.Oracle(c)
    o.write_state(0, prey_rows, None, 0)
    o.write_state(1, pred_rows, None, 0)
    o.step(1)
    return o


def _p_capture(a, n_c, z, zbar_c):
    return 1.0 - math.exp(-a * n_c * math.exp(-0.5 * (z - zbar_c) ** 2))


def test_predation_term_uses_the_consumers_mean_count_and_scale(oracle_mod):
    """All consumers at trait x, all newborns at delta != x, no stabilising term: the captured fraction
    is 1 - exp(-a N_C exp(-(delta - x)^2 / 2)) with x, N_C taken from the rows that were loaded."""
    cases = [  # (n_prey, n_pred, a*N_C, delta quanta (prey scale), x quanta (predator scale))
        (6000, 500, 0.8, 0, 1024),        # delta = 0,    x = 1.0
        (6000, 250, 0.8, -1024, 512),     # delta = -0.5, x = 0.5   (half the consumers, same a*N_C)
        (6000, 400, 1.6, 2048, 0),        # delta = 1.0,  x = 0
        (5000, 5000, 0.5, 0, -1536),      # delta = 0,    x = -1.5  (as many consumers as adults)
    ]
    for n_prey, n_pred, A, dq, xq in cases:
        a = A / n_pred
        c = _community(n_prey, n_pred, a)
        o = _step(oracle_mod, c, _rows(n_prey, dq), _rows(n_pred, xq))
        d = o.debug(0)
        m = d["m_t"]
        assert m > 18000
        delta, x = dq * PREY_SCALE, xq * PRED_SCALE
        p = _p_capture(a, n_pred, delta, x)
        se = math.sqrt(p * (1 - p) / m)
        frac = d["captured"].mean()
        assert abs(frac - p) < 4.5 * se, (n_prey, n_pred, frac, p)
        # ... and is NOT what the wrong mean (the prey's own: M1), the wrong scale (M2) or the wrong
        # count (M3) would give: each alternative is far outside the band
        for wrong in (_p_capture(a, n_pred, delta, delta),                      # M1
                      _p_capture(a, n_pred, delta, xq * PREY_SCALE),            # M2
                      _p_capture(a, n_prey, delta, x)):                          # M3
            if abs(wrong - p) > 12 * se:
                assert abs(frac - wrong) > 6 * se
        # omega = inf: the predation term is the whole survival probability; captured <=> dead
        assert np.array_equal(d["alive"], 1 - d["captured"])
        assert np.max(np.abs(d["s"].astype(np.float64) - (1 - p))) < 2e-6
        assert o.log(0)[0]["captures"] == d["captured"].sum() == o.debug(1)["cap"].sum()
    # the alternatives above are distinguishable in every case for M1 and in at least one for M2, M3
    a = 0.8 / 500
    assert abs(_p_capture(a, 500, 0.0, 0.0) - _p_capture(a, 500, 0.0, 1.0)) > 0.1
    assert abs(_p_capture(0.8 / 250, 250, -0.5, 512 * PREY_SCALE) - _p_capture(0.8 / 250, 250, -0.5, 0.5)) > 0.05
    assert abs(_p_capture(a, 6000, 0.0, 1.0) - _p_capture(a, 500, 0.0, 1.0)) > 0.3


def test_predation_term_uses_the_mean_over_consumers_of_mixed_types(oracle_mod):
    """Consumers of two types, 3/4 at x1 and 1/4 at x2: the term is evaluated at their MEAN (mean-field),
    zbar_C = (3 x1 + x2) / 4 from the loaded rows -- not at either type, not at the resource's mean."""
    n_prey, n_pred, A = 6000, 400, 1.2
    x1q, x2q = 0, 2048                                      # 0 and 2.0 in the predator's units
    xq = np.where(np.arange(n_pred) % 4 == 3, x2q, x1q)
    zbar = float(xq.astype(np.float64).sum() / n_pred * PRED_SCALE)
    assert abs(zbar - 0.5) < 1e-12
    c = _community(n_prey, n_pred, A / n_pred)
    o = _step(oracle_mod, c, _rows(n_prey, -1024), _rows(n_pred, xq))     # newborns at -0.5
    d = o.debug(0)
    p = _p_capture(A / n_pred, n_pred, -0.5, zbar)
    se = math.sqrt(p * (1 - p) / d["m_t"])
    assert abs(d["captured"].mean() - p) < 4.5 * se
    for wrong_mean in (0.0, 2.0, -0.5):
        assert abs(d["captured"].mean() - _p_capture(A / n_pred, n_pred, -0.5, wrong_mean)) > 6 * se


def test_mean_field_capture_is_credited_to_a_uniform_consumer(oracle_mod):
    """Who gets the capture.  (1) Many more captures than consumers: the counts are a uniform multinomial
    (chi-square, and no trend along the consumer index).  (2) FEWER captures than consumers, everyone
    captured: under a uniform draw the number of distinct consumers credited follows the occupancy law
    N_C (1 - (1 - 1/N_C)^M) and several consumers are credited twice; an index that is a function of j
    (j % N_C: mutant M4) credits M distinct consumers, all of them in the first M slots; a fixed consumer
    (M5) credits one."""
    # (1) a*N_C = 3 at the matched trait: 95 % captured
    n_prey, n_pred = 8000, 300
    c = _community(n_prey, n_pred, 3.0 / n_pred)
    o = _step(oracle_mod, c, _rows(n_prey, 0), _rows(n_pred, 0))
    d, dp = o.debug(0), o.debug(1)
    cap = dp["cap"].astype(np.float64)
    n_cap = int(d["captured"].sum())
    assert cap.shape[0] == n_pred and cap.sum() == n_cap > 25000
    chi2 = ((cap - cap.mean()) ** 2 / cap.mean()).sum()
    assert stats.chi2.ppf(1e-4, n_pred - 1) < chi2 < stats.chi2.ppf(1 - 1e-4, n_pred - 1)   # neither clumped nor too even
    idx = np.arange(n_pred)
    mean_idx = (cap * idx).sum() / n_cap
    assert abs(mean_idx - (n_pred - 1) / 2) < 4.5 * math.sqrt((n_pred ** 2 - 1) / 12.0 / n_cap)
    # (2) 250 adults -> about 1,000 newborns, 5,000 consumers, a*N_C = 40: every newborn is captured
    n_prey, n_pred = 250, 5000
    c = _community(n_prey, n_pred, 40.0 / n_pred)
    o = _step(oracle_mod, c, _rows(n_prey, 0), _rows(n_pred, 0))
    d, dp = o.debug(0), o.debug(1)
    m = d["m_t"]
    assert 800 < m < 1200 and d["captured"].all()
    cap = dp["cap"].astype(np.int64)
    assert cap.sum() == m
    distinct = int((cap > 0).sum())
    e_distinct = n_pred * (1.0 - (1.0 - 1.0 / n_pred) ** m)
    # variance of the occupancy count, exact: N q^m (1 - q^m) + N (N-1) (q2^m - q^2m), q = 1-1/N, q2 = 1-2/N
    q, q2 = 1.0 - 1.0 / n_pred, 1.0 - 2.0 / n_pred
    var = n_pred * q ** m * (1 - q ** m) + n_pred * (n_pred - 1) * (q2 ** m - q ** (2 * m))
    assert abs(distinct - e_distinct) < 4.5 * math.sqrt(var), (distinct, e_distinct)
    assert distinct < m - 40                                   # collisions happen (about m^2 / 2 N_C = 100)
    # the credited consumers are spread over the whole population, not packed into the first m slots
    credited = np.repeat(np.arange(n_pred), cap)
    assert abs(credited.mean() - (n_pred - 1) / 2) < 4.5 * math.sqrt((n_pred ** 2 - 1) / 12.0 / m)
    fifths = np.bincount(credited * 5 // n_pred, minlength=5)
    assert ((fifths - m / 5.0) ** 2 / (m / 5.0)).sum() < stats.chi2.ppf(1 - 1e-4, 4)
    # and the credit does not follow j: the captured newborns are j = 0..m-1, so "consumer j % N_C" would be
    # exactly the indicator of the first m consumers
    assert not np.array_equal(cap, (np.arange(n_pred) < m).astype(np.int64))


def test_consumer_fecundity_follows_its_own_captures(oracle_mod):
    """R14: a consumer with k captures draws its fecundity from table k, mean eps * k * max(0, 1 - N_C/K_C);
    here eps = 2, K_C = 2.5 N_C: mean 1.2 k.  The groups are large by construction (asserted, not skipped)."""
    n_prey, n_pred = 20000, 20000
    c = _community(n_prey, n_pred, 1.0 / n_pred, fec=2.0)
    o = _step(oracle_mod, c, _rows(n_prey, 0), _rows(n_pred, 0))
    dp = o.debug(1)
    f, cap = dp["f"].astype(np.float64), dp["cap"]
    assert f[cap == 0].sum() == 0 and dp["table_len"][0] == 0
    for k in (1, 2, 3):
        sel = cap == k
        assert sel.sum() > 300, (k, sel.sum())
        assert abs(f[sel].mean() - 1.2 * k) < 4.5 * math.sqrt(1.2 * k / sel.sum()), k
    # captures per consumer: Poisson(total / N_C) to the accuracy of the multinomial
    lam = cap.sum() / n_pred
    assert abs((cap == 0).mean() - math.exp(-lam)) < 4.5 * math.sqrt(math.exp(-lam) / n_pred)
