"""Pins for the oracle's fecundity cost of defence (reading R22; eq. S3-3, PAPER.md:471:
w_F,R <- w_F,R * n_i * exp(-rho * trait^2)).  -m "not gpu".

A Poisson count thinned egg by egg with probability c is Poisson with mean lambda*c: pinned on a
hand-built population of three trait classes (c = 1, 1/2, 1/16: mean AND variance of the eggs per
adult), by the Gaussian-selection response of the offspring mean (only mothers are selected: half of
V/(V + 1/(2 rho)) times the distance to 0), and by rho = 0 being the unchanged path."""
import math

import numpy as np

from helpers import cfg, species
from paper_1603_09255_b200 import workloads


def _cfg(n0, rho, L=16, fec_a=6.0, seed=22):
    sp = species(L=L, kind="q10", r=0.5, mu=0.0, fec_a=fec_a, K=1e12, omega=0.0, capacity=int(n0 * (fec_a + 2)))
    sp["fec_cost"] = rho
    c = cfg(sp, seed=seed)
    c["n0"] = [n0]
    c["init_sd"] = 0.1
    return c


def test_three_trait_classes_by_hand(oracle_mod):
    n0, lam = 30000, 6.0
    c = _cfg(n0, math.log(2.0), fec_a=lam)
    rows = np.zeros((n0, 32), np.int16)
    rows[:, 0] = 1024 * (np.arange(n0) % 3)
    rows[:, 16] = 1024 * (np.arange(n0) % 3)          # z = 0, 1, 2  ->  c = 1, 2^-1, 2^-4
    o = oracle_mod.Oracle(c)
    o.write_state(0, rows, None, 0)
    o.step(1)
    d = o.debug(0)
    f = d["f"].astype(np.float64)
    for k, ck in enumerate((1.0, 0.5, 1.0 / 16.0)):
        fk = f[k::3]
        m = lam * ck
        assert abs(fk.mean() - m) < 4.5 * math.sqrt(m / len(fk)), (k, fk.mean(), m)
        assert abs(fk.var() / m - 1) < 0.06, (k, fk.var(), m)      # still Poisson: variance = mean
    assert d["m_t"] == f.sum() and np.array_equal(np.bincount(d["mother"], minlength=n0), f)
    # the eggs' uniforms are not the count's word: class 0 (c = 1) keeps exactly the count that was drawn
    c0 = _cfg(n0, 0.0, fec_a=lam)
    o0 = oracle_mod.Oracle(c0)
    o0.write_state(0, rows, None, 0)
    o0.step(1)
    f0 = o0.debug(0)["f"]
    assert np.array_equal(d["f"][0::3], f0[0::3]) and (d["f"] <= f0).all()
    # thinning is independent of the count: P(keep) does not depend on how many eggs were drawn
    for cnt in (4, 8):
        sel = (f0[1::3] == cnt)
        assert abs(d["f"][1::3][sel].mean() / cnt - 0.5) < 4.5 * math.sqrt(0.25 / (cnt * sel.sum()))


def test_response_to_fecundity_selection(oracle_mod):
    """w(z) = exp(-rho z^2) is Gaussian selection of width omega^2 = 1/(2 rho) toward 0 acting on the
    mothers only: the offspring mean moves by (1/2) (0 - zbar) V / (V + omega^2)."""
    n0, rho = 40000, 0.5
    c = _cfg(n0, rho, L=64, fec_a=4.0)
    rows = workloads.initial_rows(c, 0)
    rows[:, 0] += 1600                                  # shift the mean to about +0.78
    o = oracle_mod.Oracle(c)
    o.write_state(0, rows, None, 0)
    o.step(1)
    d = o.debug(0)
    z = rows.astype(np.int64).sum(axis=1) * 2.0 ** -11
    w = np.exp(-rho * z * z)
    S = (w * z).sum() / w.sum() - z.mean()              # finite-population selection differential
    assert abs(S / (-z.mean() * z.var() / (z.var() + 1.0 / (2 * rho))) - 1) < 0.03   # the closed form
    zo = d["zi"].astype(np.float64) * 2.0 ** -11
    assert abs((zo.mean() - z.mean()) - 0.5 * S) < 4.5 * math.sqrt(z.var() / len(zo))
    assert zo.mean() < z.mean() - 10 * math.sqrt(z.var() / len(zo))
    # mothers are the selected ones, fathers are not
    assert abs(z[d["father"]].mean() - z.mean()) < 4.5 * math.sqrt(z.var() / len(zo))
    assert abs(z[d["mother"]].mean() - (z.mean() + S)) < 4.5 * math.sqrt(z.var() / n0) * 2


def test_zero_cost_is_the_unchanged_path(oracle_mod):
    a, b = workloads.config(2, scale=0.01), workloads.config(2, scale=0.01)
    b["species"][0]["fec_cost"] = 0.0
    outs = []
    for c in (a, b):
        o = oracle_mod.Oracle(c)
        o.write_state(0, workloads.initial_rows(c, 0), None, 0)
        o.step(3)
        outs.append(o)
    assert outs[0].log(0) == outs[1].log(0) and np.array_equal(outs[0].read_state(0)[0], outs[1].read_state(0)[0])
