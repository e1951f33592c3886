"""Pins for the oracle's weighted mothers (reading R24; eq. S2-9: "For each egg,
the mother and father are drawn at random from mature males and females in the population.  The
probability that the egg comes from female i is a function of the female's relative gonadal mass",
(G_i / (Omega_i + q_J Omega_i))^{v_f}).  -m "not gpu".

The weighted draw of the mother is pinned by (1) a population built by hand whose three fecundity
classes must mother eggs in the ratio 1 : 2 : 4 while the NUMBER of eggs is what the Poisson
fecundities give, (2) the exponential tilt of a Gaussian trait through the mothers only, (3) the
response of the offspring mean, half the mothers' differential, (4) separate sexes (only females
mother), patches (the mother comes from the patch that laid the egg), the zero-weight fallback, and
v_f = 0 being the unchanged path bit for bit.  A dropped weight, a wrong sign, a search over the
wrong segment, the wrong sex zeroed or a changed egg count fails one of them."""
import math

import numpy as np
import pytest
from scipy import stats

from helpers import cfg, species
from paper_1603_09255_b200 import workloads


def _cfg(n0, v, L=16, fec_a=2.0, K=1e12, omega=0.0, capacity=None, grid=(1, 1), seed=24, init_sd=0.1, mu=0.0, **extra):
    sp = species(L=L, kind="q10", r=0.5, mu=mu, fec_a=fec_a, K=K, omega=omega,
                 capacity=capacity or max(4096, int(n0 * (fec_a + 1.5))))
    sp["mother_skew"] = v
    sp.update(extra)
    c = cfg(sp, seed=seed, grid=grid)
    c["n0"] = [n0]
    c["init_sd"] = init_sd
    return c


def _z(rows):
    return rows.astype(np.int64).sum(axis=1) * 2.0 ** -11


def test_three_fecundity_classes_by_hand(oracle_mod):
    """Adults of genetic value 0, 1, 2 (100 of each, interleaved) and v_f = ln 2: Y^{v_f} = 1, 2, 4, so
    the classes mother 1/7, 2/7 and 4/7 of the eggs, every adult of a class equally often; the number
    of eggs is the sum of the Poisson fecundities and the father stays uniform."""
    n0 = 300
    c = _cfg(n0, math.log(2.0), fec_a=30.0)
    rows = np.zeros((n0, 32), np.int16)
    rows[:, 0] = 1024 * (np.arange(n0) % 3)
    rows[:, 16] = 1024 * (np.arange(n0) % 3)         # zi = 0, 2048, 4096 -> z = 0, 1, 2
    o = oracle_mod.Oracle(c)
    o.write_state(0, rows, None, 0)
    o.step(1)
    d = o.debug(0)
    m = d["m_t"]
    assert m == int(d["f"].sum()) and m > 8000        # the egg count is untouched
    assert abs(d["f"].mean() - 30.0) < 5 * math.sqrt(30.0 / n0)
    cls = np.bincount(d["mother"] % 3, minlength=3)
    expect = m * np.array([1.0, 2.0, 4.0]) / 7.0
    assert ((cls - expect) ** 2 / expect).sum() < stats.chi2.ppf(1 - 1e-4, 2)
    for k in range(3):   # uniform within a class
        cnt = np.bincount(d["mother"][d["mother"] % 3 == k] // 3, minlength=100)
        assert ((cnt - cnt.mean()) ** 2 / cnt.mean()).sum() < stats.chi2.ppf(1 - 1e-4, 99)
    fcls = np.bincount(d["father"] % 3, minlength=3)  # fathers: uniform mate (R2)
    assert ((fcls - m / 3.0) ** 2 / (m / 3.0)).sum() < stats.chi2.ppf(1 - 1e-4, 2)
    w = np.diff(np.concatenate([[0], d["mom_cum"].astype(np.float64)]))
    assert len(set(w[0::3])) == 1 and len(set(w[1::3])) == 1 and len(set(w[2::3])) == 1
    assert abs(w[1] / w[0] - 2.0) < 5e-5 and abs(w[2] / w[0] - 4.0) < 5e-5
    assert abs(w[1] / (math.exp(-16.0) * 2.0 ** 40) - 1) < 1e-5   # the adult at the mean weighs exp(-16) 2^40
    # the maternal gamete of every egg comes from the drawn mother: with two distinct alleles per
    # class at locus 0 and no mutation, the offspring's maternal allele at locus 0 is the mother's
    assert np.array_equal(d["offspring"][:, 0], rows[d["mother"], 0])


def test_exponential_tilt_through_the_mothers(oracle_mod):
    """Weights exp(v z): the chosen mothers' expected mean is sum w z / sum w (Gaussian closed form
    zbar + v V); the fathers stay at the adults' mean; the offspring mean moves by half the mothers'
    differential (no viability selection, no mutation); v < 0 the other way.  The mother of egg j is
    the first adult whose running sum exceeds the target built from words 0,1 of MOTHER block 0."""
    n0 = 30000
    for v in (2.0, -2.0):
        c = _cfg(n0, v, L=64, fec_a=2.0)
        rows = workloads.initial_rows(c, 0)
        o = oracle_mod.Oracle(c)
        o.write_state(0, rows, None, 0)
        o.step(1)
        d = o.debug(0)
        z = _z(rows)
        V = z.var()
        assert np.abs(v * (z - z.mean())).max() < 16
        w = np.exp(v * (z - z.mean()))
        expect = (w * z).sum() / w.sum()
        Vm = (w * (z - expect) ** 2).sum() / w.sum()
        zm = z[d["mother"]]
        assert abs(zm.mean() - expect) < 4.5 * math.sqrt(Vm / len(zm))
        assert abs((expect - z.mean()) / (v * V) - 1) < 0.05
        assert abs(zm.mean() - z.mean()) > 20 * math.sqrt(V / len(zm))
        zf = z[d["father"]]
        assert abs(zf.mean() - z.mean()) < 4.5 * math.sqrt(V / len(zf))
        zo = d["zi"].astype(np.float64) * 2.0 ** -11
        assert d["alive"].all()
        S = expect - z.mean()
        # offspring = mid-parent + segregation noise; sd of the mean <= sqrt(V / m)
        assert abs((zo.mean() - z.mean()) - 0.5 * S) < 5 * math.sqrt(V / len(zo))
        cum = [int(x) for x in d["mom_cum"]]
        for j in range(0, d["m_t"], max(1, d["m_t"] // 40)):
            y = oracle_mod.draw(c["seed"], 0, 7, j, 0, 0)
            u = (int(y[0]) << 32) | int(y[1])
            target = (u * cum[-1]) >> 64
            i = 0
            while cum[i] <= target:
                i += 1
            assert i == d["mother"][j]


def test_only_females_mother_and_patches_keep_their_eggs(oracle_mod):
    """With separate sexes a male's mothering weight is 0; in patches the mother is drawn inside the
    patch that laid the egg (so per-patch egg numbers, and the density regulation, are unchanged)."""
    n0, grid = 1200, (3, 2)
    c = _cfg(n0, 1.0, L=16, fec_a=6.0, grid=grid, separate_sexes=1, K_patch=[1e12] * 6)
    rows = workloads.initial_rows(c, 0)
    ps = np.array([0, 100, 300, 300, 700, 1000, 1200], np.uint32)       # one empty patch
    sex = (np.arange(n0) % 3 == 0).astype(np.uint8)                      # every third adult is male
    o = oracle_mod.Oracle(c)
    o.write_state(0, rows, ps, 0)
    o.write_sex(0, sex)
    o.step(1)
    d = o.debug(0)
    mo = d["mother"]
    assert (sex[mo] == 0).all()
    assert (d["f"][sex == 1] == 0).all()
    pat = np.searchsorted(ps, np.arange(n0), side="right") - 1
    # egg j was laid in the patch of the adult whose offspring range holds j
    layer = np.searchsorted(d["off"].astype(np.int64) + d["f"], np.arange(d["m_t"]), side="right")
    assert np.array_equal(pat[layer], pat[mo])
    assert np.array_equal(pat[d["father"]], pat[mo]) and (sex[d["father"]] == 1).all()
    # within a patch: heavier females mother more (sign of the weight)
    z = _z(rows)
    for p in (1, 3):
        fem = np.where((pat == p) & (sex == 0))[0]
        cnt = np.bincount(mo[pat[mo] == p], minlength=n0)[fem]
        assert np.corrcoef(cnt, np.exp(z[fem]))[0, 1] > 0.3


def test_zero_weight_fallback_and_unchanged_path(oracle_mod):
    """A patch whose mothering weights are all 0 (every adult 32 e-folds below the mean) keeps the
    laying adult as the mother; v_f = 0 is today's path bit for bit."""
    n0 = 400
    c = _cfg(n0, 64.0, L=16, fec_a=4.0, grid=(2, 1), K_patch=[1e12, 1e12])
    rows = np.zeros((n0, 32), np.int16)
    rows[200:, 0] = 2048                                   # patch 1 sits 1 above patch 0: zbar = 0.5
    rows[200:, 16] = 2048
    rows[200:, 1] = 2048 * 15                              # ... far above: patch 0 weighs exp(-16-16) 2^40 -> 0
    ps = np.array([0, 200, 400], np.uint32)
    o = oracle_mod.Oracle(c)
    o.write_state(0, rows, ps, 0)
    o.step(1)
    d = o.debug(0)
    w = np.diff(np.concatenate([[0], d["mom_cum"].astype(np.float64)]))
    assert (w[:200] == 0).all() and (w[200:] > 0).all()
    layer = np.searchsorted(d["off"].astype(np.int64) + d["f"], np.arange(d["m_t"]), side="right")
    in0 = layer < 200
    assert in0.any() and np.array_equal(d["mother"][in0], layer[in0])          # fallback: the laying adult
    assert (d["mother"][~in0] >= 200).all() and not np.array_equal(d["mother"][~in0], layer[~in0])
    a, b = workloads.config(1), workloads.config(1)
    b["species"][0]["mother_skew"] = 0.0
    oa, ob = oracle_mod.Oracle(a), oracle_mod.Oracle(b)
    for x, cc in ((oa, a), (ob, b)):
        x.write_state(0, workloads.initial_rows(cc, 0), None, 0)
        x.step(3)
    assert oa.log(0) == ob.log(0) and np.array_equal(oa.read_state(0)[0], ob.read_state(0)[0])


def test_rejected_combinations(oracle_mod):
    c = _cfg(100, 1.0, fec_cost=0.5)
    with pytest.raises(ValueError):
        oracle_mod.Oracle(c)
