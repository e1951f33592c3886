"""Pins for the oracle's shared-preference mating (reading R19; "shared preference across
individuals"; eq. S2-10: Pr(male i fertilizes an egg) = X_i^{v_m} / sum_j X_j^{v_m}).
-m "not gpu".

The weighted draw is pinned by (1) a population built by hand whose three size classes must father
eggs in the ratio 1 : 2 : 4, (2) the exponential tilt of a Gaussian trait: the chosen fathers' mean
exceeds the adults' mean by v_m V (finite-population form: sum w z / sum w), (3) the response of the
offspring mean, half of that (only one parent is chosen), (4) patch structure, sign and the
unchanged rest of the step.  A dropped weight, a wrong sign, an off-by-one in the search or a
running sum that restarts in the wrong place fails one of them."""
import math

import numpy as np
from scipy import stats

from helpers import cfg, species
from paper_1603_09255_b200 import workloads


def _cfg(n0, v, L=16, fec_a=2.0, K=1e12, omega=0.0, capacity=None, grid=(1, 1), seed=19, init_sd=0.1, mu=0.0):
    sp = species(L=L, kind="q10", r=0.5, mu=mu, fec_a=fec_a, K=K, omega=omega,
                 capacity=capacity or max(4096, int(n0 * (fec_a + 1.5))))
    sp["mate_skew"] = v
    c = cfg(sp, seed=seed, grid=grid)
    c["n0"] = [n0]
    c["init_sd"] = init_sd
    return c


def _z(rows):
    return rows.astype(np.int64).sum(axis=1) * 2.0 ** -11


def test_three_size_classes_by_hand(oracle_mod):
    """Adults of genetic value 0, 1, 2 (100 of each, interleaved) and v_m = ln 2: X^{v_m} = 1, 2, 4,
    so the classes father 1/7, 2/7 and 4/7 of the eggs, and within a class every adult is equally
    likely."""
    n0 = 300
    c = _cfg(n0, math.log(2.0), fec_a=30.0)
    rows = np.zeros((n0, 32), np.int16)
    rows[:, 0] = 1024 * (np.arange(n0) % 3)          # hap0 locus 0
    rows[:, 16] = 1024 * (np.arange(n0) % 3)         # hap1 locus 0: zi = 0, 2048, 4096 -> z = 0, 1, 2
    o = oracle_mod.Oracle(c)
    o.write_state(0, rows, None, 0)
    o.step(1)
    d = o.debug(0)
    m = d["m_t"]
    assert m > 8000
    cls = np.bincount(d["father"] % 3, minlength=3)
    expect = m * np.array([1.0, 2.0, 4.0]) / 7.0
    assert ((cls - expect) ** 2 / expect).sum() < stats.chi2.ppf(1 - 1e-4, 2)
    for k in range(3):   # uniform within a class
        cnt = np.bincount(d["father"][d["father"] % 3 == k] // 3, minlength=100)
        assert ((cnt - cnt.mean()) ** 2 / cnt.mean()).sum() < stats.chi2.ppf(1 - 1e-4, 99)
    # the running sum: equal steps within a class, ratio 1:2:4 between classes (to fp32 rounding)
    w = np.diff(np.concatenate([[0], d["mate_cum"].astype(np.float64)]))
    assert len(set(w[0::3])) == 1 and len(set(w[1::3])) == 1 and len(set(w[2::3])) == 1
    assert abs(w[1] / w[0] - 2.0) < 5e-5 and abs(w[2] / w[0] - 4.0) < 5e-5   # truncation to integers
    assert abs(d["zbar_self"] - 1.0) < 1e-6
    # the adult at the mean has weight exp(-16) 2^40
    assert abs(w[1] / (math.exp(-16.0) * 2.0 ** 40) - 1) < 1e-5


def test_exponential_tilt_of_a_gaussian_trait(oracle_mod):
    """Weights exp(v z) tilt the trait distribution of the chosen fathers: their expected mean is
    sum w z / sum w, which for a Gaussian trait of variance V is zbar + v V."""
    n0, v = 20000, 1.5
    c = _cfg(n0, v, L=64, fec_a=2.0)
    rows = workloads.initial_rows(c, 0)
    o = oracle_mod.Oracle(c)
    o.write_state(0, rows, None, 0)
    o.step(1)
    d = o.debug(0)
    z = _z(rows)
    V = z.var()
    assert np.abs(v * (z - z.mean())).max() < 16          # the clamp is not in play
    w = np.exp(v * (z - z.mean()))
    zf = z[d["father"]]
    expect = (w * z).sum() / w.sum()
    Vf = (w * (z - expect) ** 2).sum() / w.sum()
    assert abs(zf.mean() - expect) < 4.5 * math.sqrt(Vf / len(zf))
    assert abs((expect - z.mean()) / (v * V) - 1) < 0.05  # Gaussian closed form
    assert (zf.mean() - z.mean()) > 20 * math.sqrt(V / len(zf))   # uniform mating would give 0
    # mothers are not chosen by size: their mean stays at the adults' mean
    zm = z[d["mother"]]
    assert abs(zm.mean() - z.mean()) < 4.5 * math.sqrt(V / n0) * 2
    # the stored running sum is the definition, to the accuracy of the fp32 exp
    wi = np.diff(np.concatenate([[0], d["mate_cum"].astype(np.float64)]))
    ref = np.exp(v * (z - z.mean()) - 16.0) * 2.0 ** 40
    assert (np.abs(wi - ref) < 1.0 + 2e-5 * ref).all()     # truncation + fp32 argument rounding at |x| <= 32
    assert (np.diff(d["mate_cum"].astype(np.float64)) >= 0).all()
    # father j is the first adult whose running sum exceeds the target built from words 2,3 of
    # SCALAR block 1 (checked against a plain scan on a sample)
    cum = [int(x) for x in d["mate_cum"]]
    for j in range(0, d["m_t"], max(1, d["m_t"] // 40)):
        y = oracle_mod.draw(c["seed"], 0, 1, j, 1, 0)
        u = (int(y[2]) << 32) | int(y[3])
        target = (u * cum[-1]) >> 64
        i = 0
        while cum[i] <= target:
            i += 1
        assert i == d["father"][j]


def test_response_to_sexual_selection(oracle_mod):
    """No viability selection (omega = inf), no mutation: the offspring mean moves by half the
    fathers' selection differential, (1/2) v V; with v < 0 the other way."""
    n0 = 30000
    for v in (3.0, -3.0):
        c = _cfg(n0, v, L=64, fec_a=2.0)
        rows = workloads.initial_rows(c, 0)
        o = oracle_mod.Oracle(c)
        o.write_state(0, rows, None, 0)
        o.step(1)
        d = o.debug(0)
        z = _z(rows)
        w = np.exp(v * (z - z.mean()))
        S = (w * z).sum() / w.sum() - z.mean()
        zo = d["zi"].astype(np.float64) * 2.0 ** -11
        assert d["alive"].all()
        assert abs((zo.mean() - z.mean()) - 0.5 * S) < 4.5 * math.sqrt(z.var() / len(zo))
        assert np.sign(zo.mean() - z.mean()) == np.sign(v)
        assert abs(zo.mean() - z.mean()) > 10 * math.sqrt(z.var() / len(zo))


def test_patches_and_the_rest_of_the_step(oracle_mod):
    """In patch mode the father comes from the mother's patch, with the patch's own weights; the
    mating rule changes the father column and nothing else drawn in the step; v = 0 is R2."""
    n0, v = 4000, 5.0
    c = _cfg(n0, v, L=16, fec_a=2.0, K=1e12, grid=(2, 2), capacity=16384)
    rows = workloads.initial_rows(c, 0)
    rows[:1000] += 40                                   # patch 0 is larger than the rest on average
    ps = workloads.initial_patch_start(c, 0)
    o = oracle_mod.Oracle(c)
    o.write_state(0, rows, ps, 0)
    o.step(1)
    d = o.debug(0)
    pm = np.searchsorted(ps, d["mother"], side="right") - 1
    pf = np.searchsorted(ps, d["father"], side="right") - 1
    assert np.array_equal(pm, pf)
    z = _z(rows)
    for p in range(4):
        sl = slice(int(ps[p]), int(ps[p + 1]))
        w = np.exp(v * (z[sl] - z.mean()))
        zf = z[d["father"][pm == p]]
        expect = (w * z[sl]).sum() / w.sum()
        Vf = (w * (z[sl] - expect) ** 2).sum() / w.sum()
        assert abs(zf.mean() - expect) < 4.5 * math.sqrt(Vf / len(zf))
    # same configuration with uniform mating: only the fathers (and what descends from them) differ
    c0 = _cfg(n0, 0.0, L=16, fec_a=2.0, K=1e12, grid=(2, 2), capacity=16384)
    o0 = oracle_mod.Oracle(c0)
    o0.write_state(0, rows, ps, 0)
    o0.step(1)
    d0 = o0.debug(0)
    for k in ("f", "off", "mother", "dest", "u01"):
        assert np.array_equal(d[k], d0[k]), k
    L = 16
    assert np.array_equal(d["offspring"][:, :L], d0["offspring"][:, :L])      # maternal gametes
    assert not np.array_equal(d["father"], d0["father"])
    # v = 0 is bit-identical to a configuration without the field
    a, b = workloads.config(1), workloads.config(1)
    b["species"][0]["mate_skew"] = 0.0
    ra, rb = oracle_mod.Oracle(a), oracle_mod.Oracle(b)
    for r_, c_ in ((ra, a), (rb, b)):
        r_.write_state(0, workloads.initial_rows(c_, 0), None, 0)
        r_.step(3)
    assert ra.log(0) == rb.log(0) and np.array_equal(ra.read_state(0)[0], rb.read_state(0)[0])


def test_clamp_and_zero_weight_patch(oracle_mod):
    """|v (z - zbar)| is clamped to 16; an adult 32 e-folds below the top has integer weight 0 and is
    never chosen; a patch whose total weight is 0 falls back to the uniform mate of R2."""
    n0 = 64
    c = _cfg(n0, 100.0, L=16, fec_a=20.0, grid=(2, 1), capacity=8192)
    rows = np.zeros((n0, 32), np.int16)
    rows[:32, 0] = -2048          # patch 0: everybody at z = -1, far below the mean -> e = -16, x = -32
    rows[32:48, 0] = 2048         # patch 1: half at z = +1 (e = +16, x = 0, weight 2^40) ...
    rows[48:, 0] = -2048          # ... half at z = -1 (weight trunc(exp(-32) 2^40) = 0)
    ps = np.array([0, 32, 64], np.uint32)
    o = oracle_mod.Oracle(c)
    o.write_state(0, rows, ps, 0)
    o.step(1)
    d = o.debug(0)
    w = np.diff(np.concatenate([[0], d["mate_cum"].astype(np.float64)]))
    assert (w[:32] == 0).all() and (w[48:] == 0).all() and (w[32:48] == 2.0 ** 40).all()
    in1 = d["mother"] >= 32
    assert in1.sum() > 300 and (~in1).sum() > 300
    assert ((d["father"][in1] >= 32) & (d["father"][in1] < 48)).all()
    f0 = d["father"][~in1]
    assert f0.max() < 32
    cnt = np.bincount(f0, minlength=32)
    assert ((cnt - cnt.mean()) ** 2 / cnt.mean()).sum() < stats.chi2.ppf(1 - 1e-4, 31)
