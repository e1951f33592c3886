"""Pins for the oracle's primitives (RNG, exp specs, table samplers).  -m "not gpu".

Each test pins the oracle to something other than itself: published known-answer vectors,
libm, closed-form moments of the Poisson / rounded-normal laws."""
import math
import os

import numpy as np
import pytest
from scipy import stats

HERE = os.path.dirname(os.path.abspath(__file__))


def test_philox_known_answer_vectors(oracle_mod):
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "philox4x32_10_kat.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        out = oracle_mod.philox4x32_10(v[4:6], v[0:4])
        assert [int(x) for x in out] == v[6:10]


def test_draw_counter_layout(oracle_mod):
    # R3: key=(seed_lo,seed_hi), ctr=(entity, block, step, species<<8|stream)
    seed, sp, st, ent, blk, step = 0x123456789ABCDEF0, 3, 5, 77, 9, 1234
    a = oracle_mod.draw(seed, sp, st, ent, blk, step)
    b = oracle_mod.philox4x32_10([seed & 0xFFFFFFFF, seed >> 32], [ent, blk, step, (sp << 8) | st])
    assert (a == b).all()


def test_philox_uniformity_and_lag(oracle_mod):
    n = 20000
    w = np.concatenate([oracle_mod.draw(7, 0, 0, i, 0, 0) for i in range(n)]).astype(np.float64)
    counts, _ = np.histogram(w, bins=64, range=(0, 2.0 ** 32))
    chi2 = ((counts - counts.mean()) ** 2 / counts.mean()).sum()
    assert chi2 < stats.chi2.ppf(1 - 1e-6, 63)
    u = w / 2.0 ** 32
    assert abs(np.corrcoef(u[:-1], u[1:])[0, 1]) < 5 / math.sqrt(len(u))
    # consecutive entities / blocks / steps / streams give unrelated blocks
    base = oracle_mod.draw(7, 0, 0, 0, 0, 0)
    for other in [oracle_mod.draw(7, 0, 0, 1, 0, 0), oracle_mod.draw(7, 0, 0, 0, 1, 0),
                  oracle_mod.draw(7, 0, 0, 0, 0, 1), oracle_mod.draw(7, 0, 1, 0, 0, 0),
                  oracle_mod.draw(7, 1, 0, 0, 0, 0), oracle_mod.draw(8, 0, 0, 0, 0, 0)]:
        assert not (base == other).any()


def test_exp_neg64_matches_libm(oracle_mod):
    rng = np.random.default_rng(0)
    lams = np.concatenate([[0.0, 1.0, 2.0, 1e-300, 1e-9, 64.0, 699.0], rng.uniform(0, 5, 2000), rng.uniform(0, 700, 500)])
    for lam in lams:
        got, ref = oracle_mod.exp_neg64(lam), math.exp(-lam)
        assert abs(got - ref) <= 4 * np.spacing(ref), (lam, got, ref)
    assert oracle_mod.exp_neg64(0.0) == 1.0


def test_expf_spec_matches_libm(oracle_mod):
    rng = np.random.default_rng(1)
    xs = np.concatenate([[0.0, -1e-30, -1e-8, -87.0], -rng.uniform(0, 4, 4000), -rng.uniform(0, 87, 2000)]).astype(np.float32)
    worst = 0.0
    for x in xs:
        got, ref = oracle_mod.expf_spec(float(x)), math.exp(float(x))
        worst = max(worst, abs(got - ref) / ref)
    assert worst < 4e-7  # north_star: survival probabilities within 1e-6 relative
    assert oracle_mod.expf_spec(0.0) == 1.0
    assert oracle_mod.expf_spec(-0.0) == 1.0
    assert oracle_mod.expf_spec(-88.0) == 0.0
    # monotone over a fine grid near 0 where decisions are taken
    g = np.linspace(-3, 0, 3001).astype(np.float32)
    v = np.array([oracle_mod.expf_spec(float(x)) for x in g])
    assert (np.diff(v) >= 0).all()


@pytest.mark.parametrize("lam", [0.01024, 0.5, 1.0, 1.0607, 2.0, 7.5, 37.2])
def test_poisson_table_is_the_poisson_law(oracle_mod, lam):
    T = oracle_mod.poisson_table(lam).astype(np.float64)
    F = T / 2.0 ** 32
    # thresholds are the Poisson cdf truncated to 32 bits
    ref = stats.poisson.cdf(np.arange(len(T)), lam)
    assert np.all(np.abs(F - ref) < 2.0 ** -31)
    assert np.all(np.diff(T) >= 0)
    # the table ends before the first k whose cdf is within 2^-32 of one
    assert stats.poisson.sf(len(T), lam) < 2.0 ** -31
    assert stats.poisson.sf(len(T) - 1, lam) > 2.0 ** -33
    assert abs(F[0] - math.exp(-lam)) < 2.0 ** -31  # P(f = 0) = e^-lam


def test_poisson_table_edges(oracle_mod):
    assert len(oracle_mod.poisson_table(0.0)) == 0  # lam = 0 -> f = 0 always
    T = oracle_mod.poisson_table(1.0)
    assert oracle_mod.poisson_count(T, 0) == 0
    assert oracle_mod.poisson_count(T, int(T[0]) - 1) == 0
    assert oracle_mod.poisson_count(T, int(T[0])) == 1
    assert oracle_mod.poisson_count(T, 0xFFFFFFFF) == len(T)


def test_poisson_sampler_moments(oracle_mod):
    # mean offspring count equals the Poisson mean (north_star), variance too
    lam = 1.0607
    T = oracle_mod.poisson_table(lam)
    rng = np.random.default_rng(5)
    u = rng.integers(0, 2 ** 32, size=400000, dtype=np.uint64)
    k = np.searchsorted(T.astype(np.uint64), u, side="right")  # = #{T_k <= u}
    # the numpy shortcut equals the oracle's own search
    for i in range(0, 2000):
        assert oracle_mod.poisson_count(T, int(u[i])) == k[i]
    se = math.sqrt(lam / len(u))
    assert abs(k.mean() - lam) < 4 * se
    assert abs(k.var() - lam) < 6 * lam * math.sqrt(2.0 / len(u)) + 4 * se
    assert abs((k == 0).mean() - math.exp(-lam)) < 4 * math.sqrt(0.25 / len(u))


def test_normal_table_is_rounded_normal(oracle_mod):
    sq = 51.2  # sigma = 0.05, q = 2^-10
    R, T = oracle_mod.normal_table(sq)
    assert R == math.ceil(8 * sq) == 410 and len(T) == 820
    pk = np.diff(np.concatenate([[0.0], T.astype(np.float64) / 2.0 ** 32, [1.0]]))
    ks = np.arange(-R, R + 1)
    ref = stats.norm.cdf((ks + 0.5) / sq) - stats.norm.cdf((ks - 0.5) / sq)
    ref[0] = stats.norm.cdf((ks[0] + 0.5) / sq)
    ref[-1] = stats.norm.sf((ks[-1] - 0.5) / sq)
    assert np.all(np.abs(pk - ref) < 2.0 ** -30)
    mean = (pk * ks).sum()
    var = (pk * ks ** 2).sum() - mean ** 2
    assert abs(mean) < 1e-6
    assert abs(var - (sq ** 2 + 1.0 / 12.0)) < 1e-3  # Sheppard's correction
    assert abs(pk[R] - (2 * stats.norm.cdf(0.5 / sq) - 1)) < 1e-9  # P(delta = 0)
    # search
    assert oracle_mod.normal_delta(T, R, 0) == -R + int((T == 0).sum())
    assert oracle_mod.normal_delta(T, R, 2 ** 31) in (0, 1)
    assert oracle_mod.normal_delta(T, R, 2 ** 31 - 1) in (-1, 0)
