"""Pins for the oracle's gamete formation (readings R7-R9).  -m "not gpu".

Parents with marker haplotypes (hap0 all-A, hap1 all-B) expose the phase pattern of each gamete,
so recombination fractions, brute-force gamete probabilities and mutation rates can be checked
against their closed forms."""
import itertools
import math

import numpy as np
import pytest
from scipy import stats

from helpers import cfg, marker_parent, phase_bits, species


def gametes(oracle_mod, sp, n, gamete=0, step=0, seed=11, parent=None):
    o = oracle_mod.Oracle(cfg(sp, seed=seed))
    par = marker_parent(sp["kind"], sp["n_loci"]) if parent is None else parent
    return np.stack([o.make_gamete(0, par, gamete, j, step) for j in range(n)])


@pytest.mark.parametrize("kind,L", [("q10", 16), ("bit", 32)])
def test_interval_recombination_fraction_equals_r(oracle_mod, kind, L):
    r = np.array([0.5, 0.05, 0.2, 0.0] + [0.01 * (i % 7) for i in range(L - 5)])
    sp = species(L=L, kind=kind, r=r)
    n = 40000
    ph = np.stack([phase_bits(kind, L, g) for g in gametes(oracle_mod, sp, n)])
    rec = (ph[:, 1:] != ph[:, :-1]).mean(axis=0)
    se = np.sqrt(np.maximum(r * (1 - r), 1e-4) / n)
    assert np.all(np.abs(rec - r) < 4.5 * se)
    assert rec[3] == 0.0  # r = 0: never recombines
    assert abs(ph[:, 0].mean() - 0.5) < 4.5 * 0.5 / math.sqrt(n)  # start phase fair
    # both gamete streams obey the same law but are different draws
    ph_p = np.stack([phase_bits(kind, L, g) for g in gametes(oracle_mod, sp, 2000, gamete=1)])
    assert (ph_p != ph[:2000]).any()


def test_interval_r_zero_gives_whole_haplotype(oracle_mod):
    sp = species(L=16, r=0.0)
    ph = gametes(oracle_mod, sp, 4000)
    assert np.all((ph.sum(axis=1) == 0) | (ph.sum(axis=1) == 16))
    assert abs((ph.sum(axis=1) == 16).mean() - 0.5) < 4.5 * 0.5 / math.sqrt(4000)


def test_interval_free_recombination_is_iid_fair(oracle_mod):
    sp = species(L=16, r=0.5)
    ph = gametes(oracle_mod, sp, 30000).astype(np.float64)
    assert np.all(np.abs(ph.mean(axis=0) - 0.5) < 4.5 * 0.5 / math.sqrt(30000))
    cc = np.corrcoef(ph.T) - np.eye(16)
    assert np.abs(cc).max() < 5 / math.sqrt(30000)


@pytest.mark.parametrize("L,r", [(2, [0.3]), (3, [0.1, 0.4]), (4, [0.05, 0.5, 0.25])])
def test_bruteforce_gamete_enumeration(oracle_mod, L, r):
    # P(phase pattern) = 1/2 * prod_l (r_l if switch else 1-r_l)   (north_star: brute force at L<=4)
    sp = species(L=L, r=np.asarray(r))
    n = 200000
    ph = gametes(oracle_mod, sp, n)
    code = (ph * (1 << np.arange(L))).sum(axis=1)
    obs = np.bincount(code, minlength=1 << L).astype(np.float64)
    exp = np.zeros(1 << L)
    for pat in itertools.product([0, 1], repeat=L):
        p = 0.5
        for l in range(1, L):
            p *= r[l - 1] if pat[l] != pat[l - 1] else 1 - r[l - 1]
        exp[sum(b << i for i, b in enumerate(pat))] = p * n
    chi2 = ((obs - exp) ** 2 / exp).sum()
    assert chi2 < stats.chi2.ppf(1 - 1e-5, (1 << L) - 1)


def test_bruteforce_alleles_follow_phase(oracle_mod):
    # with arbitrary alleles the gamete is exactly the parent's alleles picked by the phase pattern
    L = 4
    sp = species(L=L, r=np.array([0.3, 0.5, 0.1]))
    o = oracle_mod.Oracle(cfg(sp, seed=11))
    par = np.array([5, -7, 11, 13, 100, 200, -300, 400], dtype=np.int16)
    mark = marker_parent("q10", L)
    for j in range(500):
        ph = o.make_gamete(0, mark, 0, j, 3)
        g = o.make_gamete(0, par, 0, j, 3)
        assert np.array_equal(g, np.where(ph == 1, par[L:], par[:L]))


def test_poisson_mode_haldane_map(oracle_mod):
    # R8: per-interval switch rate 1/2(1-exp(-2*lam/(len-1))), crossover count mean = variance = lam
    L, lam = 128, 1.0
    sp = species(L=L, kind="bit", chrom_len=[64, 64], linkage="poisson", xover_mean=lam)
    n = 40000
    ph = np.stack([phase_bits("bit", L, g) for g in gametes(oracle_mod, sp, n)])
    sw = (ph[:, 1:] != ph[:, :-1])
    within = np.r_[np.arange(0, 63), np.arange(64, 127)]
    rate = sw[:, within].mean()
    ref = 0.5 * (1 - math.exp(-2 * lam / 63))
    assert abs(rate - ref) < 4.5 * math.sqrt(ref / (n * len(within)))
    # between chromosomes: independent start phases -> 0.5
    assert abs(sw[:, 63].mean() - 0.5) < 4.5 * 0.5 / math.sqrt(n)
    # uniform along the chromosome
    per = sw[:, :63].mean(axis=0)
    assert np.all(np.abs(per - ref) < 5 * math.sqrt(ref / n))
    # observed switches per chromosome: odd/even structure of a Poisson count with coincidences
    # cancelling; P(no switch) >= P(n=0) = e^-lam and mean <= lam
    k = sw[:, :63].sum(axis=1)
    assert abs(k.mean() - 63 * ref) < 4.5 * math.sqrt(63 * ref / n) * 1.5
    assert (k == 0).mean() > math.exp(-lam) - 0.01


def test_poisson_mode_bruteforce_small(oracle_mod):
    # chromosome of 3 loci (2 intervals), lam = 0.7: switch indicators of the two intervals are
    # independent with P = 1/2(1-exp(-2*lam/2)) (Poisson thinning), start phase fair
    lam = 0.7
    sp = species(L=32, kind="bit", chrom_len=[3, 29], linkage="poisson", xover_mean=[lam, 0.0])
    n = 100000
    ph = np.stack([phase_bits("bit", 32, g) for g in gametes(oracle_mod, sp, n)])
    a = (ph[:, 0] != ph[:, 1]).astype(int)
    b = (ph[:, 1] != ph[:, 2]).astype(int)
    p = 0.5 * (1 - math.exp(-lam))
    obs = np.bincount(ph[:, 0] + 2 * a + 4 * b, minlength=8).astype(float)
    exp = np.array([0.5 * (p if x else 1 - p) * (p if y else 1 - p) for y in (0, 1) for x in (0, 1) for s in (0, 1)]) * n
    assert ((obs - exp) ** 2 / exp).sum() < stats.chi2.ppf(1 - 1e-5, 7)
    # second chromosome has mean 0 crossovers: it is one whole haplotype
    tail = ph[:, 3:]
    assert np.all((tail.sum(axis=1) == 0) | (tail.sum(axis=1) == 29))


def test_bit_mutation_flip_rate(oracle_mod):
    # R9 sparse form: per-locus flip probability 1/2(1-exp(-2mu)) ~ mu; mu=0 -> no change
    L, mu = 64, 2e-3
    homo = np.zeros(4, np.uint32)  # both haplotypes all-0: any 1 bit is a mutation
    n = 40000
    g = gametes(oracle_mod, species(L=L, kind="bit", linkage="poisson", chrom_len=[64], mu=mu), n, parent=homo)
    bits = np.unpackbits(g.view(np.uint8), bitorder="little", axis=1)[:, :L]
    ref = 0.5 * (1 - math.exp(-2 * mu))
    assert abs(bits.mean() - ref) < 4.5 * math.sqrt(ref / (n * L))
    per = bits.mean(axis=0)
    assert np.all(np.abs(per - ref) < 5.5 * math.sqrt(ref / n))
    g0 = gametes(oracle_mod, species(L=L, kind="bit", linkage="poisson", chrom_len=[64], mu=0.0), 2000, parent=homo)
    assert not g0.any()


def test_q10_mutation_effects(oracle_mod):
    # mutated allele = old + round(N(0, sd^2)/q): mean 0, variance (sd/q)^2 + 1/12
    L, mu, sd = 16, 0.02, 0.05
    homo = np.full(2 * L, 37, np.int16)
    n = 60000
    g = gametes(oracle_mod, species(L=L, mu=mu, mut_sd=sd), n, parent=homo).astype(np.int64) - 37
    hit = g != 0
    p0 = 2 * stats.norm.cdf(0.5 / 51.2) - 1  # a mutation that lands on delta = 0 is invisible
    ref = (1 - math.exp(-mu)) * (1 - p0)
    assert abs(hit.mean() - ref) < 5 * math.sqrt(ref / (n * L))
    d = g[hit]
    assert abs(d.mean()) < 5 * 51.2 / math.sqrt(len(d))
    assert abs(d.var() / (51.2 ** 2 + 1 / 12.0) - 1) < 0.06
    # saturation at +/-(2^15-1)
    top = np.full(2 * L, 32767, np.int16)
    gt = gametes(oracle_mod, species(L=L, mu=0.5, mut_sd=sd), 500, parent=top)
    assert gt.max() == 32767 and gt.min() > 32767 - 600


def test_mendelian_invariant(oracle_mod):
    # mu = 0: every gamete allele equals one of the parent's two alleles at that locus
    rng = np.random.default_rng(3)
    L = 64
    sp = species(L=L, chrom_len=[16] * 4, r=0.05)
    o = oracle_mod.Oracle(cfg(sp, seed=5))
    for j in range(300):
        par = rng.integers(-500, 500, size=2 * L).astype(np.int16)
        g = o.make_gamete(0, par, j % 2, j, 7)
        assert np.all((g == par[:L]) | (g == par[L:]))
    spb = species(L=256, kind="bit", chrom_len=[128, 128], linkage="poisson")
    ob = oracle_mod.Oracle(cfg(spb, seed=5))
    for j in range(300):
        par = rng.integers(0, 2 ** 32, size=16, dtype=np.uint64).astype(np.uint32)
        g = ob.make_gamete(0, par, j % 2, j, 7)
        h0, h1 = par[:8], par[8:]
        assert np.all(((g ^ h0) & (g ^ h1)) == 0)
    # homozygote -> gamete identical to the haplotype
    hom = np.concatenate([par[:8], par[:8]])
    assert np.array_equal(ob.make_gamete(0, hom, 0, 1, 1), par[:8])
