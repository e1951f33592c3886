"""Pins for the oracle's whole step (Fig. 1 A-F; readings R1-R16).  -m "not gpu".

Closed forms (Gaussian selection integral, Wright-Fisher drift, Beverton-Holt fixed point),
invariants (scan, parent arrays, compaction order, patch bookkeeping, capture accounting) and
determinism.  A dropped term, wrong sign/index or transposed operand fails one of them."""
import math
import os

import numpy as np
import pytest
from scipy import stats

from helpers import cfg, species
from paper_1603_09255_b200 import workloads

HERE = os.path.dirname(os.path.abspath(__file__))


def popcount_rows(rows):
    return np.unpackbits(rows.view(np.uint8), axis=1).sum(axis=1).astype(np.int64)


def zi_numpy(sp, rows):
    if sp["kind"] == "bit":
        return 2 * popcount_rows(rows) - 2 * sp["n_loci"]
    return rows.astype(np.int64).sum(axis=1)


def run(oracle_mod, c, n_steps=1, n0=None):
    o = oracle_mod.Oracle(c)
    for s in range(len(c["species"])):
        o.write_state(s, workloads.initial_rows(c, s, n=None if n0 is None else n0[s]),
                      workloads.initial_patch_start(c, s), 0)
    o.step(n_steps)
    return o


def test_scan_and_parent_arrays(oracle_mod):
    c = workloads.config(3, scale=0.02)
    o = run(oracle_mod, c)
    d = o.debug(0)
    n, m = d["n_t"], d["m_t"]
    f = d["f"].astype(np.int64)
    assert n == c["n0"][0] and m == f.sum()
    assert d["off"][0] == 0 and np.array_equal(d["off"], np.concatenate([[0], np.cumsum(f)[:-1]]))
    # every offspring has exactly one mother, mothers non-decreasing, f_i offspring each
    assert np.all(np.diff(d["mother"].astype(np.int64)) >= 0)
    assert np.array_equal(np.bincount(d["mother"], minlength=n), f)
    # fathers uniform over adults (chi-square over 50 bins), selfing allowed
    assert d["father"].max() < n
    cnt, _ = np.histogram(d["father"], bins=50, range=(0, n))
    assert ((cnt - m / 50) ** 2 / (m / 50)).sum() < stats.chi2.ppf(1 - 1e-5, 49)
    # mean offspring count equals the Poisson mean lam = 2/(1+N/K) = 1 (north_star)
    assert abs(f.mean() - 1.0) < 4.5 / math.sqrt(n)
    assert abs(f.var() - 1.0) < 0.05
    # u01 has 24 bits, in [0,1)
    assert d["u01"].min() >= 0 and d["u01"].max() < 1
    assert np.all(d["u01"] * 2 ** 24 == np.floor(d["u01"] * 2 ** 24))


def test_phenotype_is_exact_integer_sum(oracle_mod):
    for which, scale in [(1, 1.0), (3, 0.005)]:
        c = workloads.config(which, scale=scale)
        o = run(oracle_mod, c)
        d = o.debug(0)
        sp = c["species"][0]
        zi = zi_numpy(sp, d["offspring"])
        assert np.array_equal(zi, d["zi"])
        assert np.array_equal(d["z"], (zi * sp["pheno_scale"]).astype(np.float32))
        assert np.array_equal(d["z"].astype(np.float64), zi * sp["pheno_scale"])  # exact in fp32
        rows, _, zis = o.read_state(0)
        assert np.array_equal(zi_numpy(sp, rows), zis)


def test_offspring_rows_are_parent_gametes(oracle_mod):
    # offspring hap0 comes from the mother, hap1 from the father (mu = 0: Mendelian)
    c = workloads.config(3, scale=0.002)
    c["species"][0]["mu"] = 0.0
    rows0 = workloads.initial_rows(c, 0)
    o = run(oracle_mod, c)
    d = o.debug(0)
    W = 32
    mo, fa, off = rows0[d["mother"]], rows0[d["father"]], d["offspring"]
    assert not (((off[:, :W] ^ mo[:, :W]) & (off[:, :W] ^ mo[:, W:])).any())
    assert not (((off[:, W:] ^ fa[:, :W]) & (off[:, W:] ^ fa[:, W:])).any())
    # and really recombinant: most maternal gametes differ from both maternal haplotypes
    assert ((off[:, :W] != mo[:, :W]).any(axis=1) & (off[:, :W] != mo[:, W:]).any(axis=1)).mean() > 0.9


def test_survival_rule_and_compaction_order(oracle_mod):
    c = workloads.config(2, scale=0.05)
    o = run(oracle_mod, c, n_steps=3)  # step index 2 -> theta = 0.02
    d = o.debug(0)
    assert abs(d["theta_t"] - np.float32(0.02)) < 1e-9
    s64 = np.exp(-((d["z"].astype(np.float64) - d["theta_t"]) ** 2) / 2.0)
    assert np.max(np.abs(d["s"] - s64) / s64) < 1e-6  # fitness within 1e-6 relative (north_star)
    assert np.array_equal(d["alive"], (d["u01"] < d["s"]).astype(np.uint8))
    rows, _, zi = o.read_state(0)
    keep = d["alive"].astype(bool)
    assert np.array_equal(rows, d["offspring"][keep])  # stable: survivors in offspring order
    assert np.array_equal(zi, d["zi"][keep])
    le = o.log(0)[-1]
    assert le["n_next"] == keep.sum() == o.n(0) and le["m_t"] == d["m_t"]
    assert le["sum_zi"] == int(zi.astype(np.int64).sum()) and le["sum_zi2"] == int((zi.astype(np.int64) ** 2).sum())
    assert le["near_ties"] == int((np.abs(d["u01"] - d["s"]) < np.float32(1e-6)).sum())


def _closed_forms():
    out = {}
    for l in open(os.path.join(HERE, "golden", "closed_forms.txt")):
        if l.strip() and l[0] != "#":
            name, V, om, th, w = l.split()
            out[name] = (float(V), float(om), float(th), float(w))
    return out


@pytest.mark.parametrize("which,scale", [(1, 40.0), (2, 0.4), (3, 0.04), (5, 0.04)])
def test_first_step_survivor_fraction_closed_form(oracle_mod, which, scale):
    V, om, th, wref = _closed_forms()["C%d" % which]
    c = workloads.config(which, scale=scale, grid=(8, 8) if which == 5 else None)
    sp = c["species"][0]
    if which == 5:  # theta = 0 everywhere, no dispersal: the C5 row of the table
        sp["gaussian"]["theta_patch"] = np.zeros(64, np.float32)
    sp["mu"] = 0.0
    o = run(oracle_mod, c)
    d = o.debug(0)
    m = d["m_t"]
    # the closed form itself (retyped here from the textbook Gaussian integral)
    assert abs(om / math.sqrt(V + om * om) * math.exp(-th * th / (2 * (V + om * om))) - wref) < 2e-5
    z = d["z"].astype(np.float64)
    assert abs(z.var() / V - 1) < 0.05  # offspring variance = parental variance under random mating
    frac = d["alive"].mean()
    assert abs(frac - wref) < 4.5 * math.sqrt(wref * (1 - wref) / m) + 0.002
    # post-selection mean and variance: (zbar*om^2+theta*V)/(V+om^2), V*om^2/(V+om^2)
    zs = z[d["alive"].astype(bool)]
    assert abs(zs.var() / (V * om * om / (V + om * om)) - 1) < 0.05
    assert abs(zs.mean() - z.mean() * om * om / (V + om * om)) < 5 * math.sqrt(V / m)


def test_directional_selection_shifts_mean(oracle_mod):
    # theta != 0: survivors' mean moves towards theta by V/(V+omega^2) of the distance
    c = workloads.config(2, scale=0.3)
    c["species"][0]["gaussian"].update(theta0=0.8, dtheta=0.0)
    o = run(oracle_mod, c)
    d = o.debug(0)
    z = d["z"].astype(np.float64)
    zs = z[d["alive"].astype(bool)]
    V = z.var()
    assert abs((zs.mean() - z.mean()) - (0.8 - z.mean()) * V / (V + 1.0)) < 5 * math.sqrt(V / len(zs))
    w = 1 / math.sqrt(V + 1) * math.exp(-(0.8 - z.mean()) ** 2 / (2 * (V + 1)))
    assert abs(d["alive"].mean() - w) < 0.006


def test_neutral_drift_heterozygosity_and_wf_variance(oracle_mod):
    # omega = inf (c = 0), mu = 0: E[H_{t+1}] = H_t (1 - 1/(2 N_{t+1})); Var(dp) = p(1-p)/(2 N_{t+1})
    c = workloads.config(3, scale=0.001)
    sp = c["species"][0]
    sp["mu"] = 0.0
    sp["gaussian"]["omega"] = 0.0
    o = oracle_mod.Oracle(c)
    rows = workloads.initial_rows(c, 0)
    o.write_state(0, rows, None, 0)

    def freqs(r):
        b = np.unpackbits(r.view(np.uint8), axis=1, bitorder="little")  # [n, 2048]
        return (b[:, :1024] + b[:, 1024:]).sum(axis=0) / (2.0 * len(r))

    p = freqs(rows)
    H0 = (2 * p * (1 - p)).mean()
    expect = 1.0
    wf_ratio = []
    for t in range(200):
        o.step(1)
        r, _, _ = o.read_state(0)
        assert o.log(0)[-1]["n_next"] == o.log(0)[-1]["m_t"]  # everyone survives
        p2 = freqs(r)
        if t < 20:
            wf_ratio.append(((p2 - p) ** 2).mean() / ((p * (1 - p)).mean() / (2 * len(r))))
        p = p2
        expect *= 1 - 1 / (2.0 * len(r))
    H = (2 * p * (1 - p)).mean()
    assert abs(expect - 0.9048) < 0.01  # N ~ 1000, 200 steps
    # 1024 loci on 4 chromosomes: sd of the ratio ~ sqrt(Var(H)/n_eff); generous 5 %
    assert abs(H / H0 / expect - 1) < 0.05
    assert abs(np.mean(wf_ratio) - 1) < 0.08


def test_regulation_fixed_point(oracle_mod):
    # neutral: E[N_{t+1}|N_t] = 2N/(1+N/K); with selection N* = K(2w-1)
    c = workloads.config(1, scale=20.0)  # K = 20000
    c["species"][0]["gaussian"]["omega"] = 0.0
    o = run(oracle_mod, c, n_steps=1, n0=[5000])
    lam = 2 / (1 + 5000 / 20000.0)
    assert abs(o.n(0) - 5000 * lam) < 4.5 * math.sqrt(5000 * lam)
    c = workloads.config(3, scale=0.02)
    o = run(oracle_mod, c, n_steps=25)
    ns = np.array([e["n_next"] for e in o.log(0)[10:]], dtype=np.float64)
    K = c["species"][0]["K"]
    assert abs(ns.mean() / K - 0.8856) < 0.02  # K(2*0.942809-1)


def test_two_steps_equal_one_plus_one_and_checkpoint(oracle_mod):
    for which, scale, grid in [(1, 1.0, None), (3, 0.003, None), (5, 0.02, (4, 4))]:
        c = workloads.config(which, scale=scale, grid=grid)
        a = run(oracle_mod, c, n_steps=3)
        b = run(oracle_mod, c, n_steps=1)
        rows, ps, _ = b.read_state(0)
        b2 = oracle_mod.Oracle(c)  # checkpoint = rows + patch_start + step (counter-based RNG)
        b2.write_state(0, rows, ps if c["grid"] != (1, 1) else None, 1)
        b2.step(2)
        ra, pa, za = a.read_state(0)
        rb, pb, zb = b2.read_state(0)
        assert np.array_equal(ra, rb) and np.array_equal(pa, pb) and np.array_equal(za, zb)
        assert a.step_counter == b2.step_counter == 3


def test_overflow_and_extinction_flags(oracle_mod):
    c = workloads.config(1, scale=1.0)
    c["species"][0]["capacity"] = 1000
    c["species"][0]["K"] = 1e9  # lam = 2 -> M ~ 2000 > capacity
    o = run(oracle_mod, c)
    d = o.debug(0)
    assert d["m_t"] == 1000 and o.flags & 1 and o.log(0)[-1]["flags"] & 1
    full = int(d["f"].sum())
    assert full > 1000 and d["mother"][-1] == np.searchsorted(np.cumsum(d["f"]), 999, side="right")
    # fecundity mean 0 -> extinct next step, then steps are no-ops
    c = workloads.config(1, scale=1.0)
    c["species"][0]["fec_a"] = 0.0
    o = run(oracle_mod, c, n_steps=3)
    assert o.n(0) == 0 and o.flags & 2
    assert [e["n_t"] for e in o.log(0)] == [1000, 0, 0]


def test_patches_bookkeeping(oracle_mod):
    c = workloads.config(5, scale=0.05, grid=(6, 5))
    P = 30
    o = run(oracle_mod, c)
    d = o.debug(0)
    ps0 = workloads.initial_patch_start(c, 0)
    natal = np.searchsorted(ps0, d["mother"], side="right") - 1
    fa_patch = np.searchsorted(ps0, d["father"], side="right") - 1
    assert np.array_equal(natal, fa_patch)  # mating within the natal patch
    moved = d["dest"] != natal
    assert abs(moved.mean() - 0.05) < 4.5 * math.sqrt(0.05 * 0.95 / d["m_t"])
    # destination is one of the 4 torus neighbours, each direction equally likely
    x, y = natal % 6, natal // 6
    nb = np.stack([((y - 1) % 5) * 6 + x, y * 6 + (x + 1) % 6, ((y + 1) % 5) * 6 + x, y * 6 + (x - 1) % 6], axis=1)
    which = (nb[moved] == d["dest"][moved][:, None])
    assert np.all(which.sum(axis=1) == 1)
    cnt = which.sum(axis=0)
    assert ((cnt - cnt.mean()) ** 2 / cnt.mean()).sum() < stats.chi2.ppf(1 - 1e-5, 3)
    # selection uses theta of the destination patch
    th = c["species"][0]["gaussian"]["theta_patch"][d["dest"]]
    s64 = np.exp(-((d["z"].astype(np.float64) - th) ** 2) / 2.0)
    assert np.max(np.abs(d["s"] - s64) / s64) < 1e-6
    # next generation ordered by (dest, j); patch_start = histogram scan
    rows, ps, _ = o.read_state(0)
    keep = np.flatnonzero(d["alive"])
    order = keep[np.argsort(d["dest"][keep], kind="stable")]
    assert np.array_equal(rows, d["offspring"][order])
    assert np.array_equal(ps, np.concatenate([[0], np.cumsum(np.bincount(d["dest"][keep], minlength=P))]))
    # per-patch Beverton-Holt tables: lam_p = 2/(1+n_p/K_p)
    assert len(d["table_len"]) == P
    # m = 0: nobody changes patch, an emptied patch stays empty
    c0 = workloads.config(5, scale=0.05, grid=(6, 5))
    c0["species"][0]["migration"] = 0.0
    o0 = oracle_mod.Oracle(c0)
    rows0 = workloads.initial_rows(c0, 0)
    ps0 = workloads.initial_patch_start(c0, 0).copy()
    n7 = ps0[8] - ps0[7]
    rows0 = np.delete(rows0, np.arange(ps0[7], ps0[8]), axis=0)
    ps0[8:] -= n7  # patch 7 empty
    o0.write_state(0, rows0, ps0, 0)
    for _ in range(3):
        o0.step(1)
        dd = o0.debug(0)
        _, ps, _ = o0.read_state(0)
        assert ps[8] == ps[7]
        natal = np.searchsorted(ps0, dd["mother"], side="right") - 1
        assert np.array_equal(dd["dest"], natal)
        ps0 = ps


def test_two_species_capture_accounting(oracle_mod):
    c = workloads.config(4, scale=0.01)
    o = run(oracle_mod, c)
    prey, pred = o.debug(0), o.debug(1)
    le_prey = o.log(0)[-1]
    n_c = c["n0"][1]
    # R14's two scalars recomputed from the INPUT rows of the predator species and the parameters (not from
    # the oracle's own zbar_pred / attack_n): A = a*N_C is scale-free (= 0.1), zbar_C = mean predator trait
    pr = c["species"][0]["predation"]
    attack_n = pr["attack"] * n_c
    assert abs(attack_n - 0.1) < 1e-9
    rows_c = workloads.initial_rows(c, 1)
    zbar_c = float(zi_numpy(c["species"][1], rows_c).sum()) / n_c * c["species"][1]["pheno_scale"]
    rows_p = workloads.initial_rows(c, 0)
    zbar_own = float(zi_numpy(c["species"][0], rows_p).sum()) / c["n0"][0] * c["species"][0]["pheno_scale"]
    assert abs(zbar_c - zbar_own) > 1e-4                      # the two means differ, so the wrong one shows in s
    assert abs(prey["attack_n"] - attack_n) < 1e-6 and abs(prey["zbar_pred"] - zbar_c) < 1e-6
    g = np.exp(-0.5 * (prey["z"].astype(np.float64) - zbar_c) ** 2)
    s_pred = np.exp(-attack_n * g)
    cap_ref = prey["u01"] >= s_pred
    near = np.abs(prey["u01"] - s_pred) < 2e-6
    assert np.array_equal(prey["captured"].astype(bool)[~near], cap_ref[~near])
    assert le_prey["captures"] == prey["captured"].sum() == pred["cap"].sum()
    assert pred["cap"].shape[0] == n_c
    # s = s_pred * s_stab ; alive iff u01 < s ; captured individuals are dead
    s_stab = np.exp(-(prey["z"].astype(np.float64) ** 2) / 8.0)
    assert np.max(np.abs(prey["s"] - s_pred * s_stab) / (s_pred * s_stab)) < 2e-6
    assert not (prey["captured"].astype(bool) & prey["alive"].astype(bool)).any()
    # expected capture fraction = 1 - E[exp(-A g)] (numerical integral over the offspring z)
    assert abs(prey["captured"].mean() - (1 - s_pred.mean())) < 4.5 * math.sqrt(0.1 / prey["m_t"])
    # prey fecundity: logistic mean max(0, 1 + rho(1 - N/K)) = 1 + 1/3
    assert abs(prey["f"].mean() - (1 + 1 / 3.0)) < 4.5 * math.sqrt(1.34 / prey["n_t"])
    # predator fecundity table k has mean eps*k*(1 - N_C/K_C) = 1.2 k ; zero captures -> no offspring
    assert pred["table_len"][0] == 0
    f, cap = pred["f"].astype(np.float64), pred["cap"]
    assert f[cap == 0].sum() == 0
    sel = cap == 1
    assert sel.sum() > 50          # (larger capture counts: tests/test_oracle_predation.py, on a population built for it)
    assert abs(f[sel].mean() - 1.2) < 5 * math.sqrt(1.2 / sel.sum())
    assert pred["alive"].all()  # predator offspring all survive
    # A = 0 -> no captures -> predator extinct in one step
    c2 = workloads.config(4, scale=0.005)
    c2["species"][0]["predation"]["attack"] = 0.0
    o2 = run(oracle_mod, c2, n_steps=2)
    assert o2.log(0)[0]["captures"] == 0 and o2.n(1) == 0 and (o2.flags & 2)


def test_c4_reading_persists_at_small_scale(oracle_mod):
    # R14 default (prey under stabilising selection): both species persist over 60 steps at 1/200 scale
    c = workloads.config(4, scale=0.005)
    o = run(oracle_mod, c, n_steps=60)
    assert o.n(0) > 0.5 * c["n0"][0] and o.n(1) > 0.2 * c["n0"][1]


def test_residual_phenotype_noise_closed_forms(oracle_mod):
    """R17, eq. S2-14: z ~ Normal(genetic value, rho).  Pins: the residual is a
    whole number of phenotype quanta with mean 0 and variance rho^2 (+ q^2/12, Sheppard), is
    independent of the genetic value and normal; selection then sees V_P = V_G + rho^2 (survivor
    fraction: the Gaussian integral) and moves the GENETIC mean by h^2 = V_G/V_P of the phenotypic
    selection differential (breeder's equation); rho = 0 is the path without noise."""
    rho, theta = 0.5, 0.8
    c = workloads.config(2, scale=0.3)
    sp = c["species"][0]
    sp["gaussian"].update(theta0=theta, dtheta=0.0)
    sp["mu"] = 0.0
    sp["resid_sd"] = rho
    d = run(oracle_mod, c).debug(0)
    q = sp["pheno_scale"]
    g = d["zi"].astype(np.float64) * q
    z = d["z"].astype(np.float64)
    k = (z - g) / q
    assert np.array_equal(k, np.rint(k))                         # whole quanta, exact in fp32
    e = k * q
    m = len(e)
    assert abs(e.mean()) < 5 * rho / math.sqrt(m)
    assert abs(e.var() / (rho * rho + q * q / 12) - 1) < 5 * math.sqrt(2.0 / m)
    assert abs(np.corrcoef(e, g)[0, 1]) < 5 / math.sqrt(m)
    assert stats.kstest(e / rho, "norm").pvalue > 1e-3
    # the survival probability is the Gaussian of the PHENOTYPE
    assert np.allclose(d["s"], np.exp(-(z - theta) ** 2 / 2.0), rtol=2e-6, atol=1e-12)
    alive = d["alive"].astype(bool)
    VG, VP = g.var(), g.var() + rho * rho
    w = 1.0 / math.sqrt(VP + 1.0) * math.exp(-(theta - g.mean()) ** 2 / (2 * (VP + 1.0)))
    assert abs(alive.mean() - w) < 4.5 * math.sqrt(w * (1 - w) / m) + 0.002
    resp = g[alive].mean() - g.mean()
    assert abs(resp - (theta - g.mean()) * VG / (VP + 1.0)) < 5 * math.sqrt(VG / alive.sum())
    # without the noise the response would be (theta - gbar) VG / (VG + 1): a dropped term fails here
    assert abs(resp - (theta - g.mean()) * VG / (VG + 1.0)) > 5 * math.sqrt(VG / alive.sum())
    # rho = 0 is bit-identical to a configuration without the field
    c0 = workloads.config(2, scale=0.01)
    c1 = workloads.config(2, scale=0.01)
    c1["species"][0]["resid_sd"] = 0.0
    a, b = run(oracle_mod, c0, 3), run(oracle_mod, c1, 3)
    assert a.log(0) == b.log(0) and np.array_equal(a.read_state(0)[0], b.read_state(0)[0])


def _overlap_cfg(n0=2000, sA=0.975, omega=0.0, fec_a=0.0, K=1e9, L=16, capacity=8192):
    sp = species(L=L, kind="q10", r=0.5, mu=0.0, fec_a=fec_a, K=K, omega=omega, capacity=capacity)
    sp["adult_survival"] = sA
    c = cfg(sp, seed=11)
    c["n0"] = [n0]
    c["init_sd"] = 0.1
    return c


def test_overlapping_generations_lifespan(oracle_mod):
    """R18.  Pin from the paper itself: at the maximum per-step survivorship
    0.975 the average lifespan is about 40 steps (tests/golden/lifespan.txt).  A cohort
    that neither reproduces (fec_a = 0) nor is selected (omega = inf) decays as N_t ~ N_0 s^t, and
    the lifespan of its members, sum_t N_t / N_0 counting the step of birth, is 1/(1-s)."""
    sA, life = [float(x) for x in open(os.path.join(HERE, "golden", "lifespan.txt")).read().split("\n")[-2].split()]
    assert abs(1.0 / (1.0 - sA) - life) < 1e-9            # the textbook geometric mean, retyped
    n0 = 3000
    c = _overlap_cfg(n0=n0, sA=sA)
    o = oracle_mod.Oracle(c)
    o.write_state(0, workloads.initial_rows(c, 0), None, 0)
    o.step(600)
    lg = o.log(0)
    N = np.array([e["n_t"] for e in lg] + [lg[-1]["n_next"]], dtype=np.float64)
    assert all(e["m_t"] == 0 for e in lg) and N[-1] == 0   # nobody is born, everybody dies in the end
    assert (np.diff(N) <= 0).all()
    # binomial chain: N_t | N_0 has mean N_0 s^t and variance N_0 s^t (1 - s^t)
    for t in (10, 40, 100):
        mu = n0 * sA ** t
        assert abs(N[t] - mu) < 5 * math.sqrt(mu * (1 - sA ** t))
    lifespan = N[:-1].sum() / n0                           # steps lived per individual
    assert abs(lifespan - life) < 5 * math.sqrt(sA) / (1 - sA) / math.sqrt(n0)   # sd of a geometric lifetime
    # s_A = 0 is the discrete-generation path, bit for bit
    a, b = workloads.config(1), workloads.config(1)
    b["species"][0]["adult_survival"] = 0.0
    ra, rb = run(oracle_mod, a, 3), run(oracle_mod, b, 3)
    assert ra.log(0) == rb.log(0) and np.array_equal(ra.read_state(0)[0], rb.read_state(0)[0])


def test_overlapping_generations_order_selection_and_regulation(oracle_mod):
    """R18: the next generation is the staying adults (in order, rows unchanged) followed by the
    surviving offspring; an adult stays with probability s_A w(z); with overlap the Beverton-Holt
    population settles where births balance deaths."""
    sA, om = 0.6, 1.0
    c = _overlap_cfg(n0=4000, sA=sA, omega=om, fec_a=2.0, K=4000.0, L=64, capacity=32768)
    c["species"][0]["gaussian"]["theta0"] = 0.5
    o = oracle_mod.Oracle(c)
    rows0 = workloads.initial_rows(c, 0)
    o.write_state(0, rows0, None, 0)
    o.step(1)
    d = o.debug(0)
    stay = d["a_alive"].astype(bool)
    alive = d["alive"].astype(bool)
    rows1 = o.read_state(0)[0]
    assert len(rows1) == stay.sum() + alive.sum() == o.log(0)[0]["n_next"]
    assert np.array_equal(rows1[:stay.sum()], rows0[stay])
    assert np.array_equal(rows1[stay.sum():], d["offspring"][alive])
    # probability and decision
    z = rows0.astype(np.int64).sum(axis=1) * 2.0 ** -11
    assert np.allclose(d["a_s"], sA * np.exp(-(z - 0.5) ** 2 / (2 * om * om)), rtol=2e-6)
    assert np.array_equal(stay, d["a_u"] < d["a_s"])
    # the adults' uniforms are independent of their fecundity draws (two words of one block)
    assert abs(np.corrcoef(d["a_u"], d["f"].astype(np.float64))[0, 1]) < 5 / math.sqrt(len(z))
    assert stats.kstest(d["a_u"], "uniform").pvalue > 1e-3
    V = z.var()
    w = om / math.sqrt(V + om * om) * math.exp(-(0.5 - z.mean()) ** 2 / (2 * (V + om * om)))
    assert abs(stay.mean() - sA * w) < 4.5 * math.sqrt(sA * w * (1 - sA * w) / len(z))
    # regulation without selection: N* solves 1 = s_A + R0/(1 + N*/K)  =>  N* = K (R0/(1 - s_A) - 1)
    c = _overlap_cfg(n0=1000, sA=0.5, fec_a=2.0, K=1000.0, capacity=16384)
    o = oracle_mod.Oracle(c)
    o.write_state(0, workloads.initial_rows(c, 0), None, 0)
    o.step(120)
    N = np.array([e["n_t"] for e in o.log(0)[40:]], dtype=np.float64)
    assert abs(N.mean() / (1000.0 * (2.0 / 0.5 - 1.0)) - 1) < 0.03
    # the offspring get the room the adults leave: M_t <= capacity - N_t
    c = _overlap_cfg(n0=1500, sA=0.9, fec_a=2.0, K=1e9, capacity=2048)
    o = oracle_mod.Oracle(c)
    o.write_state(0, workloads.initial_rows(c, 0), None, 0)
    o.step(1)
    e = o.log(0)[0]
    assert e["m_t"] == 2048 - 1500 and e["flags"] & 1 and e["n_next"] <= 2048


def test_overlapping_generations_in_patches(oracle_mod):
    """R18 in patch mode (PAPER.md:126 patches; PAPER.md:56,170 overlapping generations -- case study
    1 is exactly this combination): an adult that stays keeps its patch and its row; patch p of the
    next generation holds its staying adults (order i) followed by the surviving offspring whose
    destination is p (order j); the adult's survival uses ITS patch's optimum; each unlinked patch
    settles at its own balance N*_p = K_p (R0 / (1 - s_A) - 1); and the paper's lifespan pin holds
    patch by patch."""
    sA, om = 0.6, 1.0
    sp = species(L=16, kind="q10", r=0.5, mu=0.0, fec_a=2.0, K=500.0, K_patch=[300.0, 500.0, 800.0, 500.0], omega=om,
                 theta_patch=[-0.3, 0.0, 0.3, 0.6], migration=0.3, capacity=16384)
    sp["adult_survival"] = sA
    c = cfg(sp, seed=12, grid=(2, 2))
    c["n0"] = [2000]
    c["init_sd"] = 0.1
    o = oracle_mod.Oracle(c)
    rows0 = workloads.initial_rows(c, 0)
    ps0 = np.array([0, 400, 1000, 1500, 2000], np.uint32)
    o.write_state(0, rows0, ps0, 0)
    o.step(1)
    d = o.debug(0)
    rows1, ps1, _ = o.read_state(0)
    stay, alive = d["a_alive"].astype(bool), d["alive"].astype(bool)
    pat0 = np.searchsorted(ps0, np.arange(2000), side="right") - 1
    k = 0
    for p in range(4):
        a = np.where(stay & (pat0 == p))[0]
        j = np.where(alive & (d["dest"] == p))[0]
        assert ps1[p] == k
        assert np.array_equal(rows1[k:k + len(a)], rows0[a])
        k += len(a)
        assert np.array_equal(rows1[k:k + len(j)], d["offspring"][j])
        k += len(j)
    assert ps1[4] == k == o.log(0)[0]["n_next"]
    z = rows0.astype(np.int64).sum(axis=1) * 2.0 ** -11
    th = np.array([-0.3, 0.0, 0.3, 0.6], np.float32)[pat0]
    assert np.allclose(d["a_s"], sA * np.exp(-(z - th) ** 2 / (2 * om * om)), rtol=2e-6)
    assert np.array_equal(stay, d["a_u"] < d["a_s"])
    # unlinked patches, no selection: per-patch balance of births and deaths
    sp2 = species(L=16, kind="q10", r=0.5, mu=0.0, fec_a=2.0, K=500.0, K_patch=[300.0, 500.0, 800.0, 500.0], omega=0.0,
                  migration=0.0, capacity=32768)
    sp2["adult_survival"] = 0.5
    c2 = cfg(sp2, seed=13, grid=(2, 2))
    c2["n0"] = [2000]
    c2["init_sd"] = 0.1
    o = oracle_mod.Oracle(c2)
    o.write_state(0, workloads.initial_rows(c2, 0), np.array([0, 500, 1000, 1500, 2000], np.uint32), 0)
    acc = np.zeros(4)
    for t in range(160):
        o.step(1)
        if t >= 60:
            acc += np.diff(o.read_state(0)[1])
    for p, K in enumerate([300.0, 500.0, 800.0, 500.0]):
        assert abs(acc[p] / 100 / (K * (2.0 / 0.5 - 1.0)) - 1) < 0.05
    # the paper's lifespan (0.975 -> 40 steps) in every patch of a non-reproducing cohort
    sp3 = species(L=16, kind="q10", r=0.5, mu=0.0, fec_a=0.0, K=1e9, omega=0.0, migration=0.5, capacity=8192)
    sp3["adult_survival"] = 0.975
    c3 = cfg(sp3, seed=14, grid=(2, 1))
    c3["n0"] = [4000]
    c3["init_sd"] = 0.1
    o = oracle_mod.Oracle(c3)
    o.write_state(0, workloads.initial_rows(c3, 0), np.array([0, 1500, 4000], np.uint32), 0)
    tot = np.zeros(2)
    prev = np.array([1500, 2500])
    for t in range(700):
        tot += prev
        o.step(1)
        now = np.diff(o.read_state(0)[1])
        assert (now <= prev).all()                       # nobody is born, adults do not move
        prev = now
    assert prev.sum() == 0
    for p, n in enumerate([1500, 2500]):
        assert abs(tot[p] / n - 40.0) < 5 * math.sqrt(0.975) / 0.025 / math.sqrt(n)
