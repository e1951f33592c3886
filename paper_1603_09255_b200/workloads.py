"""Seeded synthetic workloads: BASELINE.json's five configurations and their initial states.

This module serves BOTH the CUDA path and the oracle tests and therefore holds none of the
method's arithmetic: only parameter dicts (the neutral format both bindings accept) and numpy
random initial populations.  Recipe: the paper's case-study parameter
files are not available, so these stand in for them with the paper's structure
(multi-locus additive diploid traits PAPER.md:56, patches of equal size PAPER.md:126, two
interacting species PAPER.md:60, 1e6-1e7 individuals PAPER.md:64,122).
"""
import numpy as np

Q = 2.0 ** -10  # allelic quantum of the q10 genomes


def _interval_r(chrom_len, r_within, r_between=0.5):
    r = []
    for c, n in enumerate(chrom_len):
        if c > 0:
            r.append(r_between)
        r.extend([r_within] * (n - 1))
    return np.asarray(r, dtype=np.float64)


def smooth_theta(grid_w, grid_h, seed):
    """Per-patch optimum: U(-1,1), one 5-point torus average (fp64), rounded to fp32."""
    rng = np.random.default_rng(seed + 7919)
    th = rng.uniform(-1.0, 1.0, size=(grid_h, grid_w))
    sm = (th + np.roll(th, 1, 0) + np.roll(th, -1, 0) + np.roll(th, 1, 1) + np.roll(th, -1, 1)) / 5.0
    return sm.astype(np.float32).reshape(-1)


def config(which, scale=1.0, grid=None, seed=None):
    """BASELINE.json config `which` (1..5).  `scale` shrinks N0/K/capacity for tests; the
    two-species attack rate is divided by `scale` so that a*N_C is unchanged."""
    def cap(n0):
        c = int(np.ceil(n0 * 1.125 / 1024.0)) * 1024
        return max(c, 2048)

    if which == 1:
        n0 = max(int(round(1000 * scale)), 8)
        sp = dict(n_loci=16, kind="q10", chrom_len=[16], linkage="interval", r=_interval_r([16], 0.5),
                  xover_mean=None, mu=1e-3, mut_sd=0.05, pheno_scale=2.0 ** -11, fecundity="bh", fec_a=2.0,
                  K=float(n0), K_patch=None, gaussian=dict(theta0=0.0, dtheta=0.0, omega=1.0, theta_patch=None),
                  predation=None, migration=0.0, capacity=max(2048, cap(n0)))
        return dict(name="C1", seed=1 if seed is None else seed, grid=(1, 1), species=[sp], n0=[n0], steps=100,
                    init_sd=0.1)
    if which == 2:
        n0 = max(int(round(100_000 * scale)), 8)
        cl = [16] * 4
        sp = dict(n_loci=64, kind="q10", chrom_len=cl, linkage="interval", r=_interval_r(cl, 0.05),
                  xover_mean=None, mu=1e-4, mut_sd=0.05, pheno_scale=2.0 ** -11, fecundity="bh", fec_a=2.0,
                  K=float(n0), K_patch=None, gaussian=dict(theta0=0.0, dtheta=0.01, omega=1.0, theta_patch=None),
                  predation=None, migration=0.0, capacity=131072 if scale == 1.0 else cap(n0))
        return dict(name="C2", seed=2 if seed is None else seed, grid=(1, 1), species=[sp], n0=[n0], steps=1000,
                    init_sd=0.1)
    if which == 3:
        n0 = max(int(round(1_000_000 * scale)), 8)
        cl = [256] * 4
        sp = dict(n_loci=1024, kind="bit", chrom_len=cl, linkage="poisson", r=None, xover_mean=[1.0] * 4,
                  mu=1e-5, mut_sd=0.0, pheno_scale=2.0 ** -6, fecundity="bh", fec_a=2.0, K=float(n0),
                  K_patch=None, gaussian=dict(theta0=0.0, dtheta=0.0, omega=2.0, theta_patch=None),
                  predation=None, migration=0.0, capacity=1_179_648 if scale == 1.0 else cap(n0))
        return dict(name="C3", seed=3 if seed is None else seed, grid=(1, 1), species=[sp], n0=[n0], steps=200,
                    init_sd=None)
    if which == 4:
        n_prey = max(int(round(1_000_000 * scale)), 16)
        n_pred = max(int(round(100_000 * scale)), 8)
        cl = [32] * 8
        common = dict(n_loci=256, kind="q10", chrom_len=cl, linkage="interval", r=_interval_r(cl, 0.01),
                      xover_mean=None, mu=1e-5, mut_sd=0.05, pheno_scale=2.0 ** -11, K_patch=None, migration=0.0)
        prey = dict(common, fecundity="logistic", fec_a=1.0, K=1.5 * n_prey,
                    gaussian=dict(theta0=0.0, dtheta=0.0, omega=2.0, theta_patch=None),
                    predation=dict(attack=1e-6 / scale, predator=1),
                    capacity=1_703_936 if scale == 1.0 else cap(int(1.5 * n_prey)))
        pred = dict(common, fecundity="captures", fec_a=2.0, K=2.5 * n_pred, gaussian=None, predation=None,
                    capacity=327_680 if scale == 1.0 else cap(int(2.9 * n_pred)))
        return dict(name="C4", seed=4 if seed is None else seed, grid=(1, 1), species=[prey, pred],
                    n0=[n_prey, n_pred], steps=500, init_sd=0.1)
    if which == 5:
        gw, gh = grid if grid is not None else (64, 64)
        per = max(int(round(1000 * scale)), 4)
        P = gw * gh
        cl = [32] * 4
        sd = 5 if seed is None else seed
        sp = dict(n_loci=128, kind="q10", chrom_len=cl, linkage="interval", r=_interval_r(cl, 0.05),
                  xover_mean=None, mu=1e-5, mut_sd=0.05, pheno_scale=2.0 ** -11, fecundity="bh", fec_a=2.0,
                  K=float(per), K_patch=np.full(P, float(per)),
                  gaussian=dict(theta0=0.0, dtheta=0.0, omega=1.0, theta_patch=smooth_theta(gw, gh, sd)),
                  predation=None, migration=0.05,
                  capacity=4_718_592 if (scale == 1.0 and grid is None) else cap(per * P))
        return dict(name="C5", seed=sd, grid=(gw, gh), species=[sp], n0=[per * P], steps=200, init_sd=0.1)
    if which == 6:
        return sweep_config(scale=scale, seed=seed, n_patches=None if grid is None else grid[0] * grid[1])
    raise ValueError(which)


def sweep_config(n_patches=None, per_patch=50_000, scale=1.0, seed=None, first_patch=0, total_patches=None):
    """S6, the paper-shaped sweep (Fig. S5): P UNLINKED
    patches (m = 0), i.e. independent replicates, each governed by its own parameter combination
    (carrying capacity K_p and optimum theta_p), about 50,000 individuals per patch, few freely
    recombining loci with mutation (case study 1 has 5; rows are 16-byte multiples, so 8 here), 250
    steps.  `first_patch` / `total_patches` cut a block of patches out of a larger sweep (the
    parameters of patch p do not depend on how the sweep is split), which is how it shards."""
    P = 16 if n_patches is None else int(n_patches)
    T = P if total_patches is None else int(total_patches)
    per = max(int(round(per_patch * scale)), 4)
    sd = 6 if seed is None else seed
    idx = np.arange(first_patch, first_patch + P, dtype=np.float64)
    # the sweep's parameter grid: optimum from -1 to 1 across the sweep, capacity 60-100 % of the start size
    theta = (-1.0 + 2.0 * (idx + 0.5) / T).astype(np.float32)
    Kp = np.floor(per * (0.6 + 0.4 * ((idx * 7.0) % 10.0) / 9.0))
    cl = [1] * 8
    n0 = per * P
    cap = int(np.ceil(n0 * 1.125 / 1024.0)) * 1024
    sp = dict(n_loci=8, kind="q10", chrom_len=cl, linkage="interval", r=_interval_r(cl, 0.5),
              xover_mean=None, mu=1e-3, mut_sd=0.05, pheno_scale=2.0 ** -11, fecundity="bh", fec_a=2.0,
              K=float(per), K_patch=Kp, gaussian=dict(theta0=0.0, dtheta=0.0, omega=1.0, theta_patch=theta),
              predation=None, migration=0.0, capacity=max(cap, 2048))
    return dict(name="S6", seed=sd, grid=(P, 1), species=[sp], n0=[n0], steps=250, init_sd=0.1,
                first_patch=first_patch, total_patches=T)


def initial_rows(cfg, species, n=None, seed=None):
    """iid initial genomes: bit -> fair bits; q10 -> round(N(0, init_sd^2)/q) as int16."""
    sp = cfg["species"][species]
    n = cfg["n0"][species] if n is None else n
    rng = np.random.default_rng((cfg["seed"] if seed is None else seed) * 1000003 + species)
    L = sp["n_loci"]
    if sp["kind"] == "bit":
        return rng.integers(0, 2 ** 32, size=(n, 2 * (L // 32)), dtype=np.uint64).astype(np.uint32)
    sd = cfg.get("init_sd") or 0.1
    v = np.rint(rng.normal(0.0, sd, size=(n, 2 * L)) / Q)
    return np.clip(v, -32767, 32767).astype(np.int16)


def initial_sex(cfg, species, n=None, seed=None):
    """iid initial sexes (1 = male), probability 1/2, for species with separate_sexes (R21)."""
    n = cfg["n0"][species] if n is None else n
    rng = np.random.default_rng((cfg["seed"] if seed is None else seed) * 7919 + 17 + species)
    return rng.integers(0, 2, size=n).astype(np.uint8)


def initial_patch_start(cfg, species):
    w, h = cfg["grid"]
    P = w * h
    if P == 1:
        return None
    per = cfg["n0"][species] // P
    return (np.arange(P + 1, dtype=np.uint64) * per).astype(np.uint32)
