"""Small config builders shared by the tests (no method arithmetic)."""
import numpy as np


def species(L=16, kind="q10", chrom_len=None, linkage="interval", r=0.5, xover_mean=1.0, mu=0.0,
            mut_sd=0.05, fecundity="bh", fec_a=2.0, K=1000.0, K_patch=None, omega=1.0, theta0=0.0,
            dtheta=0.0, theta_patch=None, gaussian=True, predation=None, migration=0.0, capacity=4096,
            pheno_scale=None):
    chrom_len = [L] if chrom_len is None else list(chrom_len)
    if np.isscalar(r):
        rr = []
        for c, n in enumerate(chrom_len):
            if c > 0:
                rr.append(0.5)
            rr.extend([r] * (n - 1))
        r = np.asarray(rr, dtype=np.float64)
    xm = [xover_mean] * len(chrom_len) if np.isscalar(xover_mean) else list(xover_mean)
    if pheno_scale is None:
        pheno_scale = 2.0 ** -6 if kind == "bit" else 2.0 ** -11
    return dict(n_loci=L, kind=kind, chrom_len=chrom_len, linkage=linkage,
                r=r if linkage == "interval" else None, xover_mean=xm if linkage == "poisson" else None,
                mu=mu, mut_sd=mut_sd, pheno_scale=pheno_scale, fecundity=fecundity, fec_a=fec_a, K=K,
                K_patch=K_patch,
                gaussian=dict(theta0=theta0, dtheta=dtheta, omega=omega, theta_patch=theta_patch) if gaussian else None,
                predation=predation, migration=migration, capacity=capacity)


def cfg(sp, seed=1, grid=(1, 1)):
    if isinstance(sp, dict):
        sp = [sp]
    return dict(seed=seed, grid=grid, species=sp)


def marker_parent(kind, L):
    """hap0 = all 'A' alleles, hap1 = all 'B' alleles, so a gamete exposes its phase pattern."""
    if kind == "bit":
        W = L // 32
        return np.concatenate([np.zeros(W, np.uint32), np.full(W, 0xFFFFFFFF, np.uint32)])
    return np.concatenate([np.zeros(L, np.int16), np.ones(L, np.int16)])


def phase_bits(kind, L, gam):
    if kind == "bit":
        return np.unpackbits(gam.view(np.uint8), bitorder="little")[:L].astype(np.uint8)
    return gam.astype(np.uint8)
