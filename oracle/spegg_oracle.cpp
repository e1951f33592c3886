/*
 * spegg_oracle.cpp -- CPU ORACLE for the sPEGG per-time-step update.
 *
 * TEST INFRASTRUCTURE ONLY (see spegg_oracle.h).  Plain single-threaded C++; no
 * blocking, fusion or reordering beyond what the paper's step order and the
 * DESIGN.md readings state.  Every function cites the passage it follows:
 *   PAPER.md:48-52   Fig. 1 A-F, the per-step loop (parents -> genes -> G->P map ->
 *                    selection -> survivors -> environment)
 *   PAPER.md:54      random mating, recombination with arbitrary linkage, mutation
 *   PAPER.md:126     patches / demes
 *   PAPER.md:325     gametes carry half the parent's alleles; per-locus mutation
 *                    probability mu; Gaussian step about the old value; fusion;
 *                    midpoint additive map
 *   PAPER.md:329     eq. S2-14 additive genotype -> phenotype
 *   PAPER.md:327-330 eq. S2-14 residual phenotype noise z ~ Normal(genetic value, rho) (R17)
 *   PAPER.md:56,170,182 overlapping generations, maximum per-step survivorship 0.975 (R18)
 *   PAPER.md:54, 273-283 (eqs. S2-9, S2-10) mating systems, weighted mothers and fathers (R19, R21, R23, R24)
 *   PAPER.md:464-475 (eqs. S3-1..S3-3) individual encounters, fecundity cost of defence (R20, R22)
 *   DESIGN.md "Readings" R1-R25 for everything the paper leaves open.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): Philox known-answer vectors, exp
 * specs vs libm, Poisson/normal table moments, brute-force gamete enumeration at
 * L <= 4, recombination fraction = r, Haldane map for the Poisson mode, Mendelian
 * invariant, selection closed forms, Wright-Fisher drift, Beverton-Holt fixed point.
 * PARITY UNPINNED BY THE PAPER (each is pinned to its READING by closed forms on hand-built
 * populations, none to a number or formula the paper prints): the two-species constants and terms
 * of R14; the trait reading X = exp(z) of R19 / R24 (the paper's X is irreversible mass, G/Omega
 * gonadal over neonate mass); R20's replacement of the S3-1/S3-2 integrals by E uniform meetings;
 * R23's acceptance kernel exp(-a d^2) and its cap of 8 candidates (the paper gives the word
 * "assortative" only); R25's pairing rule (the word "monogamy" only).
 *
 * Build: g++ -O2 -ffp-contract=off -shared -fPIC (fp contraction OFF: every fp
 * value that feeds an integer decision is a stated sequence of IEEE +,-,*,/ ops).
 */
#include "spegg_oracle.h"

#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <vector>

namespace {

/* ------------------------------------------------------------------ R3: RNG */
/* Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11): 10 rounds of
 *   (hi0,lo0) = M0*c0 ; (hi1,lo1) = M1*c2 ; c <- (hi1^c1^k0, lo1, hi0^c3^k1, lo0)
 * with the key bumped by the Weyl constants between rounds. */
void philox(const uint32_t key[2], const uint32_t ctr[4], uint32_t out[4]) {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

enum Stream { FEC = 0, SCALAR = 1, RECOMB_M = 2, RECOMB_P = 3, MUT_M = 4, MUT_P = 5, MATE = 6, MOTHER = 7, PAIR = 8 };
const uint32_t ASSORT_TRIES = 8; /* R23 */

/* R3: key = (seed_lo, seed_hi); counter = (entity, block, step, species<<8 | stream) */
void draw(uint64_t seed, uint32_t species, uint32_t stream, uint32_t entity, uint32_t block,
          uint32_t step, uint32_t out[4]) {
    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    uint32_t ctr[4] = {entity, block, step, (species << 8) | stream};
    philox(key, ctr, out);
}

/* ------------------------------------------------------- R6: spec'd exp(-lam) */
/* exp(-lam) in fp64 from +,-,*,floor only: k = floor(x*log2e + 1/2),
 * r = (x - k*ln2_hi) - k*ln2_lo, degree-14 Taylor polynomial by Horner, scale by 2^k. */
double exp_neg64(double lam) {
    if (!(lam >= 0.0)) lam = 0.0;
    if (lam > 700.0) return 0.0;
    const double x = -lam;
    const double t = x * 0x1.71547652b82fep+0;
    const double kf = std::floor(t + 0.5);
    const double r = (x - kf * 0x1.62e42fee00000p-1) - kf * 0x1.a39ef35793c76p-33;
    static const double c[15] = {
        0x1.0000000000000p+0,  0x1.0000000000000p+0,  0x1.0000000000000p-1,
        0x1.5555555555555p-3,  0x1.5555555555555p-5,  0x1.1111111111111p-7,
        0x1.6c16c16c16c17p-10, 0x1.a01a01a01a01ap-13, 0x1.a01a01a01a01ap-16,
        0x1.71de3a556c734p-19, 0x1.27e4fb7789f5cp-22, 0x1.ae64567f544e4p-26,
        0x1.1eed8eff8d898p-29, 0x1.6124613a86d09p-33, 0x1.93974a8c07c9dp-37};
    double p = c[14];
    for (int i = 13; i >= 0; --i) p = p * r + c[i];
    const int k = (int)kf;
    uint64_t bits = (uint64_t)(1023 + k) << 52;
    double scale;
    std::memcpy(&scale, &bits, 8);
    return p * scale;
}

/* ----------------------------------------------------- R11: spec'd expf(x<=0) */
/* fp32, separate mul/add (no fma): k = floor(x*log2e + 1/2), Cody-Waite with
 * ln2_hi = 0.693359375, degree-7 Taylor polynomial by Horner, scale by 2^k. */
float expf_spec(float x) {
    if (!(x <= 0.0f)) x = 0.0f;
    if (x < -87.0f) return 0.0f;
    const float t = x * 0x1.715476p+0f;
    const float kf = std::floor(t + 0.5f);
    const float r = (x - kf * 0x1.63p-1f) - kf * -0x1.bd0106p-13f;
    static const float c[8] = {0x1.000000p+0f, 0x1.000000p+0f, 0x1.000000p-1f, 0x1.555556p-3f,
                               0x1.555556p-5f, 0x1.111112p-7f, 0x1.6c16c2p-10f, 0x1.a01a02p-13f};
    float p = c[7];
    for (int i = 6; i >= 0; --i) p = p * r + c[i];
    const int k = (int)kf;
    uint32_t bits = (uint32_t)(127 + k) << 23;
    float scale;
    std::memcpy(&scale, &bits, 4);
    return p * scale;
}

/* ------------------------------------------------------------ R4: thresholds */
uint64_t bernoulli_T(double p) { /* event iff u32 < T, T = floor(p*2^32) */
    if (!(p > 0.0)) return 0;
    if (p >= 1.0) return 4294967296ull;
    return (uint64_t)std::floor(p * 4294967296.0);
}
inline uint32_t uniform_index(uint32_t u, uint32_t n) { return (uint32_t)(((uint64_t)u * n) >> 32); }
inline float u01_of(uint32_t u) { return (float)(u >> 8) * 0x1p-24f; }

/* --------------------------------------------------------- R5: Poisson table */
/* p_0 = exp(-lam), p_k = (p_{k-1}*lam)/k, F_k = F_{k-1}+p_k (fp64, this order);
 * T_k = floor(F_k*2^32); the table stores T_0..T_{len-1}, ending before the first k with
 * T_k >= 2^32-1 or at maxlen.  count(u) = #{k < len : u >= T_k}. */
int poisson_table(double lam, uint32_t *T, int maxlen) {
    double p = exp_neg64(lam);
    double F = p;
    int k = 0;
    for (;;) {
        double tk = std::floor(F * 4294967296.0);
        if (tk >= 4294967295.0) break;
        if (k == maxlen) break;
        T[k] = (uint32_t)tk;
        ++k;
        p = (p * lam) / (double)k;
        F = F + p;
    }
    return k;
}
inline int poisson_count(const uint32_t *T, int len, uint32_t u) {
    int k = 0;
    while (k < len && u >= T[k]) ++k;
    return k;
}

/* ------------------------------------------- R9: discrete-normal effect table */
/* delta/q = round(N(0,sigma^2)/q): T_k = floor(Phi((k+1/2)/(sigma/q))*2^32), k=-R..R-1,
 * R = ceil(8*sigma/q); Phi(x) = erfc(-x*sqrt(1/2))/2; delta index = -R + #{k: u >= T_k}. */
int normal_table(double sq, uint32_t *T, int cap) {
    int R = (int)std::ceil(8.0 * sq);
    if (R < 1) R = 1;
    if (2 * R > cap) return -1;
    for (int k = -R; k < R; ++k) {
        double a = (double)k + 0.5;
        double x = a / sq;
        double y = -x * 0.70710678118654752440;
        double ph = 0.5 * std::erfc(y);
        double tk = std::floor(ph * 4294967296.0);
        if (tk > 4294967295.0) tk = 4294967295.0;
        T[k + R] = (uint32_t)tk;
    }
    return R;
}
inline int normal_delta(const uint32_t *T, int R, uint32_t u) {
    int cnt = 0;
    for (int i = 0; i < 2 * R; ++i) cnt += (u >= T[i]) ? 1 : 0;
    return cnt - R;
}

/* ---------------------------------------------------------------- simulator */
const int NORMAL_CAP = 8192;
const int ENV_CAP = 65536;   /* R17: residual-noise table, sd up to 4096 phenotype quanta */

struct SpeciesDebug {
    uint64_t n_t = 0, m_t = 0;
    std::vector<uint8_t> f, alive, captured, a_alive, sex_off;
    std::vector<uint32_t> off, mother, father, dest, tables, table_len, cap;
    std::vector<float> u01, s, z, a_u, a_s;
    std::vector<uint64_t> mate_cum; /* R19 */
    std::vector<uint64_t> mom_cum;  /* R24 */
    float zbar_self = 0;
    std::vector<int32_t> zi;
    std::vector<uint32_t> off_bits; /* offspring rows, BIT */
    std::vector<int16_t> off_q;     /* offspring rows, Q10 */
    float theta_t = 0, zbar_pred = 0, attack_n = 0;
};

struct Species {
    orc_species_params p;
    std::vector<uint32_t> chrom_len, chrom_start;
    std::vector<double> r, xover_mean, K_patch;
    std::vector<float> theta_patch;
    uint32_t W = 0;       /* words per haplotype (BIT) */
    size_t row_elems = 0; /* uint32 per row (BIT) or int16 per row (Q10) */
    /* constant tables built at create */
    std::vector<uint64_t> T_recomb;               /* INTERVAL: per locus switch threshold */
    std::vector<std::vector<uint32_t>> T_xover;   /* POISSON: per chromosome */
    std::vector<uint32_t> T_mut;                  /* Poisson(L*mu) */
    std::vector<uint32_t> T_norm; int R_norm = 0; /* Q10 effects */
    std::vector<uint32_t> T_env; int R_env = 0;   /* R17: residual phenotype noise, in phenotype quanta; R_env = 0: none */
    uint64_t T_mig = 0;
    float sel_c = 0.0f; /* fp32(1/(2 omega^2)) */
    /* state */
    uint64_t n = 0;
    std::vector<uint32_t> bits;
    std::vector<int16_t> q;
    std::vector<uint32_t> patch_start;
    std::vector<int32_t> zi;
    std::vector<uint8_t> sex;   /* R21: 1 = male; all 0 without separate sexes */
    std::vector<uint32_t> cap;
    std::vector<orc_log_entry> log;
    SpeciesDebug dbg;
};

} // namespace

struct orc_sim {
    uint64_t seed = 0;
    uint32_t n_species = 0, grid_w = 1, grid_h = 1, P = 1;
    uint32_t step = 0, flags = 0;
    std::vector<Species> sp;
};

namespace {

/* R10 / PAPER.md:325,329: additive map. BIT: each allele adds +/-1 unit -> zi = 2*ones - 2L.
 * Q10: zi = sum of all 2L allelic integers (midpoint 1/2 folded into pheno_scale). */
int32_t phenotype_int(const Species &S, const uint32_t *rb, const int16_t *rq) {
    const uint32_t L = S.p.n_loci;
    if (S.p.genome_kind == ORC_BIT) {
        int ones = 0;
        for (uint32_t w = 0; w < 2 * S.W; ++w) ones += __builtin_popcount(rb[w]);
        return 2 * ones - 2 * (int32_t)L;
    }
    int32_t sum = 0;
    for (uint32_t l = 0; l < 2 * L; ++l) sum += rq[l];
    return sum;
}

/* R7 / R8: phase (which parental haplotype) at every locus of one gamete. */
void gamete_phase(const orc_sim &sim, const Species &S, uint32_t species, uint32_t gamete,
                  uint32_t entity, uint32_t step, std::vector<uint8_t> &phase) {
    const uint32_t L = S.p.n_loci;
    const uint32_t stream = gamete == 0 ? RECOMB_M : RECOMB_P;
    phase.assign(L, 0);
    if (S.p.linkage_mode == ORC_INTERVAL) {
        /* R7: s_0 ~ Bern(1/2), s_l ~ Bern(r_{l-1,l}); phase_l = s_0 ^ ... ^ s_l;
         * draw for locus l = word l%4 of RECOMB block l/4 */
        uint32_t x[4] = {0, 0, 0, 0};
        uint8_t ph = 0;
        for (uint32_t l = 0; l < L; ++l) {
            if (l % 4 == 0) draw(sim.seed, species, stream, entity, l / 4, step, x);
            uint8_t sw = ((uint64_t)x[l % 4] < S.T_recomb[l]) ? 1 : 0;
            ph ^= sw;
            phase[l] = ph;
        }
    } else {
        /* R8: per chromosome c, block c*16: x0 -> crossover count, x1>>31 -> start phase,
         * crossover k lands in interval b_k = (u_k*(len-1))>>32, u_0=x2, u_1=x3, later ones
         * from the words of blocks c*16+1.. ; phase(m) = phi ^ parity(#{k: b_k < m}). */
        for (uint32_t c = 0; c < S.p.n_chrom; ++c) {
            const uint32_t len = S.chrom_len[c], s0 = S.chrom_start[c];
            uint32_t x[4];
            draw(sim.seed, species, stream, entity, c * 16, step, x);
            const int nc = poisson_count(S.T_xover[c].data(), (int)S.T_xover[c].size(), x[0]);
            const uint8_t phi = (uint8_t)(x[1] >> 31);
            std::vector<uint32_t> b(nc);
            uint32_t y[4] = {0, 0, 0, 0};
            for (int k = 0; k < nc; ++k) {
                uint32_t u;
                if (k == 0) u = x[2];
                else if (k == 1) u = x[3];
                else {
                    if ((k - 2) % 4 == 0) draw(sim.seed, species, stream, entity, c * 16 + 1 + (k - 2) / 4, step, y);
                    u = y[(k - 2) % 4];
                }
                b[k] = uniform_index(u, len - 1);
            }
            for (uint32_t m = 0; m < len; ++m) {
                int cnt = 0;
                for (int k = 0; k < nc; ++k) cnt += (b[k] < m) ? 1 : 0;
                phase[s0 + m] = phi ^ (uint8_t)(cnt & 1);
            }
        }
    }
}

/* PAPER.md:325 gamete = half the parent's alleles, then mutation (R9, sparse form):
 * n ~ Poisson(L*mu) from MUT block 0 word 0; mutation k: position (x1*L)>>32 and effect
 * word x2 of MUT block k, applied in order after recombination. */
void make_gamete(const orc_sim &sim, const Species &S, uint32_t species, const uint32_t *pb,
                 const int16_t *pq, uint32_t gamete, uint32_t entity, uint32_t step, uint32_t *ob,
                 int16_t *oq) {
    const uint32_t L = S.p.n_loci;
    std::vector<uint8_t> phase;
    gamete_phase(sim, S, species, gamete, entity, step, phase);
    if (S.p.genome_kind == ORC_BIT) {
        for (uint32_t w = 0; w < S.W; ++w) ob[w] = 0;
        for (uint32_t l = 0; l < L; ++l) {
            const uint32_t *hap = pb + (phase[l] ? S.W : 0);
            uint32_t bit = (hap[l / 32] >> (l % 32)) & 1u;
            ob[l / 32] |= bit << (l % 32);
        }
    } else {
        for (uint32_t l = 0; l < L; ++l) oq[l] = pq[(phase[l] ? L : 0) + l];
    }
    const uint32_t mstream = gamete == 0 ? MUT_M : MUT_P;
    uint32_t x[4];
    draw(sim.seed, species, mstream, entity, 0, step, x);
    const int nm = poisson_count(S.T_mut.data(), (int)S.T_mut.size(), x[0]);
    for (int k = 0; k < nm; ++k) {
        if (k > 0) draw(sim.seed, species, mstream, entity, (uint32_t)k, step, x);
        const uint32_t pos = uniform_index(x[1], L);
        if (S.p.genome_kind == ORC_BIT) {
            ob[pos / 32] ^= 1u << (pos % 32);
        } else {
            int d = normal_delta(S.T_norm.data(), S.R_norm, x[2]);
            int v = (int)oq[pos] + d;
            if (v > 32767) v = 32767;
            if (v < -32767) v = -32767;
            oq[pos] = (int16_t)v;
        }
    }
}

uint32_t patch_of(const Species &S, uint32_t P, uint64_t i) {
    if (P == 1) return 0;
    /* patch_start is a CSR over adults sorted by patch */
    uint32_t lo = 0, hi = P;
    while (hi - lo > 1) {
        uint32_t mid = (lo + hi) / 2;
        if (S.patch_start[mid] <= i) lo = mid; else hi = mid;
    }
    /* skip empty patches that share the same start */
    while (lo + 1 < P && S.patch_start[lo + 1] <= i) ++lo;
    return lo;
}

/* R13 / R14 fecundity mean, fp64 with this exact op order (R6). */
double fecundity_mean(const Species &S, double n, double K, uint32_t cap_index) {
    switch (S.p.fecundity_model) {
    case ORC_FEC_BH: { double q = n / K; double d = 1.0 + q; return S.p.fec_a / d; }
    case ORC_FEC_LOGISTIC: { double q = n / K; double a = 1.0 - q; double b = S.p.fec_a * a; double l = 1.0 + b; return l < 0.0 ? 0.0 : l; }
    default: { double q = n / K; double a = 1.0 - q; if (a < 0.0) a = 0.0; double b = S.p.fec_a * (double)cap_index; return b * a; }
    }
}

void step_species(orc_sim &sim, uint32_t si, const std::vector<uint64_t> &N0,
                  const std::vector<int64_t> &sumzi0) {
    Species &S = sim.sp[si];
    SpeciesDebug &D = S.dbg;
    const uint32_t P = sim.P, L = S.p.n_loci, t = sim.step;
    const uint64_t N = S.n;
    orc_log_entry le;
    std::memset(&le, 0, sizeof le);
    le.step = t;
    le.n_t = N;
    D = SpeciesDebug();
    D.n_t = N;
    D.cap = S.cap; /* capture counts credited during this step's prey update (R14) */
    if (N == 0) { /* extinct species is skipped */
        le.flags |= ORC_FLAG_EXTINCT;
        sim.flags |= ORC_FLAG_EXTINCT;
        S.log.push_back(le);
        return;
    }

    /* ---- a0: derived parameters from start-of-step statistics (Fig. 1F -> A) ---- */
    uint32_t n_tables = (S.p.fecundity_model == ORC_FEC_CAPTURES) ? ORC_CAP_TABLES : P;
    D.tables.assign((size_t)n_tables * ORC_TMAX, 0);
    D.table_len.assign(n_tables, 0);
    for (uint32_t k = 0; k < n_tables; ++k) {
        double lam;
        if (S.p.fecundity_model == ORC_FEC_CAPTURES) {
            lam = fecundity_mean(S, (double)N, S.p.K, k);
        } else if (P == 1) {
            lam = fecundity_mean(S, (double)N, S.K_patch.empty() ? S.p.K : S.K_patch[0], 0);
        } else {
            double np = (double)(S.patch_start[k + 1] - S.patch_start[k]);
            lam = fecundity_mean(S, np, S.K_patch.empty() ? S.p.K : S.K_patch[k], 0);
        }
        D.table_len[k] = (uint32_t)poisson_table(lam, &D.tables[(size_t)k * ORC_TMAX], ORC_TMAX);
    }
    /* R6: theta_t = fp32(theta0 + t*dtheta), fp64, never accumulated */
    D.theta_t = (float)(S.p.theta0 + (double)t * S.p.dtheta);
    if (S.p.sel_predation) {
        const uint32_t pr = S.p.predator_species;
        const uint64_t NC = N0[pr];
        /* R14: zbar_C = fp32((sum zi / N_C) * scale); A = fp32(a * N_C) */
        D.zbar_pred = NC ? (float)(((double)sumzi0[pr] / (double)NC) * (double)sim.sp[pr].p.pheno_scale) : 0.0f;
        D.attack_n = (float)(S.p.attack * (double)NC);
    }

    /* ---- R19 ("shared preference"; eq. S2-10): the probability that
     *      adult i fathers a given egg is X_i^{v_m} / sum_k X_k^{v_m}.  The trait is read as log size,
     *      X_i = exp(z_i), so the weight is exp(v_m z_i); it is taken relative to the adults' mean
     *      zbar (fp64 sum/N*scale rounded to fp32, as zbar_C in R14) and clamped to +-16 so that the
     *      spec'd expf (x <= 0) serves: fp32, this order: d = z_i - zbar; e = v*d; e = min(max(e,-16),16);
     *      x = e - 16; w = expf_spec(x); integer weight = trunc(w * 2^40) (exact scaling).  mate_cum is
     *      the inclusive running sum in adult order (uint64, no rounding anywhere). ---- */
    /* R21 (eqs. S2-9/S2-10): with separate sexes only males father eggs: a
     * female's mating weight is 0, a male's is the weight above (with v_m = 0 every male weighs
     * trunc(expf_spec(-16) * 2^40), i.e. the father is uniform over the males of the patch). */
    const bool mate_on = S.p.mate_skew != 0.0 || S.p.separate_sexes;
    if (mate_on) {
        const float v = (float)S.p.mate_skew;
        D.zbar_self = (float)(((double)sumzi0[si] / (double)N) * (double)S.p.pheno_scale);
        D.mate_cum.resize(N);
        uint64_t run = 0;
        for (uint64_t i = 0; i < N; ++i) {
            const float z = (float)S.zi[i] * S.p.pheno_scale;
            const float d = z - D.zbar_self;
            float e = v * d;
            e = std::min(std::max(e, -16.0f), 16.0f);
            const float x = e - 16.0f;
            const float w = expf_spec(x);
            if (!S.p.separate_sexes || S.sex[i]) run += (uint64_t)(w * 0x1p40f);
            D.mate_cum[i] = run;
        }
    }

    /* ---- R24 (eq. S2-9): "For each egg, the mother and father are drawn at random
     *      ... The probability that the egg comes from female i is a function of the female's relative
     *      gonadal mass", (G_i/(Omega_i + q_J Omega_i))^{v_f}.  The relative fecundity is read as
     *      Y_i = exp(z_i) (a log-fecundity trait, as X_i = exp(z_i) in R19), so the mothering weight is
     *      exp(v_f z_i), built exactly like the mating weight of R19 (same zbar, clamp, expf_spec,
     *      integer 2^40 scaling); with separate sexes a male's weight is 0.  mom_cum is its inclusive
     *      running sum in adult order. ---- */
    const bool mom_on = S.p.mother_skew != 0.0;
    if (mom_on) {
        const float v = (float)S.p.mother_skew;
        D.zbar_self = (float)(((double)sumzi0[si] / (double)N) * (double)S.p.pheno_scale);
        D.mom_cum.resize(N);
        uint64_t run = 0;
        for (uint64_t i = 0; i < N; ++i) {
            const float z = (float)S.zi[i] * S.p.pheno_scale;
            const float d = z - D.zbar_self;
            float e = v * d;
            e = std::min(std::max(e, -16.0f), 16.0f);
            const float x = e - 16.0f;
            const float w = expf_spec(x);
            if (!S.p.separate_sexes || !S.sex[i]) run += (uint64_t)(w * 0x1p40f);
            D.mom_cum[i] = run;
        }
    }

    /* ---- a1: fecundity (Fig. 1A), one FEC block per adult ---- */
    D.f.resize(N);
    D.off.resize(N);
    for (uint64_t i = 0; i < N; ++i) {
        uint32_t x[4];
        draw(sim.seed, si, FEC, (uint32_t)i, 0, t, x);
        uint32_t tab;
        if (S.p.fecundity_model == ORC_FEC_CAPTURES) tab = std::min<uint32_t>(S.cap[i], ORC_CAP_TABLES - 1);
        else tab = patch_of(S, P, i);
        D.f[i] = (uint8_t)poisson_count(&D.tables[(size_t)tab * ORC_TMAX], (int)D.table_len[tab], x[0]);
        if (S.p.separate_sexes && S.sex[i]) D.f[i] = 0; /* R21: males lay no eggs (the draw is made and ignored) */
        if (S.p.fec_cost > 0.0 && D.f[i] > 0) {
            /* R22 (eq. S3-3): fecundity times exp(-rho z_i^2), z_i the adult's genetic value.
             * A Poisson count thinned egg by egg is Poisson with the mean multiplied, so: egg k of the
             * f_i drawn is laid iff u01(word (2+k)%4 of FEC block (2+k)/4) < c_i, fp32 in this order:
             * z = zi*scale; c = expf_spec(-(rho * (z*z))).  (Words 0, 1 of block 0 are the count and R18.) */
            const float z = (float)S.zi[i] * S.p.pheno_scale;
            const float c = expf_spec(-((float)S.p.fec_cost * (z * z)));
            uint32_t keep = 0;
            for (uint32_t k = 0; k < D.f[i]; ++k) {
                uint32_t y[4];
                draw(sim.seed, si, FEC, (uint32_t)i, (2 + k) / 4, t, y);
                if (u01_of(y[(2 + k) % 4]) < c) ++keep;
            }
            D.f[i] = (uint8_t)keep;
        }
    }
    /* ---- a2: exclusive scan ---- */
    uint64_t M = 0;
    for (uint64_t i = 0; i < N; ++i) { D.off[i] = (uint32_t)M; M += D.f[i]; }
    /* R18: with overlapping generations every adult may stay, so the offspring get what is left */
    const uint64_t m_cap = S.p.adult_survival > 0.0 ? S.p.capacity - N : S.p.capacity;
    if (M > m_cap) { /* offspring j >= m_cap do not exist */
        M = m_cap;
        le.flags |= ORC_FLAG_OVERFLOW;
        sim.flags |= ORC_FLAG_OVERFLOW;
    }
    D.m_t = M;
    le.m_t = M;

    /* ---- a3: parent assignment (Fig. 1B), mother order ---- */
    D.mother.resize(M); D.father.resize(M); D.dest.resize(M);
    D.u01.resize(M); D.s.resize(M); D.z.resize(M); D.zi.resize(M);
    D.alive.resize(M); D.captured.assign(M, 0); D.sex_off.assign(M, 0);
    for (uint64_t i = 0; i < N; ++i)
        for (uint32_t k = 0; k < D.f[i]; ++k) {
            uint64_t j = (uint64_t)D.off[i] + k;
            if (j < M) D.mother[j] = (uint32_t)i;
        }
    if (S.p.genome_kind == ORC_BIT) D.off_bits.assign(M * S.row_elems, 0);
    else D.off_q.assign(M * S.row_elems, 0);

    Species *pred = S.p.sel_predation ? &sim.sp[S.p.predator_species] : nullptr;
    const uint64_t NC = pred ? N0[S.p.predator_species] : 0;

    for (uint64_t j = 0; j < M; ++j) {
        uint32_t mo = D.mother[j];
        const uint32_t pm = patch_of(S, P, mo);
        uint32_t x[4];
        draw(sim.seed, si, SCALAR, (uint32_t)j, 0, t, x);
        /* R2: father uniform over the adults of the mother's patch, selfing allowed */
        const uint32_t base = (P == 1) ? 0 : S.patch_start[pm];
        const uint32_t np = (P == 1) ? (uint32_t)N : S.patch_start[pm + 1] - S.patch_start[pm];
        if (mom_on) {
            /* R24: the egg was counted in its patch by the adult that laid it (a1-a2: the patch's
             * number of eggs is the sum of its Poisson fecundities); its MOTHER is now drawn among the
             * adults of that patch by running sum + search, as the father in R19: total = weight of
             * the patch; 64-bit uniform from words 0,1 of block 0 of stream MOTHER (entity j);
             * target = floor(u * total / 2^64); mother = first adult of the patch whose inclusive
             * running sum exceeds (running sum before the patch) + target.  Total weight 0: unchanged. */
            const uint64_t before = base ? D.mom_cum[base - 1] : 0;
            const uint64_t total = D.mom_cum[base + np - 1] - before;
            if (total > 0) {
                uint32_t y[4];
                draw(sim.seed, si, MOTHER, (uint32_t)j, 0, t, y);
                const uint64_t u = ((uint64_t)y[0] << 32) | y[1];
                const uint64_t target = before + (uint64_t)(((unsigned __int128)u * total) >> 64);
                mo = (uint32_t)(std::upper_bound(D.mom_cum.begin() + base, D.mom_cum.begin() + base + np, target) - D.mom_cum.begin());
                D.mother[j] = mo;
            }
        }
        /* R25 ("monogamy or polygynandry"): with monogamy the father's draws are addressed by
         * the MOTHER (stream PAIR, entity = her adult index: block 0 word 0 = the uniform index of R2,
         * words 2,3 = the 64-bit uniform of R19/R21, blocks 1.. = R23's candidates), so all the eggs of
         * one mother in one step have one father; otherwise by the egg (SCALAR / MATE, entity j). */
        const bool mono = S.p.monogamy != 0;
        uint32_t xp[4] = {0, 0, 0, 0};
        if (mono) draw(sim.seed, si, PAIR, mo, 0, t, xp);
        uint32_t fa = base + uniform_index(mono ? xp[0] : x[0], np);
        if (mate_on) {
            /* R19: weighted draw among the adults of the mother's patch by running sum + search:
             * total = weight of the patch; 64-bit uniform from words 2,3 of SCALAR block 1 (R25: of PAIR
             * block 0); target = floor(u * total / 2^64); father = first adult whose inclusive running sum
             * exceeds (running sum before the patch) + target.  A patch of total weight 0 keeps R2. */
            const uint64_t before = base ? D.mate_cum[base - 1] : 0;
            const uint64_t total = D.mate_cum[base + np - 1] - before;
            if (total > 0) {
                uint32_t y[4];
                if (mono) { y[2] = xp[2]; y[3] = xp[3]; }
                else draw(sim.seed, si, SCALAR, (uint32_t)j, 1, t, y);
                const uint64_t u = ((uint64_t)y[2] << 32) | y[3];
                const uint64_t target = before + (uint64_t)(((unsigned __int128)u * total) >> 64);
                /* first index in the patch with mate_cum > target (library binary search) */
                fa = (uint32_t)(std::upper_bound(D.mate_cum.begin() + base, D.mate_cum.begin() + base + np, target) - D.mate_cum.begin());
            }
        }
        if (S.p.assort > 0.0) {
            /* R23 (assortative mating): candidate t = 0..7, uniform over the adults of the
             * mother's patch (word 2(t%2) of MATE block t/2, entity j; R25: of PAIR block 1 + t/2, entity
             * the mother), is accepted iff u01(word 2(t%2)+1) < expf_spec(-(a * (d*d))), d = z_cand -
             * z_mother (genetic values, fp32, this order); the first accepted candidate is the father,
             * else the last candidate. */
            const float a = (float)S.p.assort;
            const float zm = (float)S.zi[mo] * S.p.pheno_scale;
            for (uint32_t tr = 0; tr < ASSORT_TRIES; ++tr) {
                uint32_t y[4];
                if (mono) draw(sim.seed, si, PAIR, mo, 1 + tr / 2, t, y);
                else draw(sim.seed, si, MATE, (uint32_t)j, tr / 2, t, y);
                fa = base + uniform_index(y[2 * (tr & 1)], np);
                const float d = (float)S.zi[fa] * S.p.pheno_scale - zm;
                const float p = expf_spec(-(a * (d * d)));
                const float u = u01_of(y[2 * (tr & 1) + 1]);
                if (std::fabs(u - p) < 1e-6f) le.near_ties++;
                if (u < p) break;
            }
        }
        D.father[j] = fa;
        /* R15: dispersal drawn at birth */
        uint32_t dest = pm;
        if (P > 1 && (uint64_t)x[1] < S.T_mig) {
            uint32_t px = pm % sim.grid_w, py = pm / sim.grid_w;
            switch (x[2] >> 30) {
            case 0: py = (py + sim.grid_h - 1) % sim.grid_h; break;
            case 1: px = (px + 1) % sim.grid_w; break;
            case 2: py = (py + 1) % sim.grid_h; break;
            default: px = (px + sim.grid_w - 1) % sim.grid_w; break;
            }
            dest = py * sim.grid_w + px;
        }
        D.dest[j] = dest;
        D.u01[j] = u01_of(x[3]);
        /* R21: sex at birth = bit 0 of word 2 of SCALAR block 0 (bits 30-31 of it are the dispersal direction) */
        D.sex_off[j] = S.p.separate_sexes ? (uint8_t)(x[2] & 1u) : 0;

        /* ---- a4: gametes; offspring hap0 = maternal gamete, hap1 = paternal gamete ---- */
        uint32_t *ob = nullptr; int16_t *oq = nullptr;
        if (S.p.genome_kind == ORC_BIT) {
            ob = &D.off_bits[j * S.row_elems];
            make_gamete(sim, S, si, &S.bits[(size_t)mo * S.row_elems], nullptr, 0, (uint32_t)j, t, ob, nullptr);
            make_gamete(sim, S, si, &S.bits[(size_t)fa * S.row_elems], nullptr, 1, (uint32_t)j, t, ob + S.W, nullptr);
        } else {
            oq = &D.off_q[j * S.row_elems];
            make_gamete(sim, S, si, nullptr, &S.q[(size_t)mo * S.row_elems], 0, (uint32_t)j, t, nullptr, oq);
            make_gamete(sim, S, si, nullptr, &S.q[(size_t)fa * S.row_elems], 1, (uint32_t)j, t, nullptr, oq + L);
        }
        /* ---- a5: genotype -> phenotype (Fig. 1C) ---- */
        const int32_t zi = phenotype_int(S, ob, oq);
        /* R17, eq. S2-14: z ~ Normal(genetic value, resid_sd).  The residual is a
         * whole number k of phenotype quanta from the discrete-normal table (the sampler of R9) on
         * word 1 of SCALAR block 1; it acts on this individual's selection only and is not inherited. */
        int32_t zp = zi;
        if (S.R_env > 0) {
            uint32_t y[4];
            draw(sim.seed, si, SCALAR, (uint32_t)j, 1, t, y);
            zp += normal_delta(S.T_env.data(), S.R_env, y[1]);
        }
        const float z = (float)zp * S.p.pheno_scale;
        D.zi[j] = zi; D.z[j] = z;
        /* ---- a6: selection (Fig. 1D), fp32 in this order (R11, R14) ---- */
        float s = 1.0f;
        bool captured = false;
        int met = -1; /* R20: the consumer that captured this newborn */
        if (S.p.sel_predation && S.p.encounters > 0) {
            /* R20 ("for a given individual of either species we instead simulate a random
             * subset of possible encounters"; eq. S3-2): meeting k = 0..E-1, in order, until
             * the first capture: consumer i_k uniform over the N_C consumers (word 2(k%2) of SCALAR block
             * 2 + k/2), matching m = e/(1+e), e = expf_spec(-(d*d)), d = z - z_{i_k} (the consumer's genetic
             * value), capture probability p = v * m (v = fp32(attack)), captured iff u01(word 2(k%2)+1) < p.
             * fp32, this order.  The stabilising term below is separate: alive iff not captured and u01 < s. */
            const float v = (float)S.p.attack;
            for (uint32_t k = 0; k < S.p.encounters && NC && !captured; ++k) {
                uint32_t y[4];
                draw(sim.seed, si, SCALAR, (uint32_t)j, 2 + k / 2, t, y);
                const uint32_t ik = uniform_index(y[2 * (k & 1)], (uint32_t)NC);
                const float zc = (float)pred->zi[ik] * pred->p.pheno_scale;
                const float d = z - zc;
                const float e = expf_spec(-(d * d));
                const float m = e / (1.0f + e);
                const float p = v * m;
                const float u = u01_of(y[2 * (k & 1) + 1]);
                if (std::fabs(u - p) < 1e-6f) le.near_ties++;
                if (u < p) { captured = true; met = (int)ik; }
            }
        } else if (S.p.sel_predation) {
            float d = z - D.zbar_pred;
            float g = expf_spec(-(0.5f * (d * d)));
            float sp = expf_spec(-(D.attack_n * g));
            captured = !(D.u01[j] < sp);
            s = sp;
        }
        if (S.p.sel_gaussian) {
            float th = S.theta_patch.empty() ? D.theta_t : S.theta_patch[dest];
            float d = z - th;
            float sq = d * d;
            float ss = expf_spec(-(sq * S.sel_c));
            s = (S.p.sel_predation && S.p.encounters == 0) ? s * ss : ss;
        }
        D.s[j] = s;
        D.alive[j] = (D.u01[j] < s && !(captured && S.p.encounters > 0)) ? 1 : 0;
        if (std::fabs(D.u01[j] - s) < 1e-6f) le.near_ties++;
        if (captured) {
            D.captured[j] = 1;
            le.captures++;
            if (met >= 0) pred->cap[met] += 1; /* R20: the consumer met */
            else if (NC) { /* credit a uniformly drawn predator (SCALAR block 1 word 0) */
                uint32_t y[4];
                draw(sim.seed, si, SCALAR, (uint32_t)j, 1, t, y);
                pred->cap[uniform_index(y[0], (uint32_t)NC)] += 1;
            }
        }
    }

    /* ---- R18: overlapping generations.  After reproducing, adult i stays
     *      alive with probability s_A * w(z_i): s_A the maximum per-step survivorship (the paper's
     *      0.975 gives a lifespan of 1/(1-0.975) = 40 steps), w the Gaussian term of
     *      R11 at the adult's GENETIC value (the residual of R17 is a juvenile effect).  The uniform
     *      is word 1 of the adult's FEC block.  fp32, this order: p = s_A * w. ---- */
    D.a_alive.assign(N, 0); D.a_u.assign(N, 0.0f); D.a_s.assign(N, 0.0f);
    std::vector<uint32_t> stay;
    if (S.p.adult_survival > 0.0) {
        const float sA = (float)S.p.adult_survival;
        for (uint64_t i = 0; i < N; ++i) {
            uint32_t x[4];
            draw(sim.seed, si, FEC, (uint32_t)i, 0, t, x);
            const float u = u01_of(x[1]);
            float w = 1.0f;
            if (S.p.sel_gaussian) {
                const float z = (float)S.zi[i] * S.p.pheno_scale;
                const float th = S.theta_patch.empty() ? D.theta_t : S.theta_patch[patch_of(S, P, (uint32_t)i)];   /* its own patch's optimum */
                const float d = z - th;
                const float sq = d * d;
                w = expf_spec(-(sq * S.sel_c));
            }
            const float p = sA * w;
            D.a_u[i] = u; D.a_s[i] = p;
            D.a_alive[i] = (u < p) ? 1 : 0;
            if (std::fabs(u - p) < 1e-6f) le.near_ties++;
            if (D.a_alive[i]) stay.push_back((uint32_t)i);
        }
    }

    /* ---- a7: survivors (Fig. 1E): the next generation, patch by patch (individuals are
     *      kept grouped by patch): in patch p first its adults that stay (R18; none under R1; an adult
     *      does not move), in increasing i, then the surviving offspring whose destination is p, in
     *      increasing j.  With one patch: the staying adults, then the surviving offspring. ---- */
    std::vector<uint32_t> order;
    order.reserve(M);
    for (uint64_t j = 0; j < M; ++j) if (D.alive[j]) order.push_back((uint32_t)j);
    if (P > 1) std::stable_sort(order.begin(), order.end(), [&](uint32_t a, uint32_t b) { return D.dest[a] < D.dest[b]; });
    const uint64_t Na = stay.size(), Nn = Na + order.size();
    std::vector<uint32_t> nb; std::vector<int16_t> nq;
    if (S.p.genome_kind == ORC_BIT) nb.resize(Nn * S.row_elems); else nq.resize(Nn * S.row_elems);
    std::vector<int32_t> nzi(Nn);
    std::vector<uint8_t> nsex(Nn, 0);
    std::vector<uint32_t> nps(P + 1, 0);
    {
        uint64_t k = 0, ia = 0, io = 0;   /* next position, next staying adult, next surviving offspring */
        for (uint32_t p = 0; p < P; ++p) {
            for (; ia < Na && patch_of(S, P, stay[ia]) == p; ++ia, ++k) {   /* R18: the adults that stay keep their rows */
                const uint32_t i = stay[ia];
                if (S.p.genome_kind == ORC_BIT) std::memcpy(&nb[k * S.row_elems], &S.bits[(size_t)i * S.row_elems], S.row_elems * 4);
                else std::memcpy(&nq[k * S.row_elems], &S.q[(size_t)i * S.row_elems], S.row_elems * 2);
                nzi[k] = S.zi[i];
                nsex[k] = S.sex[i];
                nps[p + 1]++;
                le.sum_zi += S.zi[i];
                le.sum_zi2 += (int64_t)S.zi[i] * S.zi[i];
            }
            for (; io < order.size() && D.dest[order[io]] == p; ++io, ++k) {
                const uint32_t j = order[io];
                if (S.p.genome_kind == ORC_BIT) std::memcpy(&nb[k * S.row_elems], &D.off_bits[(size_t)j * S.row_elems], S.row_elems * 4);
                else std::memcpy(&nq[k * S.row_elems], &D.off_q[(size_t)j * S.row_elems], S.row_elems * 2);
                nzi[k] = D.zi[j];
                nsex[k] = D.sex_off[j];
                nps[p + 1]++;
                /* ---- a8: environment reductions (Fig. 1F), exact integers ---- */
                le.sum_zi += D.zi[j];
                le.sum_zi2 += (int64_t)D.zi[j] * D.zi[j];
            }
        }
    }
    for (uint32_t p = 0; p < P; ++p) nps[p + 1] += nps[p];
    S.bits.swap(nb); S.q.swap(nq); S.zi.swap(nzi); S.sex.swap(nsex); S.patch_start.swap(nps);
    S.n = Nn;
    S.cap.assign(Nn, 0);
    le.n_next = Nn;
    S.log.push_back(le);
}

} // namespace

extern "C" {

void orc_philox4x32_10(const uint32_t key[2], const uint32_t ctr[4], uint32_t out[4]) { philox(key, ctr, out); }
void orc_draw(uint64_t seed, uint32_t species, uint32_t stream, uint32_t entity, uint32_t block,
              uint32_t step, uint32_t out[4]) { draw(seed, species, stream, entity, block, step, out); }
double orc_exp_neg64(double lam) { return exp_neg64(lam); }
float orc_expf_spec(float x) { return expf_spec(x); }
uint32_t orc_bernoulli_threshold(double p, uint64_t *T) { *T = bernoulli_T(p); return 0; }
int orc_poisson_table(double lam, uint32_t *T) { return poisson_table(lam, T, ORC_TMAX); }
int orc_poisson_count(const uint32_t *T, int len, uint32_t u) { return poisson_count(T, len, u); }
int orc_normal_table(double sq, uint32_t *T, int cap) { return normal_table(sq, T, cap); }
int orc_normal_delta(const uint32_t *T, int R, uint32_t u) { return normal_delta(T, R, u); }

orc_sim *orc_create(const orc_params *p) {
    if (!p || !p->species || p->n_species == 0 || p->n_species > 255) return nullptr;
    orc_sim *sim = new orc_sim();
    sim->seed = p->seed;
    sim->n_species = p->n_species;
    sim->grid_w = p->grid_w ? p->grid_w : 1;
    sim->grid_h = p->grid_h ? p->grid_h : 1;
    sim->P = sim->grid_w * sim->grid_h;
    sim->sp.resize(p->n_species);
    for (uint32_t s = 0; s < p->n_species; ++s) {
        Species &S = sim->sp[s];
        S.p = p->species[s];
        const uint32_t L = S.p.n_loci;
        bool ok = L > 0 && S.p.n_chrom > 0 && S.p.chrom_len;
        if (ok) {
            uint32_t acc = 0;
            for (uint32_t c = 0; c < S.p.n_chrom; ++c) { S.chrom_start.push_back(acc); S.chrom_len.push_back(S.p.chrom_len[c]); acc += S.p.chrom_len[c]; }
            ok = acc == L;
        }
        if (ok && S.p.genome_kind == ORC_BIT) ok = (L % 32 == 0);
        if (ok && S.p.linkage_mode == ORC_INTERVAL) ok = (L == 1 || S.p.r != nullptr);
        if (ok && S.p.linkage_mode == ORC_POISSON) ok = S.p.xover_mean != nullptr;
        if (ok && S.p.fecundity_model == ORC_FEC_CAPTURES) ok = sim->P == 1;
        if (ok && S.p.sel_predation) ok = S.p.predator_species < p->n_species && S.p.predator_species != s;
        if (!ok) { delete sim; return nullptr; }
        S.W = L / 32;
        S.row_elems = S.p.genome_kind == ORC_BIT ? 2 * (size_t)S.W : 2 * (size_t)L;
        if (S.p.linkage_mode == ORC_INTERVAL) {
            S.r.assign(S.p.r, S.p.r + (L - 1));
            S.T_recomb.resize(L);
            S.T_recomb[0] = 2147483648ull; /* start phase ~ Bernoulli(1/2) */
            for (uint32_t l = 1; l < L; ++l) S.T_recomb[l] = bernoulli_T(S.r[l - 1]);
        } else {
            S.xover_mean.assign(S.p.xover_mean, S.p.xover_mean + S.p.n_chrom);
            S.T_xover.resize(S.p.n_chrom);
            for (uint32_t c = 0; c < S.p.n_chrom; ++c) {
                uint32_t T[ORC_TMAX];
                int len = poisson_table(S.xover_mean[c], T, 62);
                S.T_xover[c].assign(T, T + len);
            }
        }
        {
            uint32_t T[ORC_TMAX];
            int len = poisson_table((double)L * S.p.mu, T, ORC_TMAX);
            S.T_mut.assign(T, T + len);
        }
        if (S.p.genome_kind == ORC_Q10) {
            S.T_norm.resize(NORMAL_CAP);
            /* sigma/q with q = 2^-10 */
            S.R_norm = normal_table(S.p.mut_sd * 1024.0, S.T_norm.data(), NORMAL_CAP);
            if (S.R_norm < 0) { delete sim; return nullptr; }
        }
        if (!(S.p.assort >= 0.0 && S.p.assort <= 1e6) || (S.p.assort > 0.0 && (S.p.mate_skew != 0.0 || S.p.separate_sexes))) { delete sim; return nullptr; }
        if (!(std::fabs(S.p.mate_skew) <= 1e6) || !(S.p.fec_cost >= 0.0 && S.p.fec_cost <= 1e6)) { delete sim; return nullptr; }
        if (!(std::fabs(S.p.mother_skew) <= 1e6) || (S.p.mother_skew != 0.0 && (S.p.fec_cost > 0.0 || S.p.fecundity_model == ORC_FEC_CAPTURES))) { delete sim; return nullptr; }
        if (S.p.monogamy > 1) { delete sim; return nullptr; }
        if (S.p.encounters > 16 || (S.p.encounters && (!S.p.sel_predation || !(S.p.attack >= 0.0 && S.p.attack <= 2.0)))) { delete sim; return nullptr; }
        if (!(S.p.adult_survival >= 0.0 && S.p.adult_survival <= 1.0)) { delete sim; return nullptr; }
        if (S.p.resid_sd > 0.0) {
            S.T_env.resize(ENV_CAP);
            S.R_env = normal_table(S.p.resid_sd / (double)S.p.pheno_scale, S.T_env.data(), ENV_CAP);
            if (S.R_env < 0) { delete sim; return nullptr; }
        }
        if (S.p.K_patch) S.K_patch.assign(S.p.K_patch, S.p.K_patch + sim->P);
        if (S.p.theta_patch) S.theta_patch.assign(S.p.theta_patch, S.p.theta_patch + sim->P);
        S.T_mig = bernoulli_T(S.p.migration);
        /* R11: c = fp32(1/(2 omega^2)) from fp64; omega <= 0 -> c = 0 (no selection) */
        S.sel_c = (S.p.omega > 0.0) ? (float)(1.0 / (2.0 * (S.p.omega * S.p.omega))) : 0.0f;
        S.p.chrom_len = nullptr; S.p.r = nullptr; S.p.xover_mean = nullptr; S.p.K_patch = nullptr; S.p.theta_patch = nullptr;
        S.patch_start.assign(sim->P + 1, 0);
    }
    return sim;
}

void orc_destroy(orc_sim *s) { delete s; }

int orc_write_state(orc_sim *sim, uint32_t species, uint64_t n, const void *rows,
                    const uint32_t *patch_start, uint32_t step) {
    if (!sim || species >= sim->n_species) return -1;
    Species &S = sim->sp[species];
    if (n > S.p.capacity) return -1;
    S.n = n;
    if (S.p.genome_kind == ORC_BIT) { S.bits.assign((const uint32_t *)rows, (const uint32_t *)rows + n * S.row_elems); S.q.clear(); }
    else { S.q.assign((const int16_t *)rows, (const int16_t *)rows + n * S.row_elems); S.bits.clear(); }
    if (sim->P > 1) {
        if (!patch_start) return -1;
        S.patch_start.assign(patch_start, patch_start + sim->P + 1);
        if (S.patch_start[0] != 0 || S.patch_start[sim->P] != n) return -1;
    } else { S.patch_start.assign(2, 0); S.patch_start[1] = (uint32_t)n; }
    S.zi.resize(n);
    for (uint64_t i = 0; i < n; ++i)
        S.zi[i] = phenotype_int(S, S.bits.empty() ? nullptr : &S.bits[i * S.row_elems], S.q.empty() ? nullptr : &S.q[i * S.row_elems]);
    S.cap.assign(n, 0);
    S.sex.assign(n, 0);
    sim->step = step;
    return 0;
}

int orc_write_sex(orc_sim *sim, uint32_t species, uint64_t n, const uint8_t *sex) {
    if (!sim || species >= sim->n_species || n != sim->sp[species].n || !sex) return -1;
    for (uint64_t i = 0; i < n; ++i) sim->sp[species].sex[i] = sex[i] ? 1 : 0;
    return 0;
}

int orc_read_sex(const orc_sim *sim, uint32_t species, uint8_t *sex) {
    if (!sim || species >= sim->n_species || !sex) return -1;
    if (sim->sp[species].n) std::memcpy(sex, sim->sp[species].sex.data(), sim->sp[species].n);
    return 0;
}

int orc_step(orc_sim *sim, uint32_t n_steps) {
    if (!sim) return -1;
    for (uint32_t it = 0; it < n_steps; ++it) {
        /* all start-of-step statistics are taken before any species is updated */
        std::vector<uint64_t> N0(sim->n_species);
        std::vector<int64_t> sz(sim->n_species, 0);
        for (uint32_t s = 0; s < sim->n_species; ++s) {
            N0[s] = sim->sp[s].n;
            for (uint64_t i = 0; i < sim->sp[s].n; ++i) sz[s] += sim->sp[s].zi[i];
            std::fill(sim->sp[s].cap.begin(), sim->sp[s].cap.end(), 0u);
        }
        for (uint32_t s = 0; s < sim->n_species; ++s) step_species(*sim, s, N0, sz);
        sim->step += 1;
    }
    return 0;
}

uint64_t orc_n(const orc_sim *s, uint32_t species) { return s->sp[species].n; }
uint32_t orc_step_counter(const orc_sim *s) { return s->step; }
uint32_t orc_flags(const orc_sim *s) { return s->flags; }

int orc_read_state(const orc_sim *sim, uint32_t species, void *rows, uint32_t *patch_start, int32_t *zi) {
    if (!sim || species >= sim->n_species) return -1;
    const Species &S = sim->sp[species];
    /* (an extinct species has empty vectors, whose data() may be null: memcpy is not called with it) */
    if (rows && S.n) {
        if (S.p.genome_kind == ORC_BIT) std::memcpy(rows, S.bits.data(), S.n * S.row_elems * 4);
        else std::memcpy(rows, S.q.data(), S.n * S.row_elems * 2);
    }
    if (patch_start) std::memcpy(patch_start, S.patch_start.data(), (sim->P + 1) * 4);
    if (zi && S.n) std::memcpy(zi, S.zi.data(), S.n * 4);
    return 0;
}

uint32_t orc_log_len(const orc_sim *s, uint32_t species) { return (uint32_t)s->sp[species].log.size(); }
int orc_read_log(const orc_sim *sim, uint32_t species, uint32_t first, uint32_t n, orc_log_entry *out) {
    const Species &S = sim->sp[species];
    if ((size_t)first + n > S.log.size()) return -1;
    for (uint32_t i = 0; i < n; ++i) out[i] = S.log[first + i];
    return 0;
}

int orc_make_gamete(const orc_sim *sim, uint32_t species, const void *parent_row, uint32_t gamete,
                    uint32_t entity, uint32_t step, void *out_hap) {
    if (!sim || species >= sim->n_species) return -1;
    const Species &S = sim->sp[species];
    if (S.p.genome_kind == ORC_BIT) make_gamete(*sim, S, species, (const uint32_t *)parent_row, nullptr, gamete, entity, step, (uint32_t *)out_hap, nullptr);
    else make_gamete(*sim, S, species, nullptr, (const int16_t *)parent_row, gamete, entity, step, nullptr, (int16_t *)out_hap);
    return 0;
}

int orc_debug(const orc_sim *sim, uint32_t species, orc_debug_view *o) {
    if (!sim || species >= sim->n_species) return -1;
    const Species &S = sim->sp[species];
    const SpeciesDebug &D = S.dbg;
    o->n_t = D.n_t; o->m_t = D.m_t;
    o->f = D.f.data(); o->off = D.off.data();
    o->mother = D.mother.data(); o->father = D.father.data(); o->dest = D.dest.data();
    o->u01 = D.u01.data(); o->s = D.s.data(); o->z = D.z.data(); o->zi = D.zi.data();
    o->alive = D.alive.data(); o->captured = D.captured.data();
    o->offspring = S.p.genome_kind == ORC_BIT ? (const void *)D.off_bits.data() : (const void *)D.off_q.data();
    o->tables = D.tables.data(); o->table_len = D.table_len.data(); o->n_tables = (uint32_t)D.table_len.size();
    o->theta_t = D.theta_t; o->zbar_pred = D.zbar_pred; o->attack_n = D.attack_n;
    o->cap = D.cap.data();
    o->a_alive = D.a_alive.data(); o->a_u = D.a_u.data(); o->a_s = D.a_s.data();
    o->mate_cum = D.mate_cum.data(); o->zbar_self = D.zbar_self;
    o->sex_off = D.sex_off.data();
    o->mom_cum = D.mom_cum.data();
    return 0;
}

} /* extern "C" */
