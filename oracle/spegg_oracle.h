/*
 * spegg_oracle.h -- C ABI of the CPU ORACLE for the sPEGG per-time-step update.
 *
 * TEST INFRASTRUCTURE ONLY.  This is the plain, slow, single-threaded, obviously
 * correct restatement of what the hot path computes (Fig. 1 A-F;
 * PAPER.md:321-330 genetics; the readings R1-R25 in DESIGN.md).  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load it.  It shares no code, header, table or constant generator with the CUDA
 * library (include/spegg.h, paper_1603_09255_b200/csrc/): the structs below are
 * the oracle's own and are deliberately NOT the library's.
 */
#ifndef SPEGG_ORACLE_H
#define SPEGG_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { ORC_BIT = 0, ORC_Q10 = 1 };              /* genome kind                   */
enum { ORC_INTERVAL = 0, ORC_POISSON = 1 };     /* linkage mode (R7 / R8)        */
enum { ORC_FEC_BH = 0, ORC_FEC_LOGISTIC = 1, ORC_FEC_CAPTURES = 2 }; /* R13/R14 */
enum { ORC_FLAG_OVERFLOW = 1, ORC_FLAG_EXTINCT = 2 };

#define ORC_TMAX 128      /* max stored thresholds per Poisson table (R5)        */
#define ORC_CAP_TABLES 32 /* capture-indexed fecundity tables (R14)              */

typedef struct {
    uint32_t n_loci;            /* L                                              */
    uint32_t genome_kind;       /* ORC_BIT: 2*(L/32) uint32 per row; ORC_Q10: 2*L int16 */
    uint32_t n_chrom;
    const uint32_t *chrom_len;  /* n_chrom entries, sum = L                       */
    uint32_t linkage_mode;
    const double *r;            /* INTERVAL: L-1 adjacent-locus recombination fractions */
    const double *xover_mean;   /* POISSON: n_chrom crossover-count means          */
    double mu;                  /* per-locus mutation probability   */
    double mut_sd;              /* Q10 mutational step sd (allelic units)          */
    float pheno_scale;          /* z = (float)zi * pheno_scale (R10)               */
    uint32_t fecundity_model;
    double fec_a;               /* BH: R0; LOGISTIC: rho; CAPTURES: conversion eps */
    double K;                   /* carrying capacity (global)                      */
    const double *K_patch;      /* per patch K (n_patches) or NULL                 */
    uint32_t sel_gaussian;      /* 1: Gaussian stabilising term present            */
    double theta0, dtheta, omega; /* omega <= 0 means infinite width (c = 0)       */
    const float *theta_patch;   /* per-patch optimum (n_patches) or NULL           */
    uint32_t sel_predation;     /* 1: predation term present                       */
    double attack;              /* a                                               */
    uint32_t predator_species;
    double migration;           /* m                                               */
    uint64_t capacity;          /* max rows per population buffer                  */
    double resid_sd;            /* R17: sd of the residual (environmental) phenotype noise, eq. S2-14
                                   (PAPER.md:327-330), phenotype units; 0 = none      */
    double adult_survival;      /* R18: overlapping generations: maximum per-step
                                   survivorship of an adult, e.g. 0.975; 0 = discrete generations */
    double mate_skew;           /* R19: shared-preference mating (eq. S2-10):
                                   the father of each egg is drawn with probability proportional to
                                   X_i^{v_m}, X_i = exp(z_i) the adult's size, v_m = mate_skew;
                                   0 = uniform mate (R2)                              */
    uint32_t encounters;        /* R20: individual-level interspecific encounters (eq. S3-2,
                                   PAPER.md:464): with sel_predation, each newborn meets this many
                                   randomly drawn individuals of predator_species; at each meeting it is
                                   captured with probability attack * e/(1+e), e = exp(-(x - delta)^2),
                                   x the consumer's and delta its own trait; the capture is credited to
                                   the consumer met.  0 = the mean-field term of R14.  <= 16      */
    uint32_t separate_sexes;    /* R21 (eqs. S2-9/S2-10: "the mother and father are drawn
                                   at random from mature males and females"): 1 = every individual is
                                   female (0) or male (1); only females lay eggs, only males father them.
                                   0 = hermaphrodites (R2)                                       */
    double fec_cost;            /* R22 (eq. S3-3: the resource's fecundity is multiplied by
                                   exp(-rho * trait^2), the cost of its defence): each egg of adult i is
                                   laid with probability exp(-fec_cost * z_i^2); 0 = no cost        */
    double assort;              /* R23: assortative mating ("random, shared preference across
                                   individuals, or assortative"): a candidate father, uniform over the
                                   mother's patch, is accepted with probability exp(-assort * (z_c - z_m)^2);
                                   up to 8 candidates, the last one is taken if none was accepted.
                                   0 = random mating (R2); not together with mate_skew / separate_sexes */
    double mother_skew;         /* R24 (eq. S2-9: "the probability that the egg comes from
                                   female i is a function of the female's relative gonadal mass",
                                   (G_i / (Omega_i + q_J Omega_i))^{v_f}): the mother of each egg is drawn
                                   among the (female) adults of the patch that laid it with probability
                                   proportional to Y_i^{v_f}, Y_i = exp(z_i) the adult's relative fecundity,
                                   v_f = mother_skew; the NUMBER of eggs of the patch stays the sum of the
                                   Poisson fecundities (R5).  0 = every adult mothers its own eggs (R1);
                                   not together with fec_cost or the CAPTURES fecundity model     */
    uint32_t monogamy;          /* R25 ("monogamy or polygynandry"): 1 = within a time step every
                                   mother has ONE mate -- the father of all her eggs is drawn once, by the
                                   rule in force (R2 uniform, R19 / R21 weighted, R23 assortative), on the
                                   words of stream PAIR addressed by the MOTHER; 0 = every egg draws its
                                   father independently (polygynandry: R2, R19, R21, R23 as they stand) */
} orc_species_params;

typedef struct {
    uint64_t seed;
    uint32_t n_species;
    uint32_t grid_w, grid_h;    /* n_patches = grid_w*grid_h; 1x1 = unstructured    */
    const orc_species_params *species;
} orc_params;

typedef struct {
    uint64_t n_t, m_t, n_next;
    int64_t sum_zi, sum_zi2;    /* over survivors, integer phenotype units         */
    uint64_t captures, near_ties;
    uint32_t flags, step;
} orc_log_entry;

typedef struct orc_sim orc_sim;

/* ---- primitives exposed for pinning (tests call them one by one) ---- */
void orc_philox4x32_10(const uint32_t key[2], const uint32_t ctr[4], uint32_t out[4]);
void orc_draw(uint64_t seed, uint32_t species, uint32_t stream, uint32_t entity,
              uint32_t block, uint32_t step, uint32_t out[4]);
double orc_exp_neg64(double lam);          /* spec'd exp(-lam), fp64 (R6)          */
float orc_expf_spec(float x);              /* spec'd exp(x), x <= 0, fp32 (R11)    */
uint32_t orc_bernoulli_threshold(double p, uint64_t *T);   /* floor(p*2^32) (R4)   */
int orc_poisson_table(double lam, uint32_t *T /* ORC_TMAX */);  /* returns len (R5) */
int orc_poisson_count(const uint32_t *T, int len, uint32_t u);
int orc_normal_table(double sigma_over_q, uint32_t *T, int cap); /* returns R; 2R thresholds (R9) */
int orc_normal_delta(const uint32_t *T, int R, uint32_t u);

/* ---- simulator ---- */
orc_sim *orc_create(const orc_params *p);
void orc_destroy(orc_sim *s);
/* rows: BIT -> uint32 [n][2W]; Q10 -> int16 [n][2L]; patch_start: n_patches+1 or NULL */
int orc_write_state(orc_sim *s, uint32_t species, uint64_t n, const void *rows,
                    const uint32_t *patch_start, uint32_t step);
/* R21: sexes of the current adults (1 = male), in row order; write after orc_write_state (which makes everybody female) */
int orc_write_sex(orc_sim *s, uint32_t species, uint64_t n, const uint8_t *sex);
int orc_read_sex(const orc_sim *s, uint32_t species, uint8_t *sex);
int orc_step(orc_sim *s, uint32_t n_steps);
uint64_t orc_n(const orc_sim *s, uint32_t species);
uint32_t orc_step_counter(const orc_sim *s);
uint32_t orc_flags(const orc_sim *s);
int orc_read_state(const orc_sim *s, uint32_t species, void *rows, uint32_t *patch_start,
                   int32_t *zi);
int orc_read_log(const orc_sim *s, uint32_t species, uint32_t first, uint32_t n, orc_log_entry *out);
uint32_t orc_log_len(const orc_sim *s, uint32_t species);

/* make one gamete from one parent row (R7/R8/R9); used by the brute-force pins */
int orc_make_gamete(const orc_sim *s, uint32_t species, const void *parent_row, uint32_t gamete /*0 maternal,1 paternal*/,
                    uint32_t entity, uint32_t step, void *out_hap);

/* debug arrays of the LAST step of `species` (valid until the next orc_step) */
typedef struct {
    uint64_t n_t, m_t;
    const uint8_t *f;          /* [n_t] fecundity                                  */
    const uint32_t *off;       /* [n_t] exclusive scan                             */
    const uint32_t *mother, *father, *dest; /* [m_t]                               */
    const float *u01, *s, *z;  /* [m_t]                                            */
    const int32_t *zi;         /* [m_t]                                            */
    const uint8_t *alive, *captured; /* [m_t]                                     */
    const void *offspring;     /* [m_t] rows                                       */
    const uint32_t *tables;    /* [n_tables][ORC_TMAX]                             */
    const uint32_t *table_len; /* [n_tables]                                       */
    uint32_t n_tables;
    float theta_t, zbar_pred, attack_n; /* derived scalars                         */
    const uint32_t *cap;       /* predator capture counts (species with CAPTURES)  */
    const uint8_t *a_alive;    /* [n_t] R18: adult i survives to the next step     */
    const float *a_u, *a_s;    /* [n_t] its uniform and survival probability       */
    const uint64_t *mate_cum;  /* [n_t] R19: inclusive running sum of the integer mating weights */
    float zbar_self;           /* R19: mean genetic value of the adults, the weights' reference */
    const uint8_t *sex_off;    /* [m_t] R21: sex of each offspring (1 = male)                 */
    const uint64_t *mom_cum;   /* [n_t] R24: inclusive running sum of the integer mothering weights */
} orc_debug_view;
int orc_debug(const orc_sim *s, uint32_t species, orc_debug_view *out);

#ifdef __cplusplus
}
#endif
#endif
