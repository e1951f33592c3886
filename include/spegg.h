/*
 * spegg.h -- C ABI of libspegg: the B200-native per-time-step update of an individual-based,
 * forward-time, multi-locus diploid population (the hot path of sPEGG, arXiv 1603.09255).
 *
 * One call of spegg_step() performs, for every species and entirely on the GPU, the loop of the
 * paper's Fig. 1:
 *   A  parents identified, number of neonates determined   (Poisson fecundity + exclusive scan)
 *   B  parents assigned to neonates, genes transmitted      (recombination + mutation)
 *   C  genotype -> phenotype map                             (additive, eq. S2-14)
 *   D  selection updates phenotypes incl. mortality risk    (Gaussian / predation survival)
 *   E  survivors identified, dead removed                    (stable stream compaction)
 *   F  environment updated from the survivors' phenotypes   (exact integer reductions, counts)
 * plus migration between patches.  What the paper leaves open (RNG, samplers,
 * density regulation, ...) is fixed by the readings R1-R25 in DESIGN.md.
 *
 * Conventions
 *   - Plain C, no exceptions.  Every call returns an int: 0 = SPEGG_OK, <0 = error code
 *     (spegg_strerror gives text).  A failed call leaves the simulation unchanged.
 *   - OWNERSHIP: the caller owns all device memory (one workspace block, e.g. a torch uint8
 *     tensor) and the CUDA stream.  The handle owns a small host struct, the captured CUDA graph
 *     and host copies of the parameter arrays.  spegg_destroy never frees caller memory.
 *   - Pointers named d_* are DEVICE pointers; `genomes` in write/read_state is host or device
 *     as said by the *_is_device argument; everything else is a HOST pointer.
 *   - Population rows ("one contiguous row per individual"):
 *       SPEGG_BIT : 2*W uint32, W = n_loci/32: [hap0 words | hap1 words]; locus l is bit l%32
 *                   (LSB first) of word l/32; hap0 is the haplotype received from the mother.
 *       SPEGG_Q10 : 2*L int16: [hap0 | hap1], allelic value = k * 2^-10.
 *   - spegg_step is asynchronous on the caller's stream and never touches the host afterwards;
 *     population counts stay on the device (no host sync per generation).
 */
#ifndef SPEGG_H
#define SPEGG_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SPEGG_ABI_VERSION 9u

enum { SPEGG_OK = 0, SPEGG_EINVAL = -1, SPEGG_ENOMEM = -2, SPEGG_ECUDA = -3, SPEGG_ERANGE = -4,
       SPEGG_ESTATE = -5,
       SPEGG_ELIMIT = -6 };  /* size above the fixed maximum of an entry point that owns no memory */

enum { SPEGG_BIT = 0, SPEGG_Q10 = 1 };                 /* genome_kind                        */
enum { SPEGG_INTERVAL = 0, SPEGG_POISSON = 1 };        /* linkage_mode (R7 / R8)             */
enum { SPEGG_FEC_BEVERTON_HOLT = 0,                    /* lam = R0/(1+n/K)            (R13)  */
       SPEGG_FEC_LOGISTIC = 1,                         /* lam = max(0, 1+rho(1-n/K))  (R14)  */
       SPEGG_FEC_CAPTURES = 2 };                       /* lam = eps*cap_i*max(0,1-N/K) (R14) */
enum { SPEGG_FLAG_OVERFLOW = 1u,  /* M_t exceeded capacity; offspring j >= capacity dropped */
       SPEGG_FLAG_EXTINCT = 2u }; /* a species reached N = 0; its further steps are no-ops   */

#define SPEGG_TMAX 128       /* max stored thresholds of a Poisson table (R5)                */
#define SPEGG_CAP_TABLES 32  /* capture-indexed fecundity tables (R14)                       */

/* Genetic architecture and ecology of one species (Fig. S4 :495). */
typedef struct spegg_species_params {
    uint32_t n_loci;            /* L; SPEGG_BIT needs L % 32 == 0                            */
    uint32_t genome_kind;
    uint32_t n_chrom;
    const uint32_t *chrom_len;  /* [n_chrom], sum = L; SPEGG_BIT: each a multiple of 32      */
    uint32_t linkage_mode;
    const double *r;            /* INTERVAL: [L-1] probability that the phase switches between
                                   adjacent loci: the recombination fraction, normally in [0, 0.5]
                                   (0.5 across chromosome boundaries).  Any value in [0, 1) is
                                   accepted and means what it says (above 0.5: negative interference);
                                   outside [0, 1): SPEGG_EINVAL                               */
    const double *xover_mean;   /* POISSON: [n_chrom] mean crossover count per chromosome    */
    double mu;                  /* per-locus mutation probability             */
    double mut_sd;              /* Q10: sd of the Gaussian mutational step, allelic units    */
    float pheno_scale;          /* z = (float)zi * pheno_scale; BIT: zi = 2*ones-2L (each
                                   allele +-1), Q10: zi = sum of the 2L allelic integers     */
    uint32_t fecundity_model;
    double fec_a;               /* BH: R0; LOGISTIC: rho; CAPTURES: conversion efficiency    */
    double K;                   /* carrying capacity                                         */
    const double *K_patch;      /* [n_patches] per-patch K, or NULL (then K for every patch) */
    uint32_t sel_gaussian;      /* 1: s *= exp(-(z-theta)^2/(2 omega^2))                     */
    double theta0, dtheta;      /* theta_t = theta0 + t*dtheta                               */
    double omega;               /* <= 0: infinite width (everyone passes this term)          */
    const float *theta_patch;   /* [n_patches] optimum of the DESTINATION patch, or NULL     */
    uint32_t sel_predation;     /* 1: s *= exp(-a*N_C*exp(-(z-zbar_C)^2/2)), captures counted */
    double attack;              /* a                                                         */
    uint32_t predator_species;  /* index of the species whose N_C, zbar_C enter the term     */
    double migration;           /* m: probability that a newborn disperses to one of the 4
                                   torus neighbours of its natal patch (R15)                 */
    uint64_t capacity;          /* rows per population buffer (>= any N_t, M_t), < 2^31      */
    double resid_sd;            /* rho: sd of the residual (environmental) phenotype noise,
                                   z ~ Normal(genetic value, rho), eq. S2-14,
                                   in phenotype units; 0 = none.  Sampled as whole phenotype
                                   quanta (pheno_scale); rho / pheno_scale <= 4096           */
    double adult_survival;      /* s_A: overlapping generations.  After
                                   reproducing, an adult stays alive with probability
                                   s_A * w(z) (w: the Gaussian term at its genetic value; the
                                   paper's maximum survivorship is 0.975 = a lifespan of 40
                                   steps); in every patch the next generation is its staying
                                   adults, in order (an adult keeps its patch; its survival uses
                                   that patch's optimum), then the surviving offspring that
                                   land there, and M_t <= capacity - N_t.
                                   0 = discrete generations                                  */
    double mate_skew;           /* v_m: shared-preference mating (eq. S2-10,
                                   PAPER.md:281-283): the father of each egg is drawn, among
                                   the adults of the mother's patch, with probability
                                   proportional to X_i^{v_m}, X_i = exp(z_i) (z_i the adult's
                                   genetic value), by integer running sum + search (R19).
                                   0 = uniform mate (R2).  |v_m| <= 1e6                      */
    uint32_t encounters;        /* E: individual-level interspecific encounters (
                                   eq. S3-2; R20).  With sel_predation, each
                                   newborn meets E uniformly drawn adults of predator_species,
                                   in order, until the first capture; a meeting captures with
                                   probability attack * e/(1+e), e = exp(-(x - delta)^2), x the
                                   consumer's and delta the newborn's trait (attack <= 2), and
                                   the capture is credited to the consumer met.  0 = the
                                   mean-field term of R14.  E <= 16                          */
    uint32_t separate_sexes;    /* 1: every individual is female (0) or male (1) (eqs. S2-9 /
                                   S2-10; R21): only females lay eggs, only
                                   males father them (uniform over the males of the mother's
                                   patch, or by mate_skew's weights among them); sex at birth
                                   is a fair coin; a patch without males mates as R2.
                                   spegg_write_state makes everybody female: follow it with
                                   spegg_write_sex.  0 = hermaphrodites (R2)                 */
    double fec_cost;            /* rho: fecundity cost of defence (eq. S3-3; R22): the
                                   fecundity of adult i is multiplied by exp(-rho z_i^2) -- each of
                                   the eggs drawn for it is laid with that probability (a thinned
                                   Poisson count is Poisson with the mean multiplied).  0 = none  */
    double assort;              /* a: assortative mating (R23): a candidate father,
                                   uniform over the mother's patch, is accepted with probability
                                   exp(-a (z_c - z_m)^2) (genetic values); up to 8 candidates,
                                   the last one is taken if none was accepted.  0 = random
                                   mating (R2).  Not together with mate_skew / separate_sexes    */
    double mother_skew;         /* v_f: mothers drawn by relative fecundity (eq. S2-9, PAPER.md:273-275;
                                   R24): the mother of each egg is drawn, among the (female) adults
                                   of the patch that laid it, with probability proportional to
                                   Y_i^{v_f}, Y_i = exp(z_i), by integer running sum + search as the
                                   father of R19; the NUMBER of eggs of a patch stays the sum of its
                                   adults' Poisson fecundities.  0 = every adult mothers its own eggs.
                                   |v_f| <= 1e6; not with fec_cost or SPEGG_FEC_CAPTURES          */
    uint32_t monogamy;          /* 1: within a time step every mother has ONE mate ("monogamy or polygynandry",
                                   PAPER.md:54; R25): the father of all her eggs is drawn once, by the
                                   rule in force (uniform, mate_skew, separate_sexes, assort), on draws
                                   addressed by the mother.  0 = every egg draws its father (polygynandry) */
} spegg_species_params;

typedef struct spegg_params {
    uint32_t struct_size;       /* sizeof(spegg_params)                                      */
    uint32_t abi_version;       /* SPEGG_ABI_VERSION                                         */
    uint64_t seed;              /* Philox key (R3)                                           */
    uint32_t n_species;         /* 1..8; species are updated in index order                 */
    uint32_t grid_w, grid_h;    /* torus of patches; 1x1 = unstructured                      */
    uint32_t debug;             /* 1: every intermediate of the step is materialised and can
                                   be read with spegg_read_debug (slower, same results)      */
    uint32_t log_capacity;      /* per-step log ring entries (0 -> 4096)                     */
    uint32_t flags;             /* reserved, 0                                               */
    const spegg_species_params *species;
} spegg_params;

typedef struct spegg_log_entry {
    uint64_t n_t, m_t, n_next;  /* adults at start, offspring produced, survivors            */
    int64_t sum_zi, sum_zi2;    /* over survivors, integer phenotype units (exact)           */
    uint64_t captures;          /* predation captures this step                              */
    uint64_t near_ties;         /* decisions with |u01 - s| < 1e-6 (reported, north_star)    */
    uint32_t flags, step;
} spegg_log_entry;

/* Device pointers into the workspace; valid until the next spegg_step. debug = 1 only.      */
typedef struct spegg_debug_view {
    uint64_t n_t, m_t;
    const uint8_t *d_f;         /* [n_t] fecundity                                           */
    const uint32_t *d_off;      /* [n_t] exclusive scan of f                                 */
    const uint32_t *d_mother, *d_father, *d_dest; /* [m_t]                                   */
    const float *d_u01, *d_s;   /* [m_t] survival uniform, survival probability              */
    const int32_t *d_zi;        /* [m_t] integer phenotype                                   */
    const uint8_t *d_alive, *d_captured; /* [m_t]                                            */
    const void *d_offspring;    /* [m_t] rows                                                */
    const uint32_t *d_tables;   /* [n_tables][SPEGG_TMAX] fecundity thresholds               */
    const uint32_t *d_table_len;/* [n_tables]                                                */
    uint32_t n_tables;
    float theta_t, zbar_pred, attack_n;
    const uint32_t *d_cap;      /* [n_t] capture counts (SPEGG_FEC_CAPTURES species)          */
    const uint8_t *d_a_alive;   /* [n_t] adult stays alive (adult_survival > 0)               */
    const float *d_a_u, *d_a_s; /* [n_t] its uniform and survival probability                 */
    const uint64_t *d_mate_cum; /* [n_t] inclusive running sum of the integer mating weights
                                   (mate_skew != 0, R19)                                      */
    float zbar_self;            /* the weights' reference: mean genetic value of the adults   */
    const uint8_t *d_sex_off;   /* [m_t] sex of each offspring, 1 = male (separate_sexes, R21) */
    const uint64_t *d_mom_cum;  /* [n_t] inclusive running sum of the integer mothering weights
                                   (mother_skew != 0, R24)                                    */
} spegg_debug_view;

typedef struct spegg_sim spegg_sim;

/* PAPER.md:116 ("the data for each individual ... is stored in ... vectors" of one species object) and
 * PAPER.md:122 (10^6-10^7 individuals in GPU memory): the storage of a simulation.  Validates `p` and
 * returns the device bytes spegg_create needs (two population buffers of `capacity` rows per species
 * + index / scan / table / log arrays).  p, bytes: HOST.  SPEGG_EINVAL on bad parameters (L not a
 * multiple of 32 / 64 for bit genomes, chromosome lengths not summing to L, rates outside [0,1],
 * capacity 0 or >= 2^31, combinations DESIGN.md lists as unsupported); nothing is allocated. */
int spegg_workspace_bytes(const spegg_params *p, uint64_t *bytes);

/* PAPER.md:50-54, :116 and Fig. S4: a species is a genetic architecture (loci, linkage,
 * mutation) plus an ecology (mating, fecundity, selection, migration), set up once before the loop of
 * Fig. 1.  Builds the constant threshold tables (Bernoulli, Poisson, discrete normal: readings R4-R9),
 * uploads them and captures the step graphs on `cuda_stream` (a cudaStream_t; 0 = a private stream).
 * d_workspace: DEVICE memory, 256-byte aligned, at least spegg_workspace_bytes() (else SPEGG_ENOMEM);
 * it stays the caller's.  Populations start empty.  SPEGG_ECUDA wraps CUDA errors. */
int spegg_create(const spegg_params *p, void *d_workspace, uint64_t bytes, void *cuda_stream,
                 spegg_sim **out);

/* Fig. S4 `Initialize()` (the user-supplied initial state of every individual) and
 * PAPER.md:126 (individuals belong to patches): loads a whole population of `species` (n rows in the
 * row layout above, n <= capacity else SPEGG_ERANGE) and sets the global step counter t (R16).
 * genomes: host or device as said by genomes_is_device.  patch_start: HOST [n_patches+1] CSR of the
 * rows, sorted by patch (NULL iff 1x1 grid; SPEGG_EINVAL if inconsistent with n).
 * Serves as initialisation and as "resume": with the counter-based RNG the state (rows, patch_start,
 * step, seed) is a complete checkpoint.  Resets that species' step accumulators AND ITS LOG (the next
 * step writes log index 0); with separate sexes everybody is female until spegg_write_sex.
 * Synchronises the stream. */
int spegg_write_state(spegg_sim *s, uint32_t species, uint64_t n, const void *genomes,
                      int genomes_is_device, const uint32_t *patch_start, uint32_t step);

/* Eqs. S2-9 / S2-10 (mothers and fathers are drawn from mature females and males;
 * R21): sexes of the current adults of `species` (separate_sexes = 1, else SPEGG_ESTATE), in the row
 * order of spegg_write_state / spegg_read_state: HOST [n] bytes, 0 = female, non-zero = male; n must
 * be the current population size (SPEGG_ERANGE).  Synchronises the stream. */
int spegg_write_sex(spegg_sim *s, uint32_t species, uint64_t n, const uint8_t *sex);
/* Eqs. S2-9 / S2-10 (R21): the sexes back, HOST [cap_bytes >= n] (else SPEGG_ERANGE). */
int spegg_read_sex(spegg_sim *s, uint32_t species, uint8_t *sex_out, uint64_t cap_bytes);

/* Fig. 1 A-F: n_steps passes of the per-time-step loop -- parents and neonate numbers
 * (A), genes transmitted (B; recombination and mutation PAPER.md:54, :325), genotype -> phenotype (C;
 * eq. S2-14), selection (D), survivors kept (E), environment updated (F) -- for every
 * species in index order, plus dispersal between patches.  Enqueues the steps on the
 * stream and returns; no host synchronisation, population counts never leave the device.  Never fails
 * for model reasons: overflow / extinction set sticky device flags (spegg_status).  n_steps is split
 * greedily into captured graphs of 16, 8, 4, 2 and 1 steps (inside a graph consecutive steps' kernels
 * overlap through programmatic edges); the trajectory does not depend on how n_steps is split. */
int spegg_step(spegg_sim *s, uint32_t n_steps);

/* Fig. 1 E ("surviving individuals are identified") and PAPER.md:126 (patches): synchronises,
 * then copies the current adults of `species` out in their stable order (staying adults, then offspring
 * in birth order j; patch by patch in patch mode).  Any output may be NULL.  n, step: HOST scalars.
 * genomes_out: host or device buffer of cap_bytes; SPEGG_ERANGE if too small (*n is still set).
 * patch_start_out: HOST [n_patches+1].  zi_out: HOST [n] integer genetic values (z = zi * pheno_scale,
 * eq. S2-14).  Uses the idle population buffer as staging; the simulation is unchanged. */
int spegg_read_state(spegg_sim *s, uint32_t species, uint64_t *n, uint32_t *step,
                     void *genomes_out, int genomes_is_device, uint64_t cap_bytes,
                     uint32_t *patch_start_out, int32_t *zi_out);

/* Fig. 1 F ("the environment is updated" from the survivors' phenotypes): the per-step
 * record of N_t, M_t, N_{t+1}, exact integer sums of z and z^2 over the survivors, captures, near-ties
 * and flags.  Synchronises and copies log entries [first, first + n) to HOST out (at most two device
 * copies, one per side of the ring wrap); index 0 is the first step taken since the last
 * spegg_write_state of that species.  *n_avail (nullable) receives the number of entries written so
 * far; n = 0 only queries it.  SPEGG_ERANGE if the span is not (or no longer, ring of log_capacity)
 * available. */
int spegg_read_log(spegg_sim *s, uint32_t species, uint32_t first, uint32_t n,
                   spegg_log_entry *out, uint32_t *n_avail);

/* Fig. 1 A-E intermediates: synchronises; fills DEVICE pointers (into the caller's
 * workspace, valid until the next spegg_step) to every intermediate of the last step -- fecundities,
 * offsets, parents, destinations, uniforms, survival probabilities, genetic values, decisions, offspring
 * rows, derived tables.  debug = 1 only, else SPEGG_ESTATE. */
int spegg_read_debug(spegg_sim *s, uint32_t species, spegg_debug_view *out);

/* Fig. 1 A, E: what the loop cannot express as a count -- synchronises; returns the
 * sticky flags: SPEGG_FLAG_OVERFLOW (some step's neonates exceeded `capacity`; offspring j >= capacity
 * were never born) and SPEGG_FLAG_EXTINCT (a species reached N = 0 and is skipped from then on). */
int spegg_status(spegg_sim *s, uint32_t *flags);

/* Fig. 1 as launched: number of kernel launches one step replays (graph kernel nodes);
 * bench.py's `gpu_launches` claim. */
int spegg_launches_per_step(const spegg_sim *s, uint32_t *n);

/* Fig. 1 B-E timed: CUDA-event timing of the dominant kernel.  When enabled, spegg_step
 * launches the kernels directly (no graph) and brackets the main (gamete) kernel of species 0 with
 * events on the stream; read back with the mean duration in milliseconds over the launches since
 * enabling.  For bench.py's roofline figure. */
int spegg_kernel_timing(spegg_sim *s, int enable, float *mean_ms, uint32_t *n_launches);

/* Largest n spegg_offsets_static accepts: its scratch is a fixed array inside the library image. */
#define SPEGG_STATIC_MAX_N 4194304ull

/* Fig. 1 A ("the number of neonates are determined"), step a2 on its own and WITHOUT ANY
 * ALLOCATION: from the fecundities f[0..n) of the adults, the index of each adult's first neonate,
 * d_off[i] = f[0] + ... + f[i-1] (clamped to 2^32 - 1), and the number of neonates *d_total = sum of f --
 * the same numbers spegg_step's scan produces (spegg_debug_view.d_off, m_t before capacity truncation).
 *
 * Who this is for.  Every other call works inside a workspace the caller allocated.  This one is for
 * callers that cannot allocate device memory at all at the point of the call: a plug-in running inside
 * a host application whose own allocator has claimed the GPU, code called back while an allocator lock
 * is held, a latency-critical loop that cannot afford the device-wide synchronisation cudaMalloc and
 * cudaFree imply.  The scan needs scratch (look-back status words and a tile ticket); here that scratch
 * is a fixed array of about 34 KB compiled into libspegg.so, so the call performs no cudaMalloc, no
 * cudaFree and no allocating library call.  The price: every GPU that loads the library holds those
 * 34 KB until the process ends, and n is limited to SPEGG_STATIC_MAX_N (4,194,304 adults); a larger n
 * returns SPEGG_ELIMIT and nothing is launched.
 *
 * d_f [n] uint8, d_off [n] uint32 (4-byte aligned), d_total [1] uint64 (8-byte aligned): DEVICE memory of
 * the device that is CURRENT when the call is made; they stay the caller's and must not overlap.  n = 0
 * is allowed (d_f, d_off may then be NULL; *d_total = 0).  cuda_stream: a cudaStream_t of that device
 * (0 = the default stream).  The work is enqueued on the stream and the call returns; results are
 * ready when the stream reaches that point.  SPEGG_EINVAL for NULL pointers, SPEGG_ECUDA for a CUDA error.
 *
 * Two things a caller must know.  (1) The FIRST call on each device looks up the array's device
 * address (cudaGetSymbolAddress, which may also load the module): make that first call, on every device
 * you use, before you start capturing a stream.  (2) There is one array per device and every call on
 * that device uses it, whatever the thread or stream: calls whose GPU work can overlap in time corrupt
 * each other's results -- put them on one stream or order them with events.  Each call clears the part
 * of the array it uses before scanning, so consecutive calls do not see each other's leftovers. */
int spegg_offsets_static(const uint8_t *d_f, uint64_t n, uint32_t *d_off, uint64_t *d_total,
                         void *cuda_stream);

/* PAPER.md:116 (the species object's lifetime): frees the host struct and the graphs; never frees the
 * caller's workspace or stream.  NULL is allowed. */
void spegg_destroy(spegg_sim *s);
/* Text for an error code of any call above (PAPER.md:48-52 has no error model: this is the ABI's own). */
const char *spegg_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif
