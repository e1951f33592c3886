// spegg_internal.h -- structs shared by the host orchestration and the kernels of libspegg.
#pragma once
#include <cstdint>

#include "spegg_device.cuh"

namespace spegg {

constexpr int TMAX = 128;        // thresholds per Poisson table (R5)
constexpr int XMAX = 64;         // row stride of the crossover-count tables (len <= 62, R8)
constexpr int CAP_TABLES = 32;   // R14
constexpr int SCAN_THREADS = 256;
constexpr int SCAN_ITEMS = 4;
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;
constexpr int MAX_SPECIES = 8;
constexpr uint32_t ASSORT_TRIES = 8;            // R23: candidate fathers per egg
constexpr uint32_t MATE_TILE = 1024;             // R19: adults per tile of the mating-weight running sum
constexpr uint32_t FUSED_RANGE = 1024;            // fused path: rows per scan range (32 slabs of 32 rows)

// Device-resident per-species state: counts never leave the GPU between steps.
struct DevSpecies {
    uint32_t cur;          // which population buffer holds the adults
    uint32_t n;            // adults
    uint32_t n0;           // adults at the start of the current step (snapshot)
    uint32_t m;            // offspring of the current step (after capacity truncation)
    uint32_t n_next;       // survivors of the current step
    uint32_t flags_step;   // flags raised during the current step
    uint32_t ticket_fec, done_fused;
    uint32_t log_pos;      // entries written to the log ring
    uint32_t m_phys;       // fused path: physical rows of the current buffer (32-row slabs + chunk_mask)
    long long sum_zi;      // over the current adults (survivors of the last step)
    long long sum_zi0;     // snapshot at the start of the step
    long long acc_zi, acc_zi2;  // accumulators of the current step's survivors
    unsigned long long captures, near_ties;
    float theta_t, zbar_pred, attack_n, zbar_self;
    uint32_t n_pred0;      // predator count snapshot used by this step
    // work tickets of the step kernels, each on a cache line of its own: hundreds of CTAs draw from
    // them at the same moment, and same-line atomics are served one after the other by L2
    alignas(128) uint32_t ticket_cmp;
    alignas(128) unsigned long long ticket_fused;   // (64-bit: see atom_inc_ticket)
    alignas(128) uint32_t ticket_pad;
};

struct DevGlobal {
    uint32_t step;
    uint32_t flags;        // sticky
};

struct LogEntry {          // == spegg_log_entry
    unsigned long long n_t, m_t, n_next;
    long long sum_zi, sum_zi2;
    unsigned long long captures, near_ties;
    uint32_t flags, step;
};

// Per-species constants and device pointers, passed to kernels by value.
struct SpK {
    uint32_t species, n_species;
    uint32_t L, W, kind, n_chrom, linkage;
    uint32_t row_bytes, row_u4;          // bytes / uint4 per row
    uint32_t P, grid_w, grid_h;
    uint32_t capacity;
    uint32_t fec_model;
    double fec_a, K;
    const double *K_patch;
    uint32_t sel_gaussian, sel_predation, predator;
    double theta0, dtheta, attack;
    float sel_c, pheno_scale, pred_scale;
    const float *theta_patch;
    unsigned long long T_mig;
    uint32_t n_tables;
    Key key;
    uint32_t rk[20];            // Philox round keys (k0_r, k1_r), r = 0..9: key + r * Weyl constants
    // constant tables
    const uint32_t *T_recomb;   // [L] INTERVAL switch thresholds (T_0 = 2^31)
    const uint32_t *T_xover;    // [n_chrom][XMAX]
    const uint32_t *xover_len;  // [n_chrom]
    const uint32_t *chrom_start, *chrom_len;
    const uint32_t *T_mut;
    uint32_t mut_len;
    const uint32_t *T_norm;
    int R_norm;
    const uint32_t *T_env;      // R17: residual phenotype noise, whole phenotype quanta (discrete-normal table)
    int R_env;                  // 0: no noise
    // state
    uint8_t *pop[2];
    uint32_t *patch_start[2];   // [P+1] each
    uint32_t *rowptr[2];        // logical adult index -> physical row of pop[]
    uint32_t *chunk_mask[2];    // fused path: survivor bitmask of each 32-row slab of pop[0] / pop[1]
    uint32_t *range_cnt[2];     // fused path: adults per 1,024-row range (FUSED_RANGE) of pop[0] / pop[1]
    uint32_t phys_parents;      // 1: mother[] / father[] hold physical rows (fused path)
    uint32_t solo;              // 1: single-species simulation (the gamete kernel's last CTA closes and prepares the step)
    uint32_t index_only;        // 1: offspring rows are written once, at row j of the other buffer; compaction writes rowptr[] only
    uint8_t *f;
    uint32_t *off, *mother, *father, *dest, *pos;
    float *u01, *s;
    uint8_t *offbuf;
    int32_t *zi;
    int32_t *zrow[2];           // integer genetic value of the individual in each PHYSICAL row of pop[0] / pop[1] (when zrow_on)
    uint32_t zrow_on;           // 1: some kernel of this configuration reads the adults' genetic values
    uint8_t *alive, *captured;
    // R18, overlapping generations (adult_surv > 0): per adult i of the current step
    float adult_surv;           // s_A as fp32; 0 = discrete generations
    uint8_t *a_alive;           // stays alive
    float *a_u, *a_s;           // its uniform and survival probability
    int32_t *a_zi;              // its integer genetic value
    uint32_t *a_pos;            // its position in the next generation (0xFFFFFFFF: dies)
    uint32_t *a_rank;           // patch mode: its rank among ALL staying adults (physical row M + rank of the other buffer)
    // R19, shared-preference mating (mate_v != 0): integer mating weights of the current adults
    float mate_v;               // v_m as fp32; 0 = uniform mate (R2)
    unsigned long long *mate_cum;   // [n] inclusive running sum of the weights, adult order
    unsigned long long *mate_tile;  // [n / MATE_TILE + 2] weight of each tile of MATE_TILE adults
    uint32_t mate_on;           // 1: the father comes from the running sum (mate_v != 0 or separate sexes)
    uint32_t monogamy;          // R25: 1 = the father's draws are addressed by the mother (one mate per mother per step)
    // R24, mothers drawn by relative fecundity (mom_v != 0): integer mothering weights of the current adults
    float mom_v;                // v_f as fp32; 0 = every adult mothers its own eggs
    unsigned long long *mom_cum;    // [n] inclusive running sum, adult order
    unsigned long long *mom_tile;   // [n / MATE_TILE + 2]
    // R21, separate sexes (sexes = 1): one byte per PHYSICAL row of pop[0] / pop[1], 1 = male
    uint32_t sexes;
    uint8_t *sex[2];
    uint8_t *sex_off;           // [m] sex of each offspring of the current step (staging; also I/O staging)
    // R20, individual-level encounters (enc_E > 0 on the prey; enc_zi filled on the species it meets)
    float assort;               // R23: a of the acceptance exp(-a d^2) of a candidate father; 0 = random mating (uses enc_zi)
    float fec_cost;             // R22: rho of the fecundity cost exp(-rho z^2); 0 = none (uses enc_zi of this species)
    uint32_t enc_E;             // meetings per newborn; 0 = mean-field predation term (R14)
    float enc_v;                // v = fp32(attack)
    int32_t *enc_zi;            // [n] integer genetic values of THIS species' adults (when another species meets them)
    const int32_t *pred_zi;     // enc_zi of the predator species
    uint32_t *cap;              // capture counts of THIS species' adults (CAPTURES model)
    uint32_t *cap_pred;         // capture counts of the predator species (predation term)
    uint32_t *tables, *table_len;
    unsigned long long *status_fec, *status_cmp;  // [n] tile aggregates + [n/32+2] group counters
    uint32_t status_fec_n, status_cmp_n;
    uint32_t patch_sub;         // S: segments per patch of the patch-mode compaction (1 with many small patches)
    uint32_t *patch_cnt, *patch_base;  // [P * S][6]: survivors per (natal patch, destination slot 0..4); [5]: staying adults of the patch (R18)
    // patch topology (P > 1), built once by the host: the torus never changes
    uint32_t *patch_abase;      // [P * S] R18: staying adults of the patches before this one
    const uint32_t *nbr;        // [P][4] neighbour of patch p in direction 0..3 (R15)
    const uint32_t *src_list;   // [P][6]: word 0 = number of sources n of destination d, words 1..n = source patch << 3 | slot, by source patch
    DevSpecies *st;             // this species
    DevSpecies *st_all;         // all species
    DevGlobal *glob;
    LogEntry *log;
    uint32_t log_capacity;
    uint32_t debug;
};

}  // namespace spegg
