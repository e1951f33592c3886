// spegg_kernels.cuh -- the step pipeline of libspegg as separate kernels (sm_100a).
//
// One time step of one species (Fig. 1 A-F) on the production path is
//   [k_enc_zi, k_mate_weight, k_mate_scan]  adults' genetic values / parental weights, when a widening needs them
//   k_fec_scan        a1-a3  Poisson fecundity, single-pass look-back scan, mothers, then the scalar draws
//                            (father, weighted parents, dispersal, survival uniform, sex) of the range's offspring
//   k_gamete_q10v/r   a4-a5  per-interval recombination, select, phenotype (register prefetch / cp.async ring)
//   k_select_compact  a4-a8  unstructured species: mutation, selection, scan, look-back, index -- one kernel
//   k_patch_count / k_patch_base / k_patch_pos  a4-a8  patch mode: mutation + selection + counts per
//                            segment, one flat exclusive scan, positions + index
//   [k_adult_survive, k_cmp_scan, k_cmp_scatter]  overlapping generations: the adults that stay
//   k_finish_all / k_prepare_all  a9, a0  (or the last CTA of the step's last kernel for a solo species)
// and, for debug mode (every intermediate materialised) and genomes the fast kernels do not cover,
// the plain kernels k_gamete_bit / k_gamete_q10, k_mutate, k_phenotype, k_survival, k_cmp_scan,
// k_cmp_scatter.  spegg_fused.cuh holds the fused two-kernel step of the hot configuration.
// All grids are fixed at graph-capture time and loop against device-side counts.
#pragma once
#include <algorithm>

#include "spegg_internal.h"

namespace spegg {

// ------------------------------------------------------------------------------- helpers
__device__ __forceinline__ uint32_t patch_of(const uint32_t *__restrict__ ps, uint32_t P, uint32_t i) {
    uint32_t lo = 0, hi = P;  // largest lo with ps[lo] <= i
    while (hi - lo > 1) {
        const uint32_t mid = (lo + hi) >> 1;
        if (ps[mid] <= i) lo = mid; else hi = mid;
    }
    return lo;
}

// the same search between two known patches lo <= patch(i) <= hi
__device__ __forceinline__ uint32_t patch_between(const uint32_t *__restrict__ ps, uint32_t lo, uint32_t hi, uint32_t i) {
    ++hi;
    while (hi - lo > 1) {
        const uint32_t mid = (lo + hi) >> 1;
        if (ps[mid] <= i) lo = mid; else hi = mid;
    }
    return lo;
}

// Philox4x32-10 (R3) with the ten round keys taken from the kernel parameter block: the key
// schedule k_r = k_0 + r * Weyl is the same for every draw of a simulation, so the host computes it
// once (SpK::rk) and the XORs read it straight from the constant bank -- four instructions a round.
__device__ __forceinline__ void draw_rk(const SpK &sp, uint32_t stream, uint32_t entity, uint32_t block,
                                        uint32_t step, uint32_t (&o)[4]) {
    uint32_t c0 = entity, c1 = block, c2 = step, c3 = (sp.species << 8) | stream;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ sp.rk[2 * r];
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ sp.rk[2 * r + 1];
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
    }
    o[0] = c0; o[1] = c1; o[2] = c2; o[3] = c3;
}

// R13/R14: fecundity mean, fp64 with the stated op order
__device__ __forceinline__ double fecundity_mean(const SpK &sp, double n, double K, uint32_t cap_index) {
    if (sp.fec_model == 0) {  // Beverton-Holt
        const double q = __ddiv_rn(n, K);
        const double d = __dadd_rn(1.0, q);
        return __ddiv_rn(sp.fec_a, d);
    } else if (sp.fec_model == 1) {  // logistic
        const double q = __ddiv_rn(n, K);
        const double a = __dsub_rn(1.0, q);
        const double b = __dmul_rn(sp.fec_a, a);
        const double l = __dadd_rn(1.0, b);
        return l < 0.0 ? 0.0 : l;
    }
    const double q = __ddiv_rn(n, K);
    double a = __dsub_rn(1.0, q);
    if (a < 0.0) a = 0.0;
    const double b = __dmul_rn(sp.fec_a, (double)cap_index);
    return __dmul_rn(b, a);
}

// R11/R14 survival probability in fp32, in the stated order.  Returns s; sets captured.
__device__ __forceinline__ float survival_prob(const SpK &sp, float z, float theta, float u01, bool &captured) {
    float s = 1.0f;
    captured = false;
    if (sp.sel_predation) {
        const float d = __fsub_rn(z, sp.st->zbar_pred);
        const float g = expf_spec(-__fmul_rn(0.5f, __fmul_rn(d, d)));
        const float spd = expf_spec(-__fmul_rn(sp.st->attack_n, g));
        captured = !(u01 < spd);
        s = spd;
    }
    if (sp.sel_gaussian) {
        const float d = __fsub_rn(z, theta);
        const float sq = __fmul_rn(d, d);
        const float ss = expf_spec(-__fmul_rn(sq, sp.sel_c));
        s = sp.sel_predation ? __fmul_rn(s, ss) : ss;
    }
    return s;
}

// where the offspring rows of the current step live: row j of the other population buffer when the
// compaction is index-only (they are never moved again), else the staging buffer
__device__ __forceinline__ uint8_t *offspring_rows(const SpK &sp) {
    return sp.index_only ? sp.pop[sp.st->cur ^ 1u] : sp.offbuf;
}

// ------------------------------------------------------------------------ step bookkeeping
__device__ __forceinline__ uint32_t ld_u32(const uint32_t *p) {
    uint32_t v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned long long ld_u64(const void *p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}

// a9: end of step for one species (one thread): counts stay on the device, log entry, buffer flip.
// Reads go through L2 (ld.relaxed.gpu) because the caller may be the last CTA of another kernel.
__device__ __forceinline__ void finish_species(const SpK &sp) {
    DevSpecies &st = *sp.st;
    const uint32_t nn = ld_u32(&st.n_next), n0 = ld_u32(&st.n0);
    uint32_t fl = ld_u32(&st.flags_step);
    if (n0 == 0) fl |= 2u;
    const uint32_t lp = ld_u32(&st.log_pos);
    const long long a1 = (long long)ld_u64(&st.acc_zi), a2 = (long long)ld_u64(&st.acc_zi2);
    LogEntry &e = sp.log[lp % sp.log_capacity];
    e.n_t = n0; e.m_t = ld_u32(&st.m); e.n_next = nn;
    e.sum_zi = a1; e.sum_zi2 = a2;
    e.captures = ld_u64(&st.captures); e.near_ties = ld_u64(&st.near_ties);
    e.flags = fl; e.step = ld_u32(&sp.glob->step);
    st.log_pos = lp + 1;
    if (fl) atomicOr(&sp.glob->flags, fl);
    st.n = nn;
    if (sp.phys_parents) st.m_phys = ld_u32(&st.m);   // every offspring row was stored; the masks say which live
    st.sum_zi = a1;
    const uint32_t cur = ld_u32(&st.cur) ^ 1u;
    st.cur = cur;
    if (sp.P == 1) { uint32_t *psn = sp.patch_start[cur]; psn[0] = 0; psn[1] = nn; }
}

// a0: everything the next step needs before its first kernel (Fig. 1 F -> A): start-of-step
// snapshots, fecundity tables from the device-resident counts, theta_t, predation scalars, cleared
// look-back statuses / tickets / capture counts.  g / stride: this thread's index and the number
// of threads sharing the work; N, cur, sum_zi, step: the species' finished state.
__device__ __forceinline__ void prepare_species(const SpK &sp, uint32_t g, uint32_t stride, uint32_t N,
                                                uint32_t cur, long long sum_zi, uint32_t step, uint32_t g_tab) {
    const uint32_t nf = sp.status_fec_n + sp.status_fec_n / 32 + 2, nc = sp.status_cmp_n + sp.status_cmp_n / 32 + 2;
    for (uint32_t i = g; i < nf; i += stride) sp.status_fec[i] = 0ull;
    for (uint32_t i = g; i < nc; i += stride) sp.status_cmp[i] = 0ull;
    if (sp.fec_model == 2)
        for (uint32_t i = g; i < sp.capacity; i += stride) sp.cap[i] = 0u;
    if (sp.mate_on)   // R19: tile totals of the mating weights are accumulated with atomics
        for (uint32_t i = g; i < sp.capacity / MATE_TILE + 2u; i += stride) sp.mate_tile[i] = 0ull;
    if (sp.mom_v != 0.0f)   // R24: the same for the mothering weights
        for (uint32_t i = g; i < sp.capacity / MATE_TILE + 2u; i += stride) sp.mom_tile[i] = 0ull;
    if (sp.phys_parents) {  // fused path: the coming step counts its survivors per range of the other buffer
        uint32_t *cnt_next = sp.range_cnt[cur ^ 1u];
        const uint32_t n_max = (sp.capacity + 31u) / 32u * 32u / FUSED_RANGE + 2u;
        for (uint32_t i = g; i < n_max; i += stride) cnt_next[i] = 0u;
    }
    const uint32_t *ps = sp.patch_start[cur];
    // g_tab: this thread's index for the table builds (the step-closing CTA gives table 0 to a thread of
    // another warp than the one that is busy closing the step: the fp64 chain of a table is ~2 us)
    // (fused path: k_scan_fused builds the one table itself, off the path between the kernels)
    for (uint32_t tab = sp.phys_parents ? sp.n_tables : g_tab; tab < sp.n_tables; tab += stride) {
        double lam;
        if (sp.fec_model == 2) lam = fecundity_mean(sp, (double)N, sp.K, tab);
        else if (sp.P == 1) lam = fecundity_mean(sp, (double)N, sp.K_patch ? sp.K_patch[0] : sp.K, 0);
        else lam = fecundity_mean(sp, (double)(ps[tab + 1] - ps[tab]), sp.K_patch ? sp.K_patch[tab] : sp.K, 0);
        sp.table_len[tab] = (uint32_t)build_poisson_table(lam, sp.tables + (size_t)tab * TMAX, TMAX);
    }
    if (g == 0) {
        DevSpecies &st = *sp.st;
        st.n0 = N;
        st.sum_zi0 = sum_zi;
        st.m = 0; st.n_next = 0; st.flags_step = 0;
        st.ticket_fec = 0; st.ticket_cmp = 0; st.ticket_fused = 0; st.done_fused = 0;
        st.acc_zi = 0; st.acc_zi2 = 0; st.captures = 0; st.near_ties = 0;
        // R6: theta_t = fp32(theta0 + t*dtheta), fp64, never accumulated
        st.theta_t = __double2float_rn(__dadd_rn(sp.theta0, __dmul_rn((double)step, sp.dtheta)));
        if (sp.sel_predation) {
            const DevSpecies &pr = sp.st_all[sp.predator];
            const uint32_t NC = pr.n;
            st.n_pred0 = NC;
            // R14: zbar_C = fp32((sum zi / N_C) * scale_C) ; A = fp32(a * N_C)
            st.zbar_pred = NC ? __double2float_rn(__dmul_rn(__ddiv_rn((double)pr.sum_zi, (double)NC), (double)sp.pred_scale)) : 0.0f;
            st.attack_n = __double2float_rn(__dmul_rn(sp.attack, (double)NC));
        }
    }
}

// Single block, so nothing races on glob->step.
__global__ void k_finish_all(const SpK *__restrict__ spk, uint32_t n_species) {
    if (threadIdx.x < n_species) finish_species(spk[threadIdx.x]);
    __syncthreads();
    if (threadIdx.x == 0) spk[0].glob->step += 1;
}

// grid = (blocks, n_species)
__global__ void __launch_bounds__(256) k_prepare_all(const SpK *__restrict__ spk) {
    const SpK &sp = spk[blockIdx.y];
    const DevSpecies &st = *sp.st;
    const uint32_t g = blockIdx.x * blockDim.x + threadIdx.x;
    prepare_species(sp, g, gridDim.x * blockDim.x, st.n, st.cur, st.sum_zi, sp.glob->step, g);
}

// Tail of the last kernel of a single-species step: the CTA that finishes last closes the step and
// prepares the next one, saving two launches.  Call from every CTA after its work is done.
__device__ __forceinline__ void solo_tail(const SpK &sp, uint32_t *s_flag) {
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        *s_flag = (atomicAdd(&sp.st->done_fused, 1u) == gridDim.x - 1) ? 1u : 0u;
    }
    __syncthreads();
    if (!*s_flag) return;
    __threadfence();
    // every thread reads what the next step's preparation needs straight from L2, in one round trip,
    // while thread 0 closes the step: nothing below waits for a value another thread wrote
    DevSpecies &st = *sp.st;
    const uint32_t nn = ld_u32(&st.n_next), cur1 = ld_u32(&st.cur) ^ 1u, step1 = ld_u32(&sp.glob->step) + 1u;
    const long long a1 = (long long)ld_u64(&st.acc_zi);
    __syncthreads();   // every thread holds its snapshot before thread 0 flips cur / bumps the step / zeroes the accumulators
    if (threadIdx.x == 0) {
        finish_species(sp);
        sp.glob->step = step1;
    }
    prepare_species(sp, threadIdx.x, blockDim.x, nn, cur1, a1, step1, (threadIdx.x + blockDim.x - 32u) % blockDim.x);
}

// a3: the scalar draws of offspring j: father (R2; R19 / R21 weighted; R23 assortative), mother by relative
// fecundity (R24), dispersal (R15), survival uniform (R4), sex at birth (R21).  mother[j] (and, in patch
// mode, the natal patch in dest[j]) were just written by the calling CTA of k_fec_scan.
// (pm, base, np: the natal patch of j, its first adult and its size -- loaded by the caller, who batches
// these two dependent loads over several offspring)
__device__ __forceinline__ void scalar_one(const SpK &sp, uint32_t j, uint32_t pm, uint32_t base, uint32_t np, uint32_t step,
                                           unsigned int &ties) {
    uint32_t mo = (sp.mom_v != 0.0f || sp.assort > 0.0f || sp.monogamy) ? sp.mother[j] : 0u;   // (only those read it)
    uint32_t x[4];
    draw(sp.key, sp.species, ST_SCALAR, j, 0, step, x);
    if (sp.mom_v != 0.0f) {
        // R24 (eq. S2-9): the egg was counted by the adult that laid it; its mother is
        // drawn among the adults of that patch: 64-bit uniform from words 0,1 of MOTHER block 0,
        // target = floor(u * total / 2^64), first adult whose running sum exceeds it; total 0: unchanged
        const unsigned long long before = base ? sp.mom_cum[base - 1] : 0ull;
        const unsigned long long total = sp.mom_cum[base + np - 1] - before;
        if (total) {
            uint32_t y[4];
            draw_rk(sp, ST_MOTHER, j, 0, step, y);
            const unsigned long long u = ((unsigned long long)y[0] << 32) | y[1];
            const unsigned long long target = before + __umul64hi(u, total);
            uint32_t lo = base, hi = base + np - 1;
            while (lo < hi) {
                const uint32_t mid = (lo + hi) >> 1;
                if (sp.mom_cum[mid] > target) hi = mid; else lo = mid + 1;
            }
            mo = lo;
            sp.mother[j] = mo;
        }
    }
    // R25 ("monogamy or polygynandry"): with monogamy the father's draws are addressed by the
    // MOTHER (stream PAIR, entity = her adult index: block 0 word 0 = R2's index, words 2,3 = R19's uniform,
    // blocks 1.. = R23's candidates), so all the eggs of one mother in one step have one father
    uint32_t xp[4] = {0u, 0u, 0u, 0u};
    if (sp.monogamy) draw_rk(sp, ST_PAIR, mo, 0, step, xp);
    uint32_t fa = base + uniform_index(sp.monogamy ? xp[0] : x[0], np);
    if (sp.mate_on) {
        // R19: weighted draw among the adults of the mother's patch: 64-bit uniform from words 2,3 of
        // SCALAR block 1, target = floor(u * total / 2^64), father = first adult of the patch whose
        // inclusive running sum exceeds (sum before the patch) + target; total 0 keeps the uniform mate
        const unsigned long long before = base ? sp.mate_cum[base - 1] : 0ull;
        const unsigned long long total = sp.mate_cum[base + np - 1] - before;
        if (total) {
            uint32_t y[4];
            if (sp.monogamy) { y[2] = xp[2]; y[3] = xp[3]; }
            else draw_rk(sp, ST_SCALAR, j, 1, step, y);
            const unsigned long long u = ((unsigned long long)y[2] << 32) | y[3];
            const unsigned long long target = before + __umul64hi(u, total);
            uint32_t lo = base, hi = base + np - 1;   // first index with mate_cum > target; exists since target < before + total
            while (lo < hi) {
                const uint32_t mid = (lo + hi) >> 1;
                if (sp.mate_cum[mid] > target) hi = mid; else lo = mid + 1;
            }
            fa = lo;
        }
    }
    if (sp.assort > 0.0f) {
        // R23 (assortative mating): candidate t = 0..7 uniform over the mother's patch (word
        // 2(t%2) of MATE block t/2), accepted iff u01(word 2(t%2)+1) < expf_spec(-(a * (d*d))),
        // d = z_cand - z_mother (genetic values from k_enc_zi); first accepted, else the last candidate
        const float zm = __fmul_rn((float)sp.enc_zi[mo], sp.pheno_scale);
        uint32_t y[4];
        for (uint32_t tr = 0; tr < ASSORT_TRIES; ++tr) {
            if ((tr & 1u) == 0) {
                if (sp.monogamy) draw_rk(sp, ST_PAIR, mo, 1u + (tr >> 1), step, y);
                else draw_rk(sp, ST_MATE, j, tr >> 1, step, y);
            }
            fa = base + uniform_index(y[2 * (tr & 1u)], np);
            const float d = __fsub_rn(__fmul_rn((float)sp.enc_zi[fa], sp.pheno_scale), zm);
            const float p = expf_spec(-__fmul_rn(sp.assort, __fmul_rn(d, d)));
            const float u = u01_of(y[2 * (tr & 1u) + 1]);
            if (fabsf(__fsub_rn(u, p)) < 1e-6f) ++ties;
            if (u < p) break;
        }
    }
    sp.father[j] = fa;
    uint32_t dest = pm;
    if (sp.P > 1 && (unsigned long long)x[1] < sp.T_mig) dest = sp.nbr[pm * 4u + (x[2] >> 30)];
    sp.dest[j] = dest;
    sp.u01[j] = u01_of(x[3]);
    if (sp.sexes) sp.sex_off[j] = (uint8_t)(x[2] & 1u);   // R21: sex at birth (bits 30-31 of the word are the direction)
}

// a1-a3: fecundity (one FEC block per adult), exclusive scan by decoupled look-back, mother fill.
// Each CTA takes a contiguous RANGE of adults (about N / gridDim.x, at most FEC_RANGE_MAX): pass 1
// draws the fecundities into shared memory and reduces them, ONE look-back per range gives the
// range's offspring base, pass 2 scans inside the range and writes off[], f[] and mother[].  With
// a few hundred ranges the look-back chain is a handful of hops instead of one per 1,024 adults.
constexpr int FEC_RANGE_MAX = 8192;

__device__ __forceinline__ uint32_t fec_range_size(uint32_t N, uint32_t n_ctas) {
    uint32_t R = (N + n_ctas - 1) / n_ctas;
    R = (R + SCAN_THREADS - 1) / SCAN_THREADS * SCAN_THREADS;
    return min(max(R, (uint32_t)SCAN_THREADS), (uint32_t)FEC_RANGE_MAX);
}

__global__ void __launch_bounds__(SCAN_THREADS, 4) k_fec_scan(const __grid_constant__ SpK sp) {
    __shared__ uint32_t s_tab[TMAX];
    __shared__ uint8_t s_f[FEC_RANGE_MAX];
    __shared__ uint32_t s_off[FEC_RANGE_MAX];
    __shared__ uint32_t s_warp[SCAN_THREADS / 32];
    __shared__ uint32_t s_tile, s_total;
    __shared__ unsigned long long s_excl;
    DevSpecies &st = *sp.st;
    const uint32_t N = st.n0, step = sp.glob->step;
    unsigned int ties = 0;
    // R18: with overlapping generations every adult may stay, so the offspring get the room that is left
    const uint32_t m_cap = sp.adult_surv > 0.0f ? sp.capacity - N : sp.capacity;
    const uint32_t R = fec_range_size(N, gridDim.x);
    const uint32_t n_ranges = (N + R - 1) / R;
    const uint32_t per = R / SCAN_THREADS;  // adults per thread in pass 2 (<= 32)
    const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const bool one_table = sp.n_tables == 1;
    uint32_t len0 = 0;
    if (one_table) {
        len0 = sp.table_len[0];
        for (uint32_t i = tid; i < len0; i += SCAN_THREADS) s_tab[i] = sp.tables[i];
    }
    const uint32_t *ps = sp.patch_start[st.cur];
    const uint32_t *rowptr = sp.rowptr[st.cur];
    const bool by_patch = !one_table && sp.fec_model != 2;
    for (;;) {
        if (tid == 0) s_tile = atomicAdd(&st.ticket_fec, 1u);
        __syncthreads();
        const uint32_t range = s_tile;
        if (range >= n_ranges) break;
        const uint32_t r0 = range * R;
        // patch mode: the adults of a range lie in a few consecutive patches -- every thread finds the
        // patches of the range's first and last adult (the same search in every lane: broadcast loads) and
        // then only searches between them
        uint32_t p_lo = 0, p_hi = 0;
        if (by_patch) { p_lo = patch_of(ps, sp.P, r0); p_hi = patch_of(ps, sp.P, min(r0 + R, N) - 1u); }
        // ---- pass 1: fecundity draws (coalesced in i), staged as bytes
        for (uint32_t k = tid; k < R; k += SCAN_THREADS) {
            const uint32_t i = r0 + k;
            uint32_t f = 0;
            if (i < N) {
                uint32_t x[4];
                draw(sp.key, sp.species, ST_FEC, i, 0, step, x);
                if (one_table) {
                    f = poisson_count(s_tab, len0, x[0]);
                } else {
                    const uint32_t tab = (sp.fec_model == 2) ? min(sp.cap[i], (uint32_t)(CAP_TABLES - 1)) : patch_between(ps, p_lo, p_hi, i);
                    // the first four thresholds in one 16-byte load (tables are TMAX-word rows), the rest -- rare --
                    // by the plain search
                    const uint32_t *T = sp.tables + (size_t)tab * TMAX;
                    const uint32_t len = sp.table_len[tab];
                    const uint4 t4 = *(const uint4 *)T;
                    f = (len > 0 && x[0] >= t4.x ? 1u : 0u) + (len > 1 && x[0] >= t4.y ? 1u : 0u) +
                        (len > 2 && x[0] >= t4.z ? 1u : 0u) + (len > 3 && x[0] >= t4.w ? 1u : 0u);
                    if (f == 4u) while (f < len && x[0] >= T[f]) ++f;
                }
                if (sp.sexes && sp.sex[st.cur][rowptr[i]]) f = 0;   // R21: males lay no eggs (the draw is made and ignored)
                if (sp.fec_cost > 0.0f && f) {
                    // R22 (eq. S3-3): egg k is laid iff u01(word (2+k)%4 of FEC block (2+k)/4) < c_i,
                    // c_i = expf_spec(-(rho * (z*z))), z the adult's genetic value (k_enc_zi ran before this kernel)
                    const float z = __fmul_rn((float)sp.enc_zi[i], sp.pheno_scale);
                    const float c = expf_spec(-__fmul_rn(sp.fec_cost, __fmul_rn(z, z)));
                    uint32_t keep = 0, y[4] = {x[0], x[1], x[2], x[3]};
                    for (uint32_t k = 0; k < f; ++k) {
                        const uint32_t w = 2u + k;
                        if (k > 0 && (w & 3u) == 0) draw(sp.key, sp.species, ST_FEC, i, w >> 2, step, y);
                        if (u01_of(y[w & 3u]) < c) ++keep;
                    }
                    f = keep;
                }
            }
            s_f[k] = (uint8_t)f;
        }
        __syncthreads();
        // ---- block scan over the range: per-thread slices [tid*per, tid*per+per) in shared memory
        uint32_t sum = 0;
        for (uint32_t k = 0; k < per; ++k) { s_off[tid * per + k] = sum; sum += s_f[tid * per + k]; }
        const uint32_t incl = warp_incl_scan(sum);
        if (lane == 31) s_warp[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            uint32_t w = (lane < SCAN_THREADS / 32) ? s_warp[lane] : 0u;
            const uint32_t wi = warp_incl_scan(w);
            const uint32_t total = __shfl_sync(0xffffffffu, wi, SCAN_THREADS / 32 - 1);
            const unsigned long long excl = lookback(sp.status_fec, sp.status_fec_n, range, (unsigned long long)total);
            if (lane < SCAN_THREADS / 32) s_warp[lane] = wi - w;  // exclusive warp prefix
            if (lane == 0) {
                s_excl = excl;
                s_total = total;
                if (range == n_ranges - 1) {  // the last range knows M
                    const unsigned long long Mtot = excl + total;
                    if (Mtot > (unsigned long long)m_cap) { st.m = m_cap; st.flags_step |= 1u; }
                    else st.m = (uint32_t)Mtot;
                }
            }
        }
        __syncthreads();
        {
            const uint32_t tbase = s_warp[warp] + (incl - sum);
            for (uint32_t k = 0; k < per; ++k) s_off[tid * per + k] += tbase;
        }
        __syncthreads();
        // ---- pass 2 (coalesced in i): offsets, f[], mother[]
        const unsigned long long rbase = s_excl;
        for (uint32_t k = tid; k < R; k += SCAN_THREADS) {
            const uint32_t i = r0 + k;
            if (i >= N) break;
            const uint32_t f = s_f[k];
            const unsigned long long o = rbase + s_off[k];
            sp.off[i] = (uint32_t)min(o, (unsigned long long)0xFFFFFFFFull);
            sp.f[i] = (uint8_t)f;
            if (f) {
                const uint32_t mval = sp.phys_parents ? rowptr[i] : i;
                // patch mode: the offspring's natal patch goes into dest[] (k_scalar reads it and stores the destination)
                const uint32_t pm = by_patch ? patch_between(ps, p_lo, p_hi, i) : 0u;
                for (uint32_t c = 0; c < f; ++c) {
                    const unsigned long long j = o + c;
                    if (j < (unsigned long long)m_cap) { sp.mother[j] = mval; if (sp.P > 1) sp.dest[j] = pm; }
                }
            }
        }
        __syncthreads();   // mother[] / dest[] of this range's offspring are written (same CTA: visible after the barrier)
        // ---- a3 for this range's offspring, one thread each: no separate kernel, no second pass over mother[]
        {
            const unsigned long long j_end = min(rbase + (unsigned long long)s_total, (unsigned long long)m_cap);
            // four offspring per trip: their natal patches (left in dest[] above), then the patches' bounds, travel
            // together -- a thread's trips are otherwise a chain of two dependent loads each
            for (unsigned long long j0 = rbase + tid; j0 < j_end; j0 += 4ull * SCAN_THREADS) {
                uint32_t pm[4], b0[4], b1[4];
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const unsigned long long j = j0 + (unsigned long long)q * SCAN_THREADS;
                    pm[q] = (sp.P > 1 && j < j_end) ? sp.dest[j] : 0u;
                }
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    b0[q] = 0u; b1[q] = N;
                    if (sp.P > 1) { b0[q] = ps[pm[q]]; b1[q] = ps[pm[q] + 1u]; }
                }
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const unsigned long long j = j0 + (unsigned long long)q * SCAN_THREADS;
                    if (j < j_end) scalar_one(sp, (uint32_t)j, pm[q], b0[q], b1[q] - b0[q], step, ties);
                }
            }
        }
        __syncthreads();
    }
    if (ties) atomicAdd(&st.near_ties, (unsigned long long)ties);
}

// Integer genetic values (R10) of the block of 32 consecutive adults blk * 32 .. of the current
// population, one per lane: lane l returns zi of adult blk * 32 + l (0 beyond n).  Called by a whole
// warp.  The value travels with the individual: zrow[buffer][physical row] is written when the row is
// (spegg_write_state: from the rows; every step: by the compaction, from the gamete kernel's phenotype),
// so nobody re-reads a row to get one integer.
__device__ __forceinline__ int32_t block_adult_zi(const SpK &sp, const uint8_t *__restrict__, const uint32_t *__restrict__ rowptr,
                                                  uint32_t blk, uint32_t n) {
    const uint32_t i = blk * 32u + (threadIdx.x & 31u);
    return i < n ? sp.zrow[sp.st->cur][rowptr[i]] : 0;
}

// The same from the rows themselves (spegg_write_state / spegg_read_state).  G lanes share one adult
// (128-bit loads: a row of up to 512 bytes is one load per lane), 32 / G adults per pass, four passes'
// loads in flight before the first reduction.
__device__ __forceinline__ int32_t block_adult_zi_rows(const SpK &sp, const uint8_t *__restrict__ pop,
                                                       const uint32_t *__restrict__ rowptr, uint32_t blk, uint32_t n) {
    const uint32_t lane = threadIdx.x & 31u;
    uint32_t G = 1;
    while (G < 32u && G < sp.row_u4) G <<= 1;
    const uint32_t apw = 32u / G, grp = lane / G, q = lane % G;
    const uint32_t blk_end = min(blk * 32u + 32u, n);
    int32_t my_sum = 0;
    for (uint32_t i0 = blk * 32u; i0 < blk_end; i0 += 4u * apw) {
        int32_t acc[4];
#pragma unroll
        for (int p = 0; p < 4; ++p) {
            const uint32_t i = i0 + p * apw + grp;
            acc[p] = 0;
            if (i < blk_end) {
                const uint4 *r4 = (const uint4 *)(pop + (size_t)rowptr[i] * sp.row_bytes);
                for (uint32_t k = q; k < sp.row_u4; k += G) {
                    const uint4 v = r4[k];
                    if (sp.kind == 0) acc[p] += __popc(v.x) + __popc(v.y) + __popc(v.z) + __popc(v.w);
                    else acc[p] += (int32_t)(int16_t)(v.x & 0xFFFFu) + (int32_t)(int16_t)(v.x >> 16) +
                                   (int32_t)(int16_t)(v.y & 0xFFFFu) + (int32_t)(int16_t)(v.y >> 16) +
                                   (int32_t)(int16_t)(v.z & 0xFFFFu) + (int32_t)(int16_t)(v.z >> 16) +
                                   (int32_t)(int16_t)(v.w & 0xFFFFu) + (int32_t)(int16_t)(v.w >> 16);
                }
            }
        }
#pragma unroll
        for (int p = 0; p < 4; ++p) {
            int32_t a_ = acc[p];
            for (uint32_t o = G >> 1; o > 0; o >>= 1) a_ += __shfl_xor_sync(0xffffffffu, a_, o);
            // the sum of the pass's adult number g sits in lanes g*G..; lane (base + g) of the block takes it
            const uint32_t base = (i0 - blk * 32u) + p * apw;
            const int32_t got = __shfl_sync(0xffffffffu, a_, ((lane - base) & (apw - 1u)) * G);
            if (lane >= base && lane < base + apw) my_sum = got;
        }
    }
    return sp.kind == 0 ? 2 * my_sum - 2 * (int32_t)sp.L : my_sum;
}

// R19 ("shared preference"; eq. S2-10): integer mating weight of every
// adult, w_i = trunc(expf_spec(clamp(v (z_i - zbar), -16, 16) - 16) * 2^40), fp32 in this order, zbar the
// adults' mean genetic value (fp64 sum / N * scale rounded to fp32, as zbar_C of R14).  A warp takes
// blocks of 32 consecutive adults (their genetic values are re-read from the rows), computes the 32
// weights one per lane, stores them to mate_cum[] and adds their sum to the tile's total (one integer
// atomic per block -- 32 divides MATE_TILE -- exact in any order).
__device__ __forceinline__ unsigned long long mating_weight(float v, float d) {
    float e = __fmul_rn(v, d);
    e = fminf(fmaxf(e, -16.0f), 16.0f);
    const float w = expf_spec(__fsub_rn(e, 16.0f));
    return (unsigned long long)__fmul_rn(w, 0x1p40f);
}

// (R24, eq. S2-9: the mothering weights exp(v_f z_i), zero for males, are built in the
// same pass into mom_cum[] / mom_tile[])
__global__ void __launch_bounds__(256) k_mate_weight(const __grid_constant__ SpK sp) {
    DevSpecies &st = *sp.st;
    const uint32_t N = st.n0, lane = threadIdx.x & 31u;
    const uint32_t warp0 = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = (gridDim.x * blockDim.x) >> 5;
    const uint8_t *pop = sp.pop[st.cur];
    const uint32_t *rowptr = sp.rowptr[st.cur];
    const uint8_t *sex = sp.sex[st.cur];
    const bool mom_on = sp.mom_v != 0.0f;
    const float zbar = N ? __double2float_rn(__dmul_rn(__ddiv_rn((double)st.sum_zi0, (double)N), (double)sp.pheno_scale)) : 0.0f;
    if (warp0 == 0 && lane == 0) st.zbar_self = zbar;
    for (uint32_t blk = warp0; blk < (N + 31u) / 32u; blk += nw) {
        const int32_t zi = block_adult_zi(sp, pop, rowptr, blk, N);
        const uint32_t i = blk * 32u + lane;
        unsigned long long part = 0ull, mpart = 0ull;
        if (i < N) {
            const float d = __fsub_rn(__fmul_rn((float)zi, sp.pheno_scale), zbar);
            const bool male = sp.sexes && sex[rowptr[i]];
            if (sp.mate_on) {
                unsigned long long wi = mating_weight(sp.mate_v, d);
                if (sp.sexes && !male) wi = 0ull;   // R21: only males father eggs
                sp.mate_cum[i] = wi;
                part = wi;
            }
            if (mom_on) {
                unsigned long long wi = mating_weight(sp.mom_v, d);
                if (male) wi = 0ull;                // R24 + R21: only females mother eggs
                sp.mom_cum[i] = wi;
                mpart = wi;
            }
        }
        for (int o = 16; o > 0; o >>= 1) { part += __shfl_xor_sync(0xffffffffu, part, o); mpart += __shfl_xor_sync(0xffffffffu, mpart, o); }
        if (lane == 0 && part) atomicAdd(&sp.mate_tile[blk * 32u / MATE_TILE], part);
        if (lane == 0 && mpart) atomicAdd(&sp.mom_tile[blk * 32u / MATE_TILE], mpart);
    }
}

// R19: inclusive running sum of the weights in adult order.  One CTA per tile of MATE_TILE adults:
// the tile's base is the sum of the tile totals before it (every CTA adds them up itself -- a few
// thousand L2-resident words, no chain between CTAs), then a block scan of 4 adults per thread.
__global__ void __launch_bounds__(256) k_mate_scan(const __grid_constant__ SpK sp, int mothers) {
    __shared__ unsigned long long s_red[8];
    __shared__ unsigned long long s_base;
    const uint32_t N = sp.st->n0, tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const uint32_t n_tiles = (N + MATE_TILE - 1) / MATE_TILE;
    unsigned long long *cum = mothers ? sp.mom_cum : sp.mate_cum;           // R24 / R19
    const unsigned long long *tile = mothers ? sp.mom_tile : sp.mate_tile;
    for (uint32_t t = blockIdx.x; t < n_tiles; t += gridDim.x) {
        unsigned long long b = 0;
        for (uint32_t k = tid; k < t; k += 256) b += tile[k];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) b += __shfl_xor_sync(0xffffffffu, b, o);
        if (lane == 0) s_red[warp] = b;
        __syncthreads();
        if (tid == 0) { unsigned long long a = 0; for (int k = 0; k < 8; ++k) a += s_red[k]; s_base = a; }
        __syncthreads();
        const uint32_t i0 = t * MATE_TILE + tid * 4;
        unsigned long long w[4], sum = 0;
#pragma unroll
        for (int k = 0; k < 4; ++k) { w[k] = (i0 + k < N) ? cum[i0 + k] : 0ull; sum += w[k]; w[k] = sum; }
        unsigned long long incl = sum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned long long v = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= (uint32_t)o) incl += v;
        }
        __syncthreads();                       // s_red is reused
        if (lane == 31) s_red[warp] = incl;
        __syncthreads();
        unsigned long long excl = s_base + (incl - sum);
        for (uint32_t k = 0; k < warp; ++k) excl += s_red[k];
#pragma unroll
        for (int k = 0; k < 4; ++k) if (i0 + k < N) cum[i0 + k] = excl + w[k];
        __syncthreads();
    }
}

// a4 (bit genomes, Poisson crossovers, R8): one thread per (offspring, gamete, chromosome)
__global__ void __launch_bounds__(256) k_gamete_bit(const __grid_constant__ SpK sp) {
    const DevSpecies &st = *sp.st;
    const uint32_t M = st.m, step = sp.glob->step;
    const uint32_t per = 2 * sp.n_chrom;
    const unsigned long long total = (unsigned long long)M * per;
    const uint32_t *pop = (const uint32_t *)sp.pop[st.cur];
    const uint32_t *rowptr = sp.rowptr[st.cur];
    uint32_t *out = (uint32_t *)sp.offbuf;
    const uint32_t rw = 2 * sp.W;
    for (unsigned long long idx = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
         idx += (unsigned long long)gridDim.x * blockDim.x) {
        const uint32_t j = (uint32_t)(idx / per), rem = (uint32_t)(idx % per);
        const uint32_t g = rem / sp.n_chrom, c = rem % sp.n_chrom;
        const uint32_t parent = rowptr[g == 0 ? sp.mother[j] : sp.father[j]];
        const uint32_t cs = sp.chrom_start[c] >> 5, cw = sp.chrom_len[c] >> 5, clen = sp.chrom_len[c];
        const uint32_t *h0 = pop + (size_t)parent * rw + cs, *h1 = h0 + sp.W;
        uint32_t *o = out + (size_t)j * rw + g * sp.W + cs;
        const uint32_t stream = g == 0 ? ST_RECOMB_M : ST_RECOMB_P;
        uint32_t x[4], y[4];
        draw(sp.key, sp.species, stream, j, c * 16, step, x);
        const uint32_t nc = poisson_count(sp.T_xover + c * XMAX, sp.xover_len[c], x[0]);
        const uint32_t phi = (x[1] >> 31) ? 0xFFFFFFFFu : 0u;
        for (uint32_t w = 0; w < cw; ++w) {
            uint32_t m = phi;
            int yb = -1;
            for (uint32_t k = 0; k < nc; ++k) {
                uint32_t u;
                if (k == 0) u = x[2];
                else if (k == 1) u = x[3];
                else {
                    const int blk = (int)(c * 16 + 1 + (k - 2) / 4);
                    if (blk != yb) { draw(sp.key, sp.species, stream, j, (uint32_t)blk, step, y); yb = blk; }
                    u = y[(k - 2) & 3];
                }
                // crossover in interval b (between local loci b and b+1) flips every locus > b
                const int t = (int)uniform_index(u, clen - 1) + 1 - (int)(32 * w);
                m ^= (t <= 0) ? 0xFFFFFFFFu : (t >= 32 ? 0u : (0xFFFFFFFFu << t));
            }
            o[w] = (h0[w] & ~m) | (h1[w] & m);
        }
    }
}

// a4 (q10 genomes, per-interval draws, R7): one lane per Philox block = 4 loci; the phase is a
// prefix parity over the gamete, done with a ballot inside lane groups of GS = min(nb, 32).
__global__ void __launch_bounds__(256) k_gamete_q10(const __grid_constant__ SpK sp) {
    const DevSpecies &st = *sp.st;
    const uint32_t M = st.m, step = sp.glob->step, L = sp.L;
    const uint32_t nb = (L + 3) / 4;
    uint32_t GS = 32;  // lane-group size: a power of two that holds a whole gamete, else 32
    if (nb < 32 && (nb & (nb - 1)) == 0) GS = nb;
    const uint32_t gpw = 32 / GS;          // gametes per warp pass
    const uint32_t chunks = (nb + GS - 1) / GS;
    const uint32_t lane = threadIdx.x & 31u, sub = lane / GS, sl = lane % GS;
    const uint32_t gmask = (GS == 32) ? 0xFFFFFFFFu : (((1u << GS) - 1u) << (sub * GS));
    const uint32_t lt = gmask & ((1u << lane) - 1u);
    const unsigned long long n_gam = 2ull * M;
    const unsigned long long warp0 = ((unsigned long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const unsigned long long n_warps = ((unsigned long long)gridDim.x * blockDim.x) >> 5;
    const int16_t *pop = (const int16_t *)sp.pop[st.cur];
    const uint32_t *rowptr = sp.rowptr[st.cur];
    int16_t *out = (int16_t *)sp.offbuf;
    for (unsigned long long gb = warp0 * gpw; gb < n_gam; gb += n_warps * gpw) {
        const unsigned long long gi = gb + sub;
        const bool live = gi < n_gam;
        const uint32_t j = (uint32_t)(gi >> 1), g = (uint32_t)(gi & 1);
        uint32_t parent = 0;
        if (live) parent = rowptr[g == 0 ? sp.mother[j] : sp.father[j]];
        const int16_t *h0 = pop + (size_t)parent * 2 * L, *h1 = h0 + L;
        int16_t *o = out + (size_t)j * 2 * L + (size_t)g * L;
        uint32_t carry = 0;
        for (uint32_t ch = 0; ch < chunks; ++ch) {
            const uint32_t blk = ch * GS + sl;
            const bool act = live && blk < nb;
            uint32_t p[4] = {0, 0, 0, 0};
            if (act) {
                uint32_t x[4];
                draw(sp.key, sp.species, g == 0 ? ST_RECOMB_M : ST_RECOMB_P, j, blk, step, x);
                uint32_t run = 0;
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const uint32_t l = 4 * blk + k;
                    if (l < L) run ^= (x[k] < sp.T_recomb[l]) ? 1u : 0u;
                    p[k] = run;
                }
            }
            const uint32_t bal = __ballot_sync(0xffffffffu, p[3] != 0);
            const uint32_t excl = (__popc(bal & lt) & 1u) ^ carry;
            carry ^= __popc(bal & gmask) & 1u;
            if (act) {
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const uint32_t l = 4 * blk + k;
                    if (l < L) o[l] = (excl ^ p[k]) ? h1[l] : h0[l];
                }
            }
        }
    }
}

// a4 + a5 (q10 genomes, R7 + R10) for L = 8 ... 256 a power of two: a lane owns 8 consecutive loci of
// one gamete (two RECOMB blocks, 16 bytes of each parental haplotype, one 128-bit store), GS = L / 8
// lanes make a gamete, and a warp works on whole offspring: both gametes side by side (L <= 128;
// several offspring per warp when L <= 64) or one after the other (L = 256).
//   * The lane's eight switch thresholds never change (its slot in the gamete is fixed): registers.
//   * The phase is the XOR prefix of the switch bits: within the lane by shift-and-xor on the packed
//     byte (built by a carry chain), across the lanes of the gamete by a ballot.  The select masks come
//     from the phase byte by a multiply (bit k -> sign bit of byte k) and a sign-replicating byte permute.
//   * The lane's share of the additive phenotype (sum of the 8 alleles it selected) is reduced over the
//     offspring's lanes (one REDUX), so the offspring row is never read again for a5.
//   * The parents' rows are random gathers; two ways of keeping them in flight, chosen by L on
//     measurements (C5 / C4 / C2, ms per launch):
//       k_gamete_q10v (L <= 128): the rows of the NEXT iteration are loaded into registers before this
//         one's draws are computed, the parents' indices are looked up two iterations ahead
//         (L = 128: 0.893; the ring below 1.03; C2, L = 64: 0.021 against 0.047);
//       k_gamete_q10r (L = 256, where two passes of row registers leave few warps): every lane copies
//         ITS 2 x 16 bytes per pass with cp.async into a ring of D iterations per warp in shared
//         memory and reads them back itself (no barrier: a thread only waits for its own copy
//         groups); indices one stage per iteration ahead of the copies (0.677 against 0.731).
__host__ __device__ inline bool gamete_q10v_supported(const SpK &k) {
    return k.kind == 1 && k.L >= 8 && k.L <= 256 && (k.L & (k.L - 1)) == 0;
}

__device__ __forceinline__ uint32_t prmt_sign(uint32_t a, uint32_t sel) {
    uint32_t d;
    asm("prmt.b32 %0, %1, %1, %2;" : "=r"(d) : "r"(a), "r"(sel));   // selector nibble 8 | i: sign of byte i replicated
    return d;
}

// resident CTAs per SM the register budget is set for (measured: L = 128 at 7 x 4 warps, 72 registers,
// 0.893 ms per C5 launch; 8 x 4 at 64 registers with spills 0.995; 256-thread CTAs x 3: 1.110), and the
// depth of the L = 256 ring (C4: depth 4 at 5 CTAs 0.677 ms, depth 3 at 6 CTAs 0.699, depth 2 at 7: 0.709)
constexpr int Q10V_MINB = 7, Q10V_MINB256 = 5, Q10V_DEPTH256 = 4;
constexpr int Q10V_THREADS = 128;
template <uint32_t LL> struct Q10V {
    static constexpr uint32_t GS = LL >> 3;                            // lanes per gamete
    static constexpr uint32_t LPO = (2u * GS < 32u) ? 2u * GS : 32u;   // lanes per offspring in one pass
    static constexpr uint32_t NPASS = (2u * GS) / LPO;                 // 2 when L = 256, else 1
    static constexpr uint32_t OPW = 32u / LPO;                         // offspring per warp iteration
    static constexpr uint32_t ROW = LL * 4u;                           // bytes per row
    static constexpr uint32_t D = Q10V_DEPTH256;                 // ring depth (iterations in flight), k_gamete_q10r
    static constexpr uint32_t ITEM = NPASS * 2u * 32u * 16u;           // bytes of one iteration's rows per warp
    static constexpr uint32_t SMEM = LL == 256 ? (Q10V_THREADS / 32) * D * ITEM : 0u;
};

// the lane's constants of the q10 gamete kernels
template <uint32_t LL> struct Q10Lane {
    uint32_t li, osub, slot, g0, lt, gmask, omask;
    uint4 t0, t1;
    __device__ __forceinline__ Q10Lane(const SpK &sp) {
        using C = Q10V<LL>;
        const uint32_t lane = threadIdx.x & 31u;
        li = lane & (C::LPO - 1u); osub = lane / C::LPO;
        slot = li & (C::GS - 1u); g0 = (C::NPASS == 1) ? li / C::GS : 0u;   // gamete of pass p: g0 + p
        lt = (1u << lane) - 1u;
        gmask = (C::GS == 32u ? 0xFFFFFFFFu : ((1u << C::GS) - 1u)) << (lane - slot);
        omask = (C::LPO == 32u ? 0xFFFFFFFFu : ((1u << C::LPO) - 1u)) << (lane - li);
        t0 = ((const uint4 *)sp.T_recomb)[2u * slot]; t1 = ((const uint4 *)sp.T_recomb)[2u * slot + 1u];
    }
};

// switch bit of one locus shifted into the packed byte: sub.cc sets the carry iff x >= T (no switch)
__device__ __forceinline__ void q10_push(uint32_t &ph, uint32_t x, uint32_t T) {
    asm("{\n\t.reg .u32 t;\n\tsub.cc.u32 t, %1, %2;\n\taddc.u32 %0, %0, %0;\n\t}" : "+r"(ph) : "r"(x), "r"(T));
}

// q10_push relies on the carry flag after sub.cc being 1 iff x >= T (the hardware's NOT-borrow), which the
// PTX manual does not promise in those words.  spegg_create runs this once per simulation that uses the
// vectorised q10 kernels and refuses to go on if the bit comes out the other way round (a toolkit that
// changed the translation would otherwise flip every recombination phase silently; parity tests would
// catch it, a user without the oracle would not).  v: five (x, T) pairs; expected bits 1,0,1,0,1.
struct PushProbe { uint32_t x[5], T[5]; };
__global__ void k_selftest_push(const PushProbe v, uint32_t *out) {
    uint32_t ph = 0;
#pragma unroll
    for (int i = 0; i < 5; ++i) q10_push(ph, v.x[i], v.T[i]);
    *out = ph | 0x100u;
}
constexpr uint32_t PUSH_PROBE_EXPECT = 0x100u | 0x15u;   // 1,0,1,0,1 pushed MSB-first

// one pass: gamete g of offspring j from the parental haplotype words a (hap0), b (hap1) of this lane
template <uint32_t LL>
__device__ __forceinline__ void q10_pass(const SpK &sp, const Q10Lane<LL> &ln, uint32_t j, uint32_t g, uint32_t M, uint32_t step,
                                         uint8_t *out, const uint4 &a, const uint4 &b, int &acc) {
    using C = Q10V<LL>;
    // R7: switch bits of this lane's 8 loci, packed (locus 0 in bit 0), and their running parity
    uint32_t x[4], y[4];
    const uint32_t stream = g ? ST_RECOMB_P : ST_RECOMB_M;
    draw_rk(sp, stream, j, 2u * ln.slot, step, x);
    draw_rk(sp, stream, j, 2u * ln.slot + 1u, step, y);
    uint32_t ph = 0;
    q10_push(ph, y[3], ln.t1.w); q10_push(ph, y[2], ln.t1.z); q10_push(ph, y[1], ln.t1.y); q10_push(ph, y[0], ln.t1.x);
    q10_push(ph, x[3], ln.t0.w); q10_push(ph, x[2], ln.t0.z); q10_push(ph, x[1], ln.t0.y); q10_push(ph, x[0], ln.t0.x);
    ph = ~ph & 0xFFu;                                 // bit k: locus k of the lane switches
    ph ^= ph << 1; ph ^= ph << 2; ph ^= ph << 4;      // bit k = parity of the switch bits of loci 0..k of the lane
    const uint32_t bal = __ballot_sync(0xffffffffu, (ph & 0x80u) != 0);
    if (__popc(bal & ln.gmask & ln.lt) & 1u) ph = ~ph;
    // select: allele from hap1 where the phase bit is set.  bit k of a nibble -> sign bit of byte k
    // (k + 7 + 7k = 8k + 7; the other products land on other bits), replicated over the allele's two bytes
    const uint32_t lo = (ph & 0xFu) * 0x10204080u, hi = ((ph >> 4) & 0xFu) * 0x10204080u;
    const uint32_t m0 = prmt_sign(lo, 0x9988u), m1 = prmt_sign(lo, 0xBBAAu), m2 = prmt_sign(hi, 0x9988u), m3 = prmt_sign(hi, 0xBBAAu);
    uint4 o;
    o.x = (a.x & ~m0) | (b.x & m0); o.y = (a.y & ~m1) | (b.y & m1);
    o.z = (a.z & ~m2) | (b.z & m2); o.w = (a.w & ~m3) | (b.w & m3);
    if (j < M) {
        ((uint4 *)(out + (size_t)j * C::ROW))[g * C::GS + ln.slot] = o;
        // R10: both int16 halves of a word summed by one dp2a
        acc = __dp2a_lo((int)o.x, 0x0101, acc); acc = __dp2a_lo((int)o.y, 0x0101, acc);
        acc = __dp2a_lo((int)o.z, 0x0101, acc); acc = __dp2a_lo((int)o.w, 0x0101, acc);
    }
}

template <uint32_t LL>
__global__ void __launch_bounds__(Q10V_THREADS, Q10V_MINB) k_gamete_q10v(const __grid_constant__ SpK sp) {
    using C = Q10V<LL>;
    static_assert(C::NPASS == 1, "L = 256 runs k_gamete_q10r");
    const DevSpecies &st = *sp.st;
    const uint32_t M = st.m, step = sp.glob->step;
    const Q10Lane<LL> ln(sp);
    const uint32_t gw = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, n_warps = (gridDim.x * blockDim.x) >> 5;
    const uint8_t *pop = sp.pop[st.cur];
    const uint32_t *rowptr = sp.rowptr[st.cur];
    uint8_t *out = offspring_rows(sp);
    // parents' rows of the offspring this lane works on in the iteration that starts at ob_
    // (32-bit offspring indices: M <= capacity < 2^31 and two strides are far below 2^31)
    auto parents = [&](uint32_t ob_, uint32_t &p0, uint32_t &p1) {
        const uint32_t j_ = ob_ + ln.osub;
        p0 = 0u; p1 = 0u;
        if (j_ < M) { p0 = rowptr[sp.mother[j_]]; p1 = rowptr[sp.father[j_]]; }
    };
    // (volatile asm: the loads are issued HERE, ahead of the draws, not sunk to their first use; a dead
    // lane reads row 0)
    auto rows = [&](uint32_t par, uint4 &a, uint4 &b) {
        const uint4 *h0 = (const uint4 *)(pop + (size_t)par * C::ROW) + ln.slot;
        asm volatile("ld.global.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(a.x), "=r"(a.y), "=r"(a.z), "=r"(a.w) : "l"(h0));
        asm volatile("ld.global.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(b.x), "=r"(b.y), "=r"(b.z), "=r"(b.w) : "l"(h0 + C::GS));
    };
    const uint32_t stride = n_warps * C::OPW, ob0 = gw * C::OPW;
    uint32_t pm, pf, nm, nf;
    parents(ob0, pm, pf);
    parents(ob0 + stride, nm, nf);
    // one iteration: works on the rows in (a, b), loads the next iteration's into (na, nb)
    auto iteration = [&](uint32_t ob, const uint4 &a, const uint4 &b, uint4 &na, uint4 &nb) {
        const uint32_t j = ob + ln.osub;
        uint32_t n2m, n2f;
        parents(ob + 2u * stride, n2m, n2f);
        int acc = 0;
        rows(ln.g0 ? nf : nm, na, nb);
        q10_pass<LL>(sp, ln, j, ln.g0, M, step, out, a, b, acc);
        acc = __reduce_add_sync(ln.omask, acc);
        if (j < M && ln.li == 0) sp.zi[j] = acc;
        pm = nm; pf = nf; nm = n2m; nf = n2f;
    };
    uint4 a0, b0, a1, b1;
    rows(ln.g0 ? pf : pm, a0, b0);
    for (uint32_t ob = ob0; ob < M; ob += stride) {     // two iterations per trip: the row registers ping-pong
        iteration(ob, a0, b0, a1, b1);
        ob += stride;
        if (ob >= M) break;
        iteration(ob, a1, b1, a0, b0);
    }
}

template <uint32_t LL>
__global__ void __launch_bounds__(Q10V_THREADS, Q10V_MINB256) k_gamete_q10r(const __grid_constant__ SpK sp) {
    using C = Q10V<LL>;
    constexpr uint32_t D = C::D;
    extern __shared__ __align__(16) uint8_t s_ring[];
    const DevSpecies &st = *sp.st;
    const uint32_t M = st.m, step = sp.glob->step;
    const Q10Lane<LL> ln(sp);
    const uint32_t gw = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, n_warps = (gridDim.x * blockDim.x) >> 5;
    const uint8_t *pop = sp.pop[st.cur];
    const uint32_t *rowptr = sp.rowptr[st.cur];
    uint8_t *out = offspring_rows(sp);
    // this lane's 16 bytes of (ring item k, pass p, haplotype h): lanes contiguous, so conflict-free
    const uint32_t ring = smem_u32(s_ring) + (threadIdx.x >> 5) * D * C::ITEM + (threadIdx.x & 31u) * 16u;
    // the parents of the offspring this lane works on in the iteration that starts at ob_ (32-bit offspring
    // indices: M <= capacity < 2^31 and D + 2 strides are far below 2^31): their logical indices ...
    auto parents1 = [&](uint32_t ob_, uint32_t &i0, uint32_t &i1) {
        const uint32_t j_ = ob_ + ln.osub;
        i0 = 0xFFFFFFFFu; i1 = 0xFFFFFFFFu;
        if (j_ < M) { i0 = sp.mother[j_]; i1 = sp.father[j_]; }
    };
    // ... and the rows they live in (a dead lane copies from row 0)
    auto parents2 = [&](uint32_t i0, uint32_t i1, uint32_t &p0, uint32_t &p1) {
        p0 = 0u; p1 = 0u;
        if (i0 != 0xFFFFFFFFu) { p0 = rowptr[i0]; p1 = rowptr[i1]; }
    };
    // asynchronous copy of this lane's words of both haplotypes of the rows (r_m, r_f) into ring item k
    auto copy_rows = [&](uint32_t k, uint32_t r_m, uint32_t r_f) {
#pragma unroll
        for (uint32_t p = 0; p < C::NPASS; ++p) {
            const uint32_t g = ln.g0 + p;
            const uint4 *h0 = (const uint4 *)(pop + (size_t)(g ? r_f : r_m) * C::ROW) + ln.slot;
            const uint32_t dst = ring + k * C::ITEM + p * 1024u;
            cp_async16(dst, h0);
            cp_async16(dst + 512u, h0 + C::GS);
        }
        cp_async_commit();
    };
    const uint32_t stride = n_warps * C::OPW, ob0 = gw * C::OPW;
    // prologue: the copies of iterations 0 .. D-1 are started, the rows' numbers of D and the indices of D+1
    // loaded (all index loads first, so that they travel together)
    uint32_t pi_m[D + 2], pi_f[D + 2], pr_m[D + 1], pr_f[D + 1];
#pragma unroll
    for (uint32_t k = 0; k < D + 2; ++k) parents1(ob0 + k * stride, pi_m[k], pi_f[k]);
#pragma unroll
    for (uint32_t k = 0; k < D + 1; ++k) parents2(pi_m[k], pi_f[k], pr_m[k], pr_f[k]);
#pragma unroll
    for (uint32_t k = 0; k < D; ++k) copy_rows(k, pr_m[k], pr_f[k]);
    uint32_t r_m = pr_m[D], r_f = pr_f[D], i_m = pi_m[D + 1], i_f = pi_f[D + 1];
    uint32_t k = 0;                                          // ring item of the current iteration
    for (uint32_t ob = ob0; ob < M; ob += stride) {
        const uint32_t j = ob + ln.osub;
        uint32_t i_m2, i_f2, r_m1, r_f1;
        parents1(ob + (D + 2u) * stride, i_m2, i_f2);        // indices of iteration n + D + 2
        parents2(i_m, i_f, r_m1, r_f1);                      // rows' numbers of n + D + 1
        cp_async_wait<(int)D - 1>();                         // this thread's copies of iteration n have landed
        int acc = 0;
#pragma unroll
        for (uint32_t p = 0; p < C::NPASS; ++p) {
            const uint32_t src = ring + k * C::ITEM + p * 1024u;
            const uint4 a = lds128(src), b = lds128(src + 512u);
            q10_pass<LL>(sp, ln, j, ln.g0 + p, M, step, out, a, b, acc);
        }
        copy_rows(k, r_m, r_f);                              // rows of n + D into the item just consumed
        acc = __reduce_add_sync(ln.omask, acc);
        if (j < M && ln.li == 0) sp.zi[j] = acc;
        r_m = r_m1; r_f = r_f1; i_m = i_m2; i_f = i_f2;
        k = (k + 1u == D) ? 0u : k + 1u;
    }
    cp_async_wait_all();
}

// grid: as many CTAs as are resident at once (the loop strides over the offspring), never more than
// the capacity needs.  The resident count is a property of the DEVICE AND CONTEXT a simulation lives in:
// gamete_q10v_configure is called by spegg_create with that device current (it also raises the kernel's
// dynamic shared-memory limit there) and the result is kept in the spegg_sim, not in the process.
template <uint32_t LL>
inline auto gamete_q10v_kernel() { if constexpr (LL == 256) return k_gamete_q10r<LL>; else return k_gamete_q10v<LL>; }

template <uint32_t LL>
inline cudaError_t gamete_q10v_configure_t(int *per_sm) {
    auto kern = gamete_q10v_kernel<LL>();
    cudaError_t e = cudaSuccess;
    if (Q10V<LL>::SMEM) e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Q10V<LL>::SMEM);
    if (e != cudaSuccess) return e;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(per_sm, kern, Q10V_THREADS, Q10V<LL>::SMEM);
    if (e != cudaSuccess) return e;
    if (*per_sm < 1) *per_sm = 1;
    return cudaSuccess;
}

inline cudaError_t gamete_q10v_configure(uint32_t L, int *per_sm) {
    switch (L) {
    case 8: return gamete_q10v_configure_t<8>(per_sm);
    case 16: return gamete_q10v_configure_t<16>(per_sm);
    case 32: return gamete_q10v_configure_t<32>(per_sm);
    case 64: return gamete_q10v_configure_t<64>(per_sm);
    case 128: return gamete_q10v_configure_t<128>(per_sm);
    case 256: return gamete_q10v_configure_t<256>(per_sm);
    default: return cudaErrorInvalidValue;
    }
}

template <uint32_t LL>
inline cudaError_t launch_gamete_q10v_t(const SpK &k, uint32_t n_sms, int per_sm, cudaStream_t stream) {
    const uint64_t per_cta = (uint64_t)(Q10V_THREADS / 32) * Q10V<LL>::OPW;
    const uint64_t need = ((uint64_t)k.capacity + per_cta - 1) / per_cta;
    const uint32_t grid = (uint32_t)std::max<uint64_t>(1, std::min<uint64_t>(need, (uint64_t)n_sms * (uint64_t)std::max(per_sm, 1)));
    gamete_q10v_kernel<LL>()<<<grid, Q10V_THREADS, Q10V<LL>::SMEM, stream>>>(k);
    return cudaGetLastError();
}

inline cudaError_t launch_gamete_q10v(const SpK &k, uint32_t n_sms, int per_sm, cudaStream_t stream) {
    switch (k.L) {
    case 8: return launch_gamete_q10v_t<8>(k, n_sms, per_sm, stream);
    case 16: return launch_gamete_q10v_t<16>(k, n_sms, per_sm, stream);
    case 32: return launch_gamete_q10v_t<32>(k, n_sms, per_sm, stream);
    case 64: return launch_gamete_q10v_t<64>(k, n_sms, per_sm, stream);
    case 128: return launch_gamete_q10v_t<128>(k, n_sms, per_sm, stream);
    case 256: return launch_gamete_q10v_t<256>(k, n_sms, per_sm, stream);
    default: return cudaErrorInvalidValue;
    }
}

// a4: sparse mutation (R9) of gamete g of offspring j, applied after recombination.  Returns the change
// of the offspring's integer genetic value (q10; the bit kernels take the phenotype afterwards).
// (in two halves, so that a caller with several offspring can issue all the count draws before the rare loops)
__device__ __forceinline__ uint32_t mutation_count(const SpK &sp, uint32_t j, uint32_t g, uint32_t step) {
    uint32_t x[4];
    draw_rk(sp, g == 0 ? ST_MUT_M : ST_MUT_P, j, 0, step, x);
    return poisson_count(sp.T_mut, sp.mut_len, x[0]);
}

__device__ __forceinline__ int mutate_apply(const SpK &sp, uint32_t j, uint32_t g, uint32_t step, uint32_t nm) {
    const uint32_t L = sp.L, stream = g == 0 ? ST_MUT_M : ST_MUT_P;
    int delta = 0;
    uint32_t x[4];
    for (uint32_t k = 0; k < nm; ++k) {
        draw(sp.key, sp.species, stream, j, k, step, x);
        const uint32_t pos = uniform_index(x[1], L);
        if (sp.kind == 0) {
            uint32_t *row = (uint32_t *)offspring_rows(sp) + (size_t)j * 2 * sp.W + (size_t)g * sp.W;
            row[pos >> 5] ^= 1u << (pos & 31u);
        } else {
            int16_t *row = (int16_t *)offspring_rows(sp) + (size_t)j * 2 * L + (size_t)g * L;
            const int v0 = (int)row[pos];
            int v = v0 + normal_delta(sp.T_norm, sp.R_norm, x[2]);
            v = max(-32767, min(32767, v));
            row[pos] = (int16_t)v;
            delta += v - v0;
        }
    }
    return delta;
}

__device__ __forceinline__ int mutate_one(const SpK &sp, uint32_t j, uint32_t g, uint32_t step) {
    const uint32_t nm = mutation_count(sp, j, g, step);
    return nm ? mutate_apply(sp, j, g, step, nm) : 0;
}

// one thread per (offspring, gamete)
__global__ void __launch_bounds__(256) k_mutate(const __grid_constant__ SpK sp, int zi_delta) {
    const DevSpecies &st = *sp.st;
    const uint32_t M = st.m, step = sp.glob->step;
    const unsigned long long total = 2ull * M;
    for (unsigned long long gi = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; gi < total;
         gi += (unsigned long long)gridDim.x * blockDim.x) {
        const uint32_t j = (uint32_t)(gi >> 1), g = (uint32_t)(gi & 1);
        const int d = mutate_one(sp, j, g, step);
        if (zi_delta && d) atomicAdd(&sp.zi[j], d);   // a5 was taken before the mutation
    }
}

// integer phenotype of one row, computed by a whole warp (R10)
__device__ __forceinline__ int32_t warp_row_zi(const SpK &sp, const uint8_t *row) {
    const uint32_t lane = threadIdx.x & 31u;
    int32_t acc = 0;
    const uint32_t *w = (const uint32_t *)row;
    const uint32_t nw = sp.row_bytes >> 2;
    if (sp.kind == 0) {
        for (uint32_t i = lane; i < nw; i += 32) acc += __popc(w[i]);
    } else {
        for (uint32_t i = lane; i < nw; i += 32) {
            const uint32_t v = w[i];
            acc += (int32_t)(int16_t)(v & 0xFFFFu) + (int32_t)(int16_t)(v >> 16);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    return sp.kind == 0 ? 2 * acc - 2 * (int32_t)sp.L : acc;
}

// a5: additive genotype -> phenotype map, one warp per offspring
__global__ void __launch_bounds__(256) k_phenotype(const __grid_constant__ SpK sp) {
    const uint32_t M = sp.st->m;
    const uint32_t warp0 = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = (gridDim.x * blockDim.x) >> 5;
    for (uint32_t j = warp0; j < M; j += nw) {
        const int32_t zi = warp_row_zi(sp, offspring_rows(sp) + (size_t)j * sp.row_bytes);
        if ((threadIdx.x & 31u) == 0) sp.zi[j] = zi;
    }
}

// phenotypes of the current adults (write_state / read_state): out[] (nullable) and their sum
__global__ void __launch_bounds__(256) k_adult_zi(const __grid_constant__ SpK sp, uint32_t n, int accumulate, int32_t *out) {
    const uint32_t warp0 = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = (gridDim.x * blockDim.x) >> 5;
    const uint32_t cur = sp.st->cur, lane = threadIdx.x & 31u;
    long long acc = 0;
    for (uint32_t blk = warp0; blk < (n + 31u) / 32u; blk += nw) {
        const int32_t zi = block_adult_zi_rows(sp, sp.pop[cur], sp.rowptr[cur], blk, n);
        const uint32_t i = blk * 32u + lane;
        if (i < n) { if (out) out[i] = zi; acc += zi; if (accumulate && sp.zrow_on) sp.zrow[cur][sp.rowptr[cur][i]] = zi; }
    }
    if (accumulate) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        if (lane == 0 && acc != 0) atomicAdd((unsigned long long *)&sp.st->sum_zi, (unsigned long long)acc);
    }
}

// R20: integer genetic values of this species' current adults, for the species that meets them
__global__ void __launch_bounds__(256) k_enc_zi(const __grid_constant__ SpK sp) {
    const uint32_t N = sp.st->n0, cur = sp.st->cur;
    const uint32_t warp0 = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = (gridDim.x * blockDim.x) >> 5;
    for (uint32_t blk = warp0; blk < (N + 31u) / 32u; blk += nw) {
        const int32_t zi = block_adult_zi(sp, sp.pop[cur], sp.rowptr[cur], blk, N);
        const uint32_t i = blk * 32u + (threadIdx.x & 31u);
        if (i < N) sp.enc_zi[i] = zi;
    }
}

// R21: sexes of the current adults in logical order (dir 0: gather into io[], dir 1: scatter from io[])
__global__ void __launch_bounds__(256) k_sex_io(const __grid_constant__ SpK sp, uint32_t n, uint8_t *io, int dir) {
    const uint32_t cur = sp.st->cur;
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        uint8_t *p = sp.sex[cur] + sp.rowptr[cur][i];
        if (dir) *p = io[i] ? 1 : 0; else io[i] = *p;
    }
}

// rowptr = identity for a freshly written, dense population
__global__ void __launch_bounds__(256) k_iota(uint32_t *p, uint32_t n) {
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) p[i] = i;
}

// rows of the current adults in logical order (read_state): out[i] = pop[rowptr[i]], one warp per row
__global__ void __launch_bounds__(256) k_gather_rows(const __grid_constant__ SpK sp, uint32_t n, uint8_t *out) {
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t warp0 = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = (gridDim.x * blockDim.x) >> 5;
    const uint32_t cur = sp.st->cur;
    for (uint32_t i = warp0; i < n; i += nw) {
        const uint4 *src = (const uint4 *)(sp.pop[cur] + (size_t)sp.rowptr[cur][i] * sp.row_bytes);
        uint4 *d = (uint4 *)(out + (size_t)i * sp.row_bytes);
        for (uint32_t q = lane; q < sp.row_u4; q += 32) d[q] = src[q];
    }
}

// a6: selection / survival (Fig. 1D) of offspring j with integer genetic value zgen, fp32; captures
// credited to a uniformly drawn predator (or to the consumer met, R20).  Writes s[], alive[], captured[];
// returns alive.
// STORE: s[j], alive[j], captured[j] are written for the kernels that read them back (k_cmp_scan, the patch
// pipeline, the debug view); k_select_compact consumes the decision in registers and skips the three stores.
template <bool STORE = true>
__device__ __forceinline__ bool survive_core(const SpK &sp, DevSpecies &st, uint32_t j, int32_t zgen, float u, float theta,
                                             uint32_t step, unsigned int &ties, unsigned int &caps) {
    int32_t zp = zgen;
    if (sp.R_env > 0) {   // R17, eq. S2-14: residual phenotype noise, k quanta from word 1 of SCALAR block 1
        uint32_t y[4];
        draw_rk(sp, ST_SCALAR, j, 1, step, y);
        zp += normal_delta(sp.T_env, sp.R_env, y[1]);
    }
    const float z = __fmul_rn((float)zp, sp.pheno_scale);
    bool captured;
    float s;
    uint32_t met = 0xFFFFFFFFu;
    if (sp.enc_E) {
        // R20 (eq. S3-2): meeting k = 0..E-1 until the first capture: consumer
        // i_k uniform (word 2(k%2) of SCALAR block 2 + k/2), m = e/(1+e), e = expf_spec(-(d*d)),
        // d = z - z_{i_k}; captured iff u01(word 2(k%2)+1) < v*m.  The stabilising term stays separate.
        captured = false;
        const uint32_t NC = st.n_pred0;
        uint32_t y[4];
        for (uint32_t k = 0; k < sp.enc_E && NC && !captured; ++k) {
            if ((k & 1u) == 0) draw_rk(sp, ST_SCALAR, j, 2 + (k >> 1), step, y);
            const uint32_t ik = uniform_index(y[2 * (k & 1u)], NC);
            const float d = __fsub_rn(z, __fmul_rn((float)sp.pred_zi[ik], sp.pred_scale));
            const float e = expf_spec(-__fmul_rn(d, d));
            const float p = __fmul_rn(sp.enc_v, __fdiv_rn(e, __fadd_rn(1.0f, e)));
            const float uk = u01_of(y[2 * (k & 1u) + 1]);
            if (fabsf(__fsub_rn(uk, p)) < 1e-6f) ++ties;
            if (uk < p) { captured = true; met = ik; }
        }
        s = 1.0f;
        if (sp.sel_gaussian) {
            const float d = __fsub_rn(z, theta);
            s = expf_spec(-__fmul_rn(__fmul_rn(d, d), sp.sel_c));
        }
    } else {
        s = survival_prob(sp, z, theta, u, captured);
    }
    const bool is_alive = u < s && met == 0xFFFFFFFFu;
    if (STORE) {
        sp.s[j] = s;
        sp.alive[j] = is_alive ? 1 : 0;
        sp.captured[j] = captured ? 1 : 0;
    }
    if (fabsf(__fsub_rn(u, s)) < 1e-6f) ++ties;
    if (captured) {
        ++caps;
        if (met != 0xFFFFFFFFu) atomicAdd(&sp.cap_pred[met], 1u);
        else if (st.n_pred0) {
            uint32_t y[4];
            draw(sp.key, sp.species, ST_SCALAR, j, 1, step, y);
            atomicAdd(&sp.cap_pred[uniform_index(y[0], st.n_pred0)], 1u);
        }
    }
    return is_alive;
}

__device__ __forceinline__ bool survive_one(const SpK &sp, DevSpecies &st, uint32_t j, int32_t zgen, uint32_t step,
                                            unsigned int &ties, unsigned int &caps) {
    const float theta = sp.theta_patch ? sp.theta_patch[sp.dest[j]] : st.theta_t;
    return survive_core(sp, st, j, zgen, sp.u01[j], theta, step, ties, caps);
}

__global__ void __launch_bounds__(256) k_survival(const __grid_constant__ SpK sp) {
    DevSpecies &st = *sp.st;
    const uint32_t M = st.m, step = sp.glob->step;
    unsigned int ties = 0, caps = 0;
    for (uint32_t j = blockIdx.x * blockDim.x + threadIdx.x; j < M; j += gridDim.x * blockDim.x)
        survive_one(sp, st, j, sp.zi[j], step, ties, caps);
    if (ties) atomicAdd(&st.near_ties, (unsigned long long)ties);
    if (caps) atomicAdd(&st.captures, (unsigned long long)caps);
}

// a4 (mutation) + a6 in one pass, one thread per offspring: the production q10 pipeline, where the gamete
// kernel has already taken the phenotype and the mutation only corrects it
__global__ void __launch_bounds__(256) k_mut_surv(const __grid_constant__ SpK sp) {
    DevSpecies &st = *sp.st;
    const uint32_t M = st.m, step = sp.glob->step;
    unsigned int ties = 0, caps = 0;
    for (uint32_t j = blockIdx.x * blockDim.x + threadIdx.x; j < M; j += gridDim.x * blockDim.x) {
        const int d = mutate_one(sp, j, 0, step) + mutate_one(sp, j, 1, step);
        int32_t zi = sp.zi[j];
        if (d) { zi += d; sp.zi[j] = zi; }
        survive_one(sp, st, j, zi, step, ties, caps);
    }
    if (ties) atomicAdd(&st.near_ties, (unsigned long long)ties);
    if (caps) atomicAdd(&st.captures, (unsigned long long)caps);
}

// R18, overlapping generations: adult i stays alive with probability
// s_A * w(z_i) -- w the Gaussian term of R11 at its genetic value, the uniform word 1 of its FEC
// block; fp32 in this order: p = s_A * w.  A warp per block of 32 adults, one adult per lane (the genetic values are re-read from the rows).
__global__ void __launch_bounds__(256) k_adult_survive(const __grid_constant__ SpK sp) {
    DevSpecies &st = *sp.st;
    const uint32_t N = st.n0, step = sp.glob->step, lane = threadIdx.x & 31u;
    const uint32_t warp0 = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = (gridDim.x * blockDim.x) >> 5;
    const uint8_t *pop = sp.pop[st.cur];
    const uint32_t *rowptr = sp.rowptr[st.cur];
    const uint32_t *ps = sp.patch_start[st.cur];
    unsigned int ties = 0;
    for (uint32_t blk = warp0; blk < (N + 31u) / 32u; blk += nw) {   // a warp per block of 32 adults, one adult per lane
        const int32_t zi = block_adult_zi(sp, pop, rowptr, blk, N);
        const uint32_t i = blk * 32u + lane;
        if (i < N) {
            uint32_t x[4];
            draw_rk(sp, ST_FEC, i, 0, step, x);
            const float u = u01_of(x[1]);
            float w = 1.0f;
            // (an adult keeps its patch: the optimum is its own patch's)
            const float theta = sp.theta_patch ? sp.theta_patch[sp.P > 1 ? patch_of(ps, sp.P, i) : 0u] : st.theta_t;
            if (sp.sel_gaussian) {
                const float d = __fsub_rn(__fmul_rn((float)zi, sp.pheno_scale), theta);
                w = expf_spec(-__fmul_rn(__fmul_rn(d, d), sp.sel_c));
            }
            const float p = __fmul_rn(sp.adult_surv, w);
            sp.a_zi[i] = zi; sp.a_u[i] = u; sp.a_s[i] = p;
            sp.a_alive[i] = (u < p) ? 1 : 0;
            if (fabsf(__fsub_rn(u, p)) < 1e-6f) ++ties;
        }
    }
    if (ties) atomicAdd(&st.near_ties, (unsigned long long)ties);
}

// a7 (unstructured): stable compaction positions by decoupled look-back + survivor reductions
__global__ void __launch_bounds__(SCAN_THREADS) k_cmp_scan(const __grid_constant__ SpK sp) {
    __shared__ uint32_t s_warp[SCAN_THREADS / 32];
    __shared__ uint32_t s_tile;
    __shared__ unsigned long long s_excl;
    DevSpecies &st = *sp.st;
    // items: the NA adults (R18; none when generations are discrete), then the M offspring -- which is
    // the order of the next generation
    const uint32_t NA = sp.adult_surv > 0.0f ? st.n0 : 0u, M = NA + st.m;
    const uint32_t n_tiles = (M + SCAN_TILE - 1) / SCAN_TILE;
    const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    long long a1 = 0, a2 = 0;
    if (M == 0 && blockIdx.x == 0 && tid == 0) st.n_next = 0;
    for (;;) {
        if (tid == 0) s_tile = atomicAdd(&st.ticket_cmp, 1u);
        __syncthreads();
        const uint32_t tile = s_tile;
        if (tile >= n_tiles) break;
        const uint32_t base = tile * SCAN_TILE + tid * SCAN_ITEMS;
        uint32_t a[SCAN_ITEMS], sum = 0;
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS; ++k) {
            const uint32_t j = base + k;
            a[k] = (j < M) ? (j < NA ? sp.a_alive[j] : sp.alive[j - NA]) : 0u;
            sum += a[k];
            if (a[k]) { const long long z = j < NA ? sp.a_zi[j] : sp.zi[j - NA]; a1 += z; a2 += z * z; }
        }
        const uint32_t incl = warp_incl_scan(sum);
        if (lane == 31) s_warp[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            uint32_t w = (lane < SCAN_THREADS / 32) ? s_warp[lane] : 0u;
            const uint32_t wi = warp_incl_scan(w);
            const uint32_t total = __shfl_sync(0xffffffffu, wi, SCAN_THREADS / 32 - 1);
            const unsigned long long excl = lookback(sp.status_cmp, sp.status_cmp_n, tile, (unsigned long long)total);
            if (lane < SCAN_THREADS / 32) s_warp[lane] = wi - w;
            if (lane == 0) {
                s_excl = excl;
                if (tile == n_tiles - 1) st.n_next = (uint32_t)(excl + total);
            }
        }
        __syncthreads();
        uint32_t o = (uint32_t)s_excl + s_warp[warp] + (incl - sum);
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS; ++k) {
            const uint32_t j = base + k;
            if (j < M) { (j < NA ? sp.a_pos[j] : sp.pos[j - NA]) = a[k] ? o : 0xFFFFFFFFu; o += a[k]; }
        }
        __syncthreads();
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { a1 += __shfl_xor_sync(0xffffffffu, a1, o); a2 += __shfl_xor_sync(0xffffffffu, a2, o); }
    if (lane == 0 && (a1 != 0 || a2 != 0)) {
        atomicAdd((unsigned long long *)&st.acc_zi, (unsigned long long)a1);
        atomicAdd((unsigned long long *)&st.acc_zi2, (unsigned long long)a2);
    }
}

// a4 (mutation) + a6 + a7 + a8 in ONE kernel for an unstructured species on the production q10 path with
// discrete generations: a tile of 1,024 offspring (4 per thread) is mutated, selected, scanned, placed by
// one look-back, and its survivors' index words are written -- offspring rows stay where the gamete kernel
// stored them, so nothing else moves.  alive[] / pos[] never travel through memory, and four launches
// (k_mutate, k_survival, k_cmp_scan, k_cmp_scatter) become one.
// ITEMS offspring per thread: 4 (tiles of 1,024) for large populations, 1 (tiles of 256) when the whole
// capacity is fewer tiles than the machine holds CTAs -- a population of 10^5 then spreads over all SMs
// and a thread's work is one offspring, not a chain of four
template <int ITEMS>
__global__ void __launch_bounds__(SCAN_THREADS) k_select_compact(const __grid_constant__ SpK sp) {
    constexpr uint32_t TILE = SCAN_THREADS * ITEMS;
    __shared__ uint32_t s_warp[SCAN_THREADS / 32];
    __shared__ uint32_t s_tile, s_flag;
    __shared__ unsigned long long s_excl;
    __shared__ __align__(4) uint8_t s_alive[TILE];
    DevSpecies &st = *sp.st;
    const uint32_t M = st.m, step = sp.glob->step;
    const uint32_t n_tiles = (M + TILE - 1) / TILE;
    const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    uint32_t *rp = sp.rowptr[st.cur ^ 1u];
    uint8_t *sex_next = sp.sex[st.cur ^ 1u];
    int32_t *zrow_next = sp.zrow[st.cur ^ 1u];
    const float theta = sp.theta_patch ? sp.theta_patch[0] : st.theta_t;   // one patch
    long long a1 = 0, a2 = 0;
    unsigned int ties = 0, caps = 0;
    if (M == 0 && blockIdx.x == 0 && tid == 0) st.n_next = 0;
    for (;;) {
        if (tid == 0) s_tile = atomicAdd(&st.ticket_cmp, 1u);
        __syncthreads();
        const uint32_t tile = s_tile;
        if (tile >= n_tiles) break;
        // ---- phase 1, offspring j = tile * 1024 + k * 256 + tid (coalesced): all loads and all mutation-count
        // draws of the thread's four offspring first, so that they travel together; then the rare mutations,
        // selection, and everything that is indexed by j
        const uint32_t t0 = tile * TILE + tid;
        int32_t zz[ITEMS];
        float uu[ITEMS];
        uint32_t nm[ITEMS];
#pragma unroll
        for (int k = 0; k < ITEMS; ++k) {
            const uint32_t j = t0 + k * SCAN_THREADS;
            zz[k] = 0; uu[k] = 2.0f;
            if (j < M) { zz[k] = sp.zi[j]; uu[k] = sp.u01[j]; }
        }
#pragma unroll
        for (int k = 0; k < ITEMS; ++k) {
            const uint32_t j = t0 + k * SCAN_THREADS;
            nm[k] = 0;
            if (j < M) nm[k] = mutation_count(sp, j, 0, step) | (mutation_count(sp, j, 1, step) << 16);
        }
#pragma unroll
        for (int k = 0; k < ITEMS; ++k) {
            const uint32_t j = t0 + k * SCAN_THREADS;
            bool al = false;
            if (j < M) {
                if (nm[k]) {
                    int d = 0;
                    if (nm[k] & 0xFFFFu) d += mutate_apply(sp, j, 0, step, nm[k] & 0xFFFFu);
                    if (nm[k] >> 16) d += mutate_apply(sp, j, 1, step, nm[k] >> 16);
                    if (d) { zz[k] += d; sp.zi[j] = zz[k]; }
                }
                al = survive_core<false>(sp, st, j, zz[k], uu[k], theta, step, ties, caps);
                if (al) {
                    a1 += zz[k]; a2 += (long long)zz[k] * zz[k];
                    if (sp.sexes) sex_next[j] = sp.sex_off[j];
                    if (sp.zrow_on) zrow_next[j] = zz[k];
                }
            }
            s_alive[k * SCAN_THREADS + tid] = al ? 1 : 0;
        }
        __syncthreads();
        // ---- phase 2, four consecutive offspring per thread: scan, one look-back, the index
        const uint32_t base = tile * TILE + tid * ITEMS;
        const uint32_t a4 = ITEMS == 4 ? ((const uint32_t *)s_alive)[tid] : (uint32_t)s_alive[tid];   // bytes base .. base + ITEMS - 1
        const uint32_t sum = __popc(a4);
        const uint32_t incl = warp_incl_scan(sum);
        if (lane == 31) s_warp[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            uint32_t w = (lane < SCAN_THREADS / 32) ? s_warp[lane] : 0u;
            const uint32_t wi = warp_incl_scan(w);
            const uint32_t total = __shfl_sync(0xffffffffu, wi, SCAN_THREADS / 32 - 1);
            const unsigned long long excl = lookback(sp.status_cmp, sp.status_cmp_n, tile, (unsigned long long)total);
            if (lane < SCAN_THREADS / 32) s_warp[lane] = wi - w;
            if (lane == 0) {
                s_excl = excl;
                if (tile == n_tiles - 1) st.n_next = (uint32_t)(excl + total);
            }
        }
        __syncthreads();
        uint32_t o = (uint32_t)s_excl + s_warp[warp] + (incl - sum);
#pragma unroll
        for (int k = 0; k < ITEMS; ++k)
            if ((a4 >> (8 * k)) & 1u) rp[o++] = base + k;
        __syncthreads();
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { a1 += __shfl_xor_sync(0xffffffffu, a1, o); a2 += __shfl_xor_sync(0xffffffffu, a2, o); }
    if (lane == 0 && (a1 != 0 || a2 != 0)) {
        atomicAdd((unsigned long long *)&st.acc_zi, (unsigned long long)a1);
        atomicAdd((unsigned long long *)&st.acc_zi2, (unsigned long long)a2);
    }
    if (ties) atomicAdd(&st.near_ties, (unsigned long long)ties);
    if (caps) atomicAdd(&st.captures, (unsigned long long)caps);
    if (sp.solo) solo_tail(sp, &s_flag);   // single species: the last CTA closes the step
}

// a7: move the surviving rows to their positions in the other buffer, one warp per row
__global__ void __launch_bounds__(256) k_cmp_scatter(const __grid_constant__ SpK sp) {
    const DevSpecies &st = *sp.st;
    const uint32_t M = st.m, lane = threadIdx.x & 31u;
    const uint32_t warp0 = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = (gridDim.x * blockDim.x) >> 5;
    uint8_t *dst = sp.pop[st.cur ^ 1u];
    uint32_t *rp = sp.rowptr[st.cur ^ 1u];
    uint8_t *sex_next = sp.sex[st.cur ^ 1u];   // R21: the sex travels with the row
    int32_t *zrow_next = sp.zrow[st.cur ^ 1u]; // ... and so does the integer genetic value
    __shared__ uint32_t s_flag;
    if (sp.index_only) {   // the rows stay where the gamete kernel stored them: only the index is written
        for (uint32_t j = blockIdx.x * blockDim.x + threadIdx.x; j < M; j += gridDim.x * blockDim.x) {
            const uint32_t p = sp.pos[j];
            if (p != 0xFFFFFFFFu) { rp[p] = j; if (sp.sexes) sex_next[j] = sp.sex_off[j]; if (sp.zrow_on) zrow_next[j] = sp.zi[j]; }
        }
    } else {
        for (uint32_t j = warp0; j < M; j += nw) {
            const uint32_t p = sp.pos[j];
            if (p == 0xFFFFFFFFu) continue;
            if (lane == 0) { rp[p] = p; if (sp.sexes) sex_next[p] = sp.sex_off[j]; if (sp.zrow_on) zrow_next[p] = sp.zi[j]; }  // materialised path: rows are dense, rowptr is the identity
            const uint4 *src = (const uint4 *)(sp.offbuf + (size_t)j * sp.row_bytes);
            uint4 *d = (uint4 *)(dst + (size_t)p * sp.row_bytes);
            for (uint32_t i = lane; i < sp.row_u4; i += 32) d[i] = src[i];
        }
    }
    // R18: the adults that stay are copied into the other buffer, one warp per row -- behind the
    // offspring rows (row M + rank) when the compaction is index-only, else at their position
    if (sp.adult_surv > 0.0f) {
        const uint32_t N = st.n0, cur = st.cur;
        const uint8_t *src_pop = sp.pop[cur];
        const uint32_t *rp_cur = sp.rowptr[cur];
        // G lanes share a row (a 32-byte row is two 128-bit words: sixteen rows per warp pass)
        uint32_t G = 1;
        while (G < 32u && G < sp.row_u4) G <<= 1;
        const uint32_t apw = 32u / G, grp = lane / G, q = lane % G;
        for (uint32_t i0 = warp0 * apw; i0 < N; i0 += nw * apw) {
            const uint32_t i = i0 + grp;
            if (i >= N) continue;
            const uint32_t p = sp.a_pos[i];
            if (p == 0xFFFFFFFFu) continue;
            const uint32_t row = sp.index_only ? M + (sp.P > 1 ? sp.a_rank[i] : p) : p;
            const uint32_t srow = rp_cur[i];
            if (q == 0) { rp[p] = row; if (sp.sexes) sex_next[row] = sp.sex[cur][srow]; if (sp.zrow_on) zrow_next[row] = sp.a_zi[i]; }
            const uint4 *src = (const uint4 *)(src_pop + (size_t)srow * sp.row_bytes);
            uint4 *d = (uint4 *)(dst + (size_t)row * sp.row_bytes);
            for (uint32_t k = q; k < sp.row_u4; k += G) d[k] = src[k];
        }
    }
    if (sp.solo) solo_tail(sp, &s_flag);   // single unstructured species: the last CTA closes the step
}

// ---- a7 (patches, R15): the next generation is ordered by (destination patch, j).  Offspring of
// natal patch p are a contiguous j-range and land in p or one of its 4 torus neighbours, so the
// stable order is: for destination d, the sources {d, neighbours(d)} in increasing patch index,
// each in j order.  slot = index of the destination in p's de-duplicated list [p, nb0..nb3].
__device__ __forceinline__ uint32_t dest_slot(uint32_t p, uint32_t dest, uint4 nb) {
    if (dest == p) return 0;
    if (nb.x == dest) return 1;
    if (nb.y == dest) return 2;
    if (nb.z == dest) return 3;
    if (nb.w == dest) return 4;
    return 0;
}

__device__ __forceinline__ void patch_offspring_range(const SpK &sp, const uint32_t *ps, uint32_t p, uint32_t N,
                                                      uint32_t M, uint32_t &j0, uint32_t &j1) {
    const uint32_t a0 = ps[p], a1 = ps[p + 1];
    j0 = (a0 < N) ? min(sp.off[a0], M) : M;
    j1 = (a1 < N) ? min(sp.off[a1], M) : M;
}

// A patch's offspring (and its adults) are cut into S = sp.patch_sub equal parts, "segments", so that a
// few large patches (the paper's sweeps: tens of patches of 50,000) still give every SM
// work: segment w = p * S + s is one CTA work item.  With thousands of small patches S = 1.
__device__ __forceinline__ void segment_range(uint32_t lo, uint32_t hi, uint32_t s, uint32_t S, uint32_t &a, uint32_t &b) {
    const unsigned long long len = hi - lo;
    a = lo + (uint32_t)(len * s / S);
    b = lo + (uint32_t)(len * (s + 1u) / S);
}

// counts of survivors per (segment, slot); one CTA per segment.  patch_cnt[w][0..4]: surviving
// offspring by destination slot; [5]: staying adults (R18)
// select = 1 (production q10 path): the segment's offspring are mutated and selected HERE (a4 + a6: what
// k_mut_surv does), so alive[] is produced by the kernel that counts it
__global__ void __launch_bounds__(256) k_patch_count(const __grid_constant__ SpK sp, int select) {
    __shared__ uint32_t s_cnt[6];
    DevSpecies &st = *sp.st;
    const uint32_t *ps = sp.patch_start[st.cur];
    const uint32_t S = sp.patch_sub, step = sp.glob->step;
    unsigned int ties = 0, caps = 0;
    for (uint32_t w = blockIdx.x; w < sp.P * S; w += gridDim.x) {
        const uint32_t p = w / S, sg = w % S;
        if (threadIdx.x < 6) s_cnt[threadIdx.x] = 0;
        __syncthreads();
        uint32_t j0, j1, jj0, jj1;
        patch_offspring_range(sp, ps, p, st.n0, st.m, j0, j1);
        segment_range(j0, j1, sg, S, jj0, jj1);
        const uint4 nb = ((const uint4 *)sp.nbr)[p];
        uint32_t c[5] = {0, 0, 0, 0, 0};
        for (uint32_t j = jj0 + threadIdx.x; j < jj1; j += blockDim.x) {
            bool al;
            if (select) {
                const int d = mutate_one(sp, j, 0, step) + mutate_one(sp, j, 1, step);
                int32_t zi = sp.zi[j];
                if (d) { zi += d; sp.zi[j] = zi; }
                al = survive_one(sp, st, j, zi, step, ties, caps);
            } else al = sp.alive[j] != 0;
            if (al) {
                const uint32_t sl = dest_slot(p, sp.dest[j], nb);
#pragma unroll
                for (uint32_t k = 0; k < 5; ++k) c[k] += (sl == k) ? 1u : 0u;
            }
        }
        uint32_t ca = 0;
        if (sp.adult_surv > 0.0f) {   // R18: the adults of the segment that stay
            uint32_t i0, i1;
            segment_range(ps[p], ps[p + 1], sg, S, i0, i1);
            for (uint32_t i = i0 + threadIdx.x; i < i1; i += blockDim.x) ca += sp.a_alive[i] ? 1u : 0u;
        }
#pragma unroll
        for (uint32_t k = 0; k < 5; ++k) {
            const uint32_t v = __reduce_add_sync(0xffffffffu, c[k]);
            if ((threadIdx.x & 31u) == 0 && v) atomicAdd(&s_cnt[k], v);
        }
        ca = __reduce_add_sync(0xffffffffu, ca);
        if ((threadIdx.x & 31u) == 0 && ca) atomicAdd(&s_cnt[5], ca);
        __syncthreads();
        if (threadIdx.x < 6) sp.patch_cnt[w * 6 + threadIdx.x] = s_cnt[threadIdx.x];
        __syncthreads();
    }
    if (ties) atomicAdd(&st.near_ties, (unsigned long long)ties);
    if (caps) atomicAdd(&st.captures, (unsigned long long)caps);
}

// next patch_start and the base position of every (segment, slot) group.  The next generation's order
// is one flat list: destination by destination; inside destination d its staying adults (R18), then
// source by source (natal patch order, from the host-built topology table); inside each of these the S
// segments in order.  Item q = (d * 6 + o) * S + sg (o = 0: stayers, o = 1..5: the o-th source, absent
// ones count 0) -- so the bases are ONE exclusive scan over P * 6 * S counts, done by a single CTA whose
// threads take contiguous runs of items (and a second scan over the stayers alone for their ranks).
__device__ __forceinline__ uint32_t patch_item_count(const SpK &sp, uint32_t q, uint32_t S, uint32_t &k_out) {
    const uint32_t sg = q % S, o = (q / S) % 6u, d = q / (6u * S);
    k_out = 0xFFFFFFFFu;
    if (o == 0) { k_out = (d * S + sg) * 6u + 5u; return sp.patch_cnt[k_out]; }
    const uint32_t *sl = sp.src_list + (size_t)d * 6;
    if (o > sl[0]) return 0u;
    const uint32_t e = sl[o];
    k_out = ((e >> 3) * S + sg) * 6u + (e & 7u);
    return sp.patch_cnt[k_out];
}

__global__ void __launch_bounds__(1024) k_patch_base(const __grid_constant__ SpK sp) {
    __shared__ uint32_t s_warp[32], s_awarp[32];
    DevSpecies &st = *sp.st;
    uint32_t *psn = sp.patch_start[st.cur ^ 1u];
    const uint32_t P = sp.P, S = sp.patch_sub, tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const uint32_t n = P * 6u * S, per = (n + 1023u) / 1024u;
    const uint32_t q0 = min(tid * per, n), q1 = min(q0 + per, n);
    uint32_t mine = 0, amine = 0, k;
    for (uint32_t q = q0; q < q1; ++q) {
        const uint32_t c = patch_item_count(sp, q, S, k);
        mine += c;
        if ((q / S) % 6u == 0) amine += c;
    }
    const uint32_t incl = warp_incl_scan(mine), aincl = warp_incl_scan(amine);
    if (lane == 31) { s_warp[warp] = incl; s_awarp[warp] = aincl; }
    __syncthreads();
    if (warp == 0) {
        const uint32_t w = s_warp[lane], wi = warp_incl_scan(w), aw = s_awarp[lane], awi = warp_incl_scan(aw);
        s_warp[lane] = wi - w;
        s_awarp[lane] = awi - aw;
        if (lane == 31) { st.n_next = wi; psn[P] = wi; }
    }
    __syncthreads();
    uint32_t run = s_warp[warp] + (incl - mine), arun = s_awarp[warp] + (aincl - amine);
    for (uint32_t q = q0; q < q1; ++q) {
        const uint32_t c = patch_item_count(sp, q, S, k);
        if (q % (6u * S) == 0) psn[q / (6u * S)] = run;
        if (k != 0xFFFFFFFFu) sp.patch_base[k] = run;
        if ((q / S) % 6u == 0) { sp.patch_abase[q / (6u * S) * S + q % S] = arun; arun += c; }
        run += c;
    }
}

// positions of the survivors of each segment (j order within each slot) + reductions
// index = 1 (index-only compaction, discrete generations): rowptr[position] = j (and the sex / genetic
// value that travel with the row) are written here, so no k_cmp_scatter follows
__global__ void __launch_bounds__(256) k_patch_pos(const __grid_constant__ SpK sp, int index) {
    __shared__ uint32_t s_w[8][5];
    __shared__ uint32_t s_run[5];
    DevSpecies &st = *sp.st;
    const uint32_t *ps = sp.patch_start[st.cur];
    uint32_t *rp = sp.rowptr[st.cur ^ 1u];
    uint8_t *sex_next = sp.sex[st.cur ^ 1u];
    int32_t *zrow_next = sp.zrow[st.cur ^ 1u];
    const uint32_t S = sp.patch_sub;
    const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    long long a1 = 0, a2 = 0;
    for (uint32_t wi = blockIdx.x; wi < sp.P * S; wi += gridDim.x) {
        const uint32_t p = wi / S, sg = wi % S;
        if (tid < 5) s_run[tid] = sp.patch_base[wi * 6 + tid];
        uint32_t j0, j1, jj0, jj1;
        patch_offspring_range(sp, ps, p, st.n0, st.m, j0, j1);
        segment_range(j0, j1, sg, S, jj0, jj1);
        const uint4 nb = ((const uint4 *)sp.nbr)[p];
        __syncthreads();
        for (uint32_t c0 = jj0; c0 < jj1; c0 += 256) {
            const uint32_t j = c0 + tid;
            const bool al = j < jj1 && sp.alive[j];
            const uint32_t slot = al ? dest_slot(p, sp.dest[j], nb) : 7u;
            uint32_t rank = 0;
#pragma unroll
            for (uint32_t k = 0; k < 5; ++k) {
                const uint32_t bal = __ballot_sync(0xffffffffu, slot == k);
                if (slot == k) rank = __popc(bal & ((1u << lane) - 1u));
                if (lane == 0) s_w[warp][k] = __popc(bal);
            }
            __syncthreads();
            if (al) {
                uint32_t o = s_run[slot] + rank;
                for (uint32_t w = 0; w < warp; ++w) o += s_w[w][slot];
                const int32_t zj = sp.zi[j];
                if (index) { rp[o] = j; if (sp.sexes) sex_next[j] = sp.sex_off[j]; if (sp.zrow_on) zrow_next[j] = zj; }
                else sp.pos[j] = o;
                const long long z = zj; a1 += z; a2 += z * z;
            } else if (j < jj1 && !index) sp.pos[j] = 0xFFFFFFFFu;
            __syncthreads();
            if (tid < 5) { uint32_t t = 0; for (int w = 0; w < 8; ++w) t += s_w[w][tid]; s_run[tid] += t; }
            __syncthreads();
        }
        __syncthreads();
        if (sp.adult_surv > 0.0f) {
            // R18: the staying adults of the segment, in order i, take the next positions of the patch's front;
            // a_rank = rank among all staying adults (their rows are copied behind the offspring rows)
            uint32_t run = sp.patch_base[wi * 6 + 5], arun = sp.patch_abase[wi], i0, i1;
            segment_range(ps[p], ps[p + 1], sg, S, i0, i1);
            for (uint32_t c0 = i0; c0 < i1; c0 += 256) {
                const uint32_t i = c0 + tid;
                const bool al = i < i1 && sp.a_alive[i];
                const uint32_t bal = __ballot_sync(0xffffffffu, al);
                if (lane == 0) s_w[warp][0] = __popc(bal);
                __syncthreads();
                uint32_t before = __popc(bal & ((1u << lane) - 1u)), tot = 0;
                for (uint32_t w = 0; w < 8; ++w) { const uint32_t v = s_w[w][0]; tot += v; if (w < warp) before += v; }
                if (al) {
                    sp.a_pos[i] = run + before;
                    sp.a_rank[i] = arun + before;
                    const long long z = sp.a_zi[i]; a1 += z; a2 += z * z;
                } else if (i < i1) sp.a_pos[i] = 0xFFFFFFFFu;
                run += tot; arun += tot;
                __syncthreads();
            }
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { a1 += __shfl_xor_sync(0xffffffffu, a1, o); a2 += __shfl_xor_sync(0xffffffffu, a2, o); }
    if (lane == 0 && (a1 != 0 || a2 != 0)) {
        atomicAdd((unsigned long long *)&st.acc_zi, (unsigned long long)a1);
        atomicAdd((unsigned long long *)&st.acc_zi2, (unsigned long long)a2);
    }
}

}  // namespace spegg
