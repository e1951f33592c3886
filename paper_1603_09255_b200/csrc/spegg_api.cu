// spegg_api.cu -- the C ABI of libspegg (include/spegg.h) and the step orchestration.
//
// Host side only marshals: it validates parameters, builds the constant threshold tables, lays
// the caller's workspace out, captures ONE CUDA graph of the step's kernel sequence and replays
// it.  Every step of the path runs in the kernels of spegg_kernels.cuh / spegg_fused.cuh;
// there is no CPU fallback.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <algorithm>
#include <new>
#include <vector>

#include "../../include/spegg.h"
#include "spegg_kernels.cuh"
#include "spegg_fused.cuh"

using namespace spegg;

static_assert(sizeof(LogEntry) == sizeof(spegg_log_entry), "log entry layout");
static_assert(TMAX == SPEGG_TMAX && CAP_TABLES == SPEGG_CAP_TABLES, "table constants");

namespace {

// ------------------------------------------------------------- host-side constant tables
// (the library's own builders; same specified arithmetic as the device code, R4-R9)
double h_exp_neg64(double lam) {
    if (!(lam >= 0.0)) lam = 0.0;
    if (lam > 700.0) return 0.0;
    const double x = -lam;
    const double t = x * 0x1.71547652b82fep+0;
    const double kf = std::floor(t + 0.5);
    const double r = (x - kf * 0x1.62e42fee00000p-1) - kf * 0x1.a39ef35793c76p-33;
    const double c[15] = {
        0x1.0000000000000p+0,  0x1.0000000000000p+0,  0x1.0000000000000p-1,
        0x1.5555555555555p-3,  0x1.5555555555555p-5,  0x1.1111111111111p-7,
        0x1.6c16c16c16c17p-10, 0x1.a01a01a01a01ap-13, 0x1.a01a01a01a01ap-16,
        0x1.71de3a556c734p-19, 0x1.27e4fb7789f5cp-22, 0x1.ae64567f544e4p-26,
        0x1.1eed8eff8d898p-29, 0x1.6124613a86d09p-33, 0x1.93974a8c07c9dp-37};
    double p = c[14];
    for (int i = 13; i >= 0; --i) { p = p * r; p = p + c[i]; }
    const long long bits = (long long)(1023 + (int)kf) << 52;
    double scale;
    std::memcpy(&scale, &bits, 8);
    return p * scale;
}

int h_poisson_table(double lam, uint32_t *T, int maxlen) {
    double p = h_exp_neg64(lam), F = p;
    int k = 0;
    for (;;) {
        const double tk = std::floor(F * 4294967296.0);
        if (tk >= 4294967295.0) break;
        if (k == maxlen) break;
        T[k++] = (uint32_t)tk;
        p = (p * lam) / (double)k;
        F = F + p;
    }
    return k;
}

unsigned long long h_bernoulli_T(double p) {
    if (!(p > 0.0)) return 0ull;
    if (p >= 1.0) return 4294967296ull;
    return (unsigned long long)std::floor(p * 4294967296.0);
}

int h_normal_table(double sq, std::vector<uint32_t> &T) {
    int R = (int)std::ceil(8.0 * sq);
    if (R < 1) R = 1;
    T.resize(2 * (size_t)R);
    for (int k = -R; k < R; ++k) {
        const double a = (double)k + 0.5;
        const double x = a / sq;
        const double y = -x * 0.70710678118654752440;
        const double ph = 0.5 * std::erfc(y);
        double tk = std::floor(ph * 4294967296.0);
        if (tk > 4294967295.0) tk = 4294967295.0;
        T[(size_t)(k + R)] = (uint32_t)tk;
    }
    return R;
}

// ---------------------------------------------------------------------- patch topology (R15)
// neighbour of patch p on the gw x gh torus: direction 0: y-1, 1: x+1, 2: y+1, 3: x-1
uint32_t h_neighbour(uint32_t p, uint32_t dir, uint32_t gw, uint32_t gh) {
    uint32_t px = p % gw, py = p / gw;
    switch (dir) {
    case 0: py = (py + gh - 1) % gh; break;
    case 1: px = (px + 1) % gw; break;
    case 2: py = (py + 1) % gh; break;
    default: px = (px + gw - 1) % gw; break;
    }
    return py * gw + px;
}

// slot of destination `dest` in the de-duplicated list [p, nb0 .. nb3] of natal patch p
uint32_t h_dest_slot(uint32_t p, uint32_t dest, uint32_t gw, uint32_t gh) {
    if (dest == p) return 0;
    for (uint32_t k = 0; k < 4; ++k)
        if (h_neighbour(p, k, gw, gh) == dest) return k + 1;
    return 0;
}

// nbr[p][dir] and, for every destination d, its sources (natal patch, slot), unique per natal patch,
// sorted by natal patch: the order of the next generation inside d (by (natal patch, j))
void h_topology(uint32_t gw, uint32_t gh, std::vector<uint32_t> &nbr, std::vector<uint32_t> &src) {
    const uint32_t P = gw * gh;
    nbr.assign((size_t)P * 4, 0);
    src.assign((size_t)P * 6, 0);
    for (uint32_t p = 0; p < P; ++p)
        for (uint32_t k = 0; k < 4; ++k) nbr[(size_t)p * 4 + k] = h_neighbour(p, k, gw, gh);
    for (uint32_t d = 0; d < P; ++d) {
        uint32_t n = 0, pp[5], ss[5];
        pp[n] = d; ss[n] = 0; ++n;
        for (uint32_t k = 0; k < 4; ++k) {
            const uint32_t q = h_neighbour(d, (k + 2) & 3u, gw, gh);   // the patch whose direction-k neighbour is d
            if (q == d || h_neighbour(q, k, gw, gh) != d) continue;
            bool dup = false;
            for (uint32_t i = 0; i < n; ++i) dup |= (pp[i] == q);
            if (!dup) { pp[n] = q; ss[n] = h_dest_slot(q, d, gw, gh); ++n; }
        }
        for (uint32_t i = 1; i < n; ++i)
            for (uint32_t k2 = i; k2 > 0 && pp[k2] < pp[k2 - 1]; --k2) { std::swap(pp[k2], pp[k2 - 1]); std::swap(ss[k2], ss[k2 - 1]); }
        src[(size_t)d * 6] = n;
        for (uint32_t i = 0; i < n; ++i) src[(size_t)d * 6 + 1 + i] = (pp[i] << 3) | ss[i];
    }
}

// ------------------------------------------------------------------------------ layout
constexpr uint64_t HEADER_SPK = 8192;   // workspace header: DevGlobal at 0, DevSpecies[] at 256, SpK[] here

struct Carver {
    uint64_t off = 0;
    uint64_t take(uint64_t bytes) {
        const uint64_t a = (off + 255) & ~255ull;
        off = a + bytes;
        return a;
    }
};

struct SpeciesLayout {
    uint64_t pop[2], patch_start[2], rowptr[2], chunk_mask[2], range_cnt[2], f, off, mother, father, dest, pos, u01, s, offbuf, zi, zrow[2], alive, captured, a_alive, a_u, a_s, a_zi, a_pos, a_rank, mate_cum, mate_tile, mom_cum, mom_tile, enc_zi, sex[2], sex_off,
        cap, tables, table_len, status_fec, status_cmp, patch_cnt, patch_base, patch_abase, log;
    uint64_t T_recomb, T_xover, xover_len, chrom_start, chrom_len, T_mut, T_norm, T_env, K_patch, theta_patch, nbr, src_list;
    uint32_t norm_len, env_len, n_tables, row_bytes, zrow_on;
};

struct HostSpecies {
    spegg_species_params p;
    std::vector<uint32_t> chrom_len, chrom_start, T_recomb, T_xover, xover_len, T_mut, T_norm, T_env;
    std::vector<double> K_patch;
    std::vector<float> theta_patch;
    int R_norm = 0, R_env = 0;
    SpeciesLayout lay;
    SpK k;
    int q10v_per_sm = 1;   // resident CTAs per SM of this species' vectorised gamete kernel on the sim's device
};

int validate(const spegg_params *p) {
    if (!p || p->struct_size != sizeof(spegg_params) || p->abi_version != SPEGG_ABI_VERSION) return SPEGG_EINVAL;
    if (!p->species || p->n_species == 0 || p->n_species > (uint32_t)MAX_SPECIES) return SPEGG_EINVAL;
    const uint32_t gw = p->grid_w ? p->grid_w : 1, gh = p->grid_h ? p->grid_h : 1;
    const uint64_t P = (uint64_t)gw * gh;
    if (P > (1u << 20)) return SPEGG_EINVAL;
    for (uint32_t s = 0; s < p->n_species; ++s) {
        const spegg_species_params &q = p->species[s];
        if (q.n_loci == 0 || q.n_loci > (1u << 20) || q.n_chrom == 0 || !q.chrom_len) return SPEGG_EINVAL;
        if (q.genome_kind > 1 || q.linkage_mode > 1 || q.fecundity_model > 2) return SPEGG_EINVAL;
        uint64_t acc = 0;
        for (uint32_t c = 0; c < q.n_chrom; ++c) {
            if (q.chrom_len[c] == 0) return SPEGG_EINVAL;
            if (q.genome_kind == SPEGG_BIT && q.chrom_len[c] % 32) return SPEGG_EINVAL;
            acc += q.chrom_len[c];
        }
        if (acc != q.n_loci) return SPEGG_EINVAL;
        if (q.genome_kind == SPEGG_BIT && q.n_loci % 32) return SPEGG_EINVAL;
        if (q.genome_kind == SPEGG_Q10 && q.n_loci % 4) return SPEGG_EINVAL;  // rows are 16-byte multiples
        // kernels exist for bit+Poisson-crossover and q10+per-interval genomes
        if (q.genome_kind == SPEGG_BIT && q.linkage_mode != SPEGG_POISSON) return SPEGG_EINVAL;
        if (q.genome_kind == SPEGG_Q10 && q.linkage_mode != SPEGG_INTERVAL) return SPEGG_EINVAL;
        if (q.genome_kind == SPEGG_BIT && q.n_loci % 64) return SPEGG_EINVAL;
        if (q.linkage_mode == SPEGG_INTERVAL) {
            if (q.n_loci > 1 && !q.r) return SPEGG_EINVAL;
            for (uint32_t l = 0; l + 1 < q.n_loci; ++l)
                if (!(q.r[l] >= 0.0 && q.r[l] < 1.0)) return SPEGG_EINVAL;
        } else {
            if (!q.xover_mean) return SPEGG_EINVAL;
            for (uint32_t c = 0; c < q.n_chrom; ++c)
                if (!(q.xover_mean[c] >= 0.0 && q.xover_mean[c] <= 32.0)) return SPEGG_EINVAL;
        }
        if (!(q.mu >= 0.0 && q.mu <= 1.0) || !(q.migration >= 0.0 && q.migration <= 1.0)) return SPEGG_EINVAL;
        if (q.genome_kind == SPEGG_Q10 && !(q.mut_sd > 0.0 && q.mut_sd * 1024.0 * 8.0 < 32000.0)) return SPEGG_EINVAL;
        if (!(q.K > 0.0) || !(q.fec_a >= 0.0)) return SPEGG_EINVAL;
        if (q.capacity == 0 || q.capacity >= (1ull << 31)) return SPEGG_EINVAL;
        if (!(q.adult_survival >= 0.0 && q.adult_survival <= 1.0)) return SPEGG_EINVAL;
        if (!(q.resid_sd >= 0.0) || !(q.pheno_scale > 0.0f) || q.resid_sd / (double)q.pheno_scale > 4096.0) return SPEGG_EINVAL;
        if (!(std::fabs(q.mate_skew) <= 1e6) || q.separate_sexes > 1) return SPEGG_EINVAL;
        if (!(q.fec_cost >= 0.0 && q.fec_cost <= 1e6)) return SPEGG_EINVAL;
        if (!(q.assort >= 0.0 && q.assort <= 1e6) || (q.assort > 0.0 && (q.mate_skew != 0.0 || q.separate_sexes))) return SPEGG_EINVAL;
        if (q.fecundity_model == SPEGG_FEC_CAPTURES && P != 1) return SPEGG_EINVAL;
        if (q.monogamy > 1) return SPEGG_EINVAL;
        if (!(std::fabs(q.mother_skew) <= 1e6) || (q.mother_skew != 0.0 && (q.fec_cost > 0.0 || q.fecundity_model == SPEGG_FEC_CAPTURES))) return SPEGG_EINVAL;
        if (q.sel_predation) {
            if (q.predator_species >= p->n_species || q.predator_species <= s) return SPEGG_EINVAL;
            if (p->species[q.predator_species].fecundity_model != SPEGG_FEC_CAPTURES) return SPEGG_EINVAL;
            if (!(q.attack >= 0.0)) return SPEGG_EINVAL;
            if (q.encounters > 16 || (q.encounters && !(q.attack <= 2.0))) return SPEGG_EINVAL;
        } else if (q.encounters) return SPEGG_EINVAL;
    }
    return SPEGG_OK;
}

// segments per patch of the patch-mode compaction: about 2,048 rows of capacity each, at most 64
uint32_t patch_sub_of(uint64_t capacity, uint64_t P) {
    if (P <= 1) return 1;
    const uint64_t s = (capacity + P * 2048 - 1) / (P * 2048);
    return (uint32_t)std::min<uint64_t>(std::max<uint64_t>(s, 1), 64);
}

uint32_t row_bytes_of(const spegg_species_params &q) {
    return q.genome_kind == SPEGG_BIT ? 2 * (q.n_loci / 32) * 4 : 2 * q.n_loci * 2;
}

// Lays out the whole workspace; returns total bytes.  Header: DevGlobal + DevSpecies[MAX].
uint64_t layout(const spegg_params *p, std::vector<SpeciesLayout> &out) {
    Carver c;
    c.take(HEADER_SPK + MAX_SPECIES * sizeof(SpK));  // header: DevGlobal, DevSpecies[], SpK[]
    const uint32_t gw = p->grid_w ? p->grid_w : 1, gh = p->grid_h ? p->grid_h : 1;
    const uint64_t P = (uint64_t)gw * gh;
    const uint32_t logcap = p->log_capacity ? p->log_capacity : 4096;
    out.resize(p->n_species);
    for (uint32_t s = 0; s < p->n_species; ++s) {
        const spegg_species_params &q = p->species[s];
        SpeciesLayout &l = out[s];
        const uint64_t cap = q.capacity;
        l.row_bytes = row_bytes_of(q);
        l.n_tables = q.fecundity_model == SPEGG_FEC_CAPTURES ? CAP_TABLES : (uint32_t)P;
        const uint64_t cap32 = (cap + 31) / 32 * 32;  // fused path: one 32-row slab per offspring chunk
        l.pop[0] = c.take(cap32 * l.row_bytes);
        l.pop[1] = c.take(cap32 * l.row_bytes);
        l.rowptr[0] = c.take(cap32 * 4);
        l.rowptr[1] = c.take(cap32 * 4);
        l.chunk_mask[0] = c.take((cap / 32 + 2) * 4);
        l.chunk_mask[1] = c.take((cap / 32 + 2) * 4);
        l.range_cnt[0] = c.take((cap32 / SCANF_RANGE + 2) * 4);
        l.range_cnt[1] = c.take((cap32 / SCANF_RANGE + 2) * 4);
        l.patch_start[0] = c.take((P + 1) * 4);
        l.patch_start[1] = c.take((P + 1) * 4);
        l.f = c.take(cap);
        l.off = c.take(cap * 4);
        l.mother = c.take(cap32 * 4);
        l.father = c.take(cap * 4);
        l.dest = c.take(cap * 4);
        l.pos = c.take(cap * 4);
        l.u01 = c.take(cap * 4);
        l.s = c.take(cap * 4);
        l.zi = c.take(cap * 4);
        {
            bool met = false;
            for (uint32_t o = 0; o < p->n_species; ++o)
                if (p->species[o].sel_predation && p->species[o].encounters && p->species[o].predator_species == s) met = true;
            const bool zr = met || q.mate_skew != 0.0 || q.separate_sexes || q.mother_skew != 0.0 || q.fec_cost > 0.0 || q.assort > 0.0 || q.adult_survival > 0.0;
            l.zrow[0] = c.take((zr ? cap32 : 1) * 4);
            l.zrow[1] = c.take((zr ? cap32 : 1) * 4);
            l.zrow_on = zr ? 1u : 0u;
        }
        l.alive = c.take(cap);
        l.captured = c.take(cap);
        const uint64_t acap = q.adult_survival > 0.0 ? cap : 1;   // R18 arrays only when generations overlap
        l.a_alive = c.take(acap); l.a_u = c.take(acap * 4); l.a_s = c.take(acap * 4);
        l.a_zi = c.take(acap * 4); l.a_pos = c.take(acap * 4); l.a_rank = c.take((P > 1 ? acap : 1) * 4);
        const bool mate_on = q.mate_skew != 0.0 || q.separate_sexes;
        l.mate_cum = c.take((mate_on ? cap : 1) * 8);      // R19 arrays only with weighted mating / separate sexes
        l.mate_tile = c.take((mate_on ? cap / MATE_TILE + 2 : 1) * 8);
        const bool mom_on = q.mother_skew != 0.0;            // R24
        l.mom_cum = c.take((mom_on ? cap : 1) * 8);
        l.mom_tile = c.take((mom_on ? cap / MATE_TILE + 2 : 1) * 8);
        const uint64_t scap = q.separate_sexes ? cap32 : 1;         // R21
        l.sex[0] = c.take(scap); l.sex[1] = c.take(scap); l.sex_off = c.take(scap);
        bool is_met = false;   // R20: some species meets this one individually
        for (uint32_t o = 0; o < p->n_species; ++o)
            if (p->species[o].sel_predation && p->species[o].encounters && p->species[o].predator_species == s) is_met = true;
        l.enc_zi = c.take(((is_met || q.fec_cost > 0.0 || q.assort > 0.0) ? cap : 1) * 4);   // R22, R23 use it for the species' own adults
        l.cap = c.take(cap * 4);
        l.offbuf = c.take(cap * l.row_bytes);
        l.tables = c.take((uint64_t)l.n_tables * TMAX * 4);
        l.table_len = c.take((uint64_t)l.n_tables * 4);
        l.status_fec = c.take((cap / SCAN_THREADS + 2 + (cap / SCAN_THREADS + 2) / 32 + 2) * 8);
        l.status_cmp = c.take((cap / SCAN_THREADS + 2 + (cap / SCAN_THREADS + 2) / 32 + 2) * 8);   // (tiles of 256 for small populations)
        const uint64_t PS = P * patch_sub_of(cap, P);
        l.patch_cnt = c.take(PS * 6 * 4);
        l.patch_base = c.take(PS * 6 * 4);
        l.patch_abase = c.take(PS * 4);
        l.log = c.take((uint64_t)logcap * sizeof(LogEntry));
        l.T_recomb = c.take((uint64_t)q.n_loci * 4);
        l.T_xover = c.take((uint64_t)q.n_chrom * XMAX * 4);
        l.xover_len = c.take((uint64_t)q.n_chrom * 4);
        l.chrom_start = c.take((uint64_t)q.n_chrom * 4);
        l.chrom_len = c.take((uint64_t)q.n_chrom * 4);
        l.T_mut = c.take(TMAX * 4);
        l.norm_len = q.genome_kind == SPEGG_Q10 ? 2 * (uint32_t)std::max(1.0, std::ceil(8.0 * q.mut_sd * 1024.0)) : 0;
        l.T_norm = c.take((uint64_t)l.norm_len * 4 + 16);
        l.env_len = q.resid_sd > 0.0 ? 2 * (uint32_t)std::max(1.0, std::ceil(8.0 * q.resid_sd / (double)q.pheno_scale)) : 0;
        l.T_env = c.take((uint64_t)l.env_len * 4 + 16);
        l.K_patch = c.take(P * 8);
        l.theta_patch = c.take(P * 4);
        l.nbr = c.take(P * 4 * 4);
        l.src_list = c.take(P * 6 * 4);
    }
    return (c.off + 255) & ~255ull;
}

#define CU(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { s_last_cuda = e_; return SPEGG_ECUDA; } } while (0)
thread_local cudaError_t s_last_cuda = cudaSuccess;

}  // namespace

// spegg_step replays captured graphs of 16, 8, 4, 2 and 1 steps (greedy, largest first): inside a
// multi-step graph the programmatic edge between one step's last kernel and the next step's first
// stays, so a step's first kernel is scheduled while the previous step drains -- for any n_steps,
// not only for multiples of sixteen
constexpr uint32_t N_MULTI = 4;
constexpr uint32_t MULTI_STEPS[N_MULTI] = {16, 8, 4, 2};

struct spegg_sim {
    spegg_params p;
    std::vector<HostSpecies> sp;
    uint8_t *ws = nullptr;
    uint64_t ws_bytes = 0;
    cudaStream_t stream = nullptr;
    bool own_stream = false;
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    // several steps in one graph: the programmatic edges between the kernels of consecutive steps
    // stay inside the graph, so a step's first kernel is scheduled while the previous step drains
    cudaGraph_t graph_multi[N_MULTI] = {};
    cudaGraphExec_t exec_multi[N_MULTI] = {};
    DevGlobal *d_glob = nullptr;
    DevSpecies *d_st = nullptr;
    SpK *d_spk = nullptr;
    uint32_t P = 1, n_sms = 148, launches = 0, scan_ctas = 1;
    uint32_t log_capacity = 4096;
    bool debug = false;
    // kernel timing (direct launches bracketed by events)
    bool timing = false;
    std::vector<cudaEvent_t> ev;
    uint32_t ev_used = 0;
    double timing_ms = 0.0;
    uint32_t timing_n = 0;
};

namespace {

template <typename T> T *at(spegg_sim *s, uint64_t off) { return reinterpret_cast<T *>(s->ws + off); }

int upload(spegg_sim *s, uint64_t off, const void *src, size_t bytes) {
    if (bytes == 0) return SPEGG_OK;
    CU(cudaMemcpyAsync(s->ws + off, src, bytes, cudaMemcpyHostToDevice, s->stream));
    return SPEGG_OK;
}

// true when the fused single-pass kernel covers this species (see spegg_fused.cuh)
bool fused_ok(const spegg_sim *s, const HostSpecies &h) {
    if (s->debug || s->P != 1 || !fused_bit_supported(h.k) || h.k.sexes || h.k.fec_cost != 0.0f || h.k.assort != 0.0f || h.k.mom_v != 0.0f || h.k.monogamy) return false;   // (mate_on without sexes = R19: the MATE instantiation; R_env > 0 = R17: the NOISE instantiation)
    // k_fused_bit_f<4, 8> places chromosome c at words 8c .. 8c+7 and packs crossover positions in 9 bits:
    // four chromosomes of exactly 256 loci (other splits of 1,024 loci run the general pipeline)
    for (uint32_t c = 0; c < h.p.n_chrom; ++c)
        if (h.chrom_len[c] != 256u) return false;
    // the fused kernel tests u >= T as u > T - 1 (see spegg_fused.cuh): every threshold must be >= 1
    for (uint32_t c = 0; c < h.p.n_chrom; ++c)
        for (uint32_t k = 0; k < h.xover_len[c]; ++k)
            if (h.T_xover[(size_t)c * XMAX + k] == 0) return false;
    return h.k.mut_len == 0 || h.T_mut[0] != 0;
}

void launch_prepare(spegg_sim *s) {
    uint32_t blocks = 8;
    for (auto &h : s->sp) {
        blocks = std::max(blocks, (h.k.n_tables + 255) / 256);
        if (h.p.fecundity_model == SPEGG_FEC_CAPTURES) blocks = std::max(blocks, s->n_sms);
    }
    k_prepare_all<<<dim3(std::min(blocks, 4 * s->n_sms), s->p.n_species), 256, 0, s->stream>>>(s->d_spk);
}

uint32_t ctas_of(uint64_t items, uint64_t per_cta, uint32_t per_sm, uint32_t n_sms) {
    return (uint32_t)std::max<uint64_t>(1, std::min<uint64_t>((items + per_cta - 1) / per_cta, (uint64_t)n_sms * per_sm));
}

// Enqueue the kernels of one step on the stream (captured into the graph, or launched directly
// when kernel timing is on).  Returns the number of kernel launches through *n_launch.
int enqueue_step(spegg_sim *s, uint32_t *n_launch, bool timed) {
    uint32_t nl = 0;
    const uint32_t G = s->n_sms;
    if (s->debug) { launch_prepare(s); ++nl; }
    for (size_t si = 0; si < s->sp.size(); ++si) {
        HostSpecies &h = s->sp[si];
        const SpK &k = h.k;
        const bool time_this = timed && si == 0 && s->ev_used + 2 <= s->ev.size();
        if (fused_ok(s, h)) {
            CU(launch_scan_fused(k, G, s->scan_ctas, s->stream)); ++nl;
            if (k.mate_on) {   // R19 on the fused path: the weights need this step's rowptr[] (the scan's) and last step's zrow[]
                k_mate_weight<<<ctas_of(k.capacity, 8, 8, G), 256, 0, s->stream>>>(k); ++nl;
                k_mate_scan<<<ctas_of(k.capacity, MATE_TILE, 8, G), 256, 0, s->stream>>>(k, 0); ++nl;
            }
            if (time_this) CU(cudaEventRecord(s->ev[s->ev_used], s->stream));
            CU(launch_fused_bit(k, G, s->stream)); ++nl;
            if (time_this) { CU(cudaEventRecord(s->ev[s->ev_used + 1], s->stream)); s->ev_used += 2; }
        } else {
            // grids are fixed at capture time: sized for the capacity (a thousand idle CTAs cost a small
            // population more than its work), capped at a few CTAs per SM; the kernels loop over the counts
            const uint64_t cap = k.capacity;
            auto ctas = [&](uint64_t items, uint64_t per_cta, uint32_t per_sm) {
                return (uint32_t)std::max<uint64_t>(1, std::min<uint64_t>((items + per_cta - 1) / per_cta, (uint64_t)G * per_sm));
            };
            const uint32_t g_thread = ctas(cap, 256, 8), g_warp = ctas(cap, 8, 8);   // thread / warp per offspring
            if (k.fec_cost > 0.0f || k.assort > 0.0f) { k_enc_zi<<<ctas(cap, 8, 8), 256, 0, s->stream>>>(k); ++nl; }   // R22, R23: the adults' genetic values
            if (k.mate_on || k.mom_v != 0.0f) {   // R19 / R24: mating and mothering weights of the adults and their running sums
                k_mate_weight<<<g_warp, 256, 0, s->stream>>>(k); ++nl;
                if (k.mate_on) { k_mate_scan<<<ctas(cap, MATE_TILE, 8), 256, 0, s->stream>>>(k, 0); ++nl; }
                if (k.mom_v != 0.0f) { k_mate_scan<<<ctas(cap, MATE_TILE, 8), 256, 0, s->stream>>>(k, 1); ++nl; }
            }
            // a1-a3 in one kernel: fecundity, scan, mothers, and the scalar draws of every range's offspring
            k_fec_scan<<<ctas(cap, SCAN_THREADS, 4), SCAN_THREADS, 0, s->stream>>>(k); ++nl;
            if (time_this) CU(cudaEventRecord(s->ev[s->ev_used], s->stream));
            // production q10 path: vectorised gamete kernel that also takes the phenotype (debug keeps
            // the plain kernels, so the two can be compared with each other and with the oracle)
            const bool q10v = !s->debug && gamete_q10v_supported(k);
            if (k.kind == 0) k_gamete_bit<<<ctas(cap * 2 * k.n_chrom, 256, 8), 256, 0, s->stream>>>(k);
            else if (q10v) CU(launch_gamete_q10v(k, G, h.q10v_per_sm, s->stream));
            else k_gamete_q10<<<ctas(cap * 2, 8, 8), 256, 0, s->stream>>>(k);
            ++nl;
            if (time_this) { CU(cudaEventRecord(s->ev[s->ev_used + 1], s->stream)); s->ev_used += 2; }
            if (k.enc_E) {   // R20: genetic values of the consumers this species' newborns meet
                const SpK &kp = s->sp[h.p.predator_species].k;
                k_enc_zi<<<ctas(kp.capacity, 8, 8), 256, 0, s->stream>>>(kp); ++nl;
            }
            if (q10v && s->P == 1 && k.adult_surv == 0.0f) {
                // mutation, selection, compaction and its index in one kernel (the last CTA closes a solo step)
                if (cap <= (uint64_t)G * 4 * SCAN_THREADS) k_select_compact<1><<<ctas(cap, SCAN_THREADS, 4), SCAN_THREADS, 0, s->stream>>>(k);
                else k_select_compact<SCAN_ITEMS><<<ctas(cap, SCAN_TILE, 4), SCAN_THREADS, 0, s->stream>>>(k);
                ++nl;
            } else {
                const bool patches = s->P > 1;
                if (q10v && !patches) { k_mut_surv<<<g_thread, 256, 0, s->stream>>>(k); ++nl; }   // (patches: inside k_patch_count)
                if (!q10v) {
                    k_mutate<<<ctas(cap * 2, 256, 8), 256, 0, s->stream>>>(k, 0); ++nl;
                    k_phenotype<<<g_warp, 256, 0, s->stream>>>(k); ++nl;
                    k_survival<<<g_thread, 256, 0, s->stream>>>(k); ++nl;
                }
                if (k.adult_surv > 0.0f) { k_adult_survive<<<g_warp, 256, 0, s->stream>>>(k); ++nl; }   // R18
                const bool index_here = patches && k.index_only && k.adult_surv == 0.0f;   // k_patch_pos writes the index itself
                if (!patches) {
                    k_cmp_scan<<<ctas(cap, SCAN_TILE, 4), SCAN_THREADS, 0, s->stream>>>(k); ++nl;
                } else {
                    k_patch_count<<<std::min(s->P * k.patch_sub, G * 8), 256, 0, s->stream>>>(k, q10v ? 1 : 0); ++nl;
                    k_patch_base<<<1, 1024, 0, s->stream>>>(k); ++nl;
                    k_patch_pos<<<std::min(s->P * k.patch_sub, G * 8), 256, 0, s->stream>>>(k, index_here ? 1 : 0); ++nl;
                }
                if (!index_here) { k_cmp_scatter<<<(k.index_only && k.adult_surv == 0.0f) ? g_thread : g_warp, 256, 0, s->stream>>>(k); ++nl; }
            }
        }
    }
    const bool solo = s->sp.size() == 1 && s->sp[0].k.solo;  // the last kernel closes the step itself
    if (!solo) {
        k_finish_all<<<1, 32, 0, s->stream>>>(s->d_spk, s->p.n_species); ++nl;
        if (!s->debug) { launch_prepare(s); ++nl; }  // debug: prepared at the start, so the view stays valid
    }
    CU(cudaGetLastError());
    if (n_launch) *n_launch = nl;
    return SPEGG_OK;
}

void drain_timing(spegg_sim *s) {
    for (uint32_t i = 0; i + 1 < s->ev_used; i += 2) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, s->ev[i], s->ev[i + 1]) == cudaSuccess) { s->timing_ms += ms; s->timing_n += 1; }
    }
    s->ev_used = 0;
}

}  // namespace

extern "C" {

const char *spegg_strerror(int code) {
    switch (code) {
    case SPEGG_OK: return "ok";
    case SPEGG_EINVAL: return "invalid parameter";
    case SPEGG_ENOMEM: return "workspace too small";
    case SPEGG_ECUDA: return cudaGetErrorString(s_last_cuda);
    case SPEGG_ERANGE: return "output buffer too small";
    case SPEGG_ESTATE: return "call not valid in this state";
    case SPEGG_ELIMIT: return "size above the fixed maximum of this entry point (SPEGG_STATIC_MAX_N)";
    default: return "unknown error";
    }
}

int spegg_workspace_bytes(const spegg_params *p, uint64_t *bytes) {
    const int rc = validate(p);
    if (rc != SPEGG_OK) return rc;
    if (!bytes) return SPEGG_EINVAL;
    std::vector<SpeciesLayout> l;
    *bytes = layout(p, l);
    return SPEGG_OK;
}

int spegg_create(const spegg_params *p, void *d_workspace, uint64_t bytes, void *cuda_stream, spegg_sim **out) {
    int rc = validate(p);
    if (rc != SPEGG_OK) return rc;
    if (!d_workspace || !out || ((uintptr_t)d_workspace & 255u)) return SPEGG_EINVAL;
    std::vector<SpeciesLayout> lays;
    const uint64_t need = layout(p, lays);
    if (bytes < need) return SPEGG_ENOMEM;
    spegg_sim *s = new (std::nothrow) spegg_sim();
    if (!s) return SPEGG_ENOMEM;
    s->p = *p;
    s->p.species = nullptr;
    s->ws = (uint8_t *)d_workspace;
    s->ws_bytes = bytes;
    s->debug = p->debug != 0;
    s->log_capacity = p->log_capacity ? p->log_capacity : 4096;
    const uint32_t gw = p->grid_w ? p->grid_w : 1, gh = p->grid_h ? p->grid_h : 1;
    s->P = gw * gh;
    auto fail = [&](int code) { spegg_destroy(s); return code; };
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
        s_last_cuda = cudaGetLastError();
        return fail(SPEGG_ECUDA);
    }
    s->n_sms = (uint32_t)prop.multiProcessorCount;
    if (cuda_stream) s->stream = (cudaStream_t)cuda_stream;
    else {  // the legacy default stream cannot be captured: use a private one
        if (cudaStreamCreateWithFlags(&s->stream, cudaStreamNonBlocking) != cudaSuccess) return fail(SPEGG_ECUDA);
        s->own_stream = true;
    }
    s->d_glob = at<DevGlobal>(s, 0);
    s->d_st = at<DevSpecies>(s, 256);
    s->d_spk = at<SpK>(s, HEADER_SPK);
    static_assert(256 + MAX_SPECIES * sizeof(DevSpecies) <= HEADER_SPK, "header too small");
    if (cudaMemsetAsync(s->ws, 0, HEADER_SPK + MAX_SPECIES * sizeof(SpK), s->stream) != cudaSuccess) return fail(SPEGG_ECUDA);

    s->sp.resize(p->n_species);
    for (uint32_t si = 0; si < p->n_species; ++si) {
        HostSpecies &h = s->sp[si];
        const spegg_species_params &q = p->species[si];
        h.p = q;
        h.lay = lays[si];
        const uint32_t L = q.n_loci;
        uint32_t acc = 0;
        for (uint32_t c = 0; c < q.n_chrom; ++c) { h.chrom_start.push_back(acc); h.chrom_len.push_back(q.chrom_len[c]); acc += q.chrom_len[c]; }
        h.T_recomb.assign(L, 0);
        if (q.linkage_mode == SPEGG_INTERVAL) {
            h.T_recomb[0] = 2147483648u;  // start phase ~ Bernoulli(1/2) (R7)
            for (uint32_t l = 1; l < L; ++l) h.T_recomb[l] = (uint32_t)h_bernoulli_T(q.r[l - 1]);
        }
        h.T_xover.assign((size_t)q.n_chrom * XMAX, 0);
        h.xover_len.assign(q.n_chrom, 0);
        if (q.linkage_mode == SPEGG_POISSON)
            for (uint32_t c = 0; c < q.n_chrom; ++c)
                h.xover_len[c] = (uint32_t)h_poisson_table(q.xover_mean[c], &h.T_xover[(size_t)c * XMAX], 62);
        h.T_mut.assign(TMAX, 0);
        const uint32_t mut_len = (uint32_t)h_poisson_table((double)L * q.mu, h.T_mut.data(), TMAX);
        if (q.genome_kind == SPEGG_Q10) h.R_norm = h_normal_table(q.mut_sd * 1024.0, h.T_norm);
        if (q.resid_sd > 0.0) h.R_env = h_normal_table(q.resid_sd / (double)q.pheno_scale, h.T_env);   // R17
        if (q.K_patch) h.K_patch.assign(q.K_patch, q.K_patch + s->P);
        if (q.theta_patch) h.theta_patch.assign(q.theta_patch, q.theta_patch + s->P);
        h.p.chrom_len = nullptr; h.p.r = nullptr; h.p.xover_mean = nullptr; h.p.K_patch = nullptr; h.p.theta_patch = nullptr;

        const SpeciesLayout &l = h.lay;
        if ((rc = upload(s, l.T_recomb, h.T_recomb.data(), h.T_recomb.size() * 4)) ||
            (rc = upload(s, l.T_xover, h.T_xover.data(), h.T_xover.size() * 4)) ||
            (rc = upload(s, l.xover_len, h.xover_len.data(), h.xover_len.size() * 4)) ||
            (rc = upload(s, l.chrom_start, h.chrom_start.data(), h.chrom_start.size() * 4)) ||
            (rc = upload(s, l.chrom_len, h.chrom_len.data(), h.chrom_len.size() * 4)) ||
            (rc = upload(s, l.T_mut, h.T_mut.data(), TMAX * 4)) ||
            (rc = upload(s, l.T_norm, h.T_norm.data(), h.T_norm.size() * 4)) ||
            (rc = upload(s, l.T_env, h.T_env.data(), h.T_env.size() * 4)) ||
            (rc = upload(s, l.K_patch, h.K_patch.data(), h.K_patch.size() * 8)) ||
            (rc = upload(s, l.theta_patch, h.theta_patch.data(), h.theta_patch.size() * 4)))
            return fail(rc);
        if (s->P > 1) {
            std::vector<uint32_t> nbr, src;
            h_topology(gw, gh, nbr, src);
            if ((rc = upload(s, l.nbr, nbr.data(), nbr.size() * 4)) || (rc = upload(s, l.src_list, src.data(), src.size() * 4))) return fail(rc);
            if (cudaStreamSynchronize(s->stream) != cudaSuccess) return fail(SPEGG_ECUDA);   // the vectors go out of scope
        }
        if (cudaMemsetAsync(s->ws + l.patch_start[0], 0, (s->P + 1) * 4, s->stream) != cudaSuccess ||
            cudaMemsetAsync(s->ws + l.patch_start[1], 0, (s->P + 1) * 4, s->stream) != cudaSuccess ||
            cudaMemsetAsync(s->ws + l.cap, 0, (size_t)q.capacity * 4, s->stream) != cudaSuccess)
            return fail(SPEGG_ECUDA);

        SpK &k = h.k;
        std::memset(&k, 0, sizeof k);
        k.species = si; k.n_species = p->n_species;
        k.L = L; k.W = L / 32; k.kind = q.genome_kind; k.n_chrom = q.n_chrom; k.linkage = q.linkage_mode;
        k.row_bytes = l.row_bytes; k.row_u4 = l.row_bytes / 16;
        k.P = s->P; k.grid_w = gw; k.grid_h = gh;
        k.capacity = (uint32_t)q.capacity;
        k.fec_model = q.fecundity_model; k.fec_a = q.fec_a; k.K = q.K;
        k.K_patch = q.K_patch ? at<double>(s, l.K_patch) : nullptr;
        k.sel_gaussian = q.sel_gaussian; k.sel_predation = q.sel_predation; k.predator = q.predator_species;
        k.theta0 = q.theta0; k.dtheta = q.dtheta; k.attack = q.attack;
        // R11: c = fp32(1/(2 omega^2)) from fp64; omega <= 0 -> c = 0
        k.sel_c = q.omega > 0.0 ? (float)(1.0 / (2.0 * (q.omega * q.omega))) : 0.0f;
        k.pheno_scale = q.pheno_scale;
        k.pred_scale = q.sel_predation ? p->species[q.predator_species].pheno_scale : 0.0f;
        k.theta_patch = q.theta_patch ? at<float>(s, l.theta_patch) : nullptr;
        k.T_mig = h_bernoulli_T(q.migration);
        k.n_tables = l.n_tables;
        k.key.k0 = (uint32_t)p->seed; k.key.k1 = (uint32_t)(p->seed >> 32);
        for (uint32_t r = 0; r < 10; ++r) { k.rk[2 * r] = k.key.k0 + r * 0x9E3779B9u; k.rk[2 * r + 1] = k.key.k1 + r * 0xBB67AE85u; }
        k.T_recomb = at<uint32_t>(s, l.T_recomb);
        k.T_xover = at<uint32_t>(s, l.T_xover); k.xover_len = at<uint32_t>(s, l.xover_len);
        k.chrom_start = at<uint32_t>(s, l.chrom_start); k.chrom_len = at<uint32_t>(s, l.chrom_len);
        k.T_mut = at<uint32_t>(s, l.T_mut); k.mut_len = mut_len;
        k.T_norm = at<uint32_t>(s, l.T_norm); k.R_norm = h.R_norm;
        k.T_env = at<uint32_t>(s, l.T_env); k.R_env = h.R_env;
        k.pop[0] = at<uint8_t>(s, l.pop[0]); k.pop[1] = at<uint8_t>(s, l.pop[1]);
        k.patch_start[0] = at<uint32_t>(s, l.patch_start[0]); k.patch_start[1] = at<uint32_t>(s, l.patch_start[1]);
        k.rowptr[0] = at<uint32_t>(s, l.rowptr[0]); k.rowptr[1] = at<uint32_t>(s, l.rowptr[1]);
        k.chunk_mask[0] = at<uint32_t>(s, l.chunk_mask[0]); k.chunk_mask[1] = at<uint32_t>(s, l.chunk_mask[1]);
        k.range_cnt[0] = at<uint32_t>(s, l.range_cnt[0]);
        k.range_cnt[1] = at<uint32_t>(s, l.range_cnt[1]);
        k.f = at<uint8_t>(s, l.f); k.off = at<uint32_t>(s, l.off);
        k.mother = at<uint32_t>(s, l.mother); k.father = at<uint32_t>(s, l.father);
        k.dest = at<uint32_t>(s, l.dest); k.pos = at<uint32_t>(s, l.pos);
        k.u01 = at<float>(s, l.u01); k.s = at<float>(s, l.s);
        k.offbuf = at<uint8_t>(s, l.offbuf); k.zi = at<int32_t>(s, l.zi);
        k.zrow[0] = at<int32_t>(s, l.zrow[0]); k.zrow[1] = at<int32_t>(s, l.zrow[1]); k.zrow_on = l.zrow_on;
        k.alive = at<uint8_t>(s, l.alive); k.captured = at<uint8_t>(s, l.captured);
        k.adult_surv = (float)q.adult_survival;
        k.a_alive = at<uint8_t>(s, l.a_alive); k.a_u = at<float>(s, l.a_u); k.a_s = at<float>(s, l.a_s);
        k.a_zi = at<int32_t>(s, l.a_zi); k.a_pos = at<uint32_t>(s, l.a_pos); k.a_rank = at<uint32_t>(s, l.a_rank);
        k.mate_v = (float)q.mate_skew;
        k.sexes = q.separate_sexes; k.mate_on = (q.mate_skew != 0.0 || q.separate_sexes) ? 1u : 0u;
        k.sex[0] = at<uint8_t>(s, l.sex[0]); k.sex[1] = at<uint8_t>(s, l.sex[1]); k.sex_off = at<uint8_t>(s, l.sex_off);
        k.mate_cum = at<unsigned long long>(s, l.mate_cum); k.mate_tile = at<unsigned long long>(s, l.mate_tile);
        k.mom_v = (float)q.mother_skew;
        k.monogamy = q.monogamy;
        k.mom_cum = at<unsigned long long>(s, l.mom_cum); k.mom_tile = at<unsigned long long>(s, l.mom_tile);
        k.fec_cost = (float)q.fec_cost; k.assort = (float)q.assort;
        k.enc_E = q.sel_predation ? q.encounters : 0u; k.enc_v = (float)q.attack;
        k.enc_zi = at<int32_t>(s, l.enc_zi);
        k.cap = at<uint32_t>(s, l.cap);
        k.tables = at<uint32_t>(s, l.tables); k.table_len = at<uint32_t>(s, l.table_len);
        k.status_fec = at<unsigned long long>(s, l.status_fec); k.status_cmp = at<unsigned long long>(s, l.status_cmp);
        k.status_fec_n = (uint32_t)(q.capacity / SCAN_THREADS + 2); k.status_cmp_n = (uint32_t)(q.capacity / SCAN_THREADS + 2);
        k.patch_cnt = at<uint32_t>(s, l.patch_cnt); k.patch_base = at<uint32_t>(s, l.patch_base); k.patch_abase = at<uint32_t>(s, l.patch_abase);
        k.nbr = at<uint32_t>(s, l.nbr); k.src_list = at<uint32_t>(s, l.src_list);
        k.patch_sub = patch_sub_of(q.capacity, s->P);
        k.st = s->d_st + si; k.st_all = s->d_st; k.glob = s->d_glob;
        k.log = at<LogEntry>(s, l.log); k.log_capacity = s->log_capacity;
        k.debug = p->debug;
        k.phys_parents = fused_ok(s, h) ? 1u : 0u;
        // single unstructured species, production kernels: the step's last kernel closes it and prepares
        // the next one itself (one Poisson table; per-patch tables are a grid's work, not a CTA's)
        k.solo = (!s->debug && p->n_species == 1 && s->P == 1) ? 1u : 0u;
        k.index_only = (!s->debug && !k.phys_parents && gamete_q10v_supported(k)) ? 1u : 0u;
    }
    for (uint32_t si = 0; si < p->n_species; ++si)
        if (s->sp[si].k.phys_parents && fused_bit_configure() != cudaSuccess) { s_last_cuda = cudaGetLastError(); return fail(SPEGG_ECUDA); }
    bool any_q10v = false;
    for (uint32_t si = 0; si < p->n_species; ++si)   // per simulation, on its own device and context (not cached per process)
        if (!s->debug && gamete_q10v_supported(s->sp[si].k)) {
            const cudaError_t e = gamete_q10v_configure(s->sp[si].k.L, &s->sp[si].q10v_per_sm);
            if (e != cudaSuccess) { s_last_cuda = e; return fail(SPEGG_ECUDA); }
            any_q10v = true;
        }
    if (any_q10v) {   // carry polarity of q10_push (see k_selftest_push); the probe word is a spare header word
        uint32_t *d_probe = at<uint32_t>(s, 128), got = 0;
        const PushProbe v = {{5u, 3u, 7u, 0u, 0xFFFFFFFFu}, {3u, 5u, 7u, 0xFFFFFFFFu, 0u}};
        k_selftest_push<<<1, 1, 0, s->stream>>>(v, d_probe);
        cudaError_t e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaMemcpyAsync(&got, d_probe, 4, cudaMemcpyDeviceToHost, s->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
        if (e == cudaSuccess && got != PUSH_PROBE_EXPECT) {
            std::fprintf(stderr, "libspegg: carry self-test of the q10 gamete kernel failed (got 0x%x, want 0x%x): this toolkit "
                                 "translates sub.cc/addc differently; rebuild with the setp/selp form of q10_push\n", got, PUSH_PROBE_EXPECT);
            e = cudaErrorNotSupported;
        }
        if (e != cudaSuccess) { s_last_cuda = e; return fail(SPEGG_ECUDA); }
    }
    {
        const int n = scan_fused_ctas_per_sm();
        if (n < 1) { s_last_cuda = cudaGetLastError(); return fail(SPEGG_ECUDA); }
        s->scan_ctas = (uint32_t)n;
    }
    for (uint32_t si = 0; si < p->n_species; ++si)
        if (s->sp[si].p.sel_predation) {
            s->sp[si].k.cap_pred = s->sp[s->sp[si].p.predator_species].k.cap;
            s->sp[si].k.pred_zi = s->sp[s->sp[si].p.predator_species].k.enc_zi;
        }

    for (uint32_t si = 0; si < p->n_species; ++si)
        if (cudaMemcpyAsync(s->d_spk + si, &s->sp[si].k, sizeof(SpK), cudaMemcpyHostToDevice, s->stream) != cudaSuccess) return fail(SPEGG_ECUDA);
    launch_prepare(s);
    // capture the step graph once; spegg_step replays it
    if (cudaStreamSynchronize(s->stream) != cudaSuccess) { s_last_cuda = cudaGetLastError(); return fail(SPEGG_ECUDA); }
    if (cudaStreamBeginCapture(s->stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { s_last_cuda = cudaGetLastError(); return fail(SPEGG_ECUDA); }
    rc = enqueue_step(s, &s->launches, false);
    cudaError_t ce = cudaStreamEndCapture(s->stream, &s->graph);
    if (rc != SPEGG_OK) return fail(rc);
    if (ce != cudaSuccess) { s_last_cuda = ce; return fail(SPEGG_ECUDA); }
    if ((ce = cudaGraphInstantiate(&s->exec, s->graph, 0)) != cudaSuccess) { s_last_cuda = ce; return fail(SPEGG_ECUDA); }
    (void)cudaGraphUpload(s->exec, s->stream);
    if (!s->debug) {   // several steps per graph (optional: a failure here leaves the one-step graph)
        for (uint32_t m = 0; m < N_MULTI; ++m) {
            bool ok = cudaStreamBeginCapture(s->stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
            if (ok) {
                for (uint32_t i = 0; i < MULTI_STEPS[m] && ok; ++i) ok = enqueue_step(s, nullptr, false) == SPEGG_OK;
                ok = (cudaStreamEndCapture(s->stream, &s->graph_multi[m]) == cudaSuccess) && ok;
            }
            if (ok) ok = cudaGraphInstantiate(&s->exec_multi[m], s->graph_multi[m], 0) == cudaSuccess;
            if (ok) (void)cudaGraphUpload(s->exec_multi[m], s->stream);   // not on the first replay's critical path
            if (!ok) { (void)cudaGetLastError(); s->exec_multi[m] = nullptr; }
        }
    }
    *out = s;
    return SPEGG_OK;
}

void spegg_destroy(spegg_sim *s) {
    if (!s) return;
    if (s->stream) cudaStreamSynchronize(s->stream);
    for (auto e : s->ev) cudaEventDestroy(e);
    for (uint32_t m = 0; m < N_MULTI; ++m) {
        if (s->exec_multi[m]) cudaGraphExecDestroy(s->exec_multi[m]);
        if (s->graph_multi[m]) cudaGraphDestroy(s->graph_multi[m]);
    }
    if (s->exec) cudaGraphExecDestroy(s->exec);
    if (s->graph) cudaGraphDestroy(s->graph);
    if (s->own_stream && s->stream) cudaStreamDestroy(s->stream);
    delete s;
}

int spegg_write_state(spegg_sim *s, uint32_t species, uint64_t n, const void *genomes, int genomes_is_device,
                      const uint32_t *patch_start, uint32_t step) {
    if (!s || species >= s->sp.size() || (n && !genomes)) return SPEGG_EINVAL;
    HostSpecies &h = s->sp[species];
    if (n > h.p.capacity) return SPEGG_ERANGE;
    std::vector<uint32_t> ps(s->P + 1, 0);
    if (s->P > 1) {
        if (!patch_start || patch_start[0] != 0 || patch_start[s->P] != n) return SPEGG_EINVAL;
        for (uint32_t p = 0; p < s->P; ++p) if (patch_start[p] > patch_start[p + 1]) return SPEGG_EINVAL;
        ps.assign(patch_start, patch_start + s->P + 1);
    } else ps[1] = (uint32_t)n;
    CU(cudaStreamSynchronize(s->stream));
    DevSpecies st;
    CU(cudaMemcpy(&st, s->d_st + species, sizeof st, cudaMemcpyDeviceToHost));
    const uint32_t cur = st.cur;
    CU(cudaMemcpyAsync(h.k.pop[cur], genomes, (size_t)n * h.k.row_bytes,
                       genomes_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, s->stream));
    CU(cudaMemcpyAsync(h.k.patch_start[cur], ps.data(), ps.size() * 4, cudaMemcpyHostToDevice, s->stream));
    std::memset(&st, 0, sizeof st);
    st.cur = cur;
    st.n = (uint32_t)n;
    st.m_phys = (uint32_t)n;
    CU(cudaMemcpyAsync(s->d_st + species, &st, sizeof st, cudaMemcpyHostToDevice, s->stream));
    DevGlobal g;
    CU(cudaMemcpy(&g, s->d_glob, sizeof g, cudaMemcpyDeviceToHost));
    g.step = step;
    CU(cudaMemcpyAsync(s->d_glob, &g, sizeof g, cudaMemcpyHostToDevice, s->stream));
    if (h.k.sexes) CU(cudaMemsetAsync(h.k.sex[cur], 0, (size_t)n, s->stream));   // R21: everybody female until spegg_write_sex
    if (n) {
        k_iota<<<s->n_sms * 4, 256, 0, s->stream>>>(h.k.rowptr[cur], (uint32_t)n);
        if (h.k.phys_parents) k_fill_masks<<<s->n_sms, 256, 0, s->stream>>>(h.k.chunk_mask[cur], h.k.range_cnt[cur], (uint32_t)n);
        k_adult_zi<<<s->n_sms * 8, 256, 0, s->stream>>>(h.k, (uint32_t)n, 1, nullptr);
    }
    launch_prepare(s);
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(s->stream));
    return SPEGG_OK;
}

int spegg_write_sex(spegg_sim *s, uint32_t species, uint64_t n, const uint8_t *sex) {
    if (!s || species >= s->sp.size() || (n && !sex)) return SPEGG_EINVAL;
    HostSpecies &h = s->sp[species];
    if (!h.k.sexes) return SPEGG_ESTATE;
    CU(cudaStreamSynchronize(s->stream));
    DevSpecies st;
    CU(cudaMemcpy(&st, s->d_st + species, sizeof st, cudaMemcpyDeviceToHost));
    if (n != st.n) return SPEGG_ERANGE;
    if (n == 0) return SPEGG_OK;
    CU(cudaMemcpyAsync(h.k.sex_off, sex, (size_t)n, cudaMemcpyHostToDevice, s->stream));
    k_sex_io<<<s->n_sms * 4, 256, 0, s->stream>>>(h.k, (uint32_t)n, h.k.sex_off, 1);
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(s->stream));
    return SPEGG_OK;
}

int spegg_read_sex(spegg_sim *s, uint32_t species, uint8_t *sex_out, uint64_t cap_bytes) {
    if (!s || species >= s->sp.size() || !sex_out) return SPEGG_EINVAL;
    HostSpecies &h = s->sp[species];
    if (!h.k.sexes) return SPEGG_ESTATE;
    CU(cudaStreamSynchronize(s->stream));
    DevSpecies st;
    CU(cudaMemcpy(&st, s->d_st + species, sizeof st, cudaMemcpyDeviceToHost));
    if (cap_bytes < st.n) return SPEGG_ERANGE;
    if (st.n == 0) return SPEGG_OK;
    k_sex_io<<<s->n_sms * 4, 256, 0, s->stream>>>(h.k, st.n, h.k.sex_off, 0);
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(s->stream));
    CU(cudaMemcpy(sex_out, h.k.sex_off, (size_t)st.n, cudaMemcpyDeviceToHost));
    return SPEGG_OK;
}

int spegg_step(spegg_sim *s, uint32_t n_steps) {
    if (!s) return SPEGG_EINVAL;
    uint32_t i = 0;
    if (!s->timing)
        for (uint32_t m = 0; m < N_MULTI; ++m)
            if (s->exec_multi[m])
                for (; i + MULTI_STEPS[m] <= n_steps; i += MULTI_STEPS[m]) CU(cudaGraphLaunch(s->exec_multi[m], s->stream));
    for (; i < n_steps; ++i) {
        if (s->timing) {
            if (s->ev_used + 2 > s->ev.size()) { CU(cudaStreamSynchronize(s->stream)); drain_timing(s); }
            const int rc = enqueue_step(s, nullptr, true);
            if (rc != SPEGG_OK) return rc;
        } else {
            CU(cudaGraphLaunch(s->exec, s->stream));
        }
    }
    return SPEGG_OK;
}

int spegg_read_state(spegg_sim *s, uint32_t species, uint64_t *n, uint32_t *step, void *genomes_out,
                     int genomes_is_device, uint64_t cap_bytes, uint32_t *patch_start_out, int32_t *zi_out) {
    if (!s || species >= s->sp.size()) return SPEGG_EINVAL;
    HostSpecies &h = s->sp[species];
    CU(cudaStreamSynchronize(s->stream));
    DevSpecies st;
    DevGlobal g;
    CU(cudaMemcpy(&st, s->d_st + species, sizeof st, cudaMemcpyDeviceToHost));
    CU(cudaMemcpy(&g, s->d_glob, sizeof g, cudaMemcpyDeviceToHost));
    if (n) *n = st.n;
    if (step) *step = g.step;
    if ((genomes_out || zi_out) && st.n && h.k.phys_parents) {
        // fused path: the index (rowptr) of the current buffer is built on demand
        launch_rowptr_fused(h.k, s->n_sms, s->stream);
    }
    // staging: the OTHER population buffer holds last step's dead adults and is free between steps, and
    // pos[] is rewritten by every step before it is read -- so the debug view (offspring rows, zi) survives
    uint8_t *stage_rows = h.k.pop[st.cur ^ 1u];
    int32_t *stage_zi = (int32_t *)h.k.pos;
    if (genomes_out) {
        if (cap_bytes < (uint64_t)st.n * h.k.row_bytes) return SPEGG_ERANGE;
        if (st.n) {  // rows in logical order: gather through rowptr into the staging buffer
            k_gather_rows<<<s->n_sms * 8, 256, 0, s->stream>>>(h.k, st.n, stage_rows);
            CU(cudaGetLastError());
            CU(cudaStreamSynchronize(s->stream));
            CU(cudaMemcpy(genomes_out, stage_rows, (size_t)st.n * h.k.row_bytes,
                          genomes_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost));
        }
    }
    if (patch_start_out) CU(cudaMemcpy(patch_start_out, h.k.patch_start[st.cur], (s->P + 1) * 4, cudaMemcpyDeviceToHost));
    if (zi_out && st.n) {
        k_adult_zi<<<s->n_sms * 8, 256, 0, s->stream>>>(h.k, st.n, 0, stage_zi);
        CU(cudaGetLastError());
        CU(cudaStreamSynchronize(s->stream));
        CU(cudaMemcpy(zi_out, stage_zi, (size_t)st.n * 4, cudaMemcpyDeviceToHost));
    }
    return SPEGG_OK;
}

int spegg_read_log(spegg_sim *s, uint32_t species, uint32_t first, uint32_t n, spegg_log_entry *out, uint32_t *n_avail) {
    if (!s || species >= s->sp.size()) return SPEGG_EINVAL;
    HostSpecies &h = s->sp[species];
    CU(cudaStreamSynchronize(s->stream));
    DevSpecies st;
    CU(cudaMemcpy(&st, s->d_st + species, sizeof st, cudaMemcpyDeviceToHost));
    if (n_avail) *n_avail = st.log_pos;
    if (n == 0) return SPEGG_OK;
    if (!out || (uint64_t)first + n > st.log_pos) return SPEGG_ERANGE;
    if (st.log_pos - first > s->log_capacity) return SPEGG_ERANGE;  // overwritten by the ring
    // at most two copies: the span up to the end of the ring, then the part that wrapped
    const uint32_t at0 = first % s->log_capacity, n0 = std::min(n, s->log_capacity - at0);
    CU(cudaMemcpy(out, h.k.log + at0, (size_t)n0 * sizeof(LogEntry), cudaMemcpyDeviceToHost));
    if (n > n0) CU(cudaMemcpy(out + n0, h.k.log, (size_t)(n - n0) * sizeof(LogEntry), cudaMemcpyDeviceToHost));
    return SPEGG_OK;
}

int spegg_read_debug(spegg_sim *s, uint32_t species, spegg_debug_view *o) {
    if (!s || species >= s->sp.size() || !o) return SPEGG_EINVAL;
    if (!s->debug) return SPEGG_ESTATE;
    HostSpecies &h = s->sp[species];
    CU(cudaStreamSynchronize(s->stream));
    DevSpecies st;
    CU(cudaMemcpy(&st, s->d_st + species, sizeof st, cudaMemcpyDeviceToHost));
    const SpK &k = h.k;
    o->n_t = st.n0; o->m_t = st.m;
    o->d_f = k.f; o->d_off = k.off; o->d_mother = k.mother; o->d_father = k.father; o->d_dest = k.dest;
    o->d_u01 = k.u01; o->d_s = k.s; o->d_zi = k.zi; o->d_alive = k.alive; o->d_captured = k.captured;
    o->d_offspring = k.offbuf; o->d_tables = k.tables; o->d_table_len = k.table_len; o->n_tables = k.n_tables;
    o->theta_t = st.theta_t; o->zbar_pred = st.zbar_pred; o->attack_n = st.attack_n;
    o->d_cap = k.cap;
    o->d_a_alive = k.a_alive; o->d_a_u = k.a_u; o->d_a_s = k.a_s;
    o->d_mate_cum = (const uint64_t *)k.mate_cum; o->zbar_self = st.zbar_self;
    o->d_sex_off = k.sex_off;
    o->d_mom_cum = (const uint64_t *)k.mom_cum;
    return SPEGG_OK;
}

int spegg_status(spegg_sim *s, uint32_t *flags) {
    if (!s || !flags) return SPEGG_EINVAL;
    CU(cudaStreamSynchronize(s->stream));
    DevGlobal g;
    CU(cudaMemcpy(&g, s->d_glob, sizeof g, cudaMemcpyDeviceToHost));
    *flags = g.flags;
    return SPEGG_OK;
}

int spegg_launches_per_step(const spegg_sim *s, uint32_t *n) {
    if (!s || !n) return SPEGG_EINVAL;
    *n = s->launches;
    return SPEGG_OK;
}

int spegg_kernel_timing(spegg_sim *s, int enable, float *mean_ms, uint32_t *n_launches) {
    if (!s) return SPEGG_EINVAL;
    CU(cudaStreamSynchronize(s->stream));
    drain_timing(s);
    if (mean_ms) *mean_ms = s->timing_n ? (float)(s->timing_ms / s->timing_n) : 0.0f;
    if (n_launches) *n_launches = s->timing_n;
    if (enable && s->ev.empty()) {
        s->ev.resize(512);
        for (auto &e : s->ev) CU(cudaEventCreate(&e));
    }
    if (enable && !s->timing) { s->timing_ms = 0.0; s->timing_n = 0; }
    s->timing = enable != 0;
    return SPEGG_OK;
}

}  // extern "C"
