// spegg_fused.cuh -- fused two-kernel step of the hot configuration (sm_100a).
//
// Bit-packed genomes with NC chromosomes of WPC 32-bit words each (config 3: 4 x 8 words = 1,024
// loci, 256-byte rows).  One time step is TWO launches:
//
//   k_scan_fused  a1-a3 + the index half of a7: one pass over the physical rows of the current
//                 buffer (32-row slabs, one survivor bitmask per slab, one adult count per 1,024-row
//                 range): logical adult index from the range counts -> rowptr[], Poisson fecundity
//                 of every adult, ONE look-back over the fecundities -> mother[] (physical rows), M_t.
//   k_fused_bit_f a3-a8 in one pass: father draw, asynchronous gather of the fathers' rows into
//                 shared memory (cp.async, issued before the recombination draws are computed so
//                 the gather latency hides behind the Philox work), mothers' rows prefetched into L2
//                 and loaded a pass ahead, crossover masks from the RECOMB blocks (R8), select,
//                 mutate, popcount -> phenotype -> survival; every offspring row is stored exactly
//                 once at row j of the other buffer, and only the 4-byte survivor mask of each
//                 32-offspring chunk says which rows are the next generation.  Its last CTA closes
//                 the step and prepares the next one (a0, a9).
//
// (A one-launch variant -- the scan as a first phase of the gamete kernel, which then polled the
// index words -- measured slower: the scan is latency-bound and wants the whole machine's warps,
// which the gamete kernel's 20 warps per SM do not give it.)
//
// Every draw is addressed by (stream, entity, block, step), never by thread, so the result is
// bit-identical to the materialised pipeline and to the oracle.
#pragma once
#include "spegg_kernels.cuh"

namespace spegg {

__device__ __forceinline__ uint32_t shl_clamp(uint32_t v, uint32_t n) {
    uint32_t r;
    asm("shl.b32 %0, %1, %2;" : "=r"(r) : "r"(v), "r"(n));  // PTX shl clamps n > 31 to "all out"
    return r;
}

// ones from bit s upward within word w of a 256-bit chromosome: (~0 << clamp(s - 32w, 0, 32))
__device__ __forceinline__ uint32_t mask_from(int s, int w) {
    return shl_clamp(0xFFFFFFFFu, (uint32_t)__viaddmax_s32(s, -32 * w, 0));
}

// Programmatic dependent launch: the two kernels of a step are launched with programmatic stream
// serialization, so the next kernel's CTAs are scheduled while the previous grid drains and wait
// here (before their first global access) until it has completed and its writes are visible.
__device__ __forceinline__ void pdl_prologue() {
    asm volatile("griddepcontrol.launch_dependents;");
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

constexpr int FUSED_CHUNK = 32;                 // offspring per warp iteration = rows per slab
constexpr uint32_t FUSED_ROW = 256;             // bytes per row (config 3)
constexpr int SCANF_RANGE = FUSED_RANGE;         // rows per scan range (1,024 = 32 chunks)
constexpr int SCANF_CHUNKS = SCANF_RANGE / FUSED_CHUNK;

// ---------------------------------------------------------------------------------------------
// The fused kernel.  A warp takes chunks of 32 consecutive offspring from an atomic ticket and runs
// a software pipeline over them:
//   (a) lane = offspring: SCALAR block (father -> rowptr -> row, survival uniform), the two MUT
//       blocks' counts, mother row -- for the NEXT chunk, so that no index load is ever waited for.
//   (b) 16 cp.async instructions start the gather of the chunk's 32 fathers' rows (8 KB) into this
//       warp's stage (random rows, full DRAM latency); the mothers' rows (ascending, shared by
//       siblings) are only prefetched into L2.  A stage of 8 KB instead of 16 doubles the warps.
//   (c) lane = (gamete g, chromosome c) of offspring it*4+sub, it = 0..7: the 8 RECOMB blocks,
//       decoded to a packed word (start phase, first two crossover positions); the few chromosomes
//       with more than two crossovers (8 % at mean 1) are queued for pass (x).
//   (m) rare: paternal mutations flip the bit in BOTH haplotypes of the staged private copy of the
//       father's row, which flips it in the gamete whatever the phase is (R9).
//   (d) 8 passes of 4 offspring: a lane owns HALF a chromosome (4 words = one uint4) of BOTH gametes,
//       so that every global access of a quarter warp is 128 contiguous bytes; mothers' words come
//       straight from global one pass ahead, fathers' from the stage; select, popcount, two 128-bit
//       stores of offspring row j.
//   (x) extra crossovers as a fix-up of the rows just stored.
//   (e) lane = offspring: phenotype -> fp32 survival -> decision; the ballot is the chunk's mask.
constexpr int FUSEDF_WARPS = 4;
constexpr int FUSEDF_UNROLL_C = 2;                // decode passes in flight per lane
constexpr int FUSEDF_CTAS = 5;                    // resident CTAs per SM (shared memory and registers allow 5; 4 x 122 registers measured slower)
constexpr int FUSEDF_AHEAD = 1;                   // passes the mothers' loads run ahead
constexpr uint32_t FUSEDF_SP_OFF = FUSED_CHUNK * FUSED_ROW;        // packed draws [8][4][4][2] / partial sums
constexpr uint32_t FUSEDF_Q_OFF = FUSEDF_SP_OFF + 8 * 32 * 4;      // queue of chromosomes with > 2 crossovers: draw [32], (pass, lane) [32]
constexpr uint32_t FUSEDF_MO_OFF = FUSEDF_Q_OFF + 64 * 4;          // mothers' row offsets [32]
constexpr uint32_t FUSEDF_WARP_BYTES = FUSEDF_MO_OFF + 32 * 4;
constexpr uint32_t FUSEDF_SMEM = FUSEDF_WARPS * FUSEDF_WARP_BYTES;

__device__ __forceinline__ uint4 ldg128(const void *p) {
    uint4 v;
    asm volatile("ld.global.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
    return v;
}
__device__ __forceinline__ void prefetch_l2(const void *p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
// ticket counter: a 64-bit atomic, because ptxas turns a 32-bit atom.add (and atom.inc) into its
// warp-aggregated form (vote, leader's atomic, broadcast shuffle) even for a single active lane, and
// that shuffle waits for the atomic's round trip on the spot; the ticket is consumed a chunk later
__device__ __forceinline__ uint32_t atom_inc_ticket(unsigned long long *p, uint32_t one) {
    unsigned long long r;
    asm volatile("atom.global.add.u64 %0, [%1], %2;" : "=l"(r) : "l"(p), "l"((unsigned long long)one));
    return (uint32_t)r;
}

// packed draw of one (gamete, chromosome): s0 | s1 << 9 | phase << 31; positions 1..255,
// 256 = no crossover
__device__ __forceinline__ void half_masks(uint32_t P, uint32_t half, uint32_t (&m)[4]) {
    const int s0 = (int)(P & 0x1FFu) - 128 * (int)half, s1 = (int)((P >> 9) & 0x1FFu) - 128 * (int)half;
    const uint32_t phi = (uint32_t)((int)P >> 31);
#pragma unroll
    for (int i = 0; i < 4; ++i) m[i] = phi ^ mask_from(s0, i) ^ mask_from(s1, i);
}

// crossover count of a draw already known to be >= 3 (u >= T[2]): the next four thresholds are loaded
// at once instead of one dependent load per step of the search; longer searches (count > 6) finish
// with the plain loop
__device__ __forceinline__ uint32_t xover_count_from3(const uint32_t *__restrict__ T, uint32_t len, uint32_t u) {
    const uint32_t t3 = len > 3 ? T[3] : 0xFFFFFFFFu, t4 = len > 4 ? T[4] : 0xFFFFFFFFu,
                   t5 = len > 5 ? T[5] : 0xFFFFFFFFu, t6 = len > 6 ? T[6] : 0xFFFFFFFFu;
    // (a missing threshold compares as "not reached"; T is increasing, so the tests are nested)
    uint32_t k = 3u + (len > 3 && u >= t3 ? 1u : 0u) + (len > 4 && u >= t4 ? 1u : 0u) + (len > 5 && u >= t5 ? 1u : 0u) +
                 (len > 6 && u >= t6 ? 1u : 0u);
    if (k == 7u) while (k < len && u >= T[k]) ++k;
    return k;
}

// MATE: the father comes from the running sum of the mating weights (R19, hermaphrodites) instead of the
// uniform draw: one more SCALAR block and a binary search over mate_cum[] in the scalar stage, and the
// offspring's integer genetic value is left in zrow[] for the next step's weights.  A second instantiation:
// the benchmarked kernel (MATE = false) is the same code as without it.
// NOISE: residual phenotype noise (R17, eq. S2-14): the offspring's phenotype is its genetic value plus k
// quanta from the discrete-normal table on word 1 of SCALAR block 1 -- one more Philox block and a table
// search in stage (e); sums, zrow[] and the stored row keep the GENETIC value.  Again an instantiation of
// its own, so the benchmarked kernel (false, false) is the same code as without it.
template <int NC, int WPC, bool MATE, bool NOISE>
__global__ void __launch_bounds__(FUSEDF_WARPS * 32, FUSEDF_CTAS) k_fused_bit_f(const __grid_constant__ SpK sp) {
    static_assert(NC == 4 && WPC == 8, "lane group of 8 = 2 gametes x 4 chromosomes of 8 words");
    extern __shared__ __align__(128) uint8_t s_dyn[];
    __shared__ uint32_t s_flag;
    __shared__ uint32_t s_one[FUSEDF_WARPS * 32];
    pdl_prologue();
    DevSpecies &st = *sp.st;
    const uint32_t M = st.m, N = st.n0, step = sp.glob->step;
    const uint32_t n_chunks = (M + FUSED_CHUNK - 1) / FUSED_CHUNK;
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t sub = lane >> 3, q = lane & 7u;
    const uint32_t g = q >> 2, c = q & 3u;        // role in (c): one (gamete, chromosome)
    const uint32_t hc = q >> 1, half = q & 1u;    // role in (d): half `half` of chromosome hc, both gametes
    constexpr uint32_t L = NC * WPC * 32;
    uint8_t *wbase = s_dyn + warp * FUSEDF_WARP_BYTES;
    const uint32_t stage = smem_u32(wbase);
    uint32_t *s_P = (uint32_t *)(wbase + FUSEDF_SP_OFF);
    uint32_t *s_q = (uint32_t *)(wbase + FUSEDF_Q_OFF);
    uint32_t *s_mo = (uint32_t *)(wbase + FUSEDF_MO_OFF);
    const uint8_t *pop = sp.pop[st.cur];
    uint8_t *nxt = sp.pop[st.cur ^ 1u];
    const uint32_t *rowptr = sp.rowptr[st.cur];
    uint32_t *mask_nxt = sp.chunk_mask[st.cur ^ 1u];
    uint32_t *range_cnt = sp.range_cnt[st.cur ^ 1u];   // zeroed when the previous step was closed
    const uint32_t stream = g ? ST_RECOMB_P : ST_RECOMB_M;
    // the hot path only needs "at least 1 / 2 / 3 crossovers": x >= T_k written as x > T_k - 1 so that a
    // missing threshold (table shorter than k+1; T_k >= 1 is checked at create time) is never reached
    const uint32_t xl = sp.xover_len[c];
    const uint32_t *XT = sp.T_xover + c * XMAX;
    const uint32_t U0 = xl > 0 ? XT[0] - 1u : 0xFFFFFFFFu, U1 = xl > 1 ? XT[1] - 1u : 0xFFFFFFFFu,
                   U2 = xl > 2 ? XT[2] - 1u : 0xFFFFFFFFu;
    const uint32_t clen1 = sp.chrom_len[c] - 1;
    const uint32_t Um0 = sp.mut_len ? sp.T_mut[0] - 1u : 0xFFFFFFFFu;
    const float theta = st.theta_t;
    const uint32_t cp_dst = stage + (lane >> 4) * FUSED_ROW + (lane & 15u) * 16u;   // + k * 512
    const uint32_t cp_src = (lane & 15u) * 16u;
    const uint32_t ld_fa = stage + sub * FUSED_ROW + q * 16u;                       // + it * 1024 (+ 128)
    const uint32_t sp_slot = sub * 8u + hc * 2u;                                    // + it * 32: (g=0, g=1) pair
    long long acc1 = 0, acc2 = 0;
    uint32_t ties = 0, n_alive = 0;
    // the ticket's addend, 1, read back from shared memory: a value ptxas can prove neither constant nor
    // uniform (a constant or uniform addend is what it aggregates)
    s_one[threadIdx.x] = 1u;
    __syncwarp();   // (the partner lane's store)
    const uint32_t one = ((volatile uint32_t *)s_one)[threadIdx.x ^ 1u];

    // mo / fa are the parents' physical ROW numbers exactly as loaded: nothing here depends on the
    // two index loads, so they stay in flight until the rows are needed one chunk later
    auto scalar_stage = [&](uint32_t jl, uint32_t &mo, uint32_t &fa, float &ul, uint32_t &mf) {
        uint32_t x[4], a[4], b[4];
        draw_rk(sp, ST_SCALAR, jl, 0, step, x);
        draw_rk(sp, ST_MUT_M, jl, 0, step, a);
        draw_rk(sp, ST_MUT_P, jl, 0, step, b);
        mo = 0; fa = 0; mf = 0; ul = 2.0f;
        if (jl < M) {
            mo = sp.mother[jl];
            uint32_t fi = uniform_index(x[0], N);   // R2
            if (MATE) {   // R19: weighted draw by running sum + search (words 2,3 of SCALAR block 1); total 0 keeps R2
                const unsigned long long total = sp.mate_cum[N - 1];
                if (total) {
                    uint32_t y[4];
                    draw_rk(sp, ST_SCALAR, jl, 1, step, y);
                    const unsigned long long target = __umul64hi(((unsigned long long)y[2] << 32) | y[3], total);
                    uint32_t lo = 0, hi = N - 1;
                    while (lo < hi) {
                        const uint32_t mid = (lo + hi) >> 1;
                        if (sp.mate_cum[mid] > target) hi = mid; else lo = mid + 1;
                    }
                    fi = lo;
                }
            }
            fa = rowptr[fi];
            ul = u01_of(x[3]);
            mf = (a[0] > Um0 ? 1u : 0u) | (b[0] > Um0 ? 2u : 0u);
        }
    };
    // R9 for one gamete of offspring jl: calls flip(word index 0..31, bit) for every mutation
    auto mutate = [&](uint32_t ms, uint32_t jl, auto &&flip) {
        uint32_t x[4];
        draw_rk(sp, ms, jl, 0, step, x);
        const uint32_t nm = poisson_count(sp.T_mut, sp.mut_len, x[0]);
        for (uint32_t k = 0; k < nm; ++k) {
            if (k > 0) draw_rk(sp, ms, jl, k, step, x);
            const uint32_t pos = __umulhi(x[1], L);
            flip(pos >> 5, 1u << (pos & 31u));
        }
    };

    uint32_t j0 = 0;
    // (x) for chromosome e_c of gamete e_g of offspring j0 + e_o, which drew e_nc > 2 crossovers
    auto fix_extra = [&](uint32_t e_o, uint32_t e_g, uint32_t e_c, uint32_t e_nc) {
        const uint32_t e_j = j0 + e_o;
        if (e_j >= M) return;
        // the loads first (the row this warp stored a moment ago comes back from L2; the parent's two
        // haplotypes of this chromosome: father from the stage, mother from global), the draws below hide them
        uint4 h[4];
        if (e_g) {
            const uint32_t a_ = stage + e_o * FUSED_ROW + e_c * 32u;
            h[0] = lds128(a_); h[1] = lds128(a_ + 16); h[2] = lds128(a_ + FUSED_ROW / 2); h[3] = lds128(a_ + FUSED_ROW / 2 + 16);
        } else {
            const uint8_t *a_ = pop + (s_mo[e_o] | (e_c * 32u));
            h[0] = ldg128(a_); h[1] = ldg128(a_ + 16); h[2] = ldg128(a_ + FUSED_ROW / 2); h[3] = ldg128(a_ + FUSED_ROW / 2 + 16);
        }
        uint4 *orow = (uint4 *)(nxt + (size_t)e_j * FUSED_ROW + e_g * (FUSED_ROW / 2) + e_c * 32u);
        uint4 o0 = ldg128(orow), o1 = ldg128(orow + 1);
        const uint32_t e_clen1 = sp.chrom_len[e_c] - 1;
        uint32_t xm[8];
#pragma unroll
        for (int w = 0; w < 8; ++w) xm[w] = 0;
        const uint32_t extra = e_nc - 2;
        for (uint32_t b = 0; b * 4 < extra; ++b) {
            uint32_t y[4];
            draw_rk(sp, e_g ? ST_RECOMB_P : ST_RECOMB_M, e_j, e_c * 16 + 1 + b, step, y);
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                if (b * 4 + i < extra) {
                    const int s = (int)__umulhi(y[i], e_clen1) + 1;
#pragma unroll
                    for (int w = 0; w < 8; ++w) xm[w] ^= mask_from(s, w);
                }
            }
        }
        const int before = __popc(o0.x) + __popc(o0.y) + __popc(o0.z) + __popc(o0.w) + __popc(o1.x) + __popc(o1.y) + __popc(o1.z) + __popc(o1.w);
        o0.x ^= (h[0].x ^ h[2].x) & xm[0]; o0.y ^= (h[0].y ^ h[2].y) & xm[1];
        o0.z ^= (h[0].z ^ h[2].z) & xm[2]; o0.w ^= (h[0].w ^ h[2].w) & xm[3];
        o1.x ^= (h[1].x ^ h[3].x) & xm[4]; o1.y ^= (h[1].y ^ h[3].y) & xm[5];
        o1.z ^= (h[1].z ^ h[3].z) & xm[6]; o1.w ^= (h[1].w ^ h[3].w) & xm[7];
        const int after = __popc(o0.x) + __popc(o0.y) + __popc(o0.z) + __popc(o0.w) + __popc(o1.x) + __popc(o1.y) + __popc(o1.z) + __popc(o1.w);
        orow[0] = o0; orow[1] = o1;
        atomicAdd(&s_P[e_o * 8], (uint32_t)(after - before));
    };

    // software pipeline over chunks: the first trip only runs stage (a) of the first chunk
    constexpr uint32_t NONE = 0xFFFFFFFFu;
    // the first two chunks of every warp are fixed (a burst of same-address atomics at the start of
    // the kernel would be served one by one), the later ones come from the ticket
    const uint32_t gwarp = blockIdx.x * FUSEDF_WARPS + warp, n_warps = gridDim.x * FUSEDF_WARPS;
    uint32_t chunk = NONE, chunk1 = gwarp;
    uint32_t mo = 0, fa = 0, mf = 0;
    float ul = 2.0f;
    for (;;) {
        uint32_t ticket = 0;
        const bool active = chunk != NONE;
        if (lane == 0 && active) ticket = atom_inc_ticket(&st.ticket_fused, one);   // consumed (and only then touched) at the loop end
        j0 = chunk * FUSED_CHUNK;
        const uint32_t jl = j0 + lane;
        // ---- (b) fathers: half-warp h copies the row of offspring 2k+h into the stage
        if (active) {
#pragma unroll
            for (int k = 0; k < FUSED_CHUNK / 2; ++k) {
                const uint32_t pf = __shfl_sync(0xffffffffu, fa, 2 * k + (lane >> 4)) * FUSED_ROW;
                cp_async16(cp_dst + k * 2 * FUSED_ROW, pop + (pf | cp_src));
            }
            cp_async_commit();
            //  mothers: every 32-byte sector of the 32 rows is asked into L2 (lane -> sector lane&7 of
            //  the rows of offspring (lane>>3) + 4k)
            s_mo[lane] = mo * FUSED_ROW;
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                const uint32_t pm = __shfl_sync(0xffffffffu, mo, 4 * k + (lane >> 3)) * FUSED_ROW;
                prefetch_l2(pop + (pm | ((lane & 7u) * 32u)));
            }
        }
        const uint32_t matmask = __ballot_sync(0xffffffffu, (mf & 1u) != 0);
        // ---- (a) of the next chunk
        uint32_t mo1, fa1, mf1;
        float ul1;
        scalar_stage(chunk1 * FUSED_CHUNK + lane, mo1, fa1, ul1, mf1);
        if (active) {
        // ---- (c) the 8 RECOMB blocks of this lane's (gamete, chromosome) role
        uint32_t qn = 0;
#pragma unroll FUSEDF_UNROLL_C
        for (int it = 0; it < 8; ++it) {
            const uint32_t j = j0 + it * 4 + sub;
            uint32_t x[4];
            draw_rk(sp, stream, j, c * 16, step, x);
            const uint32_t s0 = x[0] > U0 ? __umulhi(x[2], clen1) + 1 : 256u;
            const uint32_t s1 = x[0] > U1 ? __umulhi(x[3], clen1) + 1 : 256u;
            const uint32_t P = (s0 + (s1 << 9)) | (x[1] & 0x80000000u);
            // chromosomes with crossovers beyond the first two are queued for the fix-up pass (x)
            const bool need = x[0] > U2;
            const uint32_t bal = __ballot_sync(0xffffffffu, need);
            if (need) {
                const uint32_t e = qn + __popc(bal & ((1u << lane) - 1u));
                if (e < 32) { s_q[e] = x[0]; s_q[32 + e] = ((uint32_t)it << 5) | lane; }
            }
            qn += __popc(bal);
            s_P[it * 32 + sub * 8 + c * 2 + g] = P;
        }
        cp_async_wait_all();
        __syncwarp();
        // ---- (m) R9, paternal gamete: flips in the staged private copy of the father's row
        if (__any_sync(0xffffffffu, (mf & 2u) != 0)) {
            if (mf & 2u) {
                uint32_t *prow = (uint32_t *)(wbase + lane * FUSED_ROW);
                mutate(ST_MUT_P, jl, [&](uint32_t wi, uint32_t bit) { prow[wi] ^= bit; prow[L / 32 + wi] ^= bit; });
            }
            __syncwarp();
        }

        // ---- (d) 8 passes of 4 offspring; mothers' words are loaded TWO passes ahead (an L2 round trip
        // is several passes long)
        uint4 ma[FUSEDF_AHEAD], mb[FUSEDF_AHEAD];
#pragma unroll
        for (int p = 0; p < FUSEDF_AHEAD; ++p) {
            const uint8_t *mrow = pop + (s_mo[p * 4 + sub] | (q * 16u));
            ma[p] = ldg128(mrow); mb[p] = ldg128(mrow + FUSED_ROW / 2);
        }
        auto pass = [&](const uint32_t it, uint4 &ma_, uint4 &mb_) {
            const uint32_t o = it * 4 + sub, j = j0 + o;
            const uint4 ca = ma_, cb = mb_;
            if (it + FUSEDF_AHEAD < FUSED_CHUNK / 4) {
                const uint8_t *mrow = pop + (s_mo[o + 4 * FUSEDF_AHEAD] | (q * 16u));
                ma_ = ldg128(mrow); mb_ = ldg128(mrow + FUSED_ROW / 2);
            }
            const uint4 fa0 = lds128(ld_fa + it * 4 * FUSED_ROW), fa1_ = lds128(ld_fa + it * 4 * FUSED_ROW + FUSED_ROW / 2);
            const uint2 PP = *(const uint2 *)(s_P + it * 32 + sp_slot);
            // R8: masks of this lane's four words of chromosome hc, maternal and paternal gamete
            uint32_t mm[4], mp[4];
            half_masks(PP.x, half, mm);
            half_masks(PP.y, half, mp);
            // select: gamete word = hap[phase] word
            uint4 gm, gp;
            gm.x = (ca.x & ~mm[0]) | (cb.x & mm[0]); gm.y = (ca.y & ~mm[1]) | (cb.y & mm[1]);
            gm.z = (ca.z & ~mm[2]) | (cb.z & mm[2]); gm.w = (ca.w & ~mm[3]) | (cb.w & mm[3]);
            gp.x = (fa0.x & ~mp[0]) | (fa1_.x & mp[0]); gp.y = (fa0.y & ~mp[1]) | (fa1_.y & mp[1]);
            gp.z = (fa0.z & ~mp[2]) | (fa1_.z & mp[2]); gp.w = (fa0.w & ~mp[3]) | (fa1_.w & mp[3]);
            // R9, maternal gamete (rare): flip in the registers of the lane that owns the word
            if ((matmask >> o) & 1u) {
                mutate(ST_MUT_M, j, [&](uint32_t wi, uint32_t bit) {
                    if ((wi >> 2) == q) {
                        const uint32_t k = wi & 3u;
                        if (k == 0) gm.x ^= bit; else if (k == 1) gm.y ^= bit; else if (k == 2) gm.z ^= bit; else gm.w ^= bit;
                    }
                });
            }
            // a7: the row is stored once, at row j of the other buffer (alive or not)
            if (j < M) {
                uint4 *orow = (uint4 *)(nxt + (size_t)j * FUSED_ROW) + q;
                orow[0] = gm;
                orow[FUSED_ROW / 32] = gp;
            }
            // a5: this lane's share of the additive phenotype (R10), left where the draws were
            const uint32_t ones = __popc(gm.x) + __popc(gm.y) + __popc(gm.z) + __popc(gm.w) +
                                  __popc(gp.x) + __popc(gp.y) + __popc(gp.z) + __popc(gp.w);
            __syncwarp();
            s_P[it * 32 + lane] = ones;
        };
#pragma unroll(FUSEDF_AHEAD == 1 ? 2 : 1)
        for (uint32_t it = 0; it < FUSED_CHUNK / 4; it += FUSEDF_AHEAD) {
#pragma unroll
            for (int p = 0; p < FUSEDF_AHEAD; ++p) pass(it + p, ma[p], mb[p]);
        }
        __syncwarp();
        // ---- (x) R8, crossovers beyond the second (8 % of the chromosomes at mean 1): one lane per
        // queued chromosome.  A further crossover at s swaps the source haplotype of every locus >= s,
        // i.e. XORs the gamete with (hap0 ^ hap1) there -- applied to the row this warp just stored.
        if (qn <= 32) {
            if (lane < qn) {
                const uint32_t e = s_q[32 + lane], e_ln = e & 31u, e_c = e_ln & 3u;
                const uint32_t e_nc = xover_count_from3(sp.T_xover + e_c * XMAX, sp.xover_len[e_c], s_q[lane]);
                fix_extra((e >> 5) * 4 + (e_ln >> 3), (e_ln >> 2) & 1u, e_c, e_nc);
            }
        }
        else {   // queue overflow (more than 32 of the chunk's 256 chromosomes drew > 2 crossovers: about 0.3 % of the
                 // chunks at mean 1, i.e. some ninety chunks of a full-size step): every lane walks its own eight draws again
            for (uint32_t it = 0; it < 8; ++it) {
                uint32_t x[4];
                draw_rk(sp, stream, j0 + it * 4 + sub, c * 16, step, x);
                const uint32_t nc = poisson_count(XT, xl, x[0]);
                if (nc > 2) fix_extra(it * 4 + sub, g, c, nc);
            }
        }
        __syncwarp();
        // ---- (e) a5-a6: lane = offspring
        {
            const uint4 oa = ((const uint4 *)s_P)[lane * 2], ob = ((const uint4 *)s_P)[lane * 2 + 1];
            const int myzi = 2 * (int)(oa.x + oa.y + oa.z + oa.w + ob.x + ob.y + ob.z + ob.w) - 2 * (int)L;
            bool captured;
            int zp = myzi;
            if (NOISE) {   // R17: the residual acts on this individual's selection only and is not inherited
                uint32_t y[4];
                draw_rk(sp, ST_SCALAR, jl, 1, step, y);
                zp += normal_delta(sp.T_env, sp.R_env, y[1]);
            }
            const float z = __fmul_rn((float)zp, sp.pheno_scale);
            const float s = survival_prob(sp, z, theta, ul, captured);
            const bool valid = jl < M;
            const bool alive = valid && (ul < s);
            if (valid && fabsf(__fsub_rn(ul, s)) < 1e-6f) ++ties;
            if (alive) { acc1 += myzi; acc2 += (long long)myzi * myzi; ++n_alive; }
            const uint32_t bal = __ballot_sync(0xffffffffu, alive);
            if (lane == 0) {
                mask_nxt[chunk] = bal;
                if (bal) atomicAdd(range_cnt + chunk / SCANF_CHUNKS, (uint32_t)__popc(bal));
            }
            if (MATE && valid) sp.zrow[st.cur ^ 1u][jl] = myzi;   // the value travels with the row (next step's weights)
        }
        __syncwarp();   // the stage and the draw words are reused by the next chunk
        }
        chunk = chunk1;
        chunk1 = active ? 2u * n_warps + __shfl_sync(0xffffffffu, ticket, 0) : gwarp + n_warps;
        mo = mo1; fa = fa1; ul = ul1; mf = mf1;
        if (chunk >= n_chunks) break;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        acc1 += __shfl_xor_sync(0xffffffffu, acc1, o);
        acc2 += __shfl_xor_sync(0xffffffffu, acc2, o);
        ties += __shfl_xor_sync(0xffffffffu, ties, o);
        n_alive += __shfl_xor_sync(0xffffffffu, n_alive, o);
    }
    if (lane == 0) {
        if (acc1 != 0 || acc2 != 0) {
            atomicAdd((unsigned long long *)&st.acc_zi, (unsigned long long)acc1);
            atomicAdd((unsigned long long *)&st.acc_zi2, (unsigned long long)acc2);
        }
        if (ties) atomicAdd(&st.near_ties, (unsigned long long)ties);
        if (n_alive) atomicAdd(&st.n_next, n_alive);
    }
    if (sp.solo) solo_tail(sp, &s_flag);
}

// a1-a3 and the index half of a7 for a species on the fused path.  The current buffer holds m_phys
// physical rows in 32-row slabs; chunk_mask[cur] says which are adults and range_cnt[cur] how many
// adults each 1,024-row range holds (both left by the previous step's gamete kernel, or by
// spegg_write_state).  CTA b takes ranges b, b + gridDim.x, ... (4 rows per thread, so that the
// whole machine shares the FEC draws):
//   sum of range_cnt[0 .. range)       -> logical index i of every adult, rowptr[i] = row
//   FEC draw of adult i                -> fecundity f_i  (R5)
//   look-back over the fecundities     -> offspring base off_i, mother[off_i .. off_i+f_i) = row
// so the only dependence between CTAs is ONE counted look-back.  rowptr[] and mother[] are staged in
// shared memory and stored coalesced.  The launch is cooperative: every CTA of the grid is resident,
// so the look-back never waits for a range nobody has started (no ticket: a thousand same-address
// atomics at the start of a kernel are served one by one).
constexpr uint32_t SCANF_ROWS = SCANF_RANGE / SCAN_THREADS;   // rows per thread (4)
constexpr uint32_t SCANF_STAGE = 4096;                        // index words staged per range
static_assert(SCANF_ROWS == 4 && 32 % SCANF_ROWS == 0, "a thread's rows are one nibble of a slab mask");

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_fused(const __grid_constant__ SpK sp) {
    constexpr uint32_t NW = SCAN_THREADS / 32, NT = SCAN_THREADS;
    __shared__ uint32_t s_tab[TMAX];
    __shared__ uint32_t s_len;
    __shared__ uint32_t s_cnt[NW], s_pre[NW], s_f[NW];
    __shared__ unsigned long long s_excl;
    __shared__ uint32_t s_stage[SCANF_STAGE];
    pdl_prologue();
    DevSpecies &st = *sp.st;
    const uint32_t mp = st.m_phys, step = sp.glob->step, cur = st.cur;
    const uint32_t n_ranges = (mp + SCANF_RANGE - 1) / SCANF_RANGE;
    const uint32_t n_slabs = (mp + FUSED_CHUNK - 1) / FUSED_CHUNK;
    const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const uint32_t *cnt = sp.range_cnt[cur];
    const uint32_t *mask = sp.chunk_mask[cur];
    uint32_t *rp = sp.rowptr[cur];
    if (blockIdx.x >= n_ranges) return;   // (no adults at all: M_t stays 0)
    // a0: the fecundity table of this step (R5, R13) is built HERE, by one thread of every CTA, while the
    // others turn the range counts into indices -- the ~2 us fp64 chain of the table is then off the
    // path between the two kernels (the step closing of the previous gamete kernel leaves it out)
    if (tid == NT - 1) {
        const double lam = fecundity_mean(sp, (double)st.n0, sp.K_patch ? sp.K_patch[0] : sp.K, 0);
        s_len = (uint32_t)build_poisson_table(lam, s_tab, TMAX);
    }
    uint32_t T0 = 0xFFFFFFFFu, T1 = 0xFFFFFFFFu, T2 = 0xFFFFFFFFu, T3 = 0xFFFFFFFFu, len0 = 0;
    bool have_tab = false;
    for (uint32_t range = blockIdx.x; range < n_ranges; range += gridDim.x) {
        const uint32_t row0 = range * SCANF_RANGE + tid * SCANF_ROWS;
        const uint32_t ch = row0 >> 5;
        const uint32_t bits = ch < n_slabs ? (mask[ch] >> (row0 & 31u)) & ((1u << SCANF_ROWS) - 1u) : 0u;
        // ---- adults before this range (from the range counts) and before this thread's rows
        uint32_t pre = 0;
        for (uint32_t k = tid; k < range; k += NT) pre += cnt[k];
        const uint32_t c4 = __popc(bits);
        const uint32_t incl = warp_incl_scan(c4);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) pre += __shfl_xor_sync(0xffffffffu, pre, o);
        __syncthreads();   // the previous range's stage has been written out
        if (lane == 31) s_cnt[warp] = incl;
        if (lane == 0) s_pre[warp] = pre;
        __syncthreads();   // (also: the table is built)
        if (!have_tab) {   // the first thresholds in registers: the search below rarely goes past them
            have_tab = true;
            len0 = s_len;
            if (len0 > 0) T0 = s_tab[0];
            if (len0 > 1) T1 = s_tab[1];
            if (len0 > 2) T2 = s_tab[2];
            if (len0 > 3) T3 = s_tab[3];
        }
        uint32_t ibase = 0, li0 = incl - c4, n_r = 0;   // adults before the range / before this thread in it / in it
#pragma unroll
        for (uint32_t w = 0; w < NW; ++w) { ibase += s_pre[w]; n_r += s_cnt[w]; if (w < warp) li0 += s_cnt[w]; }
        // ---- fecundity of this thread's adults (first: the range's total is what the other ranges wait for)
        uint32_t fsum = 0, fpack = 0;
        {
            uint32_t i = ibase + li0;
#pragma unroll
            for (uint32_t k = 0; k < SCANF_ROWS; ++k) {
                if ((bits >> k) & 1u) {
                    uint32_t x[4];
                    draw_rk(sp, ST_FEC, i++, 0, step, x);
                    const uint32_t u = x[0];
                    // count(u) = #{k < len : u >= T_k}, T increasing (a missing threshold is never reached:
                    // the table stops before 2^32 - 1 ... see build_poisson_table; u >= T with T = 2^32 - 1 only
                    // for u = 2^32 - 1, excluded by the length test)
                    uint32_t f = (len0 > 0 && u >= T0 ? 1u : 0u) + (len0 > 1 && u >= T1 ? 1u : 0u) +
                                 (len0 > 2 && u >= T2 ? 1u : 0u) + (len0 > 3 && u >= T3 ? 1u : 0u);
                    if (f == 4u) while (f < len0 && u >= s_tab[f]) ++f;
                    fpack |= f << (8u * k);
                    fsum += f;
                }
            }
        }
        // ---- look-back over the fecundities: offspring before this range
        const uint32_t fincl = warp_incl_scan(fsum);
        if (lane == 31) s_f[warp] = fincl;
        // ---- rowptr (staged, stored coalesced below while warp 0 waits for the look-back)
        {
            uint32_t li = li0;
#pragma unroll
            for (uint32_t k = 0; k < SCANF_ROWS; ++k)
                if ((bits >> k) & 1u) s_stage[li++] = row0 + k;
        }
        __syncthreads();
        uint32_t total = 0, wbase = 0;
#pragma unroll
        for (uint32_t w = 0; w < NW; ++w) { const uint32_t v = s_f[w]; total += v; if (w < warp) wbase += v; }
        if (warp == 0) {
            const unsigned long long excl = lookback(sp.status_fec, sp.status_fec_n, range, (unsigned long long)total);
            if (lane == 0) {
                s_excl = excl;
                if (range == n_ranges - 1) {  // the last range knows M
                    const unsigned long long Mtot = excl + total;
                    if (Mtot > (unsigned long long)sp.capacity) { st.m = sp.capacity; st.flags_step |= 1u; }
                    else st.m = (uint32_t)Mtot;
                }
            }
        } else {
            for (uint32_t k = tid - 32u; k < n_r; k += NT - 32u) rp[ibase + k] = s_stage[k];
        }
        __syncthreads();   // the staged rowptr words have been read; s_excl is there
        // ---- mother[]: staged per range like rowptr (a range with more offspring than the stage holds
        // -- fecundities far above the table means of any configuration -- writes them directly)
        const bool staged = total <= SCANF_STAGE;
        uint32_t lo = wbase + (fincl - fsum);
        if (staged) {
#pragma unroll
            for (uint32_t k = 0; k < SCANF_ROWS; ++k) {
                const uint32_t f = (fpack >> (8u * k)) & 0xFFu;
                for (uint32_t cpy = 0; cpy < f; ++cpy) s_stage[lo++] = row0 + k;
            }
        }
        const unsigned long long obase = s_excl;
        __syncthreads();
        if (staged) {
            for (uint32_t k = tid; k < total; k += NT)
                if (obase + k < (unsigned long long)sp.capacity) sp.mother[obase + k] = s_stage[k];
        } else {
            unsigned long long o = obase + lo;
#pragma unroll
            for (uint32_t k = 0; k < SCANF_ROWS; ++k) {
                const uint32_t f = (fpack >> (8u * k)) & 0xFFu;
                for (uint32_t cpy = 0; cpy < f; ++cpy, ++o)
                    if (o < (unsigned long long)sp.capacity) sp.mother[o] = row0 + k;
            }
        }
    }
}

// rowptr[] of the current buffer alone (spegg_read_state): the index half of k_scan_fused.
__global__ void __launch_bounds__(SCAN_THREADS) k_rowptr_fused(const __grid_constant__ SpK sp) {
    constexpr uint32_t NW = SCAN_THREADS / 32;
    __shared__ uint32_t s_cnt[NW], s_pre[NW];
    const DevSpecies &st = *sp.st;
    const uint32_t mp = st.m_phys, cur = st.cur;
    const uint32_t n_ranges = (mp + SCANF_RANGE - 1) / SCANF_RANGE;
    const uint32_t n_slabs = (mp + FUSED_CHUNK - 1) / FUSED_CHUNK;
    const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const uint32_t *cnt = sp.range_cnt[cur];
    const uint32_t *mask = sp.chunk_mask[cur];
    uint32_t *rp = sp.rowptr[cur];
    for (uint32_t range = blockIdx.x; range < n_ranges; range += gridDim.x) {
        const uint32_t row0 = range * SCANF_RANGE + tid * SCANF_ROWS;
        const uint32_t ch = row0 >> 5;
        const uint32_t bits = ch < n_slabs ? (mask[ch] >> (row0 & 31u)) & ((1u << SCANF_ROWS) - 1u) : 0u;
        uint32_t pre = 0;
        for (uint32_t k = tid; k < range; k += SCAN_THREADS) pre += cnt[k];
        const uint32_t c = __popc(bits);
        const uint32_t incl = warp_incl_scan(c);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) pre += __shfl_xor_sync(0xffffffffu, pre, o);
        __syncthreads();
        if (lane == 31) s_cnt[warp] = incl;
        if (lane == 0) s_pre[warp] = pre;
        __syncthreads();
        uint32_t i = incl - c;
#pragma unroll
        for (uint32_t w = 0; w < NW; ++w) i += s_pre[w] + (w < warp ? s_cnt[w] : 0u);
#pragma unroll
        for (uint32_t k = 0; k < SCANF_ROWS; ++k)
            if ((bits >> k) & 1u) rp[i++] = row0 + k;
    }
}

// chunk masks and range counts of a freshly written, dense population of n rows
__global__ void __launch_bounds__(256) k_fill_masks(uint32_t *mask, uint32_t *range_cnt, uint32_t n) {
    const uint32_t n_chunks = (n + 31) / 32, n_ranges = (n + SCANF_RANGE - 1) / SCANF_RANGE;
    for (uint32_t c = blockIdx.x * blockDim.x + threadIdx.x; c < n_chunks; c += gridDim.x * blockDim.x) {
        const uint32_t r = n - c * 32;
        mask[c] = r >= 32 ? 0xFFFFFFFFu : ((1u << r) - 1u);
    }
    for (uint32_t c = blockIdx.x * blockDim.x + threadIdx.x; c < n_ranges; c += gridDim.x * blockDim.x)
        range_cnt[c] = min(n - c * SCANF_RANGE, (uint32_t)SCANF_RANGE);
}

__host__ inline bool fused_bit_supported(const SpK &k) {
    return k.kind == 0 && k.linkage == 1 && k.n_chrom == 4 && k.L == 1024 && k.P == 1 && !k.sel_predation && k.adult_surv == 0.0f &&
           k.fec_model != 2 && k.theta_patch == nullptr &&
           (unsigned long long)(k.capacity + 32) * FUSED_ROW < (1ull << 32);
}

inline cudaError_t fused_bit_configure() {
    cudaError_t e = cudaFuncSetAttribute(k_fused_bit_f<4, 8, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FUSEDF_SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_fused_bit_f<4, 8, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FUSEDF_SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_fused_bit_f<4, 8, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FUSEDF_SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_fused_bit_f<4, 8, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FUSEDF_SMEM);
    return e;
}

inline cudaError_t launch_fused_bit(const SpK &k, uint32_t n_sms, cudaStream_t stream) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(n_sms * FUSEDF_CTAS);
    cfg.blockDim = dim3(FUSEDF_WARPS * 32);
    cfg.dynamicSmemBytes = FUSEDF_SMEM;
    cfg.stream = stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    if (k.R_env > 0) return k.mate_on ? cudaLaunchKernelEx(&cfg, k_fused_bit_f<4, 8, true, true>, k) : cudaLaunchKernelEx(&cfg, k_fused_bit_f<4, 8, false, true>, k);
    return k.mate_on ? cudaLaunchKernelEx(&cfg, k_fused_bit_f<4, 8, true, false>, k) : cudaLaunchKernelEx(&cfg, k_fused_bit_f<4, 8, false, false>, k);
}

// Cooperative launch: the whole grid is resident at once (or the launch fails), which the fixed
// range -> CTA assignment of the look-back relies on.  ctas_per_sm comes from the occupancy query.
inline cudaError_t launch_scan_fused(const SpK &k, uint32_t n_sms, uint32_t ctas_per_sm, cudaStream_t stream) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(n_sms * ctas_per_sm);
    cfg.blockDim = dim3(SCAN_THREADS);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = stream;
    cudaLaunchAttribute at[2];
    at[0].id = cudaLaunchAttributeCooperative;
    at[0].val.cooperative = 1;
    at[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[1].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 2;
    return cudaLaunchKernelEx(&cfg, k_scan_fused, k);
}

inline int scan_fused_ctas_per_sm() {
    int n = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_scan_fused, SCAN_THREADS, 0) != cudaSuccess) return 0;
    return n;
}

inline void launch_rowptr_fused(const SpK &k, uint32_t n_sms, cudaStream_t stream) {
    k_rowptr_fused<<<n_sms * 4, SCAN_THREADS, 0, stream>>>(k);
}

}  // namespace spegg
