// spegg_fused.cuh -- fused single-pass kernels of the hot configuration (sm_100a).
//
// Bit-packed genomes with NC chromosomes of WPC 32-bit words each (config 3: 4 x 8 words = 1,024
// loci, 256-byte rows).  After k_fec_scan (fecundity, scan, mother[]) the step is two kernels:
//
//   k_fused_bit   a3-a8 in one pass: father draw, gather of both parents' rows, crossover masks
//                 from the RECOMB blocks (R8), select, mutate, popcount -> phenotype -> survival,
//                 survivors stored once into the other population buffer.  Offspring rows never
//                 touch memory unless they survive.
//   k_index       stable order of the next generation from 4-byte chunk masks (rowptr).
//
// Thread mapping of k_fused_bit: 8 consecutive lanes own one offspring, lane q = (gamete g = q/4,
// chromosome c = q%4): it loads the 8 words of chromosome c of both haplotypes of parent g with
// four 128-bit loads, computes that chromosome's Philox block, builds its 8 mask words in
// registers, and stores its 32 bytes of the surviving row with two 128-bit stores.  A warp handles
// 4 offspring, a 256-thread CTA a tile of 32; tiles come from an atomic ticket and the survivors'
// positions from the same decoupled look-back as the fecundity scan (stable order in j).
// Every draw is addressed by (stream, offspring j, block, step), never by thread, so the result is
// bit-identical to the materialised pipeline and to the oracle.
#pragma once
#include "spegg_kernels.cuh"

namespace spegg {


__device__ __forceinline__ uint32_t shl_clamp(uint32_t v, uint32_t n) {
    uint32_t r;
    asm("shl.b32 %0, %1, %2;" : "=r"(r) : "r"(v), "r"(n));  // PTX shl clamps n > 31 to "all out"
    return r;
}

__device__ __forceinline__ uint4 ldg_u4(const uint4 *p) {
    uint4 v;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
    return v;
}

// Warp-autonomous fused kernel.  A warp takes a chunk of FUSED_CHUNK = 32 consecutive offspring
// from an atomic ticket.
//   prologue (dense, every lane busy, independent Philox chains interleave):
//     - lane = offspring: mother row, SCALAR block (father -> rowptr -> row, survival uniform),
//       the two MUT blocks' counts
//     - lane = (gamete g, chromosome c) of offspring it*4+sub, it = 0..7: the 8 RECOMB blocks this
//       lane will need, decoded to a packed word (count, start phase, first two positions)
//     - the few chromosomes with more than two crossovers (8 % at mean 1) are queued and their
//       extra blocks / mask contributions computed one per lane, so no divergent Philox later
//   8 passes of 4 offspring (8 lanes each): four 128-bit loads of the lane's 8-word chromosome
//   from both haplotypes of its parent, mask words from the packed draw (+ queued extras), select,
//   rare mutation, popcount -> phenotype -> fp32 survival, and the surviving rows are stored,
//   packed and in j order, at the start of the chunk's own 32-row slab of the other buffer.
// Nothing waits on another warp: the stable order of the next generation is established
// afterwards by k_index, which scans the 4-byte chunk masks and writes rowptr (logical adult index
// -> physical row).  The 256-byte rows are written exactly once; only indices are compacted.
constexpr int FUSED_CHUNK = 32;
constexpr int FUSED_WARPS = 8;

template <int NC, int WPC>
__global__ void __launch_bounds__(FUSED_WARPS * 32, 3) k_fused_bit(const __grid_constant__ SpK sp) {
    static_assert(NC == 4 && WPC == 8, "lane group of 8 = 2 gametes x 4 chromosomes of 8 words");
    __shared__ uint4 s_xmask[FUSED_WARPS][32][2];   // mask contribution of queued extra crossovers
    __shared__ uint32_t s_P[FUSED_WARPS][8][32];    // packed recombination draws of the chunk
    __shared__ uint32_t s_q[FUSED_WARPS][32];       // queue of chromosomes with > 2 crossovers
    DevSpecies &st = *sp.st;
    const uint32_t M = st.m, N = st.n0, step = sp.glob->step;
    const uint32_t n_chunks = (M + FUSED_CHUNK - 1) / FUSED_CHUNK;
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t sub = lane >> 3, q = lane & 7u, g = q >> 2, c = q & 3u;
    constexpr uint32_t ROW4 = 2 * NC * WPC / 4;   // uint4 per row (16)
    constexpr uint32_t L = NC * WPC * 32;
    const uint4 *pop = (const uint4 *)sp.pop[st.cur];
    uint4 *nxt = (uint4 *)sp.pop[st.cur ^ 1u];
    const uint32_t *rowptr = sp.rowptr[st.cur];
    const uint32_t stream = g ? ST_RECOMB_P : ST_RECOMB_M;
    // this chromosome's crossover-count thresholds in registers (count <= 6 without a loop)
    const uint32_t xl = sp.xover_len[c];
    const uint32_t *XT = sp.T_xover + c * XMAX;
    uint32_t T[6];
#pragma unroll
    for (int i = 0; i < 6; ++i) T[i] = (uint32_t)i < xl ? XT[i] : 0xFFFFFFFFu;
    const bool short_table = xl <= 6;
    const uint32_t clen1 = sp.chrom_len[c] - 1;
    const uint32_t Tm0 = sp.mut_len ? sp.T_mut[0] : 0xFFFFFFFFu;
    const bool has_mut = sp.mut_len != 0;
    const float theta = st.theta_t;
    long long acc1 = 0, acc2 = 0;
    uint32_t ties = 0;

    for (;;) {
        uint32_t chunk = 0;
        if (lane == 0) chunk = atomicAdd(&st.ticket_fused, 1u);
        chunk = __shfl_sync(0xffffffffu, chunk, 0);
        if (chunk >= n_chunks) break;
        const uint32_t j0 = chunk * FUSED_CHUNK;
        // ---- prologue (a): lane = offspring j0 + lane
        uint32_t mo = 0, fa = 0, mf = 0;
        float ul = 2.0f;
        {
            const uint32_t jl = j0 + lane;
            uint32_t x[4], a[4], b[4];
            draw(sp.key, sp.species, ST_SCALAR, jl, 0, step, x);
            draw(sp.key, sp.species, ST_MUT_M, jl, 0, step, a);
            draw(sp.key, sp.species, ST_MUT_P, jl, 0, step, b);
            if (jl < M) {
                mo = sp.mother[jl];                        // physical row (phys_parents)
                fa = rowptr[uniform_index(x[0], N)];       // R2: uniform mate, selfing allowed
                ul = u01_of(x[3]);
                if (has_mut) mf = (a[0] >= Tm0 ? 1u : 0u) | (b[0] >= Tm0 ? 2u : 0u);
            }
        }
        // ---- prologue (b): the 8 RECOMB blocks of this lane's (gamete, chromosome) role
        uint32_t qn = 0;
#pragma unroll
        for (int it = 0; it < 8; ++it) {
            const uint32_t j = j0 + it * 4 + sub;
            uint32_t x[4];
            draw(sp.key, sp.species, stream, j, c * 16, step, x);
            uint32_t nc = 0;
#pragma unroll
            for (int i = 0; i < 6; ++i) nc += (x[0] >= T[i]) ? 1u : 0u;
            if (!short_table && nc == 6) nc = poisson_count(XT, xl, x[0]);
            uint32_t P = nc | ((x[1] >> 31) << 6) | ((__umulhi(x[2], clen1) + 1) << 8) | ((__umulhi(x[3], clen1) + 1) << 16);
            // queue the chromosomes that need crossovers beyond the first two
            const bool need = nc > 2;
            const uint32_t bal = __ballot_sync(0xffffffffu, need);
            uint32_t id = 63;
            if (need) {
                const uint32_t e = qn + __popc(bal & ((1u << lane) - 1u));
                if (e < 32) { id = e; s_q[warp][e] = (nc << 8) | ((uint32_t)it << 5) | lane; }
            }
            qn += __popc(bal);
            s_P[warp][it][lane] = P | (id << 24);
        }
        __syncwarp();
        // ---- prologue (c): one lane per queued chromosome computes its extra crossovers
        if (lane < min(qn, 32u)) {
            const uint32_t e = s_q[warp][lane];
            const uint32_t e_nc = e >> 8, e_it = (e >> 5) & 7u, e_ln = e & 31u;
            const uint32_t e_c = e_ln & 3u, e_g = (e_ln >> 2) & 1u;
            const uint32_t e_j = j0 + e_it * 4 + (e_ln >> 3);
            const uint32_t e_clen1 = sp.chrom_len[e_c] - 1;
            uint32_t xm[8];
#pragma unroll
            for (int w = 0; w < 8; ++w) xm[w] = 0;
            const uint32_t extra = e_nc - 2;
            for (uint32_t b = 0; b * 4 < extra; ++b) {
                uint32_t y[4];
                draw(sp.key, sp.species, e_g ? ST_RECOMB_P : ST_RECOMB_M, e_j, e_c * 16 + 1 + b, step, y);
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    if (b * 4 + i < extra) {
                        const int s = (int)__umulhi(y[i], e_clen1) + 1;
#pragma unroll
                        for (int w = 0; w < 8; ++w) xm[w] ^= shl_clamp(0xFFFFFFFFu, (uint32_t)max(s - 32 * w, 0));
                    }
                }
            }
            s_xmask[warp][lane][0] = make_uint4(xm[0], xm[1], xm[2], xm[3]);
            s_xmask[warp][lane][1] = make_uint4(xm[4], xm[5], xm[6], xm[7]);
        }
        __syncwarp();

        uint32_t cnt = 0, cmask = 0;  // survivors stored so far / survivor bitmask (warp-uniform)
#pragma unroll 1
        for (uint32_t it = 0; it < FUSED_CHUNK / 4; ++it) {
            const uint32_t src = it * 4 + sub;
            const uint32_t j = j0 + src;
            const bool valid = j < M;
            const float u01 = __shfl_sync(0xffffffffu, ul, src);
            const uint32_t mflag = (__shfl_sync(0xffffffffu, mf, src) >> g) & 1u;
            const uint32_t pm = __shfl_sync(0xffffffffu, mo, src), pf = __shfl_sync(0xffffffffu, fa, src);
            const uint32_t parent = g ? pf : pm;
            const uint4 *row = pop + (size_t)parent * ROW4 + c * 2;
            const uint4 a = ldg_u4(row), b = ldg_u4(row + 1), d = ldg_u4(row + ROW4 / 2), e = ldg_u4(row + ROW4 / 2 + 1);
            const uint32_t h0[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
            const uint32_t h1[8] = {d.x, d.y, d.z, d.w, e.x, e.y, e.z, e.w};
            // ---- R8: crossover mask of chromosome c of gamete g from the packed draw
            const uint32_t P = s_P[warp][it][lane];
            const uint32_t nc = P & 63u;
            const uint32_t phi = ((P >> 6) & 1u) ? 0xFFFFFFFFu : 0u;
            const int s0 = nc > 0 ? (int)((P >> 8) & 0xFFu) : 4096;
            const int s1 = nc > 1 ? (int)((P >> 16) & 0xFFu) : 4096;
            uint32_t m[8];
#pragma unroll
            for (int w = 0; w < 8; ++w)
                m[w] = phi ^ shl_clamp(0xFFFFFFFFu, (uint32_t)max(s0 - 32 * w, 0)) ^
                       shl_clamp(0xFFFFFFFFu, (uint32_t)max(s1 - 32 * w, 0));
            if (nc > 2) {
                const uint32_t id = (P >> 24) & 63u;
                if (id < 32) {
                    const uint4 xa = s_xmask[warp][id][0], xb = s_xmask[warp][id][1];
                    m[0] ^= xa.x; m[1] ^= xa.y; m[2] ^= xa.z; m[3] ^= xa.w;
                    m[4] ^= xb.x; m[5] ^= xb.y; m[6] ^= xb.z; m[7] ^= xb.w;
                } else {  // queue overflow (> 32 such chromosomes in one chunk): compute in place
                    const uint32_t extra = nc - 2;
                    for (uint32_t bb = 0; bb * 4 < extra; ++bb) {
                        uint32_t y[4];
                        draw(sp.key, sp.species, stream, j, c * 16 + 1 + bb, step, y);
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            if (bb * 4 + i < extra) {
                                const int s = (int)__umulhi(y[i], clen1) + 1;
#pragma unroll
                                for (int w = 0; w < 8; ++w) m[w] ^= shl_clamp(0xFFFFFFFFu, (uint32_t)max(s - 32 * w, 0));
                            }
                        }
                    }
                }
            }
            // ---- select: gamete word = hap[phase] word
            uint32_t gw[8];
#pragma unroll
            for (int w = 0; w < 8; ++w) gw[w] = (h0[w] & ~m[w]) | (h1[w] & m[w]);
            // ---- R9: mutation (rare; flagged per gamete in the prologue)
            if (mflag) {
                const uint32_t ms = g ? ST_MUT_P : ST_MUT_M;
                uint32_t x[4];
                draw(sp.key, sp.species, ms, j, 0, step, x);
                const uint32_t nm = poisson_count(sp.T_mut, sp.mut_len, x[0]);
                for (uint32_t k = 0; k < nm; ++k) {
                    if (k > 0) draw(sp.key, sp.species, ms, j, k, step, x);
                    const uint32_t pos = __umulhi(x[1], L);
                    const uint32_t wi = pos >> 5;
                    if ((wi >> 3) == c) {
#pragma unroll
                        for (int w = 0; w < 8; ++w)
                            if ((wi & 7u) == (uint32_t)w) gw[w] ^= 1u << (pos & 31u);
                    }
                }
            }
            // ---- a5: additive phenotype, exact integer (R10)
            int ones = 0;
#pragma unroll
            for (int w = 0; w < 8; ++w) ones += __popc(gw[w]);
            ones += __shfl_xor_sync(0xffffffffu, ones, 1);
            ones += __shfl_xor_sync(0xffffffffu, ones, 2);
            ones += __shfl_xor_sync(0xffffffffu, ones, 4);
            const int zi = 2 * ones - 2 * (int)L;
            // ---- a6: survival (R11), same fp32 sequence as the materialised path
            bool captured;
            const float z = __fmul_rn((float)zi, sp.pheno_scale);
            const float s = survival_prob(sp, z, theta, u01, captured);
            const bool alive = valid && (u01 < s);
            if (valid && q == 0) {
                if (fabsf(__fsub_rn(u01, s)) < 1e-6f) ++ties;
                if (alive) { acc1 += zi; acc2 += (long long)zi * zi; }
            }
            // ---- a7: store the surviving row at its rank within the chunk's slab
            const uint32_t bal = __ballot_sync(0xffffffffu, alive && q == 0);
            if (alive) {
                const uint32_t slot = j0 + cnt + __popc(bal & ((1u << (lane & 24u)) - 1u));
                uint4 *o = nxt + (size_t)slot * ROW4 + g * (ROW4 / 2) + c * 2;
                o[0] = make_uint4(gw[0], gw[1], gw[2], gw[3]);
                o[1] = make_uint4(gw[4], gw[5], gw[6], gw[7]);
            }
            cnt += __popc(bal);
            cmask |= ((bal & 1u) | ((bal >> 7) & 2u) | ((bal >> 14) & 4u) | ((bal >> 21) & 8u)) << (it * 4);
        }
        if (lane == 0) sp.chunk_mask[chunk] = cmask;
        __syncwarp();
    }
    // ---- a8: survivor reductions (exact integers)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        acc1 += __shfl_xor_sync(0xffffffffu, acc1, o);
        acc2 += __shfl_xor_sync(0xffffffffu, acc2, o);
        ties += __shfl_xor_sync(0xffffffffu, ties, o);
    }
    if (lane == 0) {
        if (acc1 != 0 || acc2 != 0) {
            atomicAdd((unsigned long long *)&st.acc_zi, (unsigned long long)acc1);
            atomicAdd((unsigned long long *)&st.acc_zi2, (unsigned long long)acc2);
        }
        if (ties) atomicAdd(&st.near_ties, (unsigned long long)ties);
    }
}

// a7: stable order of the next generation.  One thread per chunk: exclusive scan of the chunks'
// survivor counts (decoupled look-back over tiles of 256 chunks), then one warp per chunk writes
// rowptr_next[base + r] = 32*chunk + r (coalesced).  Moves 4 bytes per survivor instead of rows.
__global__ void __launch_bounds__(SCAN_THREADS) k_index(const __grid_constant__ SpK sp) {
    __shared__ uint32_t s_warp[SCAN_THREADS / 32];
    __shared__ uint32_t s_base[SCAN_THREADS], s_cnt[SCAN_THREADS];
    __shared__ uint32_t s_tile;
    __shared__ unsigned long long s_excl;
    DevSpecies &st = *sp.st;
    const uint32_t n_chunks = (st.m + FUSED_CHUNK - 1) / FUSED_CHUNK;
    const uint32_t n_tiles = (n_chunks + SCAN_THREADS - 1) / SCAN_THREADS;
    const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    uint32_t *rp = sp.rowptr[st.cur ^ 1u];
    for (;;) {
        if (tid == 0) s_tile = atomicAdd(&st.ticket_cmp, 1u);
        __syncthreads();
        const uint32_t tile = s_tile;
        if (tile >= n_tiles) break;
        const uint32_t ch = tile * SCAN_THREADS + tid;
        const uint32_t cnt = ch < n_chunks ? __popc(sp.chunk_mask[ch]) : 0u;
        const uint32_t incl = warp_incl_scan(cnt);
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
        s_base[tid] = (uint32_t)s_excl + s_warp[warp] + (incl - cnt);
        s_cnt[tid] = cnt;
        __syncthreads();
        for (uint32_t k = 0; k < 32; ++k) {
            const uint32_t t = warp * 32 + k;
            if (lane < s_cnt[t]) rp[s_base[t] + lane] = (tile * SCAN_THREADS + t) * FUSED_CHUNK + lane;
        }
        __syncthreads();
    }
    if (sp.solo) solo_tail(sp, &s_tile);
}

__host__ inline bool fused_bit_supported(const SpK &k) {
    return k.kind == 0 && k.linkage == 1 && k.n_chrom == 4 && k.L == 1024 && k.P == 1 && !k.sel_predation &&
           k.fec_model != 2 && k.theta_patch == nullptr;
}

inline void launch_fused_bit(const SpK &k, uint32_t n_sms, cudaStream_t stream) {
    k_fused_bit<4, 8><<<n_sms * 3, FUSED_WARPS * 32, 0, stream>>>(k);
}

inline void launch_index(const SpK &k, uint32_t n_sms, cudaStream_t stream) {
    k_index<<<n_sms * 2, SCAN_THREADS, 0, stream>>>(k);
}

}  // namespace spegg
