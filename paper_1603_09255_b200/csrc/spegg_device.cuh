// spegg_device.cuh -- device-side primitives of libspegg (sm_100a).
//
// Philox4x32-10 counter-based draws (R3), the two specified exponentials (R6, R11),
// integer threshold samplers (R4, R5, R9) and the single-pass decoupled look-back used by both
// scans.  Everything that feeds an integer decision is written with explicit round-to-nearest
// intrinsics so that nvcc can neither contract nor reorder it.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace spegg {

enum Stream : uint32_t { ST_FEC = 0, ST_SCALAR = 1, ST_RECOMB_M = 2, ST_RECOMB_P = 3, ST_MUT_M = 4, ST_MUT_P = 5, ST_MATE = 6, ST_MOTHER = 7, ST_PAIR = 8 };

// ---------------------------------------------------------------------------------- Philox
// Salmon et al. SC'11. One round: two 32x32->64 products, two 3-input XORs; key += Weyl.
struct Key { uint32_t k0, k1; };

__host__ __device__ __forceinline__ void philox4x32_10(Key key, uint32_t c0, uint32_t c1, uint32_t c2,
                                                       uint32_t c3, uint32_t (&o)[4]) {
    uint32_t k0 = key.k0, k1 = key.k1;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    o[0] = c0; o[1] = c1; o[2] = c2; o[3] = c3;
}

// R3: counter = (entity, block, step, species<<8 | stream)
__device__ __forceinline__ void draw(Key key, uint32_t species, uint32_t stream, uint32_t entity,
                                     uint32_t block, uint32_t step, uint32_t (&o)[4]) {
    philox4x32_10(key, entity, block, step, (species << 8) | stream, o);
}

// R4
__device__ __forceinline__ uint32_t uniform_index(uint32_t u, uint32_t n) { return __umulhi(u, n); }
__device__ __forceinline__ float u01_of(uint32_t u) { return __fmul_rn((float)(u >> 8), 0x1p-24f); }

// ------------------------------------------------------------------- specified exponentials
// R6: exp(-lam) in fp64: k = floor(x*log2e + 1/2), r = (x - k*ln2_hi) - k*ln2_lo, degree-14
// Taylor/Horner with separately rounded mul and add, exact scaling by 2^k.
__device__ __forceinline__ double exp_neg64(double lam) {
    if (!(lam >= 0.0)) lam = 0.0;
    if (lam > 700.0) return 0.0;
    const double x = -lam;
    const double t = __dmul_rn(x, 0x1.71547652b82fep+0);
    const double kf = floor(__dadd_rn(t, 0.5));
    const double r = __dsub_rn(__dsub_rn(x, __dmul_rn(kf, 0x1.62e42fee00000p-1)), __dmul_rn(kf, 0x1.a39ef35793c76p-33));
    const double c[15] = {
        0x1.0000000000000p+0,  0x1.0000000000000p+0,  0x1.0000000000000p-1,
        0x1.5555555555555p-3,  0x1.5555555555555p-5,  0x1.1111111111111p-7,
        0x1.6c16c16c16c17p-10, 0x1.a01a01a01a01ap-13, 0x1.a01a01a01a01ap-16,
        0x1.71de3a556c734p-19, 0x1.27e4fb7789f5cp-22, 0x1.ae64567f544e4p-26,
        0x1.1eed8eff8d898p-29, 0x1.6124613a86d09p-33, 0x1.93974a8c07c9dp-37};
    double p = c[14];
#pragma unroll
    for (int i = 13; i >= 0; --i) p = __dadd_rn(__dmul_rn(p, r), c[i]);
    const int k = (int)kf;
    const double scale = __longlong_as_double((long long)(1023 + k) << 52);
    return __dmul_rn(p, scale);
}

// R11: exp(x), x <= 0, fp32: Cody-Waite with ln2_hi = 0.693359375, degree-7 Taylor/Horner,
// separately rounded mul and add (no fma), exact scaling by 2^k.
__device__ __forceinline__ float expf_spec(float x) {
    if (!(x <= 0.0f)) x = 0.0f;
    if (x < -87.0f) return 0.0f;
    const float t = __fmul_rn(x, 0x1.715476p+0f);
    const float kf = floorf(__fadd_rn(t, 0.5f));
    const float r = __fsub_rn(__fsub_rn(x, __fmul_rn(kf, 0x1.63p-1f)), __fmul_rn(kf, -0x1.bd0106p-13f));
    float p = 0x1.a01a02p-13f;
    p = __fadd_rn(__fmul_rn(p, r), 0x1.6c16c2p-10f);
    p = __fadd_rn(__fmul_rn(p, r), 0x1.111112p-7f);
    p = __fadd_rn(__fmul_rn(p, r), 0x1.555556p-5f);
    p = __fadd_rn(__fmul_rn(p, r), 0x1.555556p-3f);
    p = __fadd_rn(__fmul_rn(p, r), 0x1.000000p-1f);
    p = __fadd_rn(__fmul_rn(p, r), 0x1.000000p+0f);
    p = __fadd_rn(__fmul_rn(p, r), 0x1.000000p+0f);
    const int k = (int)kf;
    const float scale = __int_as_float((127 + k) << 23);
    return __fmul_rn(p, scale);
}

// --------------------------------------------------------------------------- Poisson tables
// R5: p_0 = exp(-lam), p_k = (p_{k-1}*lam)/k, F_k = F_{k-1}+p_k; T_k = floor(F_k*2^32); stored
// until the first T_k >= 2^32-1 (or maxlen).  count(u) = #{k < len : u >= T_k}.
__device__ inline int build_poisson_table(double lam, uint32_t *T, int maxlen) {
    double p = exp_neg64(lam);
    double F = p;
    int k = 0;
    for (;;) {
        const double tk = floor(__dmul_rn(F, 4294967296.0));
        if (tk >= 4294967295.0) break;
        if (k == maxlen) break;
        T[k] = __double2uint_rz(tk);
        ++k;
        p = __ddiv_rn(__dmul_rn(p, lam), (double)k);
        F = __dadd_rn(F, p);
    }
    return k;
}

__device__ __forceinline__ uint32_t poisson_count(const uint32_t *__restrict__ T, uint32_t len, uint32_t u) {
    uint32_t k = 0;
    while (k < len && u >= T[k]) ++k;
    return k;
}

// R9: delta index = -R + #{k < 2R : u >= T_k}  (binary search; T non-decreasing)
__device__ __forceinline__ int normal_delta(const uint32_t *__restrict__ T, int R, uint32_t u) {
    int lo = 0, hi = 2 * R;  // first index with T[idx] > u
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (u >= T[mid]) lo = mid + 1; else hi = mid;
    }
    return lo - R;
}

// ----------------------------------------------------------- asynchronous copies into shared memory
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void cp_async16(uint32_t dst, const void *src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

__device__ __forceinline__ uint4 lds128(uint32_t addr) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
    return v;
}

// ------------------------------------------------------------ decoupled look-back (one warp)
// status word = flag(2 bits) << 62 | value; flag 0 = not ready, 1 = tile aggregate.  One 64-bit
// store publishes value and flag together, so no fence is needed.  Tiles are handed out by an
// atomic ticket, so every lower-numbered tile has already started (forward progress).
constexpr unsigned long long LB_MASK = (1ull << 62) - 1ull;

__device__ __forceinline__ unsigned long long ld_status(const unsigned long long *p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_status(unsigned long long *p, unsigned long long v) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// Two-level counted look-back.  Tiles are numbered by an atomic ticket; groups of 32 consecutive
// tiles share a counter word gsum[g] = (tiles arrived << 40) | (sum of their aggregates), updated
// with ONE atomicAdd per tile.  The exclusive prefix of tile r is
//     sum over complete groups g' < r/32 of gsum[g']  +  aggregates of tiles [32*(r/32), r)
// so a tile reads at most one 32-wide window of each kind, in parallel, however many tiles are in
// flight and even when they all finish at the same moment (the usual chained look-back then walks
// back window by window).  Called by all 32 lanes of one warp; returns the prefix to every lane.
// status[0..n_tiles_max) holds the per-tile aggregates, gsum = status + n_tiles_max.
__device__ __forceinline__ unsigned long long lookback(unsigned long long *status, uint32_t n_tiles_max,
                                                       uint32_t tile, unsigned long long aggregate) {
    const uint32_t lane = threadIdx.x & 31u;
    unsigned long long *gsum = status + n_tiles_max;
    const uint32_t g = tile >> 5, k = tile & 31u;
    if (lane == 0) {
        st_status(status + tile, (1ull << 62) | aggregate);
        atomicAdd(gsum + g, (1ull << 40) | aggregate);
    }
    unsigned long long v = 0ull;
    if (lane < k) {
        do { v = ld_status(status + (g << 5) + lane); } while ((v >> 62) == 0ull);
        v &= LB_MASK;
    }
    for (uint32_t gg = lane; gg < g; gg += 32) {
        unsigned long long t;
        do { t = ld_status(gsum + gg); } while ((t >> 40) != 32ull);
        v += t & ((1ull << 40) - 1ull);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t v) {
    const uint32_t lane = threadIdx.x & 31u;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, v, o);
        if (lane >= (uint32_t)o) v += t;
    }
    return v;
}

}  // namespace spegg
