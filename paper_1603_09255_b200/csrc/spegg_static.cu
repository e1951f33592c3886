// spegg_static.cu -- spegg_offsets_static: the neonate-offset scan (Fig. 1 A) for callers
// that must not allocate device memory.
//
// Everywhere else in libspegg the caller hands over one workspace block and the kernels carve their
// scratch (look-back status words, work tickets) out of it.  Some callers have no block to hand over
// and cannot make one: code that runs inside somebody else's memory budget (a plug-in of a host
// application whose allocator owns the whole GPU, a callback that runs while an allocation lock is
// held), code that must not trigger the implicit device synchronisation of cudaMalloc / cudaFree in a
// latency-critical loop, and code on systems where the allocator is simply not reachable from where the
// call is made.  For them this file keeps the scan's scratch in a fixed array that is part of the
// library image itself: the only device memory the call touches is that array plus the caller's input
// and outputs, and the call makes no cudaMalloc, cudaFree or allocating library call.
//
// Costs, stated up front:
//   - every GPU that loads libspegg.so holds SCRATCH_WORDS * 8 bytes (about 34 KB) until the process exits;
//   - the size is capped at SPEGG_STATIC_MAX_N adults per call (larger n is refused with SPEGG_ELIMIT);
//   - there is ONE array per device, shared by every call from every thread and stream: two calls whose
//     kernels overlap on the same GPU race on it and both results are garbage.  Serialise them (same stream,
//     or an event between streams).  The array keeps the previous call's contents, so each call first clears
//     the part it is going to use, on the caller's stream, in front of the scan kernel.
//
// The kernel is the a2 stage of k_fec_scan / the tile loop of k_cmp_scan (spegg_kernels.cuh) with the
// fecundities read from memory instead of drawn, and uses the same counted two-level look-back
// (spegg_device.cuh); only where its status words and ticket live is different.
#include <cstdint>
#include <mutex>

#include "../../include/spegg.h"
#include "spegg_device.cuh"

namespace {

using namespace spegg;

constexpr int ST_THREADS = 256;
constexpr int ST_ITEMS = 4;
constexpr uint32_t ST_TILE = ST_THREADS * ST_ITEMS;                        // 1,024 adults per tile
constexpr uint32_t ST_MAX_TILES = (uint32_t)(SPEGG_STATIC_MAX_N / ST_TILE);   // 4,096
// layout, in 64-bit words: [0, MAX_TILES) tile aggregates | [MAX_TILES, MAX_TILES + MAX_TILES/32 + 2) group
// counters (lookback() addresses them as status + n_tiles_max) | last word: the tile ticket
constexpr uint32_t ST_GROUP_WORDS = ST_MAX_TILES / 32 + 2;
constexpr uint32_t ST_TICKET = ST_MAX_TILES + ST_GROUP_WORDS;
constexpr uint32_t SCRATCH_WORDS = ST_TICKET + 1;
static_assert(SPEGG_STATIC_MAX_N % ST_TILE == 0, "the maximum is a whole number of tiles");

// The scratch.  In HOST code this name is only a handle for cudaGetSymbolAddress -- it is not a device
// address and must never be passed to a kernel; static_scratch() below turns it into one.
static __device__ __align__(256) unsigned long long g_static_scratch[SCRATCH_WORDS];

// off[i] = f[0] + ... + f[i-1] (saturating at 2^32 - 1 like k_fec_scan's off[]), *total = sum of all f.
// scratch: zeroed words [0, n_tiles), the group counters and the ticket (see the layout above).
__global__ void __launch_bounds__(ST_THREADS) k_offsets_static(const uint8_t *__restrict__ f, uint32_t n,
                                                               uint32_t *__restrict__ off,
                                                               unsigned long long *__restrict__ total_out,
                                                               unsigned long long *scratch) {
    __shared__ uint32_t s_warp[ST_THREADS / 32];
    __shared__ uint32_t s_tile;
    __shared__ unsigned long long s_excl;
    const uint32_t n_tiles = (n + ST_TILE - 1) / ST_TILE;
    const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    for (;;) {
        // tiles are handed out in ticket order, so every lower-numbered tile is already running
        // somewhere when a tile waits for it in the look-back
        if (tid == 0) s_tile = (uint32_t)atomicAdd(scratch + ST_TICKET, 1ull);
        __syncthreads();
        const uint32_t tile = s_tile;
        if (tile >= n_tiles) break;
        const uint32_t base = tile * ST_TILE + tid * ST_ITEMS;
        uint32_t a[ST_ITEMS], sum = 0;
        if (base + ST_ITEMS <= n) {   // f is only byte-aligned for the caller's base; tiles start at multiples of 4
            const uint32_t w = ((uintptr_t)f & 3u) == 0 ? *(const uint32_t *)(f + base)
                                                         : (uint32_t)f[base] | (uint32_t)f[base + 1] << 8 | (uint32_t)f[base + 2] << 16 | (uint32_t)f[base + 3] << 24;
#pragma unroll
            for (int k = 0; k < ST_ITEMS; ++k) { a[k] = (w >> (8 * k)) & 0xFFu; sum += a[k]; }
        } else {
#pragma unroll
            for (int k = 0; k < ST_ITEMS; ++k) { a[k] = (base + k < n) ? f[base + k] : 0u; sum += a[k]; }
        }
        const uint32_t incl = warp_incl_scan(sum);
        if (lane == 31) s_warp[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            const uint32_t w = (lane < ST_THREADS / 32) ? s_warp[lane] : 0u;
            const uint32_t wi = warp_incl_scan(w);
            const uint32_t total = __shfl_sync(0xffffffffu, wi, ST_THREADS / 32 - 1);
            const unsigned long long excl = lookback(scratch, ST_MAX_TILES, tile, (unsigned long long)total);
            if (lane < ST_THREADS / 32) s_warp[lane] = wi - w;   // exclusive warp prefix
            if (lane == 0) {
                s_excl = excl;
                if (tile == n_tiles - 1) *total_out = excl + total;   // the last tile knows the sum
            }
        }
        __syncthreads();
        unsigned long long o = s_excl + s_warp[warp] + (incl - sum);
#pragma unroll
        for (int k = 0; k < ST_ITEMS; ++k) {
            if (base + k < n) off[base + k] = (uint32_t)min(o, 0xFFFFFFFFull);
            o += a[k];
        }
        __syncthreads();   // s_tile / s_warp / s_excl are reused by the next tile
    }
}

// One-time set-up per device: resolves the array's device address on the device that is current and
// remembers it together with that device's SM count.  The runtime calls here (cudaGetSymbolAddress,
// cudaDeviceGetAttribute) may initialise the CUDA context and load the module, which is why the first
// call on a device belongs in front of any stream capture.
constexpr int ST_MAX_DEVICES = 64;
struct PerDevice { unsigned long long *scratch; int sms; };
PerDevice g_dev[ST_MAX_DEVICES];
std::mutex g_dev_lock;

int static_scratch(PerDevice *out, cudaError_t *err) {
    int dev = -1;
    *err = cudaGetDevice(&dev);
    if (*err != cudaSuccess) return SPEGG_ECUDA;
    if (dev < 0 || dev >= ST_MAX_DEVICES) return SPEGG_EINVAL;
    std::lock_guard<std::mutex> hold(g_dev_lock);
    if (g_dev[dev].scratch == nullptr) {
        void *p = nullptr;
        *err = cudaGetSymbolAddress(&p, g_static_scratch);
        if (*err != cudaSuccess || p == nullptr) return SPEGG_ECUDA;
        int sms = 0;
        *err = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (*err != cudaSuccess || sms <= 0) return SPEGG_ECUDA;
        g_dev[dev].sms = sms;
        g_dev[dev].scratch = (unsigned long long *)p;
    }
    *out = g_dev[dev];
    return SPEGG_OK;
}

}  // namespace

extern "C" int spegg_offsets_static(const uint8_t *d_f, uint64_t n, uint32_t *d_off, uint64_t *d_total,
                                    void *cuda_stream) {
    if (d_total == nullptr || (n > 0 && (d_f == nullptr || d_off == nullptr))) return SPEGG_EINVAL;
    if (n > SPEGG_STATIC_MAX_N) return SPEGG_ELIMIT;   // the scratch array has room for SPEGG_STATIC_MAX_N adults, no more
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    cudaError_t err = cudaSuccess;
    if (n == 0) {   // nothing to scan and no scratch needed: the sum is 0
        err = cudaMemsetAsync(d_total, 0, sizeof(uint64_t), stream);
        return err == cudaSuccess ? SPEGG_OK : SPEGG_ECUDA;
    }
    PerDevice dev;
    const int rc = static_scratch(&dev, &err);
    if (rc != SPEGG_OK) return rc;
    const uint32_t n_tiles = (uint32_t)((n + ST_TILE - 1) / ST_TILE);
    // the array still holds the last call's aggregates, counters and ticket: zero what this call reads.
    // Tile aggregates [0, n_tiles) and the group counters + ticket are two pieces of the array.
    err = cudaMemsetAsync(dev.scratch, 0, (size_t)n_tiles * 8u, stream);
    if (err == cudaSuccess) err = cudaMemsetAsync(dev.scratch + ST_MAX_TILES, 0, (size_t)(ST_GROUP_WORDS + 1) * 8u, stream);
    if (err != cudaSuccess) return SPEGG_ECUDA;
    const uint32_t grid = n_tiles < (uint32_t)dev.sms * 8u ? n_tiles : (uint32_t)dev.sms * 8u;
    k_offsets_static<<<grid, ST_THREADS, 0, stream>>>(d_f, (uint32_t)n, d_off, (unsigned long long *)d_total, dev.scratch);
    err = cudaGetLastError();
    return err == cudaSuccess ? SPEGG_OK : SPEGG_ECUDA;
}
