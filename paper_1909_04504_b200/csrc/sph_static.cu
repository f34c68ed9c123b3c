// sph_static.cu -- sph_cell_offsets_static (include/sph.h): the cell offsets of Sec.2.2 (L158-170), i.e. the exclusive
// prefix sum of the per-cell counts, for callers that may not allocate.  It is a variant of k_scan (sph_nnps.cu):
// the same single-pass scan with decoupled look-back over tiles of 4096 counts, but its scratch -- the ticket and
// the look-back table, which the context path keeps in memory it cudaMallocs -- lives in the file-scope device
// array below, and nothing here calls cudaMalloc, cudaFree or a routine that allocates.
//
// The array is one per GPU that loads the library and is shared by every call on that GPU.  It keeps the last call's
// contents, so every call clears the part it uses (one cudaMemsetAsync ahead of the kernel, in stream order); two
// calls that overlap on the GPU race on it (sph.h says so).
#include <cuda_runtime.h>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <mutex>

#include "sph.h"

#define SSCAN_T      512
#define SSCAN_ITEMS  8
#define SSCAN_TILE   (SSCAN_T * SSCAN_ITEMS)                          // 4096 counts per tile
#define SSCAN_MAX_TILES ((int)(SPH_STATIC_SCAN_MAX_N / SSCAN_TILE))   // 16384
#define SSCAN_HDR_WORDS 32                                            // 256 bytes: word 0 = the tile ticket
static_assert(SPH_STATIC_SCAN_MAX_N % SSCAN_TILE == 0, "maximum is a whole number of tiles");
static_assert(SPH_STATIC_SCAN_BYTES == 8 * (SSCAN_HDR_WORDS + SSCAN_MAX_TILES), "sph.h states the size of the array");

// [0, 32): header (word 0: ticket).  [32, 32 + tiles): one state word per tile = {flag << 32 | value}; flag 0 = not
// yet published, 1 = value is the tile's own sum, 2 = value is the inclusive prefix up to and including the tile.
// In HOST code this name is a host-side stand-in, not a device address: the launches below use the address that
// cudaGetSymbolAddress returns for the current device.
static __device__ __align__(256) unsigned long long g_static_scan[SSCAN_HDR_WORDS + SSCAN_MAX_TILES];

static thread_local char t_err[256] = "";
extern "C" const char* sph_static_last_error(void) { return t_err; }
static int fail(int code, const char* fmt, ...) {
    va_list ap; va_start(ap, fmt); vsnprintf(t_err, sizeof(t_err), fmt, ap); va_end(ap);
    return code;
}

__device__ __forceinline__ uint32_t sscan_block_exclusive(uint32_t v, uint32_t* total) {
    __shared__ uint32_t warp_sums[SSCAN_T / 32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    uint32_t inc = v;
    for (int o = 1; o < 32; o <<= 1) { uint32_t t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
    if (lane == 31) warp_sums[w] = inc;
    __syncthreads();
    if (w == 0) {
        uint32_t s = lane < SSCAN_T / 32 ? warp_sums[lane] : 0u, si = s;
        for (int o = 1; o < 32; o <<= 1) { uint32_t t = __shfl_up_sync(0xffffffffu, si, o); if (lane >= o) si += t; }
        if (lane < SSCAN_T / 32) warp_sums[lane] = si - s;
        if (lane == 31) *total = si;
    }
    __syncthreads();
    return warp_sums[w] + inc - v;
}

// Tiles take their number from the ticket, so every predecessor of a running tile is running or done (no deadlock
// whatever the order blocks are scheduled in).  `scratch` is the device address of g_static_scan, cleared (header
// and the first nb state words) by the memset the host issues ahead of this launch.
__global__ void __launch_bounds__(SSCAN_T)
k_scan_static(const uint32_t* __restrict__ in, long long n, uint32_t* __restrict__ out, int nb,
              unsigned long long* __restrict__ scratch) {
    __shared__ uint32_t s_tile, s_total, s_prefix;
    if (threadIdx.x == 0) s_tile = atomicAdd(reinterpret_cast<uint32_t*>(scratch), 1u);
    __syncthreads();
    const uint32_t tile = s_tile;
    volatile unsigned long long* vs = scratch + SSCAN_HDR_WORDS;
    const long long i0 = (long long)tile * SSCAN_TILE + (long long)threadIdx.x * SSCAN_ITEMS;
    uint32_t v[SSCAN_ITEMS], s = 0;
    const bool vec = i0 + SSCAN_ITEMS <= n && ((reinterpret_cast<uintptr_t>(in) & 15) == 0);
    if (vec) {
#pragma unroll
        for (int k = 0; k < SSCAN_ITEMS; k += 4) {
            const uint4 q = *reinterpret_cast<const uint4*>(in + i0 + k);
            v[k] = q.x; v[k + 1] = q.y; v[k + 2] = q.z; v[k + 3] = q.w; s += q.x + q.y + q.z + q.w;
        }
    } else {
#pragma unroll
        for (int k = 0; k < SSCAN_ITEMS; ++k) { v[k] = (i0 + k < n) ? in[i0 + k] : 0u; s += v[k]; }
    }
    uint32_t ex = sscan_block_exclusive(s, &s_total);
    const uint32_t total = s_total;
    if (threadIdx.x < 32) {
        const int lane = threadIdx.x;
        uint32_t prefix = 0u;
        if (tile > 0) {
            if (lane == 0) vs[tile] = (1ull << 32) | total;
            long long p = (long long)tile - 1;                      // look back over tiles p, p-1, ... (lane = distance)
            for (;;) {
                const long long q = p - lane;
                unsigned long long w = 0ull; uint32_t f = 2u;       // tiles before 0 count as "inclusive, 0"
                if (q >= 0) { do { w = vs[q]; f = (uint32_t)(w >> 32); } while (f == 0u); }
                const unsigned inc = __ballot_sync(0xffffffffu, f == 2u);
                const int stop = inc ? __ffs(inc) - 1 : 32;          // nearest tile whose inclusive prefix is known
                uint32_t add = (lane <= stop && q >= 0) ? (uint32_t)w : 0u;
                for (int o = 16; o > 0; o >>= 1) add += __shfl_xor_sync(0xffffffffu, add, o);
                prefix += add;
                if (inc) break;
                p -= 32;
            }
        }
        if (lane == 0) {
            vs[tile] = (2ull << 32) | (prefix + total);
            s_prefix = prefix;
            if ((int)tile == nb - 1) out[n] = prefix + total;
        }
    }
    __syncthreads();
    ex += s_prefix;
#pragma unroll
    for (int k = 0; k < SSCAN_ITEMS; ++k) { const uint32_t e = ex; ex += v[k]; v[k] = e; }
    if (i0 + SSCAN_ITEMS <= n && ((reinterpret_cast<uintptr_t>(out) & 15) == 0)) {
#pragma unroll
        for (int k = 0; k < SSCAN_ITEMS; k += 4) *reinterpret_cast<uint4*>(out + i0 + k) = make_uint4(v[k], v[k + 1], v[k + 2], v[k + 3]);
    } else {
#pragma unroll
        for (int k = 0; k < SSCAN_ITEMS; ++k) if (i0 + k < n) out[i0 + k] = v[k];
    }
}

// Set-up, once per device, with that device current: the device address of g_static_scan.
#define SSCAN_MAX_DEVICES 64
static std::mutex g_mu;
static unsigned long long* g_dev_ptr[SSCAN_MAX_DEVICES];

static int scratch_of_current_device(unsigned long long** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(SPH_ERR_CUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= SSCAN_MAX_DEVICES) return fail(SPH_ERR_BAD_ARG, "device ordinal %d not in [0, %d)", dev, SSCAN_MAX_DEVICES);
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_dev_ptr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_scan);
        if (e != cudaSuccess || !p) return fail(SPH_ERR_CUDA, "cudaGetSymbolAddress(g_static_scan) on device %d: %s", dev, cudaGetErrorString(e));
        g_dev_ptr[dev] = static_cast<unsigned long long*>(p);
    }
    *out = g_dev_ptr[dev];
    return SPH_OK;
}

extern "C" int sph_cell_offsets_static(const uint32_t* d_counts, int64_t n, uint32_t* d_offsets, void* stream) {
    if (!d_offsets || (n > 0 && !d_counts)) return fail(SPH_ERR_NULL, "sph_cell_offsets_static: NULL pointer");
    if (n < 0) return fail(SPH_ERR_BAD_ARG, "sph_cell_offsets_static: n = %lld < 0", (long long)n);
    if (n > SPH_STATIC_SCAN_MAX_N)
        return fail(SPH_ERR_CAPACITY, "sph_cell_offsets_static: n = %lld exceeds SPH_STATIC_SCAN_MAX_N = %lld (the static scratch "
                    "array holds one word per 4096 counts; use the context path for larger tables)", (long long)n, (long long)SPH_STATIC_SCAN_MAX_N);
    unsigned long long* scratch = nullptr;
    int rc = scratch_of_current_device(&scratch);
    if (rc) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    cudaError_t e;
    if (n == 0) {
        e = cudaMemsetAsync(d_offsets, 0, sizeof(uint32_t), st);
        return e == cudaSuccess ? SPH_OK : fail(SPH_ERR_CUDA, "cudaMemsetAsync: %s", cudaGetErrorString(e));
    }
    const int nb = (int)((n + SSCAN_TILE - 1) / SSCAN_TILE);
    e = cudaMemsetAsync(scratch, 0, sizeof(unsigned long long) * (size_t)(SSCAN_HDR_WORDS + nb), st);   // ticket + the nb state words
    if (e != cudaSuccess) return fail(SPH_ERR_CUDA, "cudaMemsetAsync(scratch): %s", cudaGetErrorString(e));
    k_scan_static<<<nb, SSCAN_T, 0, st>>>(d_counts, (long long)n, d_offsets, nb, scratch);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(SPH_ERR_CUDA, "k_scan_static launch: %s", cudaGetErrorString(e));
    return SPH_OK;
}
