// scan.cu -- single-pass exclusive prefix sum with decoupled look-back (step a5 of the hot path:
// bin counts -> bin offsets; also pair offsets of the absorb-mode expansion).
//
// Each CTA takes a ticket (so that tile t can only wait on tiles that already run), scans a
// tile of 2048 items with warp shuffles, publishes its aggregate, and walks back over the
// predecessors' descriptors one warp-load (32 tiles) at a time until it meets an inclusive
// prefix.  A descriptor is one 64-bit word: status in the top two bits, value below, so one
// store publishes both.
#include "common.cuh"
#include "splotch.h"

namespace splotch {

namespace {

constexpr int kScanThreads = 256;
constexpr int kScanItems = 8;
constexpr int kScanTile = kScanThreads * kScanItems;

constexpr unsigned long long kStatusAggregate = 1ull << 62;
constexpr unsigned long long kStatusPrefix = 2ull << 62;
constexpr unsigned long long kValueMask = (1ull << 62) - 1;

__device__ __forceinline__ unsigned long long ld_desc(const unsigned long long *p)
{
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}

__device__ __forceinline__ void st_desc(unsigned long long *p, unsigned long long v)
{
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

template <typename OutT>
__global__ void __launch_bounds__(kScanThreads)
scan_lookback_kernel(const uint32_t *__restrict__ in, OutT *__restrict__ out, long long n,
                     unsigned long long *desc, uint32_t *ticket)
{
    __shared__ uint32_t s_tile;
    __shared__ unsigned long long s_warp[kScanThreads / 32];
    __shared__ unsigned long long s_exclusive;

    if (threadIdx.x == 0) s_tile = atomicAdd(ticket, 1u);
    __syncthreads();
    const uint32_t tile = s_tile;
    const long long base = (long long)tile * kScanTile + (long long)threadIdx.x * kScanItems;

    uint32_t v[kScanItems];
    if (base + kScanItems <= n && ((reinterpret_cast<uintptr_t>(in + base) & 15u) == 0)) {
        const uint4 a = __ldg(reinterpret_cast<const uint4 *>(in + base));
        const uint4 b = __ldg(reinterpret_cast<const uint4 *>(in + base) + 1);
        v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w;
        v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
    } else {
#pragma unroll
        for (int k = 0; k < kScanItems; ++k) v[k] = (base + k < n) ? __ldg(in + base + k) : 0u;
    }
    unsigned long long tsum = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) tsum += v[k];

    // inclusive scan of the thread sums inside the warp
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned long long inc = tsum;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        unsigned long long o = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= d) inc += o;
    }
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    unsigned long long warp_off = 0, block_total = 0;
#pragma unroll
    for (int w = 0; w < kScanThreads / 32; ++w) {
        const unsigned long long s = s_warp[w];
        if (w < warp) warp_off += s;
        block_total += s;
    }

    // publish, then look back (warp 0)
    if (warp == 0) {
        if (lane == 0) st_desc(desc + tile, (tile == 0 ? kStatusPrefix : kStatusAggregate) | block_total);
        unsigned long long exclusive = 0;
        if (tile > 0) {
            long long idx = (long long)tile - 1;
            while (true) {
                const long long mine = idx - lane;
                unsigned long long d = kStatusPrefix;            // lanes before tile 0 read "prefix 0"
                if (mine >= 0) {
                    do { d = ld_desc(desc + mine); } while ((d >> 62) == 0ull);
                }
                const unsigned is_prefix = __ballot_sync(0xffffffffu, (d >> 62) == 2ull);
                const int first = is_prefix ? (__ffs(is_prefix) - 1) : 32;   // nearest inclusive prefix
                unsigned long long contrib = (lane <= first) ? (d & kValueMask) : 0ull;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) contrib += __shfl_xor_sync(0xffffffffu, contrib, o);
                exclusive += contrib;
                if (is_prefix) break;
                idx -= 32;
            }
            if (lane == 0) st_desc(desc + tile, kStatusPrefix | ((exclusive + block_total) & kValueMask));
        }
        if (lane == 0) s_exclusive = exclusive;
    }
    __syncthreads();

    unsigned long long run = s_exclusive + warp_off + (inc - tsum);
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        if (base + k < n) out[base + k] = (OutT)run;
        run += v[k];
    }
    // the tile that holds item n-1 (or tile 0 when n == 0) writes the total
    const long long last_tile = n > 0 ? (n - 1) / kScanTile : 0;
    if ((long long)tile == last_tile && threadIdx.x == kScanThreads - 1) out[n] = (OutT)(s_exclusive + block_total);
}

template <typename OutT>
int launch_scan(const uint32_t *in, OutT *out, int64_t n, void *scratch, cudaStream_t st)
{
    const int64_t tiles = n > 0 ? (n + kScanTile - 1) / kScanTile : 1;
    SPLOTCH_CUDA_TRY(cudaMemsetAsync(scratch, 0, scan_scratch_bytes(n), st));
    uint32_t *ticket = reinterpret_cast<uint32_t *>(scratch);
    unsigned long long *desc = reinterpret_cast<unsigned long long *>(reinterpret_cast<char *>(scratch) + 256);
    scan_lookback_kernel<OutT><<<(unsigned)tiles, kScanThreads, 0, st>>>(in, out, (long long)n, desc, ticket);
    SPLOTCH_LAUNCH_CHECK();
    return 0;
}

}  // namespace

uint64_t scan_scratch_bytes(int64_t n)
{
    const int64_t tiles = n > 0 ? (n + kScanTile - 1) / kScanTile : 1;
    return align_up(256 + (uint64_t)(tiles + 1) * 8, 256);
}

int launch_scan_u32_u64(const uint32_t *in, uint64_t *out, int64_t n, void *scratch, cudaStream_t st)
{
    return launch_scan<unsigned long long>(in, reinterpret_cast<unsigned long long *>(out), n, scratch, st);
}

int launch_scan_u32_u32(const uint32_t *in, uint32_t *out, int64_t n, void *scratch, cudaStream_t st)
{
    return launch_scan<uint32_t>(in, out, n, scratch, st);
}

// ---------------------------------------------------------------------------------------------
// splotch_scan_static: the same scan for callers that have no device memory to hand over as scratch and may not
// ask the CUDA allocator for any (include/splotch.h says who they are).  The ticket and the tile descriptors live
// in the array below, which is part of the library image: every GPU that loads the library carries these
// 66,048 bytes until the process exits, whether the entry point is ever called or not.
// ---------------------------------------------------------------------------------------------
namespace {

constexpr int64_t kStaticScanMaxN = 1 << 24;                                  // = SPLOTCH_SCAN_STATIC_MAX_N
constexpr int64_t kStaticScanTiles = kStaticScanMaxN / kScanTile;             // 8192
constexpr size_t kStaticScanBytes = (256 + (kStaticScanTiles + 1) * 8 + 255) / 256 * 256;   // same layout as launch_scan

static __device__ __align__(256) unsigned char g_static_scan_scratch[kStaticScanBytes];

// On the host the name g_static_scan_scratch is only a handle for the runtime, not a device address; the address
// differs per device and has to be asked for with that device current.  Looked up once per device and kept.
std::atomic<void *> g_static_scan_ptr[kMaxDevices];

int static_scan_scratch(void **out)
{
    int dev = -1;
    SPLOTCH_CUDA_TRY(cudaGetDevice(&dev));
    const bool slot = dev >= 0 && dev < kMaxDevices;
    void *p = slot ? g_static_scan_ptr[dev].load(std::memory_order_acquire) : nullptr;
    if (!p) {
        SPLOTCH_CUDA_TRY(cudaGetSymbolAddress(&p, g_static_scan_scratch));
        if (!p) return -3;
        if (slot) g_static_scan_ptr[dev].store(p, std::memory_order_release);   // racing threads store the same value
    }
    *out = p;
    return 0;
}

}  // namespace

}  // namespace splotch

extern "C" int splotch_scan_static(const uint32_t *in, uint64_t *out, int64_t n, void *stream)
{
    using namespace splotch;
    static_assert(kStaticScanMaxN == SPLOTCH_SCAN_STATIC_MAX_N, "header and kernel file disagree on the limit");
    static_assert(kStaticScanBytes == 66048, "the size the header and README quote");
    if (n < 0 || !out || (n > 0 && !in)) return SPLOTCH_ERR_INVALID_ARG;
    if (n > kStaticScanMaxN) return SPLOTCH_ERR_LIMIT;      // the descriptor array has no room for more tiles
    void *scratch = nullptr;
    const int rc = static_scan_scratch(&scratch);
    if (rc) return rc;
    // launch_scan zeroes the ticket and the descriptors it is about to use (a memset enqueued on the stream, not an
    // allocation), so what the previous call left in the array does not matter.
    return launch_scan_u32_u64(in, out, n, scratch, reinterpret_cast<cudaStream_t>(stream));
}
