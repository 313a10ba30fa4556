// sort.cu -- stable LSD radix sort of (uint32 key, uint32 value) pairs, 8 bits per pass (step a7:
// the absorb mode's depth ordering, and the order-preserving split of depth-ordered pairs by bin).
//
// Per pass: (1) per-tile digit histogram, (2) one decoupled look-back scan over the
// digit-major histogram matrix, (3) scatter with ranks computed on chip: each warp ranks its 256
// keys with match.any and warp-private shared-memory counters, then a 256 x 16 scan across the
// warps of the CTA places every key.  Order inside a tile is (warp, round, lane) = index order,
// so the sort is stable: equal depth keys keep ascending particle index (reading R11).
#include "common.cuh"

namespace splotch {

namespace {

constexpr int kSortThreads = 512;
constexpr int kSortWarps = kSortThreads / 32;
constexpr int kSortItems = 8;
constexpr int kSortTile = kSortThreads * kSortItems;   // 4096 keys per CTA
constexpr int kRadix = 256;

__global__ void __launch_bounds__(kSortThreads)
sort_hist_kernel(const uint32_t *__restrict__ keys, long long n_cap, const unsigned long long *__restrict__ n_dev,
                 int shift, uint32_t *__restrict__ hist, long long n_tiles, const int32_t *__restrict__ status)
{
    __shared__ uint32_t s_hist[kRadix];
    // item count may live on the device; a failed render (status != 0: pair capacity exceeded) sorts nothing
    const long long n = (status && *status != 0) ? 0 : n_dev ? min((long long)*n_dev, n_cap) : n_cap;
    const long long tile = blockIdx.x;
    if (threadIdx.x < kRadix) s_hist[threadIdx.x] = 0u;
    __syncthreads();
    const long long base = tile * kSortTile;
#pragma unroll
    for (int j = 0; j < kSortItems; ++j) {
        const long long i = base + (long long)j * kSortThreads + threadIdx.x;
        if (i < n) atomicAdd(&s_hist[(__ldg(keys + i) >> shift) & (kRadix - 1)], 1u);
    }
    __syncthreads();
    if (threadIdx.x < kRadix) hist[(long long)threadIdx.x * n_tiles + tile] = s_hist[threadIdx.x];
}

__global__ void __launch_bounds__(kSortThreads)
sort_scatter_kernel(const uint32_t *__restrict__ keys_in, const uint32_t *__restrict__ vals_in,
                    uint32_t *__restrict__ keys_out, uint32_t *__restrict__ vals_out, long long n_cap,
                    const unsigned long long *__restrict__ n_dev, int shift,
                    const uint32_t *__restrict__ hist_scanned, long long n_tiles, int write_keys,
                    const int32_t *__restrict__ status)
{
    __shared__ uint32_t s_wcnt[kSortWarps][kRadix];
    __shared__ uint32_t s_gbase[kRadix];
    const long long n = (status && *status != 0) ? 0 : n_dev ? min((long long)*n_dev, n_cap) : n_cap;
    const long long tile = blockIdx.x;
    if (tile * kSortTile >= n) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int i = threadIdx.x; i < kSortWarps * kRadix; i += kSortThreads) (&s_wcnt[0][0])[i] = 0u;
    if (threadIdx.x < kRadix) s_gbase[threadIdx.x] = hist_scanned[(long long)threadIdx.x * n_tiles + tile];
    __syncthreads();

    const long long base = tile * kSortTile + (long long)warp * (32 * kSortItems);
    uint32_t key[kSortItems], val[kSortItems], rank[kSortItems];
    const unsigned lt = (1u << lane) - 1u;
#pragma unroll
    for (int j = 0; j < kSortItems; ++j) {
        const long long i = base + j * 32 + lane;
        const bool valid = i < n;
        key[j] = valid ? __ldg(keys_in + i) : 0u;
        val[j] = valid ? __ldg(vals_in + i) : 0u;
        const uint32_t d = valid ? ((key[j] >> shift) & (kRadix - 1)) : (uint32_t)kRadix;   // invalid lanes group apart
        const unsigned peers = __match_any_sync(0xffffffffu, d);
        uint32_t before = 0;
        if (valid) before = s_wcnt[warp][d];
        __syncwarp();
        if (valid && (peers & lt) == 0u) s_wcnt[warp][d] = before + __popc(peers);   // lowest lane of the group
        __syncwarp();
        rank[j] = before + __popc(peers & lt);
    }
    __syncthreads();
    // exclusive scan over the warps, per digit
    if (threadIdx.x < kRadix) {
        uint32_t run = 0;
#pragma unroll
        for (int w = 0; w < kSortWarps; ++w) {
            const uint32_t c = s_wcnt[w][threadIdx.x];
            s_wcnt[w][threadIdx.x] = run;
            run += c;
        }
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < kSortItems; ++j) {
        const long long i = base + j * 32 + lane;
        if (i < n) {
            const uint32_t d = (key[j] >> shift) & (kRadix - 1);
            const uint32_t pos = s_gbase[d] + s_wcnt[warp][d] + rank[j];
            if (write_keys) keys_out[pos] = key[j];
            vals_out[pos] = val[j];
        }
    }
}

}  // namespace

uint64_t sort_scratch_bytes(int64_t n)
{
    const int64_t n_tiles = n > 0 ? (n + kSortTile - 1) / kSortTile : 1;
    const int64_t m = (int64_t)kRadix * n_tiles;
    return align_up((uint64_t)(m + 1) * 4, 256) * 2 + scan_scratch_bytes(m);
}

// Sorts on key bits [0, key_bits).  Ping-pongs between (keys, vals) and (keys_tmp, vals_tmp);
// *result_in_tmp tells where the result ended.  `n` is the capacity the grids are sized for; when
// n_dev != NULL the actual item count min(*n_dev, n) is read on the device (no host sync); when status_dev != NULL and
// *status_dev != 0 (a render that already failed) every pass returns at once.
int launch_sort_pairs(uint32_t *keys, uint32_t *vals, uint32_t *keys_tmp, uint32_t *vals_tmp, int64_t n,
                      const unsigned long long *n_dev, int key_bits, void *scratch, cudaStream_t st, bool *result_in_tmp,
                      const int32_t *status_dev)
{
    *result_in_tmp = false;
    if (n <= 0 || key_bits <= 0) return 0;
    if (n >= (1ll << 32)) return -4;
    const long long n_tiles = (n + kSortTile - 1) / kSortTile;
    const long long m = (long long)kRadix * n_tiles;
    char *sc = reinterpret_cast<char *>(scratch);
    uint32_t *hist = reinterpret_cast<uint32_t *>(sc);
    uint32_t *hist_scanned = reinterpret_cast<uint32_t *>(sc + align_up((uint64_t)(m + 1) * 4, 256));
    void *scan_scratch = sc + align_up((uint64_t)(m + 1) * 4, 256) * 2;
    const int passes = (key_bits + 7) / 8;
    uint32_t *ki = keys, *vi = vals, *ko = keys_tmp, *vo = vals_tmp;
    for (int p = 0; p < passes; ++p) {
        const int shift = p * 8;
        sort_hist_kernel<<<(unsigned)n_tiles, kSortThreads, 0, st>>>(ki, (long long)n, n_dev, shift, hist, n_tiles, status_dev);
        SPLOTCH_LAUNCH_CHECK();
        int rc = launch_scan_u32_u32(hist, hist_scanned, m, scan_scratch, st);
        if (rc) return rc;
        sort_scatter_kernel<<<(unsigned)n_tiles, kSortThreads, 0, st>>>(ki, vi, ko, vo, (long long)n, n_dev, shift,
                                                                        hist_scanned, n_tiles, 1, status_dev);
        SPLOTCH_LAUNCH_CHECK();
        uint32_t *t = ki; ki = ko; ko = t;
        t = vi; vi = vo; vo = t;
    }
    *result_in_tmp = (passes & 1) != 0;
    return 0;
}

}  // namespace splotch
