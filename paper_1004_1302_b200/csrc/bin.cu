// bin.cu -- K2: binning (steps a4-a6): offsets -> work units, scatter of splat ids into per-bin
// lists with big splats duplicated into every bin their pixel box touches (B-rules), and the
// depth-ordered pair expansion of the absorb mode.  PAPER.md:105 "determining screen areas
// affected by individual particles"; the paper's own load-balancing device is the
// "split particles" pass of PAPER.md:109, which this replaces.
#include "common.cuh"

namespace splotch {

namespace {

constexpr int kBinThreads = 256;
constexpr int kSmemBinsMax = 4096;          // two u32 arrays of this size live in shared memory

struct BinBox {
    int x0, x1, y0, y1;
    __device__ __forceinline__ int width() const { return x1 - x0 + 1; }
    __device__ __forceinline__ int count() const { return (x1 - x0 + 1) * (y1 - y0 + 1); }
};

__device__ __forceinline__ BinBox unpack(uint32_t b)
{
    BinBox o;
    o.x0 = b & 255; o.x1 = (b >> 8) & 255; o.y0 = (b >> 16) & 255; o.y1 = (b >> 24) & 255;
    return o;
}

// Calls f(bin_index, local_index, pa, pb) once for every bin of the splat's box, where (pa, pb)
// is the payload of the lane that owns the splat.  Boxes larger than 8 bins are walked by the
// whole warp; the owner's box and payload are broadcast while all lanes are converged.  Must be
// called by all 32 lanes (lanes without a splat pass kInvisible).
template <typename F>
__device__ __forceinline__ void for_each_bin(uint32_t bins, uint32_t pa, unsigned long long pb, int nbx, F f)
{
    const int lane = threadIdx.x & 31;
    const bool vis = bins != kInvisible;
    const BinBox bb = unpack(bins);
    const bool big = vis && bb.count() > 8;
    if (vis && !big) {
        int k = 0;
        for (int by = bb.y0; by <= bb.y1; ++by)
            for (int bx = bb.x0; bx <= bb.x1; ++bx) f(by * nbx + bx, k++, pa, pb);
    }
    unsigned m = __ballot_sync(0xffffffffu, big);
    while (m) {
        const int src = __ffs(m) - 1;
        m &= m - 1;
        const BinBox cb = unpack(__shfl_sync(0xffffffffu, bins, src));
        const uint32_t opa = __shfl_sync(0xffffffffu, pa, src);
        const unsigned long long opb = __shfl_sync(0xffffffffu, pb, src);
        const int cw = cb.width(), ctot = cb.count();
        for (int i = lane; i < ctot; i += 32) f((cb.y0 + i / cw) * nbx + cb.x0 + i % cw, i, opa, opb);
    }
}

// ---------------------------------------------------------------------------------------------
// offsets -> status head + raster work units (one CTA)
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(1024)
finish_offsets_kernel(const uint32_t *__restrict__ bin_count, const uint64_t *__restrict__ bin_offset, int n_bins,
                      unsigned long long max_pairs, uint32_t chunk, uint32_t *__restrict__ unit_prefix, WorkHead *head)
{
    __shared__ uint32_t s_part[1024];
    const int t = threadIdx.x;
    const int per = (n_bins + 1023) / 1024;
    const int b0 = min(t * per, n_bins), b1 = min(b0 + per, n_bins);
    uint32_t sum = 0;
    for (int b = b0; b < b1; ++b) sum += (bin_count[b] + chunk - 1) / chunk;
    s_part[t] = sum;
    __syncthreads();
    // Hillis-Steele inclusive scan over the 1024 partial sums
    for (int d = 1; d < 1024; d <<= 1) {
        const uint32_t v = (t >= d) ? s_part[t - d] : 0u;
        __syncthreads();
        s_part[t] += v;
        __syncthreads();
    }
    uint32_t run = s_part[t] - sum;
    for (int b = b0; b < b1; ++b) {
        unit_prefix[b] = run;
        run += (bin_count[b] + chunk - 1) / chunk;
    }
    if (t == 1023) unit_prefix[n_bins] = s_part[1023];
    if (t == 0) {
        const unsigned long long D = bin_offset[n_bins];
        head->pairs = D;
        head->n_units = 0;
        head->work_counter = 0;
        head->mma_counter = 0;
        head->tensor_on = head->area_tensor >= kTensorShare * head->area_total && head->area_total > 0.0f ? 1u : 0u;
        if (D > max_pairs) head->status = -2;   // SPLOTCH_ERR_WORKSPACE
    }
    __syncthreads();
    if (t == 0 && head->status == 0) head->n_units = s_part[1023];
}

// ---------------------------------------------------------------------------------------------
// scatter: list[bin_offset[b] + k] = particle index, any order inside a bin (additive mode).
// A CTA takes a chunk of 1024 particles, counts its pairs per bin in shared memory, reserves
// one range per touched bin with a single global atomic, then writes ids into the ranges.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kBinThreads)
scatter_kernel(const void *__restrict__ records, int record_bytes, long long n, int nbx, int n_bins,
               const uint64_t *__restrict__ bin_offset, uint32_t *__restrict__ bin_cursor,
               uint32_t *__restrict__ list, const WorkHead *head, int use_smem)
{
    extern __shared__ uint32_t s_mem[];
    if (head->status != 0) return;
    uint32_t *s_cnt = s_mem, *s_base = s_mem + n_bins;
    constexpr int kPer = 4;
    const long long chunk = (long long)kBinThreads * kPer;
    const long long n_chunks = (n + chunk - 1) / chunk;
    for (long long c = blockIdx.x; c < n_chunks; c += gridDim.x) {
        uint32_t bins[kPer];
#pragma unroll
        for (int k = 0; k < kPer; ++k) {
            const long long i = c * chunk + (long long)k * kBinThreads + threadIdx.x;
            bins[k] = i < n ? record_bins(records, record_bytes, i) : kInvisible;
        }
        if (use_smem) {
            for (int i = threadIdx.x; i < n_bins; i += kBinThreads) s_cnt[i] = 0u;
            __syncthreads();
#pragma unroll
            for (int k = 0; k < kPer; ++k)
                for_each_bin(bins[k], 0u, 0ull, nbx, [&](int b, int, uint32_t, unsigned long long) { atomicAdd(&s_cnt[b], 1u); });
            __syncthreads();
            for (int i = threadIdx.x; i < n_bins; i += kBinThreads) {
                const uint32_t cnt = s_cnt[i];
                if (cnt) {
                    s_base[i] = atomicAdd(&bin_cursor[i], cnt);
                    s_cnt[i] = 0u;
                }
            }
            __syncthreads();
#pragma unroll
            for (int k = 0; k < kPer; ++k) {
                const long long i = c * chunk + (long long)k * kBinThreads + threadIdx.x;
                const uint32_t id = (uint32_t)i;
                for_each_bin(bins[k], id, 0ull, nbx, [&](int b, int, uint32_t owner_id, unsigned long long) {
                    const uint32_t pos = s_base[b] + atomicAdd(&s_cnt[b], 1u);
                    list[bin_offset[b] + pos] = owner_id;
                });
            }
            __syncthreads();
        } else {
#pragma unroll
            for (int k = 0; k < kPer; ++k) {
                const long long i = c * chunk + (long long)k * kBinThreads + threadIdx.x;
                const uint32_t id = (uint32_t)i;
                for_each_bin(bins[k], id, 0ull, nbx, [&](int b, int, uint32_t owner_id, unsigned long long) {
                    const uint32_t pos = atomicAdd(&bin_cursor[b], 1u);
                    list[bin_offset[b] + pos] = owner_id;
                });
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// debug statistic: exact count of (splat, covered pixel-centre) pairs, one warp per splat
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
count_updates_kernel(const void *__restrict__ records, int record_bytes, long long n, CameraConst cam, WorkHead *head)
{
    const int lane = threadIdx.x & 31;
    const long long warp0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const long long n_warps = ((long long)gridDim.x * blockDim.x) >> 5;
    unsigned long long total = 0;
    for (long long i = warp0; i < n; i += n_warps) {
        if (record_bins(records, record_bytes, i) == kInvisible) continue;
        const float4 g = __ldg(reinterpret_cast<const float4 *>(reinterpret_cast<const char *>(records) +
                                                                (size_t)i * record_bytes));
        const float sx = g.x, sy = g.y, R = g.w;
        const int i0 = (int)fminf(fmaxf(ceilf((sx - R) - 0.5f), 0.0f), cam.Wf);
        const int i1 = (int)fmaxf(fminf(floorf((sx + R) - 0.5f), cam.Wf - 1.0f), -1.0f);
        const int j0 = (int)fminf(fmaxf(ceilf((sy - R) - 0.5f), 0.0f), cam.Hf);
        const int j1 = (int)fmaxf(fminf(floorf((sy + R) - 0.5f), cam.Hf - 1.0f), -1.0f);
        const double R2 = (double)R * (double)R;
        for (int j = j0 + lane; j <= j1; j += 32) {
            const double dy = ((double)j + 0.5) - (double)sy;
            const double h2 = R2 - dy * dy;
            if (h2 < 0.0) continue;
            const double h = sqrt(h2);
            int a = (int)ceil((double)sx - h - 0.5), b = (int)floor((double)sx + h - 0.5);
            a = max(a, i0); b = min(b, i1);
            if (b >= a) total += (unsigned long long)(b - a + 1);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) total += __shfl_xor_sync(0xffffffffu, total, o);
    if (lane == 0 && total) atomicAdd(&head->updates, total);
}

// ---------------------------------------------------------------------------------------------
// absorb mode: pairs emitted in depth order so that a stable sort by bin keeps that order
// ---------------------------------------------------------------------------------------------
__global__ void iota_kernel(uint32_t *v, long long n)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) v[i] = (uint32_t)i;
}

__global__ void __launch_bounds__(kBinThreads)
pair_counts_kernel(const void *__restrict__ records, int record_bytes, const uint32_t *__restrict__ sorted_ids,
                   long long n, uint32_t *__restrict__ pair_count)
{
    const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const uint32_t bins = record_bins(records, record_bytes, sorted_ids[k]);
    pair_count[k] = bins == kInvisible ? 0u : (uint32_t)unpack(bins).count();
}

__global__ void __launch_bounds__(kBinThreads)
expand_pairs_kernel(const void *__restrict__ records, int record_bytes, const uint32_t *__restrict__ sorted_ids,
                    long long n, const uint64_t *__restrict__ pair_offset, int nbx, uint32_t *__restrict__ pair_bin,
                    uint32_t *__restrict__ pair_id, const WorkHead *head)
{
    if (head->status != 0) return;
    const long long k0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long kw = k0 - (threadIdx.x & 31); kw < n; kw += stride) {
        const long long k = kw + (threadIdx.x & 31);
        uint32_t id = 0, bins = kInvisible;
        unsigned long long off = 0;
        if (k < n) {
            id = sorted_ids[k];
            bins = record_bins(records, record_bytes, id);
            off = pair_offset[k];
        }
        for_each_bin(bins, id, off, nbx, [&](int b, int local, uint32_t oid, unsigned long long ooff) {
            pair_bin[ooff + local] = (uint32_t)b;
            pair_id[ooff + local] = oid;
        });
    }
}

}  // namespace

int launch_finish_offsets(const uint32_t *bin_count, const uint64_t *bin_offset, int n_bins, uint64_t max_pairs,
                          uint32_t chunk, uint32_t *unit_prefix, WorkHead *head, cudaStream_t st)
{
    finish_offsets_kernel<<<1, 1024, 0, st>>>(bin_count, bin_offset, n_bins, (unsigned long long)max_pairs, chunk,
                                              unit_prefix, head);
    SPLOTCH_LAUNCH_CHECK();
    return 0;
}

int launch_scatter(const void *records, int record_bytes, int64_t n, const RenderConst &rc,
                   const uint64_t *bin_offset, uint32_t *bin_cursor, uint32_t *list, uint64_t max_pairs,
                   const WorkHead *head, cudaStream_t st)
{
    (void)max_pairs;
    if (n <= 0) return 0;
    const int n_bins = rc.nbx * rc.nby;
    const int use_smem = n_bins <= kSmemBinsMax ? 1 : 0;
    const size_t smem = use_smem ? (size_t)n_bins * 2 * sizeof(uint32_t) : 0;
    const long long chunk = (long long)kBinThreads * 4;
    long long blocks = (n + chunk - 1) / chunk;
    const long long cap = (long long)sm_count() * 6;
    if (blocks > cap) blocks = cap;
    scatter_kernel<<<(unsigned)blocks, kBinThreads, smem, st>>>(records, record_bytes, (long long)n, rc.nbx, n_bins,
                                                                bin_offset, bin_cursor, list, head, use_smem);
    SPLOTCH_LAUNCH_CHECK();
    return 0;
}

int launch_count_updates(const void *records, int record_bytes, int64_t n, const CameraConst &cam, float thr,
                         WorkHead *head, cudaStream_t st)
{
    (void)thr;
    if (n <= 0) return 0;
    count_updates_kernel<<<sm_count() * 8, 256, 0, st>>>(records, record_bytes, (long long)n, cam, head);
    SPLOTCH_LAUNCH_CHECK();
    return 0;
}

int launch_iota(uint32_t *v, int64_t n, cudaStream_t st)
{
    if (n <= 0) return 0;
    iota_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(v, (long long)n);
    SPLOTCH_LAUNCH_CHECK();
    return 0;
}

int launch_pair_counts(const void *records, int record_bytes, const uint32_t *sorted_ids, int64_t n,
                       uint32_t *pair_count, cudaStream_t st)
{
    if (n <= 0) return 0;
    pair_counts_kernel<<<(unsigned)((n + kBinThreads - 1) / kBinThreads), kBinThreads, 0, st>>>(
        records, record_bytes, sorted_ids, (long long)n, pair_count);
    SPLOTCH_LAUNCH_CHECK();
    return 0;
}

int launch_expand_pairs(const void *records, int record_bytes, const uint32_t *sorted_ids, int64_t n,
                        const uint64_t *pair_offset, const RenderConst &rc, uint32_t *pair_bin, uint32_t *pair_id,
                        uint64_t max_pairs, const WorkHead *head, cudaStream_t st)
{
    (void)max_pairs;
    if (n <= 0) return 0;
    long long blocks = (n + kBinThreads - 1) / kBinThreads;
    const long long cap = (long long)sm_count() * 8;
    if (blocks > cap) blocks = cap;
    expand_pairs_kernel<<<(unsigned)blocks, kBinThreads, 0, st>>>(records, record_bytes, sorted_ids, (long long)n,
                                                                  pair_offset, rc.nbx, pair_bin, pair_id, head);
    SPLOTCH_LAUNCH_CHECK();
    return 0;
}

}  // namespace splotch
