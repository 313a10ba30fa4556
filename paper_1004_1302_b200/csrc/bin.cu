// bin.cu -- K2: binning (steps a4-a6): offsets -> work units, scatter of splat ids into per-bin
// lists with big splats duplicated into every bin their pixel box touches (B-rules), and the
// depth-ordered pair expansion of the absorb mode.  PAPER.md:105 "determining screen areas
// affected by individual particles"; the paper's own load-balancing device is the
// "split particles" pass of PAPER.md:109, which this replaces.
#include "common.cuh"

namespace splotch {

namespace {

constexpr int kBinThreads = 256;

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
// scatter (a6): list[bin_offset[b] + k] = particle index, any order inside a bin (additive mode).
// A CTA takes a chunk of 1024 consecutive particles (each warp 128 of them) and
//   1. counts the chunk's pairs per bin with the difference-array trick of K1 (four shared atomics per
//      splat, then a 2-D prefix sum over the (nbx + 1) x (nby + 1) grid in shared memory),
//   2. reserves one range per touched bin with a single global atomic,
//   3. enumerates the pairs DENSELY: every warp lays the boxes of its 128 splats end to end (warp scan of
//      the box sizes) and lane l takes pairs l, l + 32, ...: owner by binary search in the 128 starts,
//      bin by one reciprocal multiplication.  All 32 lanes work whatever the box sizes are (the first
//      version let the owning lane walk small boxes and the warp walk big ones: 6 warp instructions per
//      pair on C3, most of them idle lanes and integer divisions).
// The packed bin boxes come from the compact array K1 writes beside the records (4 B per particle).
// ---------------------------------------------------------------------------------------------
constexpr int kScatWarps = kBinThreads / 32;
constexpr int kScatPerLane = 4;                                  // splats per lane and chunk
constexpr int kScatPerWarp = 32 * kScatPerLane;                  // 128
constexpr int kScatChunk = kBinThreads * kScatPerLane;           // 1024
constexpr int kScatDiffMax = 4608;                               // (nbx + 1)(nby + 1) entries in shared memory: up to 4096^2 images

template <bool kSmem>
__global__ void __launch_bounds__(kBinThreads)
scatter_kernel(const uint32_t *__restrict__ binsw, long long n, int nbx, int nby,
               const uint64_t *__restrict__ bin_offset, uint32_t *__restrict__ bin_cursor,
               uint32_t *__restrict__ list, const WorkHead *head)
{
    extern __shared__ uint32_t s_mem[];
    if (head->status != 0) return;
    const int stride = nbx + 1, n_diff = kSmem ? stride * (nby + 1) : 0;
    int *s_cnt = reinterpret_cast<int *>(s_mem);                 // difference grid -> counts -> running cursor of the chunk
    uint32_t *s_base = s_mem + n_diff;                           // start of the chunk's range inside the bin's list
    uint32_t *s_start = s_mem + 2 * n_diff;                      // [warp][129]: starts of the warp's boxes in its pair space
    uint32_t *s_box = s_start + kScatWarps * (kScatPerWarp + 4); // [warp][128]: packed bin boxes
    int *s_bb = reinterpret_cast<int *>(s_box + kScatWarps * kScatPerWarp);   // bounding box of the chunk on the grid
    if (threadIdx.x == 0) { s_bb[0] = s_bb[1] = 1 << 20; s_bb[2] = s_bb[3] = -1; }
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t *w_start = s_start + warp * (kScatPerWarp + 4), *w_box = s_box + warp * kScatPerWarp;
    const long long n_chunks = (n + kScatChunk - 1) / kScatChunk;
    for (long long c = blockIdx.x; c < n_chunks; c += gridDim.x) {
        const long long first = c * kScatChunk + (long long)warp * kScatPerWarp;
        uint32_t bins[kScatPerLane];
#pragma unroll
        for (int k = 0; k < kScatPerLane; ++k) {
            const long long i = first + k * 32 + lane;
            bins[k] = i < n ? __ldg(binsw + i) : kInvisible;
        }
        if (kSmem) {
            // bounding box of the chunk's bin boxes: all sweeps below touch only that part of the grid (a chunk of
            // spatially coherent particles covers a few bins of a 33 x 33 .. 65 x 65 grid)
            int mnx = 1 << 20, mny = 1 << 20, mxx = -1, mxy = -1;
#pragma unroll
            for (int k = 0; k < kScatPerLane; ++k) {
                if (bins[k] == kInvisible) continue;
                const BinBox bb = unpack(bins[k]);
                mnx = min(mnx, bb.x0); mny = min(mny, bb.y0); mxx = max(mxx, bb.x1 + 1); mxy = max(mxy, bb.y1 + 1);
            }
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) {
                mnx = min(mnx, __shfl_xor_sync(0xffffffffu, mnx, d)); mny = min(mny, __shfl_xor_sync(0xffffffffu, mny, d));
                mxx = max(mxx, __shfl_xor_sync(0xffffffffu, mxx, d)); mxy = max(mxy, __shfl_xor_sync(0xffffffffu, mxy, d));
            }
            if (lane == 0 && mxx >= 0) {
                atomicMin(&s_bb[0], mnx); atomicMin(&s_bb[1], mny); atomicMax(&s_bb[2], mxx); atomicMax(&s_bb[3], mxy);
            }
            __syncthreads();
            const int rx0 = s_bb[0], ry0 = s_bb[1], rx1 = s_bb[2], ry1 = s_bb[3];     // grid region [rx0, rx1] x [ry0, ry1], inclusive
            for (int y = ry0 + warp; y <= ry1; y += kScatWarps)          // (an empty chunk has ry1 < ry0)
                for (int x = rx0 + lane; x <= rx1; x += 32) s_cnt[y * stride + x] = 0;
            __syncthreads();
            if (threadIdx.x == 0) { s_bb[0] = s_bb[1] = 1 << 20; s_bb[2] = s_bb[3] = -1; }    // for the next chunk
#pragma unroll
            for (int k = 0; k < kScatPerLane; ++k) {
                if (bins[k] == kInvisible) continue;
                const BinBox bb = unpack(bins[k]);
                atomicAdd(&s_cnt[bb.y0 * stride + bb.x0], 1);
                atomicAdd(&s_cnt[bb.y0 * stride + bb.x1 + 1], -1);
                atomicAdd(&s_cnt[(bb.y1 + 1) * stride + bb.x0], -1);
                atomicAdd(&s_cnt[(bb.y1 + 1) * stride + bb.x1 + 1], 1);
            }
            __syncthreads();
            for (int y = ry0 + warp; y < ry1; y += kScatWarps) {    // prefix sums along x (row ry1 holds only closing impulses)
                int carry = 0;
                for (int x0 = rx0; x0 < rx1; x0 += 32) {
                    const int x = x0 + lane;
                    int v = x < rx1 ? s_cnt[y * stride + x] : 0;
#pragma unroll
                    for (int d = 1; d < 32; d <<= 1) {
                        const int u = __shfl_up_sync(0xffffffffu, v, d);
                        if (lane >= d) v += u;
                    }
                    v += carry;
                    if (x < rx1) s_cnt[y * stride + x] = v;
                    carry = __shfl_sync(0xffffffffu, v, 31);
                }
            }
            __syncthreads();
            for (int x = rx0 + threadIdx.x; x < rx1; x += kBinThreads) {   // prefix sums along y
                int run = 0;
                for (int y = ry0; y < ry1; ++y) {
                    run += s_cnt[y * stride + x];
                    s_cnt[y * stride + x] = run;
                }
            }
            __syncthreads();
            for (int y = ry0 + warp; y <= ry1; y += kScatWarps)
                for (int x = rx0 + lane; x <= rx1; x += 32) {
                    const int cnt = (x < rx1 && y < ry1) ? s_cnt[y * stride + x] : 0;
                    if (cnt > 0) s_base[y * stride + x] = atomicAdd(&bin_cursor[y * nbx + x], (uint32_t)cnt);
                    s_cnt[y * stride + x] = 0;
                }
            __syncthreads();
        }
        // the warp's pair space: boxes of splat o = 32 k + lane laid end to end
        uint32_t run = 0;
#pragma unroll
        for (int k = 0; k < kScatPerLane; ++k) {
            const uint32_t cnt = bins[k] == kInvisible ? 0u : (uint32_t)unpack(bins[k]).count();
            uint32_t inc = cnt;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const uint32_t u = __shfl_up_sync(0xffffffffu, inc, d);
                if (lane >= d) inc += u;
            }
            w_start[k * 32 + lane] = run + inc - cnt;
            w_box[k * 32 + lane] = bins[k];
            run += __shfl_sync(0xffffffffu, inc, 31);
        }
        const uint32_t total = run;
        __syncwarp();
        // pair t of the warp: owner = largest o with start[o] <= t (empty boxes share a start with their successor), bin by
        // one reciprocal multiplication: boxes have at most 256 x 256 bins, so (local + 1/2) / cw is at least 1/512 away
        // from an integer and the approximate reciprocal (1 ulp) cannot move the quotient across one
        auto locate = [&](uint32_t t, int &owner, int &bx, int &y) {
            int lo = 0, hi = kScatPerWarp;
#pragma unroll
            for (int it = 0; (1 << it) < kScatPerWarp; ++it) {
                const int mid = (lo + hi) >> 1;
                if (w_start[mid] <= t) lo = mid; else hi = mid;
            }
            const uint32_t local = t - w_start[lo];
            const BinBox bb = unpack(w_box[lo]);
            const int cw = bb.width();
            const int by = (int)(((float)local + 0.5f) * __fdividef(1.0f, (float)cw));
            owner = lo;
            bx = bb.x0 + (int)local - by * cw;
            y = bb.y0 + by;
        };
        if (total > 3u * kScatPerWarp) {
            // big boxes: the 32 pairs of a step lie in (mostly) different bins; one atomic and one store per pair
            auto emit = [&](int o, int bx, int y) {
                uint32_t pos;
                if (kSmem) pos = s_base[y * stride + bx] + (uint32_t)atomicAdd(&s_cnt[y * stride + bx], 1);
                else pos = atomicAdd(&bin_cursor[y * nbx + bx], 1u);
                list[__ldg(bin_offset + y * nbx + bx) + pos] = (uint32_t)(first + o);
            };
            uint32_t t = lane;
            for (; t + 32 < total; t += 64) {                    // two pairs per lane and step: two independent search chains
                int o0, bx0, y0, o1, bx1, y1;
                locate(t, o0, bx0, y0);
                locate(t + 32, o1, bx1, y1);
                emit(o0, bx0, y0);
                emit(o1, bx1, y1);
            }
            if (t < total) {
                int o, bx, y;
                locate(t, o, bx, y);
                emit(o, bx, y);
            }
        } else {
            // small boxes: neighbouring particles hit the same bins; lanes with the same bin in a step share one atomic and
            // get consecutive positions, so their stores coalesce
            for (uint32_t t0 = 0; t0 < total; t0 += 32) {        // warp-uniform trip count
                const uint32_t t = t0 + lane;
                const bool valid = t < total;
                int o = 0, bx = 0, y = 0;
                if (valid) locate(t, o, bx, y);
                const int key = valid ? y * stride + bx : -1 - lane;
                const unsigned peers = __match_any_sync(0xffffffffu, key);
                const int leader = __ffs(peers) - 1;
                uint32_t base = 0;
                if (valid && lane == leader) {
                    const uint32_t cnt = (uint32_t)__popc(peers);
                    if (kSmem) base = s_base[key] + (uint32_t)atomicAdd(&s_cnt[key], (int)cnt);
                    else base = atomicAdd(&bin_cursor[y * nbx + bx], cnt);
                }
                base = __shfl_sync(0xffffffffu, base, leader);
                if (valid)
                    list[__ldg(bin_offset + y * nbx + bx) + base + (uint32_t)__popc(peers & ((1u << lane) - 1u))] = (uint32_t)(first + o);
            }
        }
        __syncthreads();
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

int launch_scatter(const uint32_t *binsw, int64_t n, const RenderConst &rc,
                   const uint64_t *bin_offset, uint32_t *bin_cursor, uint32_t *list, uint64_t max_pairs,
                   const WorkHead *head, cudaStream_t st)
{
    (void)max_pairs;
    if (n <= 0) return 0;
    const int n_diff = (rc.nbx + 1) * (rc.nby + 1);
    const bool use_smem = n_diff <= kScatDiffMax;
    const size_t smem = ((use_smem ? 2 * (size_t)n_diff : 0) + kScatWarps * (kScatPerWarp + 4) + kScatWarps * kScatPerWarp + 4) *
                        sizeof(uint32_t);
    long long blocks = (n + kScatChunk - 1) / kScatChunk;
    const long long cap = (long long)sm_count() * 8;
    if (blocks > cap) blocks = cap;
    if (use_smem)
        scatter_kernel<true><<<(unsigned)blocks, kBinThreads, smem, st>>>(binsw, (long long)n, rc.nbx, rc.nby, bin_offset,
                                                                          bin_cursor, list, head);
    else
        scatter_kernel<false><<<(unsigned)blocks, kBinThreads, smem, st>>>(binsw, (long long)n, rc.nbx, rc.nby, bin_offset,
                                                                           bin_cursor, list, head);
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
