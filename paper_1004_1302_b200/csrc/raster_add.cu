// raster_add.cu -- K3 tile rasteriser of the additive mode + K4 output map (steps a8, a9).
//
// One CTA (8 warps) owns a 64x64-pixel block of the screen for the duration of a work unit (a
// chunk of that block's splat list).  Each warp owns a 32x16 tile, each lane 8 consecutive
// pixels in each of 2 rows: 48 accumulators in REGISTERS.  Per batch of 32 splats the CTA
//   (i)   gathers the 32-byte splat records into shared memory with cp.async, double buffered;
//   (ii)  evaluates the separable Gaussian once per splat: exp(-d^2/s^2) = gx[i] * gy[j]; it
//         stores gx[64] and, per row j, the record (a_r gy[j], a_g gy[j], a_b gy[j], thr / gy[j]),
//         and classifies every (splat, tile) pair as outside / rim / inside the truncation circle;
//   (iii) lets every warp walk only the splats that touch its tile.  Inside tiles cost 3 FMA per
//         pixel update (acc_c += (a_c gy[j]) * gx[i]); rim tiles add one compare per pixel
//         (d^2 <= R^2  <=>  gx[i] >= thr / gy[j],  thr = exp(-f^2)) and predicate the FMAs.
// The block is added to the raw image once per unit with vector red.global.add: any summation
// order is legal when A = E.
#include "raster_common.cuh"

namespace splotch {

namespace {

constexpr int kRasThreads = 256;
constexpr int kWarps = kRasThreads / 32;
constexpr int kTileW = 32, kTileH = 16;         // warp tile; lane = 8 columns x 2 rows (rows r and r + 8)

// packed fp32x2 arithmetic (sm_100+): one FFMA2 issues two FMAs, halving the issue slots of the
// inner loop; the FMA pipe rate is unchanged (measured: 36 Tlane-FMA/s either way)
__device__ __forceinline__ unsigned long long pack2(float lo, float hi)
{
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(unsigned long long v, float &lo, float &hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ void fma2_acc(unsigned long long &c, unsigned long long a, unsigned long long b)
{
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(c) : "l"(a), "l"(b));      // c += a * b, in place
}

struct SmemAdd {
    float4 row[2][kBatch][kBlockPx];            // (a_r gy, a_g gy, a_b gy, thr / gy) per splat and block row
    float gx[2][kBatch][kBlockPx];              // per splat and block column
    SplatAdd rec[2][kBatch];
    uint32_t ids[kChunkAdd];
    unsigned char cls[2][kBatch][kWarps];
    UnitInfo unit;
    uint32_t unit_id;
};

__global__ void __launch_bounds__(kRasThreads, 2)
raster_additive_kernel(const SplatAdd *__restrict__ records, const uint32_t *__restrict__ list,
                       const uint64_t *__restrict__ bin_offset, const uint32_t *__restrict__ unit_prefix, int n_bins,
                       int nbx, int W, int H, float thr, float *__restrict__ S, WorkHead *head, int vec_ok)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    SmemAdd &sm = *reinterpret_cast<SmemAdd *>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int lx = (warp & 1) * kTileW + (lane & 3) * 8;     // first of this lane's 8 columns inside the block
    const int ly = (warp >> 1) * kTileH + (lane >> 2);       // this lane's rows inside the block: ly and ly + 8
    const uint32_t n_units = head->n_units;

    while (true) {
        if (tid == 0) {
            const uint32_t u = atomicAdd(&head->work_counter, 1u);
            sm.unit_id = u;
            if (u < n_units) {
                const int b = find_bin(unit_prefix, n_bins, u);
                const unsigned long long lo = bin_offset[b] + (unsigned long long)(u - unit_prefix[b]) * kChunkAdd;
                const unsigned long long rest = bin_offset[b + 1] - lo;
                sm.unit.bin = b;
                sm.unit.first = lo;
                sm.unit.count = (uint32_t)(rest < kChunkAdd ? rest : kChunkAdd);
            }
        }
        __syncthreads();
        if (sm.unit_id >= n_units) break;
        const int bin = sm.unit.bin;
        const uint32_t count = sm.unit.count;
        const unsigned long long first = sm.unit.first;
        const int px0 = (bin % nbx) * kBlockPx, py0 = (bin / nbx) * kBlockPx;

        for (uint32_t i = tid; i < count; i += kRasThreads) sm.ids[i] = __ldg(list + first + i);
        __syncthreads();
        const int n_batches = (int)((count + kBatch - 1) / kBatch);

        auto gather = [&](int b, int slot) {        // 64 threads copy 32 records of 32 B
            if (tid < 2 * kBatch) {
                const uint32_t e = (uint32_t)b * kBatch + (tid >> 1);
                if (b < n_batches && e < count)
                    cp_async16(reinterpret_cast<char *>(&sm.rec[slot][tid >> 1]) + (tid & 1) * 16,
                               reinterpret_cast<const char *>(records + sm.ids[e]) + (tid & 1) * 16);
            }
            cp_async_commit();
        };
        // 8 threads per splat: each 8 gx values, 8 row records and the class of one warp tile
        auto produce = [&](int b, int slot) {
            const int s = tid >> 3, part = tid & 7;
            const uint32_t e = (uint32_t)b * kBatch + s;
            if (b >= n_batches || e >= count) {
                sm.cls[slot][s][part] = 0;
                return;
            }
            const float4 g = *reinterpret_cast<const float4 *>(&sm.rec[slot][s]);        // sx, sy, c, R
            const float4 a = *(reinterpret_cast<const float4 *>(&sm.rec[slot][s]) + 1);  // a_r, a_g, a_b, bins
#pragma unroll
            for (int h = 0; h < 2; ++h) {           // columns part*4 + 32h .. +3
                const float x0 = (float)(px0 + part * 4 + 32 * h) + 0.5f;
                float4 v;
                float t;
                t = (x0 - g.x) * g.z;          v.x = ex2_approx(-t * t);
                t = (x0 + 1.0f - g.x) * g.z;   v.y = ex2_approx(-t * t);
                t = (x0 + 2.0f - g.x) * g.z;   v.z = ex2_approx(-t * t);
                t = (x0 + 3.0f - g.x) * g.z;   v.w = ex2_approx(-t * t);
                *reinterpret_cast<float4 *>(&sm.gx[slot][s][part * 4 + 32 * h]) = v;
            }
#pragma unroll
            for (int k = 0; k < 8; ++k) {           // rows part + 8k: conflict-free 128-bit stores
                const int j = part + 8 * k;
                const float t = ((float)(py0 + j) + 0.5f - g.y) * g.z;
                const float gy = ex2_approx(-t * t);
                sm.row[slot][s][j] = make_float4(a.x * gy, a.y * gy, a.z * gy, __fdividef(thr, gy));
            }
            const int tpx = px0 + (part & 1) * kTileW, tpy = py0 + (part >> 1) * kTileH;
            sm.cls[slot][s][part] = (unsigned char)classify_tile(g.x, g.y, g.w, (float)tpx + 0.5f, (float)tpy + 0.5f, W, H,
                                                                 tpx, tpy, (float)kTileW, (float)kTileH);
        };

        gather(0, 0);
        gather(1, 1);
        cp_async_wait_all();
        __syncthreads();
        produce(0, 0);
        __syncthreads();

        // accumulators: acc[h][c][q] = pixels (2q, 2q+1) of row h, channel c, packed as f32x2
        unsigned long long acc[2][3][4];
#pragma unroll
        for (int h = 0; h < 2; ++h)
#pragma unroll
            for (int c = 0; c < 3; ++c)
#pragma unroll
                for (int q = 0; q < 4; ++q) acc[h][c][q] = 0ull;

        for (int b = 0; b < n_batches; ++b) {
            const int slot = b & 1;
            gather(b + 2, slot);                 // rec[slot] held batch b, already turned into factors
            produce(b + 1, slot ^ 1);
            const unsigned char c = sm.cls[slot][lane][warp];
            unsigned m_in = __ballot_sync(0xffffffffu, c == 2);
            unsigned m_rim = __ballot_sync(0xffffffffu, c == 1);
            while (m_in) {                       // tiles entirely inside the circle: no coverage test
                const int s = __ffs(m_in) - 1;
                m_in &= m_in - 1;
                const float4 g0 = *reinterpret_cast<const float4 *>(&sm.gx[slot][s][lx]);
                const float4 g1 = *reinterpret_cast<const float4 *>(&sm.gx[slot][s][lx + 4]);
                const float4 r0 = sm.row[slot][s][ly];
                const float4 r1 = sm.row[slot][s][ly + 8];
                const unsigned long long gp[4] = { pack2(g0.x, g0.y), pack2(g0.z, g0.w), pack2(g1.x, g1.y), pack2(g1.z, g1.w) };
                const float w0[3] = { r0.x, r0.y, r0.z }, w1[3] = { r1.x, r1.y, r1.z };
#pragma unroll
                for (int ch = 0; ch < 3; ++ch) {
                    const unsigned long long b0 = pack2(w0[ch], w0[ch]), b1 = pack2(w1[ch], w1[ch]);
#pragma unroll
                    for (int q = 0; q < 4; ++q) {    // two pixels per FFMA2: half the issue slots of scalar FFMA
                        fma2_acc(acc[0][ch][q], gp[q], b0);
                        fma2_acc(acc[1][ch][q], gp[q], b1);
                    }
                }
            }
            while (m_rim) {                      // tiles cut by the circle: d^2 <= R^2 <=> gx >= thr / gy
                const int s = __ffs(m_rim) - 1;
                m_rim &= m_rim - 1;
                const float4 g0 = *reinterpret_cast<const float4 *>(&sm.gx[slot][s][lx]);
                const float4 g1 = *reinterpret_cast<const float4 *>(&sm.gx[slot][s][lx + 4]);
                const float4 r0 = sm.row[slot][s][ly];
                const float4 r1 = sm.row[slot][s][ly + 8];
                const float gx[8] = { g0.x, g0.y, g0.z, g0.w, g1.x, g1.y, g1.z, g1.w };
                const float w0[3] = { r0.x, r0.y, r0.z }, w1[3] = { r1.x, r1.y, r1.z };
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    float lo, hi;
#pragma unroll
                    for (int ch = 0; ch < 3; ++ch) {
                        unpack2(acc[0][ch][q], lo, hi);
                        if (gx[2 * q] >= r0.w) lo = fmaf(w0[ch], gx[2 * q], lo);
                        if (gx[2 * q + 1] >= r0.w) hi = fmaf(w0[ch], gx[2 * q + 1], hi);
                        acc[0][ch][q] = pack2(lo, hi);
                        unpack2(acc[1][ch][q], lo, hi);
                        if (gx[2 * q] >= r1.w) lo = fmaf(w1[ch], gx[2 * q], lo);
                        if (gx[2 * q + 1] >= r1.w) hi = fmaf(w1[ch], gx[2 * q + 1], hi);
                        acc[1][ch][q] = pack2(lo, hi);
                    }
                }
            }
            cp_async_wait_all();
            __syncthreads();
        }

        // write the block once: S += acc (RGB interleaved in the image)
        const int X0 = px0 + lx;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            float v[24];
#pragma unroll
            for (int ch = 0; ch < 3; ++ch)
#pragma unroll
                for (int q = 0; q < 4; ++q) unpack2(acc[h][ch][q], v[3 * (2 * q) + ch], v[3 * (2 * q + 1) + ch]);
            const int Y = py0 + ly + 8 * h;
            if (Y < H && X0 < W) {
                float *dst = S + ((size_t)Y * W + X0) * 3;
                if (vec_ok && X0 + 8 <= W) {
#pragma unroll
                    for (int k = 0; k < 6; ++k) red_add_v4(dst + 4 * k, v[4 * k], v[4 * k + 1], v[4 * k + 2], v[4 * k + 3]);
                } else {
#pragma unroll
                    for (int k = 0; k < 8; ++k) {
                        if (X0 + k < W) {
                            atomicAdd(dst + 3 * k + 0, v[3 * k + 0]);
                            atomicAdd(dst + 3 * k + 1, v[3 * k + 1]);
                            atomicAdd(dst + 3 * k + 2, v[3 * k + 2]);
                        }
                    }
                }
            }
        }
        __syncthreads();
    }
}

// K4: additive output map out = 1 - exp(-S) (reading R13; exact solution of Eq. 1 for A = E)
__global__ void __launch_bounds__(256)
normalize_kernel(const float *__restrict__ S, float *__restrict__ out, long long n, int vec_ok)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    const long long t0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (vec_ok) {
        const long long n4 = n >> 2;
        for (long long i = t0; i < n4; i += stride) {
            const float4 v = reinterpret_cast<const float4 *>(S)[i];
            reinterpret_cast<float4 *>(out)[i] = make_float4(-expm1f(-v.x), -expm1f(-v.y), -expm1f(-v.z), -expm1f(-v.w));
        }
        for (long long i = (n4 << 2) + t0; i < n; i += stride) out[i] = -expm1f(-S[i]);
    } else {
        for (long long i = t0; i < n; i += stride) out[i] = -expm1f(-S[i]);
    }
}

}  // namespace

int launch_raster_additive(const SplatAdd *records, const uint32_t *list, const uint64_t *bin_offset,
                           const uint32_t *unit_prefix, const RenderConst &rc, const CameraConst &cam, float *S,
                           WorkHead *head, cudaStream_t st)
{
    static bool attr_set = false;
    if (!attr_set) {
        SPLOTCH_CUDA_TRY(cudaFuncSetAttribute(raster_additive_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                              (int)sizeof(SmemAdd)));
        attr_set = true;
    }
    const int vec_ok = (cam.W % 4 == 0) && ((reinterpret_cast<uintptr_t>(S) & 15u) == 0);
    raster_additive_kernel<<<sm_count() * 2, kRasThreads, sizeof(SmemAdd), st>>>(
        records, list, bin_offset, unit_prefix, rc.nbx * rc.nby, rc.nbx, cam.W, cam.H, rc.thr, S, head, vec_ok);
    SPLOTCH_LAUNCH_CHECK();
    return 0;
}

int launch_normalize(const float *S, float *out, int64_t n_values, cudaStream_t st)
{
    if (n_values <= 0) return 0;
    const int vec_ok = ((reinterpret_cast<uintptr_t>(S) & 15u) == 0) && ((reinterpret_cast<uintptr_t>(out) & 15u) == 0);
    long long blocks = (n_values / 4 + 255) / 256 + 1;
    const long long cap = (long long)sm_count() * 8;
    if (blocks > cap) blocks = cap;
    normalize_kernel<<<(unsigned)blocks, 256, 0, st>>>(S, out, (long long)n_values, vec_ok);
    SPLOTCH_LAUNCH_CHECK();
    return 0;
}

}  // namespace splotch
