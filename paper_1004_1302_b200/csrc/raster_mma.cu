// raster_mma.cu -- K3t: the interior of big splats on the 5th-generation tensor cores (step a8).
//
// In the additive mode (A = E) a pixel of a 64x64 block receives
//     S_c(i, j) = sum_p  a_{p,c} * gx_p(i) * gy_p(j) * [pixel (i, j) inside the truncation circle of p],
// gx_p(i) = exp(-(i + 1/2 - sx_p)^2 / sigma_p^2), gy_p(j) likewise (the Gaussian of PAPER.md:69 is
// separable).  Wherever the indicator is 1 for a whole 32-pixel row segment this is a sum of rank-1
// updates, i.e. a dense contraction over the splat index p:
//     D_g[(c, i), j] = sum_p  A_g[(c, i), p] * B_g[p, j],
//     A_g[(c, i), p] = a_{p,c} gx_p(32 g + i)            (128 rows: 3 channels x 32 columns, 32 rows of padding)
//     B_g[p, j]      = gy_p(j) * handled(p, j, g)        (64 columns: the rows of the block)
// with g = 0, 1 the two column groups of the block.  handled(p, j, g) (raster_common.cuh) is 1 when
// the whole segment lies inside the circle; the remaining (rim) pixels are accumulated by the ALU
// kernel of raster_add.cu, which evaluates the same predicate bit for bit and skips what is done here.
//
// The contraction runs as tcgen05.mma kind::tf32 (M = 128, N = 64, K = 8) with A in tensor memory
// (written by the producing warps with tcgen05.st), B in shared memory (K-major, no swizzle) and the
// fp32 accumulators D_0, D_1 in tensor memory.  Precision: every operand is split into two numbers,
// v = hi + lo with hi a TF32 number (Veltkamp split with 2^13 + 1 in packed f32x2 arithmetic: hi has 11
// significant bits, lo = v - hi exactly; the tensor core ignores the 13 low bits of lo), and three
// products are accumulated (hi*hi + lo*hi + hi*lo), which leaves a relative error of ~2^-21 per term
// instead of 2^-11 -- fp32 class, inside the 1e-4 parity tolerance for any amplitude.  A batch of
// splats that are all faint (|a_c| <= kFaintAmp, see below) needs one product of rounded operands.
//
// One CTA (11 warps, 2 CTAs per SM, 256 of the 512 TMEM columns each) owns a block for up to
// kUnitsPerTicket consecutive work units of its splat list:
//   filter   : one thread per list entry (ids and records prefetched one and two chunks ahead) tests
//              seg_admit() and appends admitted splats to a ring queue in shared memory; entries whose
//              block is missed by the circle or entirely handled here get kListDone set in the list,
//              so the ALU kernel (which runs next) drops them without fetching the record;
//   batch    : 16 queued splats (32 when two consecutive faint batches are available).  Warps 0-2 / 4-6
//              (channel = warp & 3, group = warp >> 2) produce A into tensor memory, warps 3, 7, 8, 9 produce
//              B (32 block rows x 8 of every 16 splats each), warp 10 issues the MMAs of the batch (12 with
//              split operands, 4 or 8 for faint batches).  Two buffers; producers -> issuer through an mbarrier `full`,
//              issuer -> producers through tcgen05.commit on an mbarrier `free`; no CTA-wide barrier
//              inside a filter chunk, so the MMAs of batch b run while batch b + 1 is produced;
//   flush    : tcgen05.ld of D, transposed through shared memory, vector red.global.add into the raw
//              image (any summation order is legal when A = E).
#include <type_traits>

#include "raster_common.cuh"

namespace splotch {

namespace {

constexpr int kMmaThreads = 352;          // 11 warps
constexpr int kProducerWarps = 10;
constexpr int kIssuerWarp = 10;
constexpr int kMmaBatch = 16;             // splats per batch = two K = 8 steps
constexpr int kFilterThreads = 256;       // warps 0-7 filter
constexpr int kPerThread = 2;             // list entries per filter thread and pass
constexpr int kFilterChunk = kFilterThreads * kPerThread;   // list entries per filter pass
constexpr int kQueue = 1024;              // ring of admitted splats (power of two, > kFilterChunk + a batch)
// Ring of per-batch "bright" flags, indexed by the unwrapped batch number: TWICE the queue's batch count, so that the
// flags a filter pass sets (batches from the tail on, at most kFilterChunk + kMmaBatch - 1 entries ahead) can never be
// the ones the previous pass's consumed batches are still being cleared from (no barrier separates the two).
constexpr int kFlagRing = 2 * kQueue / kMmaBatch;
// The tensor core adds every K = 8 dot product into the fp32 accumulator with truncation: a relative deficit of
// ~2^-25 per MMA (measured on C3: -7e-5 with ~3700 MMAs per accumulator between flushes).  One unit of 4096 list
// entries (~900 MMAs) keeps it near 1e-5, a tenth of the parity tolerance, for ~4 % more flush work.
constexpr int kUnitsPerTicket = 1;
// A batch whose 16 splats all have |a_c| <= kFaintAmp runs as ONE TF32 product per K step (operands cut to TF32, no lo
// parts: a third of the MMAs, no operand split).  The cut is a DITHERED rounding (dither_tf32 below): a 13-bit offset that
// depends on the splat's queue position, the work unit and the thread, never on the value, is added to the bit pattern
// before the tensor core drops the 13 low bits.  Each operand is then unbiased (the expected value of the cut number is the
// number itself) whatever the input is, and the errors of different splats cancel by construction: N coincident
// splats, whose operand bits are all equal, do not repeat one rounding error N times (round-to-nearest does: up to
// 2 x 2^-11 relative per term, the same sign every time, 5.5 x the parity tolerance at S = 1.2;
// tests/test_gpu_parity.py::test_tensor_path_coincident_and_lattice_faint_splats).  Bounds: one term a w is off by less
// than 2^-9 a w <= 9.6e-7 (two operands, under one TF32 ulp = 2^-10 relative each); the error of an operand has variance
// f (1 - f) ulp^2 <= ulp^2 / 4 (f = the dropped fraction), so a pixel summing N terms is off by about
// 2^-10.5 sqrt(sum (a w)^2) <= 6.9e-4 sqrt(kFaintAmp S) = 1.5e-5 sqrt(S) rms at the very worst (every amplitude at the
// threshold, every fraction 1/2): 6 sigma stay inside 1e-4 max(1, S).  All configs have a_c ~ 1e-5.  Any brighter (or
// non-finite) splat in the batch keeps the three-product split (2^-21 per term, exact enough for any sum).
constexpr float kFaintAmp = 0.00048828125f;   // 2^-11
constexpr int kTmemCols = 256;
constexpr int kDCol = 0;                  // D_g at columns 64 g .. 64 g + 63
constexpr int kACol = 128;                // A at 128 + 64 buf + 32 g + 16 (hi | lo) + k

struct Range { int bin; uint32_t count; unsigned long long first; };

struct SmemMma {
    union {
        struct {
            float B[2][2][2][kMmaBatch * kBlockPx];          // [buf][g][hi | lo][((p / 4) * 64 + j) * 4 + p % 4]
            // queue of admitted splats, stored by PAIRS (2 q, 2 q + 1) for the packed f32x2 arithmetic
            float4 qG[kQueue / 2];                           // -sx0, -sx1, c0, c1
            float2 qAmp[3][kQueue / 2];                      // per channel: a0, a1
            float4 qBg[kQueue / 2];                          // -sy0, -sy1, c0, c1
            float4 qBm[kQueue / 2];                          // folded segment minima: group 0 (splat 0, 1), group 1 (splat 0, 1)
        } w;
        float stage[kBlockPx][kBlockPx * 3];                 // flush only
    };
    unsigned long long bar_full[2], bar_free[2];
    uint32_t bright[kFlagRing];                              // per queued batch: some splat above kFaintAmp (or not finite)
    uint32_t tmem_base;
    uint32_t q_tail;
    uint32_t ticket;
    int n_ranges;
    Range range[kUnitsPerTicket];
};

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_wait(unsigned long long *bar, uint32_t parity)
{
    const uint32_t a = smem_u32(bar);
    uint32_t done = 0;
    while (!done) {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(a), "r"(parity) : "memory");
    }
}

__device__ __forceinline__ void mbar_arrive(unsigned long long *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&r)[16])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};"
                 ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]),
                   "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
                 : "memory");
}

__device__ __forceinline__ void tmem_st8(uint32_t taddr, const uint32_t (&r)[8])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};"
                 ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7])
                 : "memory");
}

__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&v)[16])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
                   "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
                 : "r"(taddr));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

// D[tmem d] (+)= A[tmem a] (128 x 8 tf32) * B[smem descriptor] (8 x 64 tf32)
__device__ __forceinline__ void mma_tf32_ts(uint32_t d, uint32_t a, uint64_t bdesc, uint32_t idesc, uint32_t accumulate)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t}"
                 ::"r"(d), "r"(a), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}

// K-major, no swizzle: 16-byte units ((8, n), 2) : ((1, SBO), LBO); here [k / 4][j][k % 4] floats
__device__ __forceinline__ uint64_t b_descriptor(const float *b)
{
    const uint64_t lbo = (uint64_t)(kBlockPx * 16) >> 4, sbo = 128 >> 4;
    return (uint64_t)((smem_u32(b) >> 4) & 0x3FFFu) | (lbo << 16) | (sbo << 32) | (1ull << 46);
}

constexpr uint32_t kIdesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(kBlockPx >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);

__device__ __forceinline__ void queue_put(SmemMma &sm, uint32_t s, float sx, float sy, float c, float ar, float ag, float ab,
                                          float m0, float m1)
{
    const uint32_t q = s >> 1, h = s & 1u;
    float *G = reinterpret_cast<float *>(&sm.w.qG[q]), *Bg = reinterpret_cast<float *>(&sm.w.qBg[q]);
    float *Bm = reinterpret_cast<float *>(&sm.w.qBm[q]);
    G[h] = -sx;  G[2 + h] = c;
    Bg[h] = -sy; Bg[2 + h] = c;
    Bm[h] = m0;  Bm[2 + h] = m1;
    reinterpret_cast<float *>(&sm.w.qAmp[0][q])[h] = ar;
    reinterpret_cast<float *>(&sm.w.qAmp[1][q])[h] = ag;
    reinterpret_cast<float *>(&sm.w.qAmp[2][q])[h] = ab;
}

// v = hi + lo for both halves of a packed pair (Veltkamp split with 2^13 + 1: hi has 11 significant bits,
// i.e. it is a TF32 number; lo = v - hi is exact; the tensor core ignores the 13 low bits of lo)
// Dithered cut to TF32 of a finite value well inside the fp32 range: the tensor core ignores the 13 low bits of an
// operand, so adding t >> 19 (13 bits, uniform over the splats of a Weyl sequence t) to the bit pattern rounds the value up
// with probability (dropped fraction) and down otherwise.  t is never a function of v.
constexpr uint32_t kDitherStride = 0x9E3779B1u;      // 2^32 / golden ratio, odd
__device__ __forceinline__ uint32_t dither_tf32(float v, uint32_t t) { return __float_as_uint(v) + (t >> 19); }

__device__ __forceinline__ void split_tf32x2(float2 v, float2 &hi, float2 &lo)
{
    const float2 m1 = make_float2(-1.0f, -1.0f);
    const float2 gm = __fmul2_rn(v, make_float2(8193.0f, 8193.0f));
    const float2 d = __ffma2_rn(v, m1, gm);          // gm - v
    hi = __ffma2_rn(d, m1, gm);                      // gm - (gm - v)
    lo = __ffma2_rn(hi, m1, v);                      // v - hi
}

__global__ void __launch_bounds__(kMmaThreads, 2)
raster_additive_mma_kernel(const SplatAdd *__restrict__ records, uint32_t *__restrict__ list,
                           const uint64_t *__restrict__ bin_offset, const uint32_t *__restrict__ unit_prefix, int n_bins,
                           int nbx, int W, int H, float thr, float *__restrict__ S, WorkHead *head, int vec_ok, int tensor)
{
    if (tensor == 2 && head->tensor_on == 0u) return;     // auto: too little of the work is in full segments
    extern __shared__ __align__(128) unsigned char smem_raw[];
    SmemMma &sm = *reinterpret_cast<SmemMma *>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int quarter = warp & 3, grp = (warp >> 2) & 1;   // TMEM lane quarter (= channel for quarter < 3), column group
    const bool a_warp = warp < 8 && quarter < 3;
    const int b_rows = warp == 3 ? 0 : warp == 7 ? 1 : warp == 8 ? 0 : 1;     // which 32 block rows
    const int b_half = warp < 8 ? 0 : 1;                                      // which 8 splats of the batch
    const uint32_t n_units = head->n_units;

    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&sm.tmem_base)), "r"(kTmemCols));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    if (tid == 0) {
        for (int b = 0; b < 2; ++b) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(&sm.bar_full[b])), "r"(kProducerWarps));
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&sm.bar_free[b])));
        }
        asm volatile("fence.mbarrier_init.release.cluster;");
        sm.q_tail = 0;
    }
    if (tid < kFlagRing) sm.bright[tid] = 0u;
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    const uint32_t tmem = sm.tmem_base;
    const uint32_t lane_addr = tmem + ((uint32_t)(quarter * 32) << 16);
    if (warp == 3) {                                      // rows 96..127 of A are padding: zero them once
        uint32_t z[16];
#pragma unroll
        for (int k = 0; k < 16; ++k) z[k] = 0u;
#pragma unroll
        for (int c0 = 0; c0 < 128; c0 += 16) tmem_st16(lane_addr + kACol + c0, z);
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
        asm volatile("tcgen05.fence::before_thread_sync;");
    }

    // dither of the faint path: splat number p of this CTA's queue, in work unit (ticket) u, gets
    // t = (p + u k1) * kDitherStride + dither_salt in this thread.  Over the splats t walks the golden-ratio Weyl sequence,
    // whose discrepancy is about 2 / N: of N coincident operands the share that is rounded up differs from the dropped
    // fraction by ~2 / N, i.e. their SUM is off by about two TF32 ulps of one operand however large N is (a random dither
    // would give sqrt(N); a per-thread stride can be degenerate).  The per-thread salt only shifts the sequence, so that
    // the A and B producers, the channels and the pixels do not all round up for the same splats.
    uint32_t dither_salt = (uint32_t)tid * 0x85EBCA6Bu;
    dither_salt ^= dither_salt >> 15;
    dither_salt *= 0xC2B2AE35u;
    dither_salt ^= dither_salt >> 16;
    uint32_t dither_unit = 0u;

    uint32_t uses0 = 0u, uses1 = 0u;                      // batches issued into buffer 0 / 1
    uint32_t n_batches = 0;                               // batches so far (buffer = parity)
    uint32_t q_head = 0;
    bool fresh = true;                                    // D holds nothing yet: the first MMAs overwrite it
    int px0 = 0, py0 = 0;

    constexpr uint32_t kBBytes = kMmaBatch * kBlockPx * 4;             // one B operand (16 splats x 64 rows)
    constexpr uint64_t kStepUnits = (8 * kBlockPx * 4) >> 4;           // 16-byte units per K step (two K chunks)
    const uint64_t bdesc0 = b_descriptor(&sm.w.B[0][0][0][0]);

    // ---- nb batches of 16 queued splats; every role walks the same sequence ----
    // one batch, compiled twice: tag = true_type: three-product split; false_type: one product of rounded operands
    auto one_batch = [&](auto tag) {
        constexpr int mode = decltype(tag)::value;           // 0: 16 faint splats, 1: 16 splats split, 2: 32 faint splats
        constexpr bool bright = mode == 1;
        constexpr int n_splats = mode == 2 ? 2 * kMmaBatch : kMmaBatch;
        {
            const uint32_t buf = n_batches & 1u;
            const uint32_t uses = buf ? uses1 : uses0;
            if (warp == kIssuerWarp) {
                if (lane == 0) {
                    mbar_wait(&sm.bar_full[buf], uses & 1u);
                    asm volatile("tcgen05.fence::after_thread_sync;");
#pragma unroll
                    for (int g = 0; g < 2; ++g) {
                        const uint32_t d = tmem + kDCol + g * 64;
                        const uint32_t a0 = tmem + kACol + buf * 64 + g * 32;
                        const uint64_t b_hi = bdesc0 + (uint64_t)(((buf * 2 + g) * 2 + 0) * kBBytes >> 4);
                        const uint64_t b_lo = bdesc0 + (uint64_t)(((buf * 2 + g) * 2 + 1) * kBBytes >> 4);
                        mma_tf32_ts(d, a0, b_hi, kIdesc, fresh ? 0u : 1u);                 // K step 0: splats 0..7
                        if (bright) {
                            mma_tf32_ts(d, a0 + 16, b_hi, kIdesc, 1u);
                            mma_tf32_ts(d, a0, b_lo, kIdesc, 1u);
                        }
                        mma_tf32_ts(d, a0 + 8, b_hi + kStepUnits, kIdesc, 1u);             // K step 1: splats 8..15
                        if (bright) {
                            mma_tf32_ts(d, a0 + 24, b_hi + kStepUnits, kIdesc, 1u);
                            mma_tf32_ts(d, a0 + 8, b_lo + kStepUnits, kIdesc, 1u);
                        }
                        if (mode == 2) {                                                   // splats 16..31 sit where the lo parts would
                            mma_tf32_ts(d, a0 + 16, b_hi + 2 * kStepUnits, kIdesc, 1u);
                            mma_tf32_ts(d, a0 + 24, b_hi + 3 * kStepUnits, kIdesc, 1u);
                        }
                    }
                    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];"
                                 ::"r"(smem_u32(&sm.bar_free[buf])) : "memory");
                }
                __syncwarp();
            } else {
                if (uses > 0) mbar_wait(&sm.bar_free[buf], (uses - 1u) & 1u);     // the MMAs that read this buffer are done
                if (a_warp) {
                    asm volatile("tcgen05.fence::after_thread_sync;");
                    const float x = pixel_centre(px0 + kSegPx * grp + lane);
                    const float2 xx = make_float2(x, x);
                    const uint32_t qp = (q_head & (kQueue - 1)) >> 1;              // a batch never wraps: 16 | kQueue
                    const float4 *qg = &sm.w.qG[qp];
                    const float2 *qa = &sm.w.qAmp[quarter][qp];
                    // Every channel warp evaluates the column exponentials itself.  Sharing them through shared memory (the
                    // channel-0 warp computes, a named barrier, the other two read) removes two thirds of the MUFU work but
                    // puts the three warps in series: measured K3t 96 -> 105 ms on C3; the batch pipeline is latency-bound.
                    const uint32_t a = lane_addr + kACol + buf * 64 + grp * 32;
                    const uint32_t t0 = (q_head + dither_unit) * kDitherStride + dither_salt;   // splat i of the batch: t0 + i * kDitherStride
#pragma unroll
                    for (int half = 0; half < n_splats / 8; ++half) {              // 8 splats at a time: two splats per step, f32x2 arithmetic
                        uint32_t hi[8], lo[8];
#pragma unroll
                        for (int k = 0; k < 4; ++k) {
                            const float4 q = qg[4 * half + k];
                            float2 t = __fmul2_rn(__fadd2_rn(xx, make_float2(q.x, q.y)), make_float2(q.z, q.w));
                            t = __fmul2_rn(t, t);
                            const float2 v = __fmul2_rn(qa[4 * half + k], make_float2(ex2_approx(-t.x), ex2_approx(-t.y)));
                            if (bright) {
                                float2 h, l;
                                split_tf32x2(v, h, l);
                                hi[2 * k] = __float_as_uint(h.x);  hi[2 * k + 1] = __float_as_uint(h.y);
                                lo[2 * k] = __float_as_uint(l.x);  lo[2 * k + 1] = __float_as_uint(l.y);
                            } else {
                                hi[2 * k] = dither_tf32(v.x, t0 + (uint32_t)(8 * half + 2 * k) * kDitherStride);
                                hi[2 * k + 1] = dither_tf32(v.y, t0 + (uint32_t)(8 * half + 2 * k + 1) * kDitherStride);
                            }
                        }
                        tmem_st8(a + 8 * half, hi);                                // faint splats 16..31 land in the columns of the lo parts
                        if (bright) tmem_st8(a + 16 + 8 * half, lo);
                    }
                    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
                    asm volatile("tcgen05.fence::before_thread_sync;");
                } else {
                    const int j = b_rows * 32 + lane;
                    const float y = pixel_centre(py0 + j);
                    const float2 yy = make_float2(y, y);
                    const uint32_t qp = (q_head & (kQueue - 1)) >> 1;
                    const float4 *qg = &sm.w.qBg[qp], *qm = &sm.w.qBm[qp];
                    const uint32_t t0 = (q_head + dither_unit) * kDitherStride + dither_salt;
#pragma unroll
                    for (int qq = 0; qq < n_splats / 8; ++qq) {
                        const int q4 = 2 * b_half + (qq & 1) + 4 * (qq >> 1);     // group of 4 splats = 2 pairs; this warp's 8 of every 16
                        float2 bh[2][2], bl[2][2];                                // [group][pair]
#pragma unroll
                        for (int k = 0; k < 2; ++k) {
                            const float4 q = qg[2 * q4 + k], m = qm[2 * q4 + k];
                            // same operations, same roundings as gauss1d / seg_covered (raster_common.cuh), two splats at a time
                            float2 t = __fmul2_rn(__fadd2_rn(yy, make_float2(q.x, q.y)), make_float2(q.z, q.w));
                            t = __fmul2_rn(t, t);
                            const float2 gy = make_float2(ex2_approx(-t.x), ex2_approx(-t.y));
                            const float2 c0 = __fmul2_rn(make_float2(m.x, m.y), gy), c1 = __fmul2_rn(make_float2(m.z, m.w), gy);
                            const float2 f0 = make_float2(c0.x >= thr ? 1.0f : 0.0f, c0.y >= thr ? 1.0f : 0.0f);
                            const float2 f1 = make_float2(c1.x >= thr ? 1.0f : 0.0f, c1.y >= thr ? 1.0f : 0.0f);
                            float2 h, l = make_float2(0.0f, 0.0f);
                            if (bright) split_tf32x2(gy, h, l);
                            else h = make_float2(__uint_as_float(dither_tf32(gy.x, t0 + (uint32_t)(4 * q4 + 2 * k) * kDitherStride)),
                                                 __uint_as_float(dither_tf32(gy.y, t0 + (uint32_t)(4 * q4 + 2 * k + 1) * kDitherStride)));
                            bh[0][k] = __fmul2_rn(h, f0);  bl[0][k] = __fmul2_rn(l, f0);
                            bh[1][k] = __fmul2_rn(h, f1);  bl[1][k] = __fmul2_rn(l, f1);
                        }
                        const int at = (q4 * kBlockPx + j) * 4;
#pragma unroll
                        for (int g = 0; g < 2; ++g) {
                            float *Bg = &sm.w.B[buf][g][0][0];             // hi operand, then the lo operand (or faint splats 16..31)
                            *reinterpret_cast<float4 *>(Bg + at) = make_float4(bh[g][0].x, bh[g][0].y, bh[g][1].x, bh[g][1].y);
                            if (bright)
                                *reinterpret_cast<float4 *>(Bg + kMmaBatch * kBlockPx + at) = make_float4(bl[g][0].x, bl[g][0].y, bl[g][1].x, bl[g][1].y);
                        }
                    }
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&sm.bar_full[buf]);
            }
            if (buf) uses1 += 1u; else uses0 += 1u;
            n_batches += 1u;
            q_head += n_splats;
            fresh = false;
        }
    };
    auto process_batches = [&](uint32_t nb) {
        for (uint32_t it = 0; it < nb;) {
            // the flags are set by the filter and stable while the batches run; the choice is uniform over the CTA
            const uint32_t at = q_head & (kQueue - 1), fb = q_head / kMmaBatch;
            if (sm.bright[fb & (kFlagRing - 1)] != 0u) {
                one_batch(std::integral_constant<int, 1>{});
                it += 1;
            } else if (it + 1 < nb && at + 2 * kMmaBatch <= kQueue && sm.bright[(fb + 1) & (kFlagRing - 1)] == 0u) {
                one_batch(std::integral_constant<int, 2>{});      // two faint batches as one: half the hand-offs per splat
                it += 2;
            } else {
                one_batch(std::integral_constant<int, 0>{});
                it += 1;
            }
        }
    };

    // ---- pad the queue to a whole batch and run it (all threads; ends every range) ----
    auto drain = [&]() {
        __syncthreads();
        const uint32_t tail = sm.q_tail;
        const uint32_t rem = tail - q_head;
        if (rem == 0) return;
        const uint32_t pad = kMmaBatch - rem;
        if ((uint32_t)tid < pad) {
            const uint32_t s = (tail + tid) & (kQueue - 1);
            queue_put(sm, s, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, kSegNever, kSegNever);
        }
        if (tid == 0) sm.q_tail = tail + pad;
        __syncthreads();
        const uint32_t slot = (q_head / kMmaBatch) & (kFlagRing - 1);
        process_batches(1u);
        __syncthreads();                                  // every role has read the batch's flag
        if (tid == 0) sm.bright[slot] = 0u;
    };

    // ---- wait for every MMA, add D to the raw image ----
    auto flush = [&]() {
        if (fresh) return;
        if (uses0 > 0) mbar_wait(&sm.bar_free[0], (uses0 - 1u) & 1u);
        if (uses1 > 0) mbar_wait(&sm.bar_free[1], (uses1 - 1u) & 1u);
        asm volatile("tcgen05.fence::after_thread_sync;");
        __syncthreads();                                  // B and the queue are dead: the stage may overwrite them
        if (a_warp) {
#pragma unroll
            for (int c0 = 0; c0 < kBlockPx; c0 += 16) {
                uint32_t v[16];
                tmem_ld16(lane_addr + kDCol + grp * 64 + c0, v);
#pragma unroll
                for (int q = 0; q < 16; ++q) sm.stage[c0 + q][(kSegPx * grp + lane) * 3 + quarter] = __uint_as_float(v[q]);
            }
            asm volatile("tcgen05.fence::before_thread_sync;");
        }
        __syncthreads();
        const bool vec = vec_ok && px0 + kBlockPx <= W;
        for (int idx = tid; idx < kBlockPx * (kBlockPx * 3 / 4); idx += kMmaThreads) {
            const int row = idx / (kBlockPx * 3 / 4), q4 = idx % (kBlockPx * 3 / 4);
            const int Y = py0 + row;
            if (Y >= H) continue;
            const float4 v = *reinterpret_cast<const float4 *>(&sm.stage[row][4 * q4]);
            float *dst = S + ((size_t)Y * W + px0) * 3;
            if (vec) {
                red_add_v4(dst + 4 * q4, v.x, v.y, v.z, v.w);
            } else {
                const float e[4] = { v.x, v.y, v.z, v.w };
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const int f = 4 * q4 + k;
                    if (px0 + f / 3 < W) atomicAdd(dst + f, e[k]);
                }
            }
        }
        __syncthreads();
        fresh = true;
    };

    while (true) {
        // ---- ticket: kUnitsPerTicket consecutive work units = at most that many list ranges, one per bin ----
        __syncthreads();
        if (tid == 0) {
            const uint32_t t = atomicAdd(&head->mma_counter, 1u);
            sm.ticket = t;
            int nr = 0;
            uint32_t u = t * kUnitsPerTicket;
            const uint32_t u1 = min(u + (uint32_t)kUnitsPerTicket, n_units);
            while (u < u1) {
                const int b = find_bin(unit_prefix, n_bins, u);
                const unsigned long long lo = bin_offset[b] + (unsigned long long)(u - unit_prefix[b]) * kChunkAdd;
                const unsigned long long want = (unsigned long long)(u1 - u) * kChunkAdd, rest = bin_offset[b + 1] - lo;
                const unsigned long long len = rest < want ? rest : want;
                sm.range[nr].bin = b;
                sm.range[nr].first = lo;
                sm.range[nr].count = (uint32_t)len;
                ++nr;
                u += (uint32_t)((len + kChunkAdd - 1) / kChunkAdd);
            }
            sm.n_ranges = nr;
        }
        __syncthreads();
        if (sm.ticket * (uint32_t)kUnitsPerTicket >= n_units) break;
        dither_unit = sm.ticket * 0x632BE5ABu;
        const int n_ranges = sm.n_ranges;
        for (int r = 0; r < n_ranges; ++r) {
            const int bin = sm.range[r].bin;
            const uint32_t count = sm.range[r].count;
            const unsigned long long first = sm.range[r].first;
            px0 = (bin % nbx) * kBlockPx;
            py0 = (bin / nbx) * kBlockPx;
            // software-pipelined filter: ids two chunks ahead, records one chunk ahead; kPerThread entries per thread
            const bool filt = tid < kFilterThreads;
            uint32_t id_cur[kPerThread], id_next[kPerThread];
            float4 geo[kPerThread];
#pragma unroll
            for (int e = 0; e < kPerThread; ++e) {
                const uint32_t i = (uint32_t)(e * kFilterThreads + tid);
                id_cur[e] = id_next[e] = 0u;
                geo[e] = make_float4(0.f, 0.f, 0.f, 0.f);
                if (filt) {
                    if (i < count) id_cur[e] = list[first + i];
                    if (i + kFilterChunk < count) id_next[e] = list[first + kFilterChunk + i];
                    if (i < count) geo[e] = __ldg(reinterpret_cast<const float4 *>(records + id_cur[e]));
                }
            }
            for (uint32_t off = 0; off < count; off += kFilterChunk) {
                if (filt) {
#pragma unroll
                    for (int e = 0; e < kPerThread; ++e) {
                        const uint32_t i = off + (uint32_t)(e * kFilterThreads + tid);
                        const float4 g = geo[e];
                        const uint32_t id = id_cur[e];
                        const bool have = i < count;
                        // prefetch for the next two chunks before the batches of this one
                        id_cur[e] = id_next[e];
                        if (i + kFilterChunk < count) geo[e] = __ldg(reinterpret_cast<const float4 *>(records + id_cur[e]));
                        if (i + 2 * kFilterChunk < count) id_next[e] = list[first + i + 2 * kFilterChunk];
                        bool adm = false;
                        float m0 = kSegNever, m1 = kSegNever;
                        bool done = false;                     // nothing left for the ALU kernel in this block
                        if (have) {                            // the circle misses the block (bins are pixel boxes: B-rules)
                            const float x_lo = pixel_centre(px0), x_hi = pixel_centre(px0 + kBlockPx - 1);
                            const float y_lo = pixel_centre(py0), y_hi = pixel_centre(py0 + kBlockPx - 1);
                            const float nx = fmaxf(fmaxf(x_lo - g.x, g.x - x_hi), 0.0f), ny = fmaxf(fmaxf(y_lo - g.y, g.y - y_hi), 0.0f);
                            done = __fmaf_rn(nx, nx, __fmul_rn(ny, ny)) > __fmul_rn(__fmul_rn(g.w, g.w), 1.00001f);
                        }
                        if (have && g.w >= 15.5f) {
                            const float e0 = gauss1d(pixel_centre(px0), g.x, g.z);
                            const float e1 = gauss1d(pixel_centre(px0 + kSegPx - 1), g.x, g.z);
                            const float e2 = gauss1d(pixel_centre(px0 + kSegPx), g.x, g.z);
                            const float e3 = gauss1d(pixel_centre(px0 + 2 * kSegPx - 1), g.x, g.z);
                            m0 = fminf(e0, e1);
                            m1 = fminf(e2, e3);
                            const unsigned a = seg_admit(g.y, g.z, g.w, thr, py0, m0, m1);
                            const unsigned f = seg_full(a, g.y, g.z, thr, py0, m0, m1);
                            adm = a != 0u;
                            done = done || f == 3u;
                            m0 = (f & 1u) ? kSegAlways : (a & 1u) ? m0 : kSegNever;
                            m1 = (f & 2u) ? kSegAlways : (a & 2u) ? m1 : kSegNever;
                        }
                        if (done) list[first + i] = id | kListDone;
                        const unsigned bal = __ballot_sync(0xffffffffu, adm);
                        uint32_t base = 0;
                        if (lane == 0 && bal) base = atomicAdd(&sm.q_tail, (uint32_t)__popc(bal));
                        base = __shfl_sync(0xffffffffu, base, 0);
                        if (adm) {
                            const uint32_t pos = base + __popc(bal & ((1u << lane) - 1u));   // unwrapped queue position
                            const uint32_t s = pos & (kQueue - 1);
                            const float4 amp = __ldg(reinterpret_cast<const float4 *>(records + id) + 1);
                            queue_put(sm, s, g.x, g.y, g.z, amp.x, amp.y, amp.z, m0, m1);
                            // written so that a NaN amplitude counts as bright (fmaxf would drop it): the split path carries
                            // non-finite values through like the ALU kernel, the integer TF32 rounding does not
                            if (!(fabsf(amp.x) <= kFaintAmp && fabsf(amp.y) <= kFaintAmp && fabsf(amp.z) <= kFaintAmp))
                                atomicOr(&sm.bright[(pos / kMmaBatch) & (kFlagRing - 1)], 1u);
                        }
                    }
                }
                __syncthreads();
                const uint32_t tail = sm.q_tail;
                const uint32_t head0 = q_head;
                process_batches((tail - q_head) / kMmaBatch);
                __syncthreads();                          // every warp is done reading the queue before it is refilled
                for (uint32_t b = head0 / kMmaBatch + tid; b < q_head / kMmaBatch; b += kMmaThreads)
                    sm.bright[b & (kFlagRing - 1)] = 0u;    // the next pass sets flags from the tail on: other slots (kFlagRing)
            }
            drain();
            flush();
        }
    }

    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(kTmemCols));
}

// Statistic for bench.py (not part of a render): the number of pixel updates inside the image that the
// tensor-core kernel performs, i.e. 32 x (handled row segments), evaluated with the same predicates.
// One warp per splat; lanes share the rows of every block of the splat's bin box.
__global__ void __launch_bounds__(256)
count_tensor_updates_kernel(const SplatAdd *__restrict__ records, long long n, int W, int H, float thr, WorkHead *head)
{
    const int lane = threadIdx.x & 31;
    const long long warp0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const long long n_warps = ((long long)gridDim.x * blockDim.x) >> 5;
    unsigned long long total = 0;
    for (long long i = warp0; i < n; i += n_warps) {
        const float4 g = __ldg(reinterpret_cast<const float4 *>(records + i));
        const uint32_t bins = __ldg(reinterpret_cast<const uint32_t *>(records + i) + 7);
        if (bins == kInvisible || !(g.w >= 15.5f)) continue;
        const int bx0 = bins & 255, bx1 = (bins >> 8) & 255, by0 = (bins >> 16) & 255, by1 = bins >> 24;
        for (int by = by0; by <= by1; ++by)
            for (int bx = bx0; bx <= bx1; ++bx) {
                const int px0 = bx * kBlockPx, py0 = by * kBlockPx;
                const float m0 = fminf(gauss1d(pixel_centre(px0), g.x, g.z), gauss1d(pixel_centre(px0 + kSegPx - 1), g.x, g.z));
                const float m1 = fminf(gauss1d(pixel_centre(px0 + kSegPx), g.x, g.z),
                                       gauss1d(pixel_centre(px0 + 2 * kSegPx - 1), g.x, g.z));
                const unsigned adm = seg_admit(g.y, g.z, g.w, thr, py0, m0, m1);
                if (adm == 0u) continue;
                const unsigned full = seg_full(adm, g.y, g.z, thr, py0, m0, m1);
                const int w0 = min(max(W - px0, 0), kSegPx), w1 = min(max(W - px0 - kSegPx, 0), kSegPx);
                for (int j = lane; j < kBlockPx; j += 32) {
                    if (py0 + j >= H) continue;
                    const unsigned hd = seg_handled(adm, full, m0, m1, gauss1d(pixel_centre(py0 + j), g.y, g.z), thr);
                    total += (unsigned long long)(((hd & 1u) ? w0 : 0) + ((hd & 2u) ? w1 : 0));
                }
            }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) total += __shfl_xor_sync(0xffffffffu, total, o);
    if (lane == 0 && total) atomicAdd(&head->updates_tensor, total);
}

}  // namespace

int launch_count_tensor_updates(const SplatAdd *records, int64_t n, const RenderConst &rc, const CameraConst &cam,
                                WorkHead *head, cudaStream_t st)
{
    if (n <= 0) return 0;
    count_tensor_updates_kernel<<<sm_count() * 8, 256, 0, st>>>(records, (long long)n, cam.W, cam.H, rc.thr, head);
    SPLOTCH_LAUNCH_CHECK();
    return 0;
}

int launch_raster_additive_mma(const SplatAdd *records, uint32_t *list, const uint64_t *bin_offset,
                               const uint32_t *unit_prefix, const RenderConst &rc, const CameraConst &cam, float *S,
                               WorkHead *head, int tensor, cudaStream_t st)
{
    static SmemOptIn opt;
    if (int rc = smem_opt_in(opt, raster_additive_mma_kernel, (int)sizeof(SmemMma))) return rc;
    const int vec_ok = (cam.W % 4 == 0) && ((reinterpret_cast<uintptr_t>(S) & 15u) == 0);
    raster_additive_mma_kernel<<<sm_count() * 2, kMmaThreads, sizeof(SmemMma), st>>>(
        records, list, bin_offset, unit_prefix, rc.nbx * rc.nby, rc.nbx, cam.W, cam.H, rc.thr, S, head, vec_ok, tensor);
    SPLOTCH_LAUNCH_CHECK();
    return 0;
}

}  // namespace splotch
