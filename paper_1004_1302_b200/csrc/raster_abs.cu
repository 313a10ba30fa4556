// raster_abs.cu -- K3 tile rasteriser of the absorb mode + the depth-ordered merge of unit partials.
// Front-to-back compositing of Eq. (1) of PAPER.md:73 integrated across one particle at a time
// (slab reading R10).  Same block geometry and producer pipeline as raster_add.cu.
#include "raster_common.cuh"

namespace splotch {

namespace {

constexpr int kRasThreads = 512;

// =============================================================================================
// absorb mode: front-to-back compositing, state per pixel = colour C and optical depth L
//   C_c += exp(-L_c) * E_c tau phi(A_c tau);  L_c += A_c tau;   phi(u) = (1 - exp(-u)) / u
// =============================================================================================
struct SmemAbs {
    float fac[2][kBatch][128];
    float4 amp0[2][kBatch];             // tau0, E_r, E_g, E_b
    float4 amp1[2][kBatch];             // A_r, A_g, A_b, max|A| * |tau0|
    unsigned char cls[2][kBatch][16];
    SplatAbs rec[2][kBatch];
    uint32_t ids[kChunkAbs];
    UnitInfo unit;
    uint32_t unit_id;
};

__device__ __forceinline__ float phi_small(float u)   // (1 - exp(-u)) / u for u < 0.25, error < 5e-8
{
    float p = -1.0f / 720.0f;
    p = fmaf(p, u, 1.0f / 120.0f);
    p = fmaf(p, u, -1.0f / 24.0f);
    p = fmaf(p, u, 1.0f / 6.0f);
    p = fmaf(p, u, -0.5f);
    return fmaf(p, u, 1.0f);
}

// one splat with every u = A tau below 0.25 on this lane's 8 pixels: phi of degree kDeg in tau
template <int kDeg>
__device__ __forceinline__ void small_u(const float2 (&tau)[4], const float (&E)[3], const float (&A)[3], float2 (&C)[3][4],
                                        float2 (&T)[3][4])
{
    float2 tau2[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) tau2[q] = __fmul2_rn(tau[q], tau[q]);
#pragma unroll
    for (int ch = 0; ch < 3; ++ch) {
        const float nA = -A[ch], c1 = 0.5f * nA, c2 = (1.0f / 3.0f) * nA * c1, c3 = 0.25f * nA * c2;
        const float c4 = 0.2f * nA * c3, c5 = (1.0f / 6.0f) * nA * c4;
        const float2 nA2 = make_float2(nA, nA), E2 = make_float2(E[ch], E[ch]), k1 = make_float2(c1, c1);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            // s = tau phi(A tau) = tau + tau^2 (c1 + c2 tau + ...):  z = T s,  C += z E,  T -= z A   (two pixels per instruction)
            float2 pl;
            if (kDeg == 1) pl = k1;
            else if (kDeg == 2) pl = __ffma2_rn(make_float2(c2, c2), tau[q], k1);
            else if (kDeg == 3) pl = __ffma2_rn(__ffma2_rn(make_float2(c3, c3), tau[q], make_float2(c2, c2)), tau[q], k1);
            else pl = __ffma2_rn(__ffma2_rn(__ffma2_rn(__ffma2_rn(make_float2(c5, c5), tau[q], make_float2(c4, c4)), tau[q],
                                                       make_float2(c3, c3)), tau[q], make_float2(c2, c2)), tau[q], k1);
            const float2 z = __fmul2_rn(T[ch][q], __ffma2_rn(pl, tau2[q], tau[q]));
            C[ch][q] = __ffma2_rn(z, E2, C[ch][q]);
            T[ch][q] = __ffma2_rn(z, nA2, T[ch][q]);
        }
    }
}

__global__ void __launch_bounds__(kRasThreads, 1)
raster_absorb_kernel(const SplatAbs *__restrict__ records, const uint32_t *__restrict__ list,
                     const uint64_t *__restrict__ bin_offset, const uint32_t *__restrict__ unit_prefix, int n_bins,
                     int nbx, int W, int H, float thr, float *__restrict__ partials, WorkHead *head)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    SmemAbs &sm = *reinterpret_cast<SmemAbs *>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int lx = (warp & 3) * 16 + (lane & 1) * 8;
    const int ly = (warp >> 2) * 16 + (lane >> 1);
    const uint32_t n_units = head->n_units;

    while (true) {
        if (tid == 0) {
            const uint32_t u = atomicAdd(&head->work_counter, 1u);
            sm.unit_id = u;
            if (u < n_units) {
                const int b = find_bin(unit_prefix, n_bins, u);
                const unsigned long long lo = bin_offset[b] + (unsigned long long)(u - unit_prefix[b]) * kChunkAbs;
                const unsigned long long rest = bin_offset[b + 1] - lo;
                sm.unit.bin = b;
                sm.unit.first = lo;
                sm.unit.count = (uint32_t)(rest < kChunkAbs ? rest : kChunkAbs);
            }
        }
        __syncthreads();
        const uint32_t unit = sm.unit_id;
        if (unit >= n_units) break;
        const int bin = sm.unit.bin;
        const uint32_t count = sm.unit.count;
        const unsigned long long first = sm.unit.first;
        const int px0 = (bin % nbx) * kBlockPx, py0 = (bin / nbx) * kBlockPx;

        for (uint32_t i = tid; i < count; i += kRasThreads) sm.ids[i] = __ldg(list + first + i);
        __syncthreads();
        const int n_batches = (int)((count + kBatch - 1) / kBatch);

        auto gather = [&](int b, int slot) {        // 96 threads copy 32 records of 48 B
            if (tid < 3 * kBatch) {
                const int s = tid / 3, q = tid - 3 * s;
                const uint32_t e = (uint32_t)b * kBatch + s;
                if (b < n_batches && e < count)
                    cp_async16(reinterpret_cast<char *>(&sm.rec[slot][s]) + q * 16,
                               reinterpret_cast<const char *>(records + sm.ids[e]) + q * 16);
            }
            cp_async_commit();
        };
        auto produce = [&](int b, int slot) {
            const int s = tid >> 4, part = tid & 15;
            const uint32_t e = (uint32_t)b * kBatch + s;
            if (b >= n_batches || e >= count) {
                sm.cls[slot][s][part] = 0;
                return;
            }
            const float4 g = *reinterpret_cast<const float4 *>(&sm.rec[slot][s]);
            const float x0 = (float)(px0 + part * 4) + 0.5f, y0 = (float)(py0 + part * 4) + 0.5f;
            float4 vx, vy;
            float t;
            t = (x0 - g.x) * g.z;          vx.x = ex2_approx(-t * t);
            t = (x0 + 1.0f - g.x) * g.z;   vx.y = ex2_approx(-t * t);
            t = (x0 + 2.0f - g.x) * g.z;   vx.z = ex2_approx(-t * t);
            t = (x0 + 3.0f - g.x) * g.z;   vx.w = ex2_approx(-t * t);
            t = (y0 - g.y) * g.z;          vy.x = ex2_approx(-t * t);
            t = (y0 + 1.0f - g.y) * g.z;   vy.y = ex2_approx(-t * t);
            t = (y0 + 2.0f - g.y) * g.z;   vy.z = ex2_approx(-t * t);
            t = (y0 + 3.0f - g.y) * g.z;   vy.w = ex2_approx(-t * t);
            *reinterpret_cast<float4 *>(&sm.fac[slot][s][part * 4]) = vx;
            *reinterpret_cast<float4 *>(&sm.fac[slot][s][64 + part * 4]) = vy;
            const int tpx = px0 + (part & 3) * 16, tpy = py0 + (part >> 2) * 16;
            sm.cls[slot][s][part] =
                (unsigned char)classify_tile(g.x, g.y, g.w, (float)tpx + 0.5f, (float)tpy + 0.5f, W, H, tpx, tpy);
            if (part == 0) {
                const float4 r1 = *(reinterpret_cast<const float4 *>(&sm.rec[slot][s]) + 1);   // tau0, E
                const float4 r2 = *(reinterpret_cast<const float4 *>(&sm.rec[slot][s]) + 2);   // A, bins
                sm.amp0[slot][s] = r1;
                // bound on |u| = |A tau| over the splat: absolute values, so that negative (unphysical, but accepted: reading
                // R20) A or I never select a polynomial tier whose truncation bound does not hold
                sm.amp1[slot][s] = make_float4(r2.x, r2.y, r2.z, fmaxf(fmaxf(fabsf(r2.x), fabsf(r2.y)), fabsf(r2.z)) * fabsf(r1.x));
            }
        };

        gather(0, 0);
        gather(1, 1);
        cp_async_wait_all();
        __syncthreads();
        produce(0, 0);
        __syncthreads();

        // state per pixel and channel: colour C and transmittance T = exp(-L).  T is carried as a product, so the common
        // case (every u = A tau of the splat below 0.25) needs no exponential at all: exp(-u) = 1 - u phi(u) by the
        // definition of phi, i.e.  q = T phi(u);  C += q E tau;  T -= q u   (the MUFU pipe runs at a quarter of the FMA rate
        // and used to bound this loop with one ex2 per update).
        float2 C[3][4], T[3][4];                    // [channel][pixel pair]: two neighbouring pixels share every packed instruction
#pragma unroll
        for (int ch = 0; ch < 3; ++ch)
#pragma unroll
            for (int q = 0; q < 4; ++q) { C[ch][q] = make_float2(0.0f, 0.0f); T[ch][q] = make_float2(1.0f, 1.0f); }

        for (int b = 0; b < n_batches; ++b) {
            const int slot = b & 1;
            gather(b + 2, slot);
            produce(b + 1, slot ^ 1);
            const unsigned char c = sm.cls[slot][lane][warp];
            unsigned any = __ballot_sync(0xffffffffu, c != 0);
            const unsigned inside = __ballot_sync(0xffffffffu, c == 2);
            while (any) {                                   // ascending s = depth order inside the batch
                const int s = __ffs(any) - 1;
                any &= any - 1;
                const float4 g0 = *reinterpret_cast<const float4 *>(&sm.fac[slot][s][lx]);
                const float4 g1 = *reinterpret_cast<const float4 *>(&sm.fac[slot][s][lx + 4]);
                const float gy = sm.fac[slot][s][64 + ly];
                const float4 a0 = sm.amp0[slot][s];
                const float4 a1 = sm.amp1[slot][s];
                const float ty = a0.x * gy;                 // tau0 * gy
                float gx[8] = { g0.x, g0.y, g0.z, g0.w, g1.x, g1.y, g1.z, g1.w };
                if (!((inside >> s) & 1u)) {
#pragma unroll
                    for (int k = 0; k < 8; ++k) gx[k] = (gx[k] * gy >= thr) ? gx[k] : 0.0f;
                }
                const float E[3] = { a0.y, a0.z, a0.w }, A[3] = { a1.x, a1.y, a1.z };
                if (a1.w < 0.25f) {
                    // Every u = A tau of this splat is small: no exponential.  phi(A tau) is a polynomial in tau whose
                    // coefficients c_m = (-A)^m / (m+1)! are per splat and channel;  q = T phi,  z = q tau,  C += z E,  T -= z A.
                    // The degree follows the bound a1.w on u so that the truncation error of phi stays below 2e-7 (the loop
                    // is bound by the FMA pipe, every dropped term is a dropped instruction per update).
                    float2 tau[4];
#pragma unroll
                    for (int q = 0; q < 4; ++q) tau[q] = __fmul2_rn(make_float2(ty, ty), make_float2(gx[2 * q], gx[2 * q + 1]));
                    if (a1.w < 1.1e-3f) small_u<1>(tau, E, A, C, T);
                    else if (a1.w < 0.017f) small_u<2>(tau, E, A, C, T);
                    else if (a1.w < 0.047f) small_u<3>(tau, E, A, C, T);
                    else small_u<5>(tau, E, A, C, T);
                } else {
#pragma unroll
                    for (int k = 0; k < 8; ++k) {
                        const float tau = ty * gx[k];
#pragma unroll
                        for (int ch = 0; ch < 3; ++ch) {
                            float &Ck = (k & 1) ? C[ch][k >> 1].y : C[ch][k >> 1].x;
                            float &Tk = (k & 1) ? T[ch][k >> 1].y : T[ch][k >> 1].x;
                            const float u = A[ch] * tau;
                            const float e = ex2_approx(-kLog2e * u);
                            const float phi = (fabsf(u) < 0.25f) ? phi_small(u) : __fdividef(1.0f - e, u);
                            Ck = fmaf(Tk * (E[ch] * tau), phi, Ck);
                            Tk *= e;
                        }
                    }
                }
            }
            cp_async_wait_all();
            __syncthreads();
        }

        // partial of this unit: planes C_r, C_g, C_b, T_r, T_g, T_b of 64x64 floats
        float *dst = partials + (size_t)unit * (6 * kBlockPx * kBlockPx) + (size_t)ly * kBlockPx + lx;
#pragma unroll
        for (int ch = 0; ch < 3; ++ch) {
            float4 *pc = reinterpret_cast<float4 *>(dst + (size_t)ch * kBlockPx * kBlockPx);
            float4 *pl = reinterpret_cast<float4 *>(dst + (size_t)(3 + ch) * kBlockPx * kBlockPx);
            pc[0] = make_float4(C[ch][0].x, C[ch][0].y, C[ch][1].x, C[ch][1].y);
            pc[1] = make_float4(C[ch][2].x, C[ch][2].y, C[ch][3].x, C[ch][3].y);
            pl[0] = make_float4(T[ch][0].x, T[ch][0].y, T[ch][1].x, T[ch][1].y);
            pl[1] = make_float4(T[ch][2].x, T[ch][2].y, T[ch][3].x, T[ch][3].y);
        }
        __syncthreads();
    }
}

// merge the unit partials of each block in depth order and write the image (every pixel)
__global__ void __launch_bounds__(256)
merge_absorb_kernel(const float *__restrict__ partials, const uint32_t *__restrict__ unit_prefix, int nbx, int W,
                    int H, float *__restrict__ out, const WorkHead *head)
{
    const int bin = blockIdx.x;
    const bool ok = head->status == 0;
    const uint32_t u0 = ok ? unit_prefix[bin] : 0u, u1 = ok ? unit_prefix[bin + 1] : 0u;
    const int px0 = (bin % nbx) * kBlockPx, py0 = (bin / nbx) * kBlockPx;
    for (int p = threadIdx.x; p < kBlockPx * kBlockPx; p += blockDim.x) {
        const int X = px0 + (p & (kBlockPx - 1)), Y = py0 + (p >> kBlockShift);
        if (X >= W || Y >= H) continue;
        float C[3] = { 0.f, 0.f, 0.f }, T[3] = { 1.f, 1.f, 1.f };
        for (uint32_t u = u0; u < u1; ++u) {
            const float *src = partials + (size_t)u * (6 * kBlockPx * kBlockPx) + p;
#pragma unroll
            for (int ch = 0; ch < 3; ++ch) {
                const float cu = __ldg(src + (size_t)ch * kBlockPx * kBlockPx);
                const float tu = __ldg(src + (size_t)(3 + ch) * kBlockPx * kBlockPx);
                C[ch] = fmaf(T[ch], cu, C[ch]);
                T[ch] *= tu;
            }
        }
        float *o = out + ((size_t)Y * W + X) * 3;
        o[0] = C[0]; o[1] = C[1]; o[2] = C[2];
    }
}

}  // namespace

int launch_raster_absorb(const SplatAbs *records, const uint32_t *list, const uint64_t *bin_offset,
                         const uint32_t *unit_prefix, const RenderConst &rc, const CameraConst &cam, float *partials,
                         WorkHead *head, cudaStream_t st)
{
    static SmemOptIn opt;
    if (int rc = smem_opt_in(opt, raster_absorb_kernel, (int)sizeof(SmemAbs))) return rc;
    raster_absorb_kernel<<<sm_count(), kRasThreads, sizeof(SmemAbs), st>>>(records, list, bin_offset, unit_prefix,
                                                                           rc.nbx * rc.nby, rc.nbx, cam.W, cam.H, rc.thr,
                                                                           partials, head);
    SPLOTCH_LAUNCH_CHECK();
    return 0;
}

int launch_merge_absorb(const float *partials, const uint32_t *unit_prefix, const RenderConst &rc,
                        const CameraConst &cam, float *out, const WorkHead *head, cudaStream_t st)
{
    merge_absorb_kernel<<<rc.nbx * rc.nby, 256, 0, st>>>(partials, unit_prefix, rc.nbx, cam.W, cam.H, out, head);
    SPLOTCH_LAUNCH_CHECK();
    return 0;
}

}  // namespace splotch
