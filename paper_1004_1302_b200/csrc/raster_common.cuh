// raster_common.cuh -- helpers shared by the two tile rasterisers (additive, absorb).
#pragma once
#include "common.cuh"

namespace splotch {

namespace {

constexpr int kBatch = 32;
constexpr float kLog2e = 1.4426950408889634f;

__device__ __forceinline__ float ex2_approx(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__device__ __forceinline__ float rcp_approx(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gmem_src)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

__device__ __forceinline__ void red_add_v4(float *addr, float a, float b, float c, float d)
{
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(a), "f"(b), "f"(c), "f"(d)
                 : "memory");
}

// class of a tw x th tile of pixel centres against the truncation circle: 0 outside, 1 rim, 2 inside.
// The margins make the classification conservative: a tile is only called inside/outside when
// every pixel of it is, whatever the rounding of the per-pixel test.
__device__ __forceinline__ int classify_tile(float sx, float sy, float R, float x_lo, float y_lo, int W, int H,
                                             int px0, int py0, float tw = 16.0f, float th = 16.0f)
{
    if (px0 >= W || py0 >= H) return 0;
    const float x_hi = x_lo + (tw - 1.0f), y_hi = y_lo + (th - 1.0f);
    const float nx = fmaxf(fmaxf(x_lo - sx, sx - x_hi), 0.0f), ny = fmaxf(fmaxf(y_lo - sy, sy - y_hi), 0.0f);
    const float fx = fmaxf(sx - x_lo, x_hi - sx), fy = fmaxf(sy - y_lo, y_hi - sy);
    const float R2 = __fmul_rn(R, R);
    if (__fmaf_rn(nx, nx, __fmul_rn(ny, ny)) > __fmul_rn(R2, 1.00001f)) return 0;
    if (__fmaf_rn(fx, fx, __fmul_rn(fy, fy)) < __fmul_rn(R2, 0.99999f)) return 2;
    return 1;
}

// ---------------------------------------------------------------------------------------------
// Split of the additive work between the tensor-core kernel (raster_mma.cu) and the ALU kernel
// (raster_add.cu).  A 64x64 block has two column groups g (32 pixels each); the row segment
// (row j, group g) of a splat is HANDLED by the tensor-core kernel when the splat is admitted
// for g and both end pixels of the segment pass the coverage test (the circle is convex, so
// every pixel between them passes too).  Both kernels evaluate the functions below on the same
// record words; every operation is an explicitly rounded intrinsic or a single hardware
// approximation, so the two kernels take bit-identical decisions and every covered pixel is
// accumulated exactly once.
// ---------------------------------------------------------------------------------------------
constexpr int kSegPx = 32;

__device__ __forceinline__ float pixel_centre(int p) { return __fadd_rn((float)p, 0.5f); }

// exp(-((x - s) / sigma)^2) with c = sqrt(log2 e) / sigma
__device__ __forceinline__ float gauss1d(float x, float s, float c)
{
    const float t = __fmul_rn(__fsub_rn(x, s), c);
    return ex2_approx(-__fmul_rn(t, t));
}

// per-pixel coverage threshold of the ALU kernel on gx for a row whose factor is gy:  gx >= thr / gy
__device__ __forceinline__ float row_threshold(float thr, float gy) { return __fdividef(thr, gy); }

// segment test: m = min of gx over the two end pixels of the segment, gy = factor of the row
__device__ __forceinline__ bool seg_covered(float m, float gy, float thr) { return __fmul_rn(m, gy) >= thr; }

// bit g set: the splat has (at the block row nearest to its centre) a fully covered segment in group g
__device__ __forceinline__ unsigned seg_admit(float sy, float c, float R, float thr, int py0, float m0, float m1)
{
    if (!(R >= 15.5f)) return 0u;                      // half chord of a 32-pixel segment
    const float jf = fminf(fmaxf(floorf(__fsub_rn(sy, (float)py0)), 0.0f), (float)(kBlockPx - 1));
    const float gy = gauss1d(__fadd_rn(__fadd_rn((float)py0, jf), 0.5f), sy, c);
    return (seg_covered(m0, gy, thr) ? 1u : 0u) | (seg_covered(m1, gy, thr) ? 2u : 0u);
}

// bit g set: every row of the block is covered in group g (tested on the two extreme rows; the
// circle is convex).  Part of the DEFINITION of "handled", so both kernels agree whatever the rounding.
__device__ __forceinline__ unsigned seg_full(unsigned adm, float sy, float c, float thr, int py0, float m0, float m1)
{
    if (adm == 0u) return 0u;
    const float gy = fminf(gauss1d(pixel_centre(py0), sy, c), gauss1d(pixel_centre(py0 + kBlockPx - 1), sy, c));
    return adm & ((seg_covered(m0, gy, thr) ? 1u : 0u) | (seg_covered(m1, gy, thr) ? 2u : 0u));
}

// bit g set: row segment (row with factor gy, group g) is accumulated by the tensor-core kernel
__device__ __forceinline__ unsigned seg_handled(unsigned adm, unsigned full, float m0, float m1, float gy, float thr)
{
    return adm & (full | (seg_covered(m0, gy, thr) ? 1u : 0u) | (seg_covered(m1, gy, thr) ? 2u : 0u));
}

// The tensor-core kernel folds (adm, full) into the segment minima it queues: -1 never passes
// seg_covered, kSegAlways always does (gy >= thr on the extreme rows of a full group).
constexpr float kSegNever = -1.0f, kSegAlways = 1.0e30f;

struct UnitInfo {
    int bin;
    uint32_t count;
    unsigned long long first;
};

// largest b with unit_prefix[b] <= unit (bins without units share their prefix with the next one)
__device__ __forceinline__ int find_bin(const uint32_t *__restrict__ unit_prefix, int n_bins, uint32_t unit)
{
    int lo = 0, hi = n_bins;            // invariant: prefix[lo] <= unit < prefix[hi]
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (__ldg(unit_prefix + mid) <= unit) lo = mid; else hi = mid;
    }
    return lo;
}

}  // namespace
}  // namespace splotch
