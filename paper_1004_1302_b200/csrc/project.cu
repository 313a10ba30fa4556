// project.cu -- K1: fused transform / cull / colour kernel (steps a1-a3 of the hot path) with the
// bin count (a4) folded in as a 2-D difference array.
//
// Reads the particle SoA (x, y, z, r, I, colval [, type]) with 128-bit coalesced loads, four
// consecutive particles per thread, and writes one 32-byte (additive) or 48-byte (absorb) splat
// record per particle.  The projection follows the canonical fp32 sequence of DESIGN.md
// ("Canonical sequence") with explicitly rounded intrinsics so that every integer derived from
// it (visible set, pixel box, bin membership, depth key) is reproducible bit for bit.
// PAPER.md:105 "transformation into screen coordinates, assigning of colours".
#include "common.cuh"

namespace splotch {

namespace {

constexpr int kProjThreads = 256;
constexpr int kSmemBinsMax = 8192;       // entries of the difference grid kept in shared memory when they fit
constexpr float kSqrtPi = 1.7724538509055160273f;
constexpr float kSqrtLog2e = 1.2011224087864498f;

struct Projected {
    float sx, sy, ss, R, zc;
    int i0, i1, j0, j1;
    bool visible;
};

__device__ __forceinline__ bool finite_f(float v) { return fabsf(v) <= 3.402823466e38f; }

// canonical fp32 projection: one correctly rounded operation per line
__device__ __forceinline__ Projected project_one(float x, float y, float z, float r, float I, float cv, int type,
                                                 const CameraConst &cam, const RenderConst &rc)
{
    Projected o;
    o.sx = o.sy = o.ss = o.R = o.zc = 0.0f;
    o.i0 = o.i1 = o.j0 = o.j1 = 0;
    o.visible = false;
    if (!(finite_f(x) && finite_f(y) && finite_f(z) && finite_f(r) && finite_f(I) && finite_f(cv))) return o;
    if (!(r > 0.0f) || type >= rc.n_types) return o;
    const float dx = __fsub_rn(x, cam.ex), dy = __fsub_rn(y, cam.ey), dz = __fsub_rn(z, cam.ez);
    const float xc = __fmaf_rn(dz, cam.rz, __fmaf_rn(dy, cam.ry, __fmul_rn(dx, cam.rx)));
    const float yc = __fmaf_rn(dz, cam.uz, __fmaf_rn(dy, cam.uy, __fmul_rn(dx, cam.ux)));
    const float zc = __fmaf_rn(dz, cam.fz, __fmaf_rn(dy, cam.fy, __fmul_rn(dx, cam.fx)));
    if (!(zc > rc.z_near)) return o;
    const float q = __fdiv_rn(cam.F, zc);
    const float sx = __fmaf_rn(xc, q, cam.cx);
    const float sy = __fmaf_rn(-yc, q, cam.cy);
    const float ss = __fmul_rn(r, q);
    const float R = __fmul_rn(rc.support_f, ss);
    if (!(ss > 0.0f) || !finite_f(R)) return o;
    const float i0f = fminf(fmaxf(ceilf(__fsub_rn(__fsub_rn(sx, R), 0.5f)), 0.0f), cam.Wf);
    const float i1f = fmaxf(fminf(floorf(__fsub_rn(__fadd_rn(sx, R), 0.5f)), __fsub_rn(cam.Wf, 1.0f)), -1.0f);
    const float j0f = fminf(fmaxf(ceilf(__fsub_rn(__fsub_rn(sy, R), 0.5f)), 0.0f), cam.Hf);
    const float j1f = fmaxf(fminf(floorf(__fsub_rn(__fadd_rn(sy, R), 0.5f)), __fsub_rn(cam.Hf, 1.0f)), -1.0f);
    if (!(i0f <= i1f) || !(j0f <= j1f)) return o;
    o.sx = sx; o.sy = sy; o.ss = ss; o.R = R; o.zc = zc;
    o.i0 = (int)i0f; o.i1 = (int)i1f; o.j0 = (int)j0f; o.j1 = (int)j1f;
    o.visible = true;
    return o;
}

// piece-wise linear colour table (reading R7)
__device__ __forceinline__ void lut_sample(const float *__restrict__ tab, int n_entries, int type, float cv,
                                           float scale, float &cr, float &cg, float &cb)
{
    const float c = fminf(fmaxf(cv, 0.0f), 1.0f);
    const float u = c * (float)(n_entries - 1);
    int k = (int)floorf(u);
    k = min(k, n_entries - 2);
    const float t = u - (float)k;
    const float *e0 = tab + ((size_t)type * n_entries + k) * 3;
    const float a0 = __ldg(e0), a1 = __ldg(e0 + 1), a2 = __ldg(e0 + 2);
    const float b0 = __ldg(e0 + 3), b1 = __ldg(e0 + 4), b2 = __ldg(e0 + 5);
    cr = scale * fmaf(t, b0 - a0, a0);
    cg = scale * fmaf(t, b1 - a1, a1);
    cb = scale * fmaf(t, b2 - a2, a2);
}

__device__ __forceinline__ uint32_t pack_bins(const Projected &o, int shift)
{
    return (uint32_t)(o.i0 >> shift) | ((uint32_t)(o.i1 >> shift) << 8) | ((uint32_t)(o.j0 >> shift) << 16) |
           ((uint32_t)(o.j1 >> shift) << 24);
}

// Bin counts (a4, B-rules: every bin of the splat's bin box gets one count) as a 2-D DIFFERENCE ARRAY: a box
// (x0..x1) x (y0..y1) is four signed unit impulses at its corners on a (nbx + 1) x (nby + 1) grid, and the 2-D prefix
// sum of the grid (bins_from_diff_kernel) is the count of every bin.  Four atomics per splat whatever the size of its
// box (the first version walked the box: 9.4 atomics per splat on C3, and a screen-filling splat cost 1024).
__device__ __forceinline__ void count_box(uint32_t bins, int *hist, int stride)
{
    const int x0 = bins & 255, x1 = (bins >> 8) & 255, y0 = (bins >> 16) & 255, y1 = (bins >> 24) & 255;
    atomicAdd(&hist[y0 * stride + x0], 1);
    atomicAdd(&hist[y0 * stride + x1 + 1], -1);
    atomicAdd(&hist[(y1 + 1) * stride + x0], -1);
    atomicAdd(&hist[(y1 + 1) * stride + x1 + 1], 1);
}

template <bool kAbsorb>
__global__ void __launch_bounds__(kProjThreads, 4)
project_kernel(ParticlePtrs p, long long n, CameraConst cam, RenderConst rc, const float *__restrict__ lutE,
               const float *__restrict__ lutA, void *__restrict__ records, int *__restrict__ bin_diff,
               uint32_t *__restrict__ binsw, uint32_t *__restrict__ zkeys, WorkHead *head, DebugProjectOut dbg,
               int has_dbg, int vec_ok, int smem_hist)
{
    extern __shared__ int s_hist[];
    __shared__ unsigned int s_visible;
    __shared__ float s_area[2];
    const int diff_stride = rc.nbx + 1, n_diff = diff_stride * (rc.nby + 1);
    if (smem_hist)
        for (int i = threadIdx.x; i < n_diff; i += blockDim.x) s_hist[i] = 0;
    if (threadIdx.x == 0) { s_visible = 0u; s_area[0] = s_area[1] = 0.0f; }
    __syncthreads();
    int *hist = smem_hist ? s_hist : bin_diff;

    unsigned int my_visible = 0;
    float my_area = 0.0f, my_tensor = 0.0f;     // heuristic for WorkHead::tensor_on, not part of the result
    const long long groups = (n + 3) / 4;
    const long long stride = (long long)gridDim.x * blockDim.x;
    // warp-uniform trip count: every lane of a warp runs the same number of iterations
    const long long first = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long warp_first = first - (threadIdx.x & 31);
    for (long long g0 = warp_first; g0 < groups; g0 += stride) {
        const long long g = g0 + (threadIdx.x & 31);
        const long long base = g * 4;
        float xv[4], yv[4], zv[4], rv[4], Iv[4], cvv[4];
        int tv[4];
        const bool full = g < groups && base + 4 <= n;
        if (full && vec_ok) {
            const float4 a = __ldg(reinterpret_cast<const float4 *>(p.x) + g);
            const float4 b = __ldg(reinterpret_cast<const float4 *>(p.y) + g);
            const float4 c = __ldg(reinterpret_cast<const float4 *>(p.z) + g);
            const float4 d = __ldg(reinterpret_cast<const float4 *>(p.r) + g);
            const float4 e = __ldg(reinterpret_cast<const float4 *>(p.I) + g);
            const float4 f = p.colval ? __ldg(reinterpret_cast<const float4 *>(p.colval) + g) : make_float4(0.f, 0.f, 0.f, 0.f);
            xv[0] = a.x; xv[1] = a.y; xv[2] = a.z; xv[3] = a.w;
            yv[0] = b.x; yv[1] = b.y; yv[2] = b.z; yv[3] = b.w;
            zv[0] = c.x; zv[1] = c.y; zv[2] = c.z; zv[3] = c.w;
            rv[0] = d.x; rv[1] = d.y; rv[2] = d.z; rv[3] = d.w;
            Iv[0] = e.x; Iv[1] = e.y; Iv[2] = e.z; Iv[3] = e.w;
            cvv[0] = f.x; cvv[1] = f.y; cvv[2] = f.z; cvv[3] = f.w;
            if (p.type) {
                const uchar4 t = __ldg(reinterpret_cast<const uchar4 *>(p.type) + g);
                tv[0] = t.x; tv[1] = t.y; tv[2] = t.z; tv[3] = t.w;
            } else {
                tv[0] = tv[1] = tv[2] = tv[3] = 0;
            }
        } else {
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const long long i = base + k;
                const bool in = g < groups && i < n;
                xv[k] = in ? __ldg(p.x + i) : 0.0f;
                yv[k] = in ? __ldg(p.y + i) : 0.0f;
                zv[k] = in ? __ldg(p.z + i) : 0.0f;
                rv[k] = in ? __ldg(p.r + i) : -1.0f;      // r <= 0: culled
                Iv[k] = in ? __ldg(p.I + i) : 0.0f;
                cvv[k] = (in && p.colval) ? __ldg(p.colval + i) : 0.0f;
                tv[k] = (in && p.type) ? (int)__ldg(p.type + i) : 0;
            }
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const long long i = base + k;
            const bool in = g < groups && i < n;
            float v0 = 0.0f, v1 = 0.0f, v2 = 0.0f;
            if (p.vr) {                          // vector colouring (reading R19): a non-finite component culls the particle
                if (in) { v0 = __ldg(p.vr + i); v1 = __ldg(p.vg + i); v2 = __ldg(p.vb + i); }
                cvv[k] = (finite_f(v0) && finite_f(v1) && finite_f(v2)) ? 0.0f : __int_as_float(0x7fc00000);
            }
            const Projected o = project_one(xv[k], yv[k], zv[k], rv[k], Iv[k], cvv[k], tv[k], cam, rc);
            const uint32_t bins = o.visible ? pack_bins(o, rc.bin_shift) : kInvisible;
            if (in) {
                my_visible += o.visible ? 1u : 0u;
                if (o.visible) {
                    const float area = 0.78539816f * (float)(o.i1 - o.i0 + 1) * (float)(o.j1 - o.j0 + 1);
                    my_area += area;
                    if (o.R >= 15.5f) my_tensor += fmaxf(area - 64.0f * o.R, 0.0f);   // minus a 16-pixel band on both edges of every row
                }
                const float tau0 = (Iv[k] * rv[k]) * kSqrtPi;
                const float cw = o.visible ? kSqrtLog2e / o.ss : 0.0f;
                float er = 0.f, eg = 0.f, eb = 0.f;
                if (o.visible) {
                    if (p.vr) { const float sc = rc.brightness[tv[k]]; er = sc * v0; eg = sc * v1; eb = sc * v2; }
                    else lut_sample(lutE, rc.n_entries, tv[k], cvv[k], rc.brightness[tv[k]], er, eg, eb);
                }
                if (!kAbsorb) {
                    float4 *rec = reinterpret_cast<float4 *>(reinterpret_cast<SplatAdd *>(records) + i);
                    rec[0] = make_float4(o.sx, o.sy, cw, o.R);
                    rec[1] = make_float4(er * tau0, eg * tau0, eb * tau0, __uint_as_float(bins));
                } else {
                    float ar = 0.f, ag = 0.f, ab = 0.f;
                    if (o.visible) {
                        if (p.vr) { const float sc = rc.abs_brightness[tv[k]]; ar = sc * v0; ag = sc * v1; ab = sc * v2; }
                        else lut_sample(lutA, rc.n_entries, tv[k], cvv[k], rc.abs_brightness[tv[k]], ar, ag, ab);
                    }
                    float4 *rec = reinterpret_cast<float4 *>(reinterpret_cast<SplatAbs *>(records) + i);
                    rec[0] = make_float4(o.sx, o.sy, cw, o.R);
                    rec[1] = make_float4(o.visible ? tau0 : 0.0f, er, eg, eb);
                    rec[2] = make_float4(ar, ag, ab, __uint_as_float(bins));
                }
                if (binsw) binsw[i] = bins;          // the packed bin box once more as a compact array: the scatter reads 4 B, not a 32-B record
                if (zkeys) zkeys[i] = o.visible ? __float_as_uint(o.zc) : 0xFFFFFFFFu;
                if (has_dbg) {
                    if (dbg.sx) dbg.sx[i] = o.sx;
                    if (dbg.sy) dbg.sy[i] = o.sy;
                    if (dbg.sigma_s) dbg.sigma_s[i] = o.ss;
                    if (dbg.R) dbg.R[i] = o.R;
                    if (dbg.zkey) dbg.zkey[i] = o.visible ? __float_as_uint(o.zc) : 0u;
                    if (dbg.pix_bbox) {
                        reinterpret_cast<int4 *>(dbg.pix_bbox)[i] = make_int4(o.i0, o.i1, o.j0, o.j1);
                    }
                    if (dbg.visible) dbg.visible[i] = o.visible ? 1 : 0;
                }
            }
            if (bin_diff && in && o.visible) count_box(bins, hist, diff_stride);
        }
    }
    atomicAdd(&s_visible, my_visible);
    for (int d = 16; d > 0; d >>= 1) {
        my_area += __shfl_xor_sync(0xffffffffu, my_area, d);
        my_tensor += __shfl_xor_sync(0xffffffffu, my_tensor, d);
    }
    if ((threadIdx.x & 31) == 0) { atomicAdd(&s_area[0], my_area); atomicAdd(&s_area[1], my_tensor); }
    __syncthreads();
    if (smem_hist && bin_diff) {
        for (int i = threadIdx.x; i < n_diff; i += blockDim.x) {
            const int c = s_hist[i];
            if (c) atomicAdd(&bin_diff[i], c);
        }
    }
    if (threadIdx.x == 0 && s_visible) {
        atomicAdd(&head->visible, (unsigned long long)s_visible);
        atomicAdd(&head->area_total, s_area[0]);
        atomicAdd(&head->area_tensor, s_area[1]);
    }
}

// counts of all bins from the difference grid: prefix sums along x (one warp per grid row), then along y (one thread per
// column).  One CTA: the grid has at most 257 x 257 entries and lives in L2.
__global__ void __launch_bounds__(1024)
bins_from_diff_kernel(int *__restrict__ diff, int nbx, int nby, uint32_t *__restrict__ bin_count)
{
    const int stride = nbx + 1, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int y = warp; y < nby; y += 32) {
        int carry = 0;
        for (int x0 = 0; x0 < nbx; x0 += 32) {
            const int x = x0 + lane;
            int v = x < nbx ? diff[y * stride + x] : 0;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int u = __shfl_up_sync(0xffffffffu, v, d);
                if (lane >= d) v += u;
            }
            v += carry;
            if (x < nbx) diff[y * stride + x] = v;
            carry = __shfl_sync(0xffffffffu, v, 31);
        }
    }
    __syncthreads();
    for (int x = threadIdx.x; x < nbx; x += blockDim.x) {
        int run = 0;
        for (int y = 0; y < nby; ++y) {
            run += diff[y * stride + x];
            bin_count[y * nbx + x] = (uint32_t)run;
        }
    }
}

}  // namespace

int launch_bins_from_diff(int *bin_diff, const RenderConst &rc, uint32_t *bin_count, cudaStream_t st)
{
    bins_from_diff_kernel<<<1, 1024, 0, st>>>(bin_diff, rc.nbx, rc.nby, bin_count);
    SPLOTCH_LAUNCH_CHECK();
    return 0;
}

int launch_project(const ParticlePtrs &p, int64_t n, const CameraConst &cam, const RenderConst &rc,
                   const float *lutE, const float *lutA, void *records, int *bin_diff, uint32_t *binsw, uint32_t *zkeys,
                   WorkHead *head, const DebugProjectOut *dbg, cudaStream_t st)
{
    if (n <= 0) return 0;
    const int n_diff = (rc.nbx + 1) * (rc.nby + 1);
    const int smem_hist = (bin_diff && n_diff <= kSmemBinsMax) ? 1 : 0;
    const size_t smem = smem_hist ? (size_t)n_diff * sizeof(int) : 0;
    auto aligned16 = [](const void *q) { return (reinterpret_cast<uintptr_t>(q) & 15u) == 0; };
    const int vec_ok = aligned16(p.x) && aligned16(p.y) && aligned16(p.z) && aligned16(p.r) && aligned16(p.I) &&
                       aligned16(p.colval) && (!p.type || (reinterpret_cast<uintptr_t>(p.type) & 3u) == 0);
    const long long groups = (n + 3) / 4;
    long long blocks = (groups + kProjThreads - 1) / kProjThreads;
    const long long cap = (long long)sm_count() * 8;
    if (blocks > cap) blocks = cap;
    DebugProjectOut d = {};
    if (dbg) d = *dbg;
    if (rc.mode == 1)
        project_kernel<true><<<(unsigned)blocks, kProjThreads, smem, st>>>(p, (long long)n, cam, rc, lutE, lutA, records,
                                                                           bin_diff, binsw, zkeys, head, d, dbg ? 1 : 0,
                                                                           vec_ok, smem_hist);
    else
        project_kernel<false><<<(unsigned)blocks, kProjThreads, smem, st>>>(p, (long long)n, cam, rc, lutE, lutA, records,
                                                                            bin_diff, binsw, zkeys, head, d, dbg ? 1 : 0,
                                                                            vec_ok, smem_hist);
    SPLOTCH_LAUNCH_CHECK();
    return 0;
}

}  // namespace splotch
