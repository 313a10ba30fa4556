// project.cu -- K1: fused transform / cull / colour kernel (steps a1-a3 of the hot path) with the
// bin count (a4) folded in.
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
constexpr int kSmemBinsMax = 8192;       // bins counted in shared memory when they fit
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

// Every bin of the splat's bin box gets one count (B-rules).  Small boxes are counted by the
// owning lane, big ones by the whole warp so that one screen-filling splat does not stall 31 lanes.
__device__ __forceinline__ void count_bins(uint32_t bins, uint32_t *hist, int nbx)
{
    const int lane = threadIdx.x & 31;
    const bool vis = bins != kInvisible;
    const int bx0 = bins & 255, bx1 = (bins >> 8) & 255, by0 = (bins >> 16) & 255, by1 = (bins >> 24) & 255;
    const int w = bx1 - bx0 + 1, tot = w * (by1 - by0 + 1);
    const bool big = vis && tot > 8;
    if (vis && !big) {
        for (int by = by0; by <= by1; ++by)
            for (int bx = bx0; bx <= bx1; ++bx) atomicAdd(&hist[by * nbx + bx], 1u);
    }
    unsigned m = __ballot_sync(0xffffffffu, big);
    while (m) {
        const int src = __ffs(m) - 1;
        m &= m - 1;
        const uint32_t b = __shfl_sync(0xffffffffu, bins, src);
        const int cx0 = b & 255, cx1 = (b >> 8) & 255, cy0 = (b >> 16) & 255, cy1 = (b >> 24) & 255;
        const int cw = cx1 - cx0 + 1, ctot = cw * (cy1 - cy0 + 1);
        for (int i = lane; i < ctot; i += 32) atomicAdd(&hist[(cy0 + i / cw) * nbx + cx0 + i % cw], 1u);
    }
}

template <bool kAbsorb>
__global__ void __launch_bounds__(kProjThreads, 4)
project_kernel(ParticlePtrs p, long long n, CameraConst cam, RenderConst rc, const float *__restrict__ lutE,
               const float *__restrict__ lutA, void *__restrict__ records, uint32_t *__restrict__ bin_count,
               uint32_t *__restrict__ zkeys, WorkHead *head, DebugProjectOut dbg, int has_dbg, int vec_ok,
               int smem_hist)
{
    extern __shared__ uint32_t s_hist[];
    __shared__ unsigned int s_visible;
    __shared__ float s_area[2];
    const int n_bins = rc.nbx * rc.nby;
    if (smem_hist)
        for (int i = threadIdx.x; i < n_bins; i += blockDim.x) s_hist[i] = 0u;
    if (threadIdx.x == 0) { s_visible = 0u; s_area[0] = s_area[1] = 0.0f; }
    __syncthreads();
    uint32_t *hist = smem_hist ? s_hist : bin_count;

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
            if (bin_count) count_bins(in ? bins : kInvisible, hist, rc.nbx);
        }
    }
    atomicAdd(&s_visible, my_visible);
    for (int d = 16; d > 0; d >>= 1) {
        my_area += __shfl_xor_sync(0xffffffffu, my_area, d);
        my_tensor += __shfl_xor_sync(0xffffffffu, my_tensor, d);
    }
    if ((threadIdx.x & 31) == 0) { atomicAdd(&s_area[0], my_area); atomicAdd(&s_area[1], my_tensor); }
    __syncthreads();
    if (smem_hist && bin_count) {
        for (int i = threadIdx.x; i < n_bins; i += blockDim.x) {
            const uint32_t c = s_hist[i];
            if (c) atomicAdd(&bin_count[i], c);
        }
    }
    if (threadIdx.x == 0 && s_visible) {
        atomicAdd(&head->visible, (unsigned long long)s_visible);
        atomicAdd(&head->area_total, s_area[0]);
        atomicAdd(&head->area_tensor, s_area[1]);
    }
}

}  // namespace

int launch_project(const ParticlePtrs &p, int64_t n, const CameraConst &cam, const RenderConst &rc,
                   const float *lutE, const float *lutA, void *records, uint32_t *bin_count, uint32_t *zkeys,
                   WorkHead *head, const DebugProjectOut *dbg, cudaStream_t st)
{
    if (n <= 0) return 0;
    const int n_bins = rc.nbx * rc.nby;
    const int smem_hist = (bin_count && n_bins <= kSmemBinsMax) ? 1 : 0;
    const size_t smem = smem_hist ? (size_t)n_bins * sizeof(uint32_t) : 0;
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
                                                                           bin_count, zkeys, head, d, dbg ? 1 : 0,
                                                                           vec_ok, smem_hist);
    else
        project_kernel<false><<<(unsigned)blocks, kProjThreads, smem, st>>>(p, (long long)n, cam, rc, lutE, lutA, records,
                                                                            bin_count, zkeys, head, d, dbg ? 1 : 0,
                                                                            vec_ok, smem_hist);
    SPLOTCH_LAUNCH_CHECK();
    return 0;
}

}  // namespace splotch
