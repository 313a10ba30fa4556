// field.cu -- stage (b) "process data (e.g. for normalization)" of PAPER.md:81, the step just before the
// render path; on the GPU the paper's kernel "involves normalizing of some particle values".
// Reading R17: a scalar field (colval, I) is mapped to [0, 1] by its own range,
//     out = clamp((f(v) - lo) / (hi - lo), 0, 1),   f = identity or log10,   lo / hi = min / max of f over the
// values where f is defined and finite; where it is not (NaN, inf, v <= 0 under log10) out = NaN, which the
// transform kernel culls (R6); hi == lo gives 0.  Both kernels are HBM-bound streams: 4 B read per value for the
// range, 8 B per value for the map.  The range stays on the device: no host synchronisation.
#include "common.cuh"

namespace splotch {

namespace {

constexpr int kFieldThreads = 256;

// order-preserving map float -> uint32 (so that atomicMin / atomicMax on the code order the floats)
__device__ __forceinline__ uint32_t encode_ordered(float v)
{
    const uint32_t u = __float_as_uint(v);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float decode_ordered(uint32_t c)
{
    return __uint_as_float((c & 0x80000000u) ? (c & 0x7fffffffu) : ~c);
}

__device__ __forceinline__ bool in_domain(float v, int log_scale)
{
    return fabsf(v) <= 3.402823466e38f && (!log_scale || v > 0.0f);
}

__global__ void field_range_init_kernel(uint32_t *code)
{
    code[0] = 0xFFFFFFFFu;      // min: larger than every code
    code[1] = 0u;               // max: smaller than every code
}

__global__ void __launch_bounds__(kFieldThreads)
field_range_kernel(const float *__restrict__ v, long long n, int log_scale, int vec_ok, uint32_t *code)
{
    float lo = __int_as_float(0x7f800000), hi = __int_as_float(0xff800000);
    const long long stride = (long long)gridDim.x * blockDim.x, t0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    auto take = [&](float x) {
        if (in_domain(x, log_scale)) { lo = fminf(lo, x); hi = fmaxf(hi, x); }
    };
    long long done = 0;
    if (vec_ok) {
        const long long n4 = n >> 2;
        for (long long i = t0; i < n4; i += stride) {
            const float4 q = __ldg(reinterpret_cast<const float4 *>(v) + i);
            take(q.x); take(q.y); take(q.z); take(q.w);
        }
        done = n4 << 2;
    }
    for (long long i = done + t0; i < n; i += stride) take(__ldg(v + i));
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        lo = fminf(lo, __shfl_xor_sync(0xffffffffu, lo, d));
        hi = fmaxf(hi, __shfl_xor_sync(0xffffffffu, hi, d));
    }
    if ((threadIdx.x & 31) == 0 && lo <= hi) {
        atomicMin(code, encode_ordered(lo));
        atomicMax(code + 1, encode_ordered(hi));
    }
}

// codes -> (lo, hi) of f; log10 is monotone, so the range of f is f of the range.  No value in the domain: (0, 0).
__global__ void field_range_finish_kernel(uint32_t *code, int log_scale)
{
    float lo = 0.0f, hi = 0.0f;
    if (code[0] != 0xFFFFFFFFu) {
        lo = decode_ordered(code[0]);
        hi = decode_ordered(code[1]);
        if (log_scale) { lo = log10f(lo); hi = log10f(hi); }
    }
    reinterpret_cast<float *>(code)[0] = lo;
    reinterpret_cast<float *>(code)[1] = hi;
}

__device__ __forceinline__ float map_one(float x, int log_scale, float lo, float span)
{
    if (!in_domain(x, log_scale)) return __int_as_float(0x7fc00000);
    const float f = log_scale ? log10f(x) : x;
    if (!(span > 0.0f)) return 0.0f;
    return fminf(fmaxf(__fdiv_rn(f - lo, span), 0.0f), 1.0f);
}

__global__ void __launch_bounds__(kFieldThreads)
field_normalize_kernel(const float *__restrict__ v, long long n, int log_scale, const float *__restrict__ range,
                       float *__restrict__ out, int vec_ok)
{
    const float lo = __ldg(range), span = __ldg(range + 1) - lo;
    const long long stride = (long long)gridDim.x * blockDim.x, t0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    long long done = 0;
    if (vec_ok) {
        const long long n4 = n >> 2;
        for (long long i = t0; i < n4; i += stride) {
            const float4 q = __ldg(reinterpret_cast<const float4 *>(v) + i);
            reinterpret_cast<float4 *>(out)[i] = make_float4(map_one(q.x, log_scale, lo, span), map_one(q.y, log_scale, lo, span),
                                                             map_one(q.z, log_scale, lo, span), map_one(q.w, log_scale, lo, span));
        }
        done = n4 << 2;
    }
    for (long long i = done + t0; i < n; i += stride) out[i] = map_one(__ldg(v + i), log_scale, lo, span);
}

// Stage (d) input ("save the final image"): 8-bit code of an image value, reading R18:
// code = rint(255 * clamp(x, 0, 1)^(1/gamma)), NaN -> 0; fp32 throughout (the integer is decided in fp32).
__device__ __forceinline__ unsigned tone_one(float x, float inv_gamma)
{
    float y = fminf(fmaxf(x, 0.0f), 1.0f);          // fmaxf(NaN, 0) = 0
    if (inv_gamma != 1.0f) y = powf(y, inv_gamma);
    return (unsigned)__float2int_rn(__fmul_rn(255.0f, y));
}

__global__ void __launch_bounds__(kFieldThreads)
tonemap_rgb8_kernel(const float *__restrict__ v, long long n, float inv_gamma, uint8_t *__restrict__ out, int vec_ok)
{
    const long long stride = (long long)gridDim.x * blockDim.x, t0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    long long done = 0;
    if (vec_ok) {
        const long long n4 = n >> 2;
        for (long long i = t0; i < n4; i += stride) {
            const float4 q = __ldg(reinterpret_cast<const float4 *>(v) + i);
            reinterpret_cast<uint32_t *>(out)[i] = tone_one(q.x, inv_gamma) | (tone_one(q.y, inv_gamma) << 8) |
                                                   (tone_one(q.z, inv_gamma) << 16) | (tone_one(q.w, inv_gamma) << 24);
        }
        done = n4 << 2;
    }
    for (long long i = done + t0; i < n; i += stride) out[i] = (uint8_t)tone_one(__ldg(v + i), inv_gamma);
}

unsigned field_grid(int64_t n)
{
    long long blocks = (n / 4 + kFieldThreads - 1) / kFieldThreads + 1;
    const long long cap = (long long)sm_count() * 8;
    return (unsigned)(blocks > cap ? cap : blocks);
}

}  // namespace

int launch_field_range(const float *v, int64_t n, int log_scale, float *range, cudaStream_t st)
{
    uint32_t *code = reinterpret_cast<uint32_t *>(range);
    field_range_init_kernel<<<1, 1, 0, st>>>(code);
    SPLOTCH_LAUNCH_CHECK();
    if (n > 0) {
        const int vec_ok = (reinterpret_cast<uintptr_t>(v) & 15u) == 0;
        field_range_kernel<<<field_grid(n), kFieldThreads, 0, st>>>(v, (long long)n, log_scale, vec_ok, code);
        SPLOTCH_LAUNCH_CHECK();
    }
    field_range_finish_kernel<<<1, 1, 0, st>>>(code, log_scale);
    SPLOTCH_LAUNCH_CHECK();
    return 0;
}

int launch_tonemap_rgb8(const float *v, int64_t n, float gamma, uint8_t *out, cudaStream_t st)
{
    if (n <= 0) return 0;
    const int vec_ok = (reinterpret_cast<uintptr_t>(v) & 15u) == 0 && (reinterpret_cast<uintptr_t>(out) & 3u) == 0;
    tonemap_rgb8_kernel<<<field_grid(n), kFieldThreads, 0, st>>>(v, (long long)n, 1.0f / gamma, out, vec_ok);
    SPLOTCH_LAUNCH_CHECK();
    return 0;
}

int launch_field_normalize(const float *v, int64_t n, int log_scale, const float *range, float *out, cudaStream_t st)
{
    if (n <= 0) return 0;
    const int vec_ok = ((reinterpret_cast<uintptr_t>(v) | reinterpret_cast<uintptr_t>(out)) & 15u) == 0;
    field_normalize_kernel<<<field_grid(n), kFieldThreads, 0, st>>>(v, (long long)n, log_scale, range, out, vec_ok);
    SPLOTCH_LAUNCH_CHECK();
    return 0;
}

}  // namespace splotch
