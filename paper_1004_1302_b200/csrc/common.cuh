// common.cuh -- shared declarations of the sm_100a Splotch render library (product code).
// Nothing here is shared with oracle/ (the CPU oracle is an independent restatement).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>

namespace splotch {

// ---------------------------------------------------------------------------------------------
// geometry of the rasteriser: one CTA owns a 64x64-pixel block, one warp a 16x16 tile of it,
// one lane a strip of 8 consecutive pixels of one tile row.
// ---------------------------------------------------------------------------------------------
constexpr int kBlockShift = 6;             // production bins: 64x64 pixels
constexpr int kBlockPx = 1 << kBlockShift;
constexpr int kTilePx = 16;
constexpr int kMaxBinsPerAxis = 256;       // packed 8-bit bin coordinates in the splat record
constexpr int kMaxImage = 16384;

// ---------------------------------------------------------------------------------------------
// camera constants, computed on the host in double and rounded once to fp32 (DESIGN.md
// "Canonical sequence"); passed to kernels by value.
// ---------------------------------------------------------------------------------------------
struct CameraConst {
    float ex, ey, ez;
    float rx, ry, rz;      // right
    float ux, uy, uz;      // upv
    float fx, fy, fz;      // fwd
    float F, cx, cy;       // focal length in pixels, W/2, H/2
    float Wf, Hf;
    int W, H;
};

struct RenderConst {
    float brightness[4];
    float abs_brightness[4];
    float support_f;
    float z_near;
    float thr;             // exp(-f^2): coverage threshold on the Gaussian weight
    int n_entries, n_types;
    int mode;              // 0 additive, 1 absorb
    int bin_shift;         // bins of 2^bin_shift pixels
    int nbx, nby;          // bins per axis
};

// ---------------------------------------------------------------------------------------------
// splat records written by the transform / cull / colour kernel (step a1-a3)
// ---------------------------------------------------------------------------------------------
constexpr uint32_t kInvisible = 0xFFFFFFFFu;
constexpr uint32_t kListDone = 0x80000000u;   // pair-list flag set by the tensor-core kernel: no ALU work left (n < 2^31)

struct __align__(16) SplatAdd {     // 32 B, additive mode
    float sx, sy;                   // screen position (pixels)
    float c;                        // sqrt(log2 e) / sigma_s : weight = exp2(-((d * c)^2))
    float R;                        // f * sigma_s
    float ar, ag, ab;               // a_c = E_c * I * r * sqrt(pi)
    uint32_t bins;                  // bx0 | bx1 << 8 | by0 << 16 | by1 << 24, or kInvisible
};

struct __align__(16) SplatAbs {     // 48 B, absorb mode
    float sx, sy, c, R;
    float tau0;                     // I * r * sqrt(pi)
    float Er, Eg, Eb;
    float Ar, Ag, Ab;
    uint32_t bins;
};

// record field access shared by the binning kernels: the packed bin box is the last word
__device__ __forceinline__ uint32_t record_bins(const void *records, int record_bytes, long long i)
{
    return __ldg(reinterpret_cast<const uint32_t *>(reinterpret_cast<const char *>(records) +
                                                    (size_t)i * record_bytes + record_bytes - 4));
}

// device-side status head at the start of every workspace (256 B reserved)
struct WorkHead {
    int32_t status;                 // SPLOTCH_OK or SPLOTCH_ERR_WORKSPACE
    uint32_t n_units;               // raster work units
    unsigned long long visible;     // particles that passed culling
    unsigned long long pairs;       // (particle, bin) pairs
    unsigned long long updates;     // debug_stats: (particle, covered pixel) updates
    uint32_t work_counter;          // persistent-kernel ticket
    uint32_t scan_ticket;           // decoupled look-back tile ticket
    uint32_t mma_counter;           // ticket of the tensor-core rasteriser
    float area_total;               // K1: sum of pi/4 x pixel-box areas of the visible splats (~ pixel updates)
    float area_tensor;              // K1: estimate of the part of it inside fully covered 32-pixel row segments
    uint32_t tensor_on;             // finish_offsets: area_tensor >= kTensorShare * area_total
    unsigned long long updates_tensor;   // debug_tensor_stats: updates the tensor-core kernel performs
};

// ---------------------------------------------------------------------------------------------
// error plumbing
// ---------------------------------------------------------------------------------------------
extern thread_local int g_last_cuda_error;

#define SPLOTCH_CUDA_TRY(expr)                                   \
    do {                                                         \
        cudaError_t e__ = (expr);                                \
        if (e__ != cudaSuccess) {                                \
            ::splotch::g_last_cuda_error = (int)e__;             \
            return -3; /* SPLOTCH_ERR_CUDA */                    \
        }                                                        \
    } while (0)

extern std::atomic<unsigned long long> g_launch_count;   // kernels this library has launched (bench.py "gpu_launches")
#define SPLOTCH_LAUNCH_CHECK()                                                      \
    do {                                                                            \
        ::splotch::g_launch_count.fetch_add(1ull, std::memory_order_relaxed);       \
        SPLOTCH_CUDA_TRY(cudaGetLastError());                                       \
    } while (0)

inline uint64_t align_up(uint64_t v, uint64_t a) { return (v + a - 1) / a * a; }

// Per-DEVICE state (function attributes and the SM count belong to a device, not to the process): caches are keyed by
// the ordinal of the calling thread's current device, so one process may render on several GPUs.
constexpr int kMaxDevices = 64;
int current_device();                                   // ordinal of the current device, 0 if it cannot be read
int sm_count();                                         // SMs of the current device

// opt a kernel in to `bytes` of dynamic shared memory once per device
struct SmemOptIn {
    std::atomic<unsigned char> done[kMaxDevices];
};
template <typename Kernel>
inline int smem_opt_in(SmemOptIn &state, Kernel kernel, int bytes)
{
    const int dev = current_device();
    if (dev >= 0 && dev < kMaxDevices && state.done[dev].load(std::memory_order_acquire)) return 0;
    SPLOTCH_CUDA_TRY(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    if (dev >= 0 && dev < kMaxDevices) state.done[dev].store(1, std::memory_order_release);
    return 0;
}

// ---------------------------------------------------------------------------------------------
// launchers (each only enqueues on `st`)
// ---------------------------------------------------------------------------------------------
struct ParticlePtrs {
    const float *x, *y, *z, *r, *I, *colval;
    const uint8_t *type;
    const float *vr, *vg, *vb;      // optional vector colouring (reading R19)
};

struct DebugProjectOut {
    float *sx, *sy, *sigma_s, *R;
    uint32_t *zkey;
    int32_t *pix_bbox;
    uint8_t *visible;
};

// scan.cu: out[k] = sum_{m<k} in[m], k = 0..n (n+1 outputs)
uint64_t scan_scratch_bytes(int64_t n);
int launch_scan_u32_u64(const uint32_t *in, uint64_t *out, int64_t n, void *scratch, cudaStream_t st);
int launch_scan_u32_u32(const uint32_t *in, uint32_t *out, int64_t n, void *scratch, cudaStream_t st);

// sort.cu
uint64_t sort_scratch_bytes(int64_t n);
int launch_sort_pairs(uint32_t *keys, uint32_t *vals, uint32_t *keys_tmp, uint32_t *vals_tmp, int64_t n,
                      const unsigned long long *n_dev, int key_bits, void *scratch, cudaStream_t st,
                      bool *result_in_tmp, const int32_t *status_dev = nullptr);

// project.cu (K1): records + fused bin counts (+ optional debug outputs, + depth keys in absorb mode)
// bin_diff: (nbx + 1) x (nby + 1) signed difference grid (zeroed by the caller), binsw: n packed bin boxes
int launch_project(const ParticlePtrs &p, int64_t n, const CameraConst &cam, const RenderConst &rc,
                   const float *lutE, const float *lutA, void *records, int *bin_diff, uint32_t *binsw, uint32_t *zkeys,
                   WorkHead *head, const DebugProjectOut *dbg, cudaStream_t st);
int launch_bins_from_diff(int *bin_diff, const RenderConst &rc, uint32_t *bin_count, cudaStream_t st);

// bin.cu (K2)
int launch_finish_offsets(const uint32_t *bin_count, const uint64_t *bin_offset, int n_bins, uint64_t max_pairs,
                          uint32_t chunk, uint32_t *unit_prefix, WorkHead *head, cudaStream_t st);
int launch_scatter(const uint32_t *binsw, int64_t n, const RenderConst &rc,
                   const uint64_t *bin_offset, uint32_t *bin_cursor, uint32_t *list, uint64_t max_pairs,
                   const WorkHead *head, cudaStream_t st);
int launch_count_updates(const void *records, int record_bytes, int64_t n, const CameraConst &cam, float thr,
                         WorkHead *head, cudaStream_t st);
// absorb: pair expansion in depth order
int launch_pair_counts(const void *records, int record_bytes, const uint32_t *sorted_ids, int64_t n,
                       uint32_t *pair_count, cudaStream_t st);
int launch_expand_pairs(const void *records, int record_bytes, const uint32_t *sorted_ids, int64_t n,
                        const uint64_t *pair_offset, const RenderConst &rc, uint32_t *pair_bin, uint32_t *pair_id,
                        uint64_t max_pairs, const WorkHead *head, cudaStream_t st);
int launch_iota(uint32_t *v, int64_t n, cudaStream_t st);

// raster.cu (K3, K4)
constexpr uint32_t kChunkAdd = 4096;   // splats per additive work unit
// Additive mode: the tensor-core kernel pays off when most pixel updates lie in fully covered row segments
// (measured: C3, share 0.83, step 476 -> 402 ms; C2, share 0.65, step 37 -> 45 ms).  tensor: 0 off, 1 on, 2 auto.
constexpr float kTensorShare = 0.75f;
constexpr uint32_t kChunkAbs = 4096;   // splats per absorb work unit
int launch_raster_additive(const SplatAdd *records, const uint32_t *list, const uint64_t *bin_offset,
                           const uint32_t *unit_prefix, const RenderConst &rc, const CameraConst &cam, float *S,
                           WorkHead *head, int tensor, cudaStream_t st);
// raster_mma.cu: the fully covered row segments of the additive mode on the tensor cores
int launch_raster_additive_mma(const SplatAdd *records, uint32_t *list, const uint64_t *bin_offset,
                               const uint32_t *unit_prefix, const RenderConst &rc, const CameraConst &cam, float *S,
                               WorkHead *head, int tensor, cudaStream_t st);
int launch_raster_absorb(const SplatAbs *records, const uint32_t *list, const uint64_t *bin_offset,
                         const uint32_t *unit_prefix, const RenderConst &rc, const CameraConst &cam,
                         float *partials, WorkHead *head, cudaStream_t st);
int launch_merge_absorb(const float *partials, const uint32_t *unit_prefix, const RenderConst &rc,
                        const CameraConst &cam, float *out, const WorkHead *head, cudaStream_t st);
int launch_count_tensor_updates(const SplatAdd *records, int64_t n, const RenderConst &rc, const CameraConst &cam,
                                WorkHead *head, cudaStream_t st);
// field.cu: stage (b), range normalisation of a scalar field
int launch_field_range(const float *v, int64_t n, int log_scale, float *range, cudaStream_t st);
int launch_field_normalize(const float *v, int64_t n, int log_scale, const float *range, float *out, cudaStream_t st);
int launch_tonemap_rgb8(const float *v, int64_t n, float gamma, uint8_t *out, cudaStream_t st);
int launch_normalize(const float *S, float *out, int64_t n_values, cudaStream_t st);

}  // namespace splotch
