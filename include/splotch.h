/*
 * splotch.h -- C ABI of the B200-native Splotch render hot path.
 *
 * What the library computes (arxiv 1004.1302, "High-performance astrophysical visualization
 * using Splotch"; citations are lines of /root/reference/PAPER.md):
 *
 *   - every particle is a Gaussian blob rho_p(r) = rho_0p exp(-r^2/sigma_p^2), set to zero
 *     beyond f*sigma_p; a ray farther than f*sigma_p from it is unaffected
 *   - R, G, B are three independent "frequencies"
 *   - along a ray  dI/dx = (E_p - A_p I) rho_p(x)                          (Eq. 1)
 *   - E_p, A_p come from a scalar through a colour look-up table; the optical depth can be
 *     modulated by another scalar; E_p = A_p is the recommended setting
 *   - "displaying involves transformation into screen coordinates, assigning of colours and
 *     rendering for determining screen areas affected by individual particles and
 *     subsequently combining them for final imaging"
 *
 * The readings of everything the paper leaves open (camera model, image orientation, point
 * sampling at pixel centres, rho_0 = I, sigma = r, truncation by impact parameter, slab
 * compositing in depth order when A != E, tie order) are listed in DESIGN.md "Readings".
 *
 * Conventions
 *   - All array arguments of splotch_render / splotch_debug_* are DEVICE pointers unless the
 *     name says host.  Structs themselves are host memory, passed by pointer, read during
 *     the call only.
 *   - Ownership: every buffer is caller-owned.  The library never allocates or frees device
 *     memory and keeps no pointer after a call returns.  Particle arrays and colour tables
 *     are read-only.  `out_rgb` is overwritten.  The workspace content is undefined after a
 *     call except for its status head (splotch_workspace_status).
 *   - Asynchrony: splotch_render, splotch_normalize and the debug calls only enqueue work on
 *     `stream` (a cudaStream_t passed as void*, NULL = default stream) and return without
 *     synchronising.  Calls whose name ends in _sync or that return host values synchronise
 *     the stream; they say so below.  splotch_render and splotch_render_batch issue only
 *     memsets and kernel launches on `stream`, so they can be captured into a CUDA graph
 *     and replayed over the same buffers (tests/test_gpu_parity.py does).
 *   - Image layout: out_rgb[(row * width + col) * 3 + c], float32, row 0 = top of the image,
 *     c = 0,1,2 = R,G,B.  Pixel (col i, row j) is sampled at its centre (i + 1/2, j + 1/2).
 *   - Errors: 0 = SPLOTCH_OK, negative = error, nothing is ever reported through the image.
 *     Particles with a non-finite field, r <= 0, type >= n_types, behind the near plane or
 *     covering no pixel centre are culled silently; they are not errors.
 *   - No CPU fallback exists: without a CUDA device every compute entry point returns
 *     SPLOTCH_ERR_CUDA.
 */
#ifndef SPLOTCH_H
#define SPLOTCH_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SPLOTCH_MAX_TYPES 4

/* status codes */
#define SPLOTCH_OK 0
#define SPLOTCH_ERR_INVALID_ARG (-1) /* NULL required pointer, n < 0, bad camera, bad params    */
#define SPLOTCH_ERR_WORKSPACE (-2)   /* workspace_bytes too small, or pair count > max_pairs    */
#define SPLOTCH_ERR_CUDA (-3)        /* a CUDA call failed; see splotch_last_cuda_error()        */
#define SPLOTCH_ERR_LIMIT (-4)       /* a size exceeds what the library supports (see below)    */

/* Limits: n < 2^31; width, height <= 16384; n_entries >= 2; n_types in 1..SPLOTCH_MAX_TYPES;
 * max_pairs < 2^32. */

/* Particle arrays, structure-of-arrays as in the paper's files ("x coordinates of all
 * particles, then y coordinates and so on").  Length n each. */
typedef struct {
    const float *x, *y, *z;   /* world position                                               */
    const float *r;           /* smoothing length = sigma_p of PAPER.md:69                    */
    const float *I;           /* optical-depth modulation = rho_0p (last sentence) */
    const float *colval;      /* scalar mapped through the colour table, clamped to [0, 1]    */
    const uint8_t *type;      /* particle type 0..n_types-1; NULL means all type 0            */
    /* Optional vector colouring ("the three components of the vectors can be mapped to the three
     * components of E and A"; reading R19): when vr is not NULL, vr / vg / vb (length n, all three required) give
     * E_p = brightness[type] * (vr, vg, vb) and A_p = abs_brightness[type] * (vr, vg, vb) directly, used as given
     * (no clamp); colval and the colour tables are ignored (colval and the table pointers of splotch_colormap may then be
     * NULL; n_types is still read); a particle with a non-finite component is culled.  Zero-initialise the struct to keep
     * the scalar path. */
    const float *vr, *vg, *vb;
} splotch_particles;

/* Pinhole perspective camera (reading R1, R2): fwd = normalise(lookat - eye),
 * right = normalise(fwd x up), upv = right x fwd, focal length F = (width/2) / tan(fov/2)
 * pixels, fov the full horizontal angle in degrees, 0 < fov < 180. */
typedef struct {
    float eye[3], lookat[3], up[3];
    float fov_deg;
    int32_t width, height;
} splotch_camera;

/* Colour look-up tables: n_types * n_entries * 3 floats, RGB interleaved, type
 * major.  Sampled piece-wise linearly between n_entries equally spaced nodes on [0, 1]. */
typedef struct {
    const float *emission;    /* E table                                                      */
    const float *absorption;  /* A table; ignored (may be NULL) in additive mode              */
    int32_t n_entries, n_types;
} splotch_colormap;

typedef enum { SPLOTCH_ADDITIVE = 0, SPLOTCH_ABSORB = 1 } splotch_mode;

#define SPLOTCH_RAW_SUM 1u /* additive mode writes S_c = sum_p E_pc tau_p, not 1 - exp(-S_c)   */
#define SPLOTCH_NO_TENSOR 2u /* additive mode: accumulate every pixel on the FP32 ALUs */
#define SPLOTCH_FORCE_TENSOR 4u /* additive mode: always run the fully covered 32-pixel row segments of big
                              splats as split-TF32 tcgen05 MMAs.  With neither flag the library decides on the
                              device (no host sync): tensor cores when >= 75 % of the estimated pixel updates
                              lie in such segments.  The image is the same within rounding either way. */

typedef struct {
    float brightness[SPLOTCH_MAX_TYPES];     /* scales E per type                             */
    float abs_brightness[SPLOTCH_MAX_TYPES]; /* scales A per type (absorb mode)               */
    int32_t mode;                            /* splotch_mode                                  */
    float support_f;                         /* f of PAPER.md:69; > 0; the configs use 3      */
    float z_near;                            /* cull view-space depth <= z_near               */
    uint32_t flags;                          /* SPLOTCH_RAW_SUM | NO_TENSOR | FORCE_TENSOR     */
} splotch_params;

/* ------------------------------------------------------------------------------------------
 * The render call.
 *
 * SPLOTCH_ADDITIVE (A_p = E_p): out_c = 1 - exp(-S_c), S_c = sum over particles of
 *   E_pc * I_p r_p sqrt(pi) * exp(-d^2 / sigma_s^2) for pixels with d^2 <= (f sigma_s)^2, the
 *   exact solution of Eq. (1) when absorption equals emission; any summation order.
 * SPLOTCH_ABSORB (A_p != E_p): particles composited front to back in order of ascending
 *   (fp32 view depth, particle index):  C_c += T_c E_pc tau phi(A_pc tau),  T_c *= exp(-A_pc tau),
 *   phi(u) = (1 - exp(-u))/u; out_c = C_c.  This is Eq. (1) integrated across one particle
 *   at a time (slab reading R10).
 *
 * workspace: device memory, >= splotch_workspace_bytes(...) bytes, 256-byte aligned.
 * max_pairs: capacity of the (particle, 64x64-pixel block) pair list; use
 *   splotch_count_pairs() or an upper bound.  If the scene needs more, the image is
 *   zero-filled and SPLOTCH_ERR_WORKSPACE is recorded in the workspace status head.
 * Returns after enqueueing on `stream`; does not synchronise.
 * ---------------------------------------------------------------------------------------- */
int splotch_workspace_bytes(int64_t n, const splotch_camera *camera, const splotch_params *params,
                            uint64_t max_pairs, uint64_t *bytes);

int splotch_render(const splotch_particles *particles, int64_t n, const splotch_camera *camera,
                   const splotch_colormap *colormap, const splotch_params *params, float *out_rgb,
                   void *workspace, uint64_t workspace_bytes, uint64_t max_pairs, void *stream);

/* Multi-camera batch over ONE resident particle set: the orbit use case, stage (c) "render data"
 * feeding stage (d) frame after frame (section 3 pipeline; BASELINE config 5 renders
 * "an orbit of 8 camera positions over the resident particle set").
 *   cameras      HOST array of n_cameras cameras; all must have the same width and height
 *   out_rgb      DEVICE buffer of n_cameras images, image k at out_rgb + k * height * width * 3
 *   frame_status DEVICE array of n_cameras * 4 uint64 (may be NULL): per frame {status (as int64),
 *                visible, pairs, 0}, copied from the workspace status head after each frame, so that
 *                one synchronisation after the call tells which frames (if any) needed more than
 *                max_pairs pairs (those images are zero-filled; the others are complete)
 *   workspace    ONE workspace of splotch_workspace_bytes(n, &cameras[0], params, max_pairs) bytes,
 *                reused by every frame; max_pairs = the capacity every frame gets (use the largest
 *                splotch_count_pairs over the cameras)
 * Every argument is validated for EVERY camera before anything is enqueued: an invalid camera k
 * fails the whole call with no work done.  Frame k is exactly splotch_render(cameras[k]); the
 * frames are enqueued back to back on `stream` with no host synchronisation in between (the
 * per-frame status copy is device to device).  Enqueue only; does not synchronise. */
int splotch_render_batch(const splotch_particles *particles, int64_t n, const splotch_camera *cameras,
                         int32_t n_cameras, const splotch_colormap *colormap, const splotch_params *params,
                         float *out_rgb, uint64_t *frame_status, void *workspace, uint64_t workspace_bytes,
                         uint64_t max_pairs, void *stream);

/* Reads the status head the last call left in `workspace`.  SYNCHRONISES `stream`.
 * status: SPLOTCH_OK or SPLOTCH_ERR_WORKSPACE; visible: particles that passed culling;
 * pairs: (particle, block) pairs the scene needs.  Any output pointer may be NULL. */
int splotch_workspace_status(const void *workspace, void *stream, int32_t *status, uint64_t *visible,
                             uint64_t *pairs);

/* Runs the transform / cull / bin-count steps only and returns the pair count and the
 * visible count to the host.  SYNCHRONISES `stream`.  workspace must be at least
 * splotch_workspace_bytes(n, camera, params, 0, ...) bytes. */
int splotch_count_pairs(const splotch_particles *particles, int64_t n, const splotch_camera *camera,
                        const splotch_colormap *colormap, const splotch_params *params, void *workspace,
                        uint64_t workspace_bytes, uint64_t *pairs_host, uint64_t *visible_host, void *stream);

/* Stage (b) of the paper's pipeline, "process data (e.g. for normalization)" (on the GPU
 * "the processing involves normalizing of some particle values"): map a scalar field
 * (the colval or I array) to [0, 1] by its own range before splotch_render (reading R17):
 *     out[k] = clamp((f(values[k]) - lo) / (hi - lo), 0, 1),   f(v) = v or log10(v) (log_scale != 0),
 * lo / hi = min / max of f over the values where f is defined and finite.  Where it is not (NaN, inf,
 * v <= 0 under log10) out[k] = NaN, which splotch_render culls; hi == lo gives 0.
 * splotch_field_range writes (lo, hi) to `range` (device, 2 floats; (0, 0) when no value is in the
 * domain); splotch_field_normalize reads it from there.  Both only enqueue on `stream`; values and out
 * are device arrays of n floats (out may equal values), caller-owned. */
int splotch_field_range(const float *values, int64_t n, int32_t log_scale, float *range, void *stream);
int splotch_field_normalize(const float *values, int64_t n, int32_t log_scale, const float *range, float *out,
                            void *stream);

/* The input of stage (d) "save the final image": 8-bit codes of an image written by
 * splotch_render (reading R18): out[k] = rint(255 * clamp(rgb[k], 0, 1)^(1/gamma)), decided in fp32, NaN -> 0;
 * gamma = 1 is the linear map.  rgb: device, n_values floats; out: device, n_values bytes; enqueue only. */
int splotch_tonemap_rgb8(const float *rgb, int64_t n_values, float gamma, uint8_t *out, void *stream);

/* out[k] = 1 - exp(-S[k]) for k < n_values (the additive output map, reading R13); S may
 * equal out.  Exposed for the multi-GPU path, which sums raw S images before this step. */
int splotch_normalize(const float *S, float *out, int64_t n_values, void *stream);

/* End-to-end variant with HOST buffers: copies the particle arrays and colour tables to the
 * device (staging areas inside `workspace`), renders, copies the image back to
 * `out_rgb_host` and SYNCHRONISES.  All pointers inside `particles_host` and
 * `colormap_host` and `out_rgb_host` are host pointers (pinned memory gives the best copy
 * rate).  workspace must be at least splotch_workspace_bytes_host(...) bytes of device memory.
 * Scalar colouring only: particles_host->vr must be NULL. */
int splotch_workspace_bytes_host(int64_t n, const splotch_camera *camera, const splotch_colormap *colormap_host,
                                 const splotch_params *params, uint64_t max_pairs, uint64_t *bytes);

int splotch_render_host(const splotch_particles *particles_host, int64_t n, const splotch_camera *camera,
                        const splotch_colormap *colormap_host, const splotch_params *params,
                        float *out_rgb_host, void *workspace, uint64_t workspace_bytes, uint64_t max_pairs,
                        void *stream);

/* The same, ENQUEUE ONLY: host-to-device copies, render and the device-to-host copy of the image are
 * enqueued on `stream` and the call returns.  The host buffers must stay valid and unchanged (and
 * out_rgb_host unread) until the stream has passed the call; splotch_workspace_status(workspace,
 * stream, ...) then synchronises and returns the status head (it sits at the start of the workspace
 * in this layout too).  With two streams and two workspaces a sequence of frames (the snapshots of a
 * time-dependent run: stage (a) "read" feeding (c) "render") is pipelined: the copies of
 * frame k + 1 run on the copy engines while frame k is rasterised.  Pinned host memory is required
 * for the copies to be asynchronous. */
int splotch_render_host_async(const splotch_particles *particles_host, int64_t n, const splotch_camera *camera,
                              const splotch_colormap *colormap_host, const splotch_params *params,
                              float *out_rgb_host, void *workspace, uint64_t workspace_bytes, uint64_t max_pairs,
                              void *stream);

/* ------------------------------------------------------------------------------------------
 * Test-only exports for the bit-exact checks (north_star: "Tile/bin indices and counts must be
 * bit-exact").  They run the SAME kernels as splotch_render with extra outputs.
 *
 * splotch_debug_project: per particle (device arrays of length n; any may be NULL)
 *   sx, sy     screen position in pixels;  sigma_s = F r / z_c;  R = f sigma_s
 *   zkey       bit pattern of the fp32 view depth z_c (the depth key, R11)
 *   pix_bbox   n*4 int32: i0, i1, j0, j1, inclusive box of candidate pixels
 *   visible    1 if the particle passed culling, else 0 (all other outputs 0)
 *
 * splotch_debug_bins: bins of 2^bin_shift x 2^bin_shift pixels (4 = the 16x16 tiles of
 *   north_star, 6 = the 64x64 blocks the rasteriser consumes).  A visible particle belongs to
 *   every bin its pixel box touches; bin index = by * ceil(width / 2^bin_shift) + bx.
 *   tile_count   T uint32;  tile_offset  T+1 uint64 (exclusive prefix sum, last = D)
 *   member_ids   D uint32 particle indices, bin by bin (may be NULL).  Additive mode: order
 *                inside a bin is unspecified.  Absorb mode: ascending (zkey, index).
 *   max_members  capacity of member_ids; if D exceeds it member_ids is left untouched.
 *   Limits: width, height <= 256 * 2^bin_shift.
 *
 * splotch_debug_stats (SYNCHRONISES): host outputs: visible count, pair count at
 *   `bin_shift`, and the exact number of (particle, covered pixel) updates U.
 * ---------------------------------------------------------------------------------------- */
int splotch_debug_project(const splotch_particles *particles, int64_t n, const splotch_camera *camera,
                          const splotch_colormap *colormap, const splotch_params *params, void *workspace,
                          uint64_t workspace_bytes, float *sx, float *sy, float *sigma_s, float *R,
                          uint32_t *zkey, int32_t *pix_bbox, uint8_t *visible, void *stream);

int splotch_debug_bins(const splotch_particles *particles, int64_t n, const splotch_camera *camera,
                       const splotch_colormap *colormap, const splotch_params *params, void *workspace,
                       uint64_t workspace_bytes, int32_t bin_shift, uint32_t *tile_count,
                       uint64_t *tile_offset, uint32_t *member_ids, uint64_t max_members, void *stream);

int splotch_debug_workspace_bytes(int64_t n, const splotch_camera *camera, const splotch_params *params,
                                  int32_t bin_shift, uint64_t max_members, uint64_t *bytes);

int splotch_debug_stats(const splotch_particles *particles, int64_t n, const splotch_camera *camera,
                        const splotch_colormap *colormap, const splotch_params *params, void *workspace,
                        uint64_t workspace_bytes, int32_t bin_shift, uint64_t *visible_host,
                        uint64_t *pairs_host, uint64_t *updates_host, void *stream);

/* splotch_debug_tensor_stats (SYNCHRONISES; additive mode, production 64x64 bins; workspace as for
 * splotch_debug_stats with bin_shift 6): host outputs: the number of pixel updates inside the image
 * that the tensor-core rasteriser performs when it runs (32-pixel row segments for which its
 * `handled` predicate holds), the library's own choice for this scene (1 = tensor cores), and the
 * estimated share of updates in such segments on which that choice rests. */
int splotch_debug_tensor_stats(const splotch_particles *particles, int64_t n, const splotch_camera *camera,
                               const splotch_colormap *colormap, const splotch_params *params, void *workspace,
                               uint64_t workspace_bytes, uint64_t *updates_tensor_host, int32_t *tensor_on_host,
                               float *share_host, void *stream);

/* Device-wide building blocks, exported so that tests can check them in isolation.
 * splotch_debug_scan: out[k] = sum_{m<k} in[k] for k <= n (n+1 outputs, 64-bit), the
 *   single-pass decoupled look-back scan used for bin offsets.  scratch: >= (n/2048 + 2) * 8 + 256 bytes.
 * splotch_debug_sort_pairs: stable LSD radix sort of (key, value) uint32 pairs on key bits
 *   [0, key_bits); keys_tmp / vals_tmp are ping-pong buffers of length n; the sorted result
 *   ends in (keys, vals).  scratch: >= splotch_sort_scratch_bytes(n). */
int splotch_debug_scan(const uint32_t *in, uint64_t *out, int64_t n, void *scratch, uint64_t scratch_bytes,
                       void *stream);
uint64_t splotch_sort_scratch_bytes(int64_t n);
int splotch_debug_sort_pairs(uint32_t *keys, uint32_t *vals, uint32_t *keys_tmp, uint32_t *vals_tmp, int64_t n,
                             int32_t key_bits, void *scratch, uint64_t scratch_bytes, void *stream);

/* ------------------------------------------------------------------------------------------
 * splotch_scan_static: the bin-offset scan (step a5, bin counts -> bin offsets) with NO caller-supplied
 * scratch and NO allocation of any kind.
 *
 * Who needs it.  A renderer of this kind can be run "in situ": linked into the simulation that produces the
 * particles and called between its time steps.  Such a host program has normally handed all of the GPU's memory
 * to its own pool at start-up and forbids its plug-ins to call cudaMalloc: the call could fail, or succeed and make the
 * simulation's next step run out of memory, and cudaMalloc / cudaFree stall every stream of the device while
 * they run, the simulation's included.  A caller in that position has device buffers for its data (the counts
 * and the offsets) but nothing to spare for the scan's tile descriptors, and cannot get any.  For it, the
 * descriptors live in a fixed 66,048-byte __device__ array that is part of the library image.
 *
 *   in   DEVICE, n uint32 (may be NULL when n == 0)        out  DEVICE, n + 1 uint64, caller-owned
 *   out[k] = in[0] + ... + in[k-1] for k = 0..n (out[n] = total), the same values splotch_debug_scan writes.
 *
 * Limit: n <= SPLOTCH_SCAN_STATIC_MAX_N (2^24 counts; a 16384 x 16384 image has 65,536 production bins and
 *   1,048,576 16x16 tiles).  A larger n returns SPLOTCH_ERR_LIMIT and enqueues nothing; use splotch_debug_scan
 *   with your own scratch instead.
 * Cost: every GPU on which this library is loaded holds the 66,048 bytes until the process exits, used or not.
 * Allocation: the call issues one memset and one kernel on `stream` (enqueue only, no synchronisation).  It
 *   calls no cudaMalloc, cudaFree, or any library routine that allocates.
 * First call on a device: looks up that device's address of the array (cudaGetSymbolAddress, with the calling
 *   thread's current device) and keeps it for later calls.  Make this first call during set-up, with the right
 *   device current and before any stream capture is begun.
 * Sharing: there is one array per device and every call uses it.  The call clears the part it needs before the
 *   kernel runs, so earlier contents never matter; but two calls that can overlap on the GPU (different streams
 *   without an ordering between them, or two host threads on one device) corrupt each other's descriptors and
 *   may hang.  Calls on one stream, or ordered by events, are safe.
 * Errors: SPLOTCH_ERR_INVALID_ARG (n < 0, NULL out, NULL in with n > 0), SPLOTCH_ERR_LIMIT, SPLOTCH_ERR_CUDA.
 * ---------------------------------------------------------------------------------------- */
#define SPLOTCH_SCAN_STATIC_MAX_N (1 << 24)
int splotch_scan_static(const uint32_t *in, uint64_t *out, int64_t n, void *stream);

/* Per-stage timing of splotch_render with CUDA events recorded on the caller's stream (used by
 * bench.py for the roofline of the dominant kernel).  splotch_profile_enable(1) resets the
 * record; while enabled every splotch_render records 7 events (up to 256 calls).
 * splotch_profile_read SYNCHRONISES on the last recorded event and returns the mean
 * milliseconds per call of the 6 stages: [0] transform/cull/colour + bin count (K1),
 * [1] offsets scan + work units, [2] lists (scatter, or depth sort + ordered split),
 * [3] tensor-core rasteriser (K3t; 0 in absorb mode and with SPLOTCH_NO_TENSOR),
 * [4] ALU tile rasteriser (K3), [5] output map / merge (K4).
 * splotch_launch_count: kernels launched by this library in this process so far. */
int splotch_profile_enable(int on);
int splotch_profile_read(double *stage_ms /* host, 6 doubles */, int64_t *calls /* host */);
unsigned long long splotch_launch_count(void);

const char *splotch_status_string(int status);
int splotch_last_cuda_error(void);  /* cudaError_t of the last failing CUDA call in this thread */
int splotch_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SPLOTCH_H */
