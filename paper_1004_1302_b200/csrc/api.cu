// api.cu -- the C ABI of include/splotch.h: argument checks, camera constants, workspace layout
// and the launch sequence of the hot path.  Every entry point only enqueues on the caller's
// stream unless its declaration says it synchronises.
#include <math.h>
#include <string.h>

#include <mutex>

#include "../../include/splotch.h"
#include "common.cuh"

namespace splotch {

thread_local int g_last_cuda_error = 0;
std::atomic<unsigned long long> g_launch_count{0};

// ---------------------------------------------------------------------------------------------
// optional per-stage timing of splotch_render with CUDA events on the caller's stream
// ---------------------------------------------------------------------------------------------
namespace {
constexpr int kStages = 6;          // project+count | offsets | lists | raster (tensor cores) | raster (ALU) | output map
constexpr int kMaxProfiledCalls = 256;
struct Profile {
    bool on = false;
    int calls = 0;
    cudaEvent_t ev[kMaxProfiledCalls][kStages + 1];
    bool created[kMaxProfiledCalls] = {};
} g_prof;
std::mutex g_prof_mutex;            // the profile is one per process: calls from several threads are serialised

void prof_mark(int stage, cudaStream_t st)
{
    std::lock_guard<std::mutex> lock(g_prof_mutex);
    if (!g_prof.on || g_prof.calls >= kMaxProfiledCalls) return;
    const int c = g_prof.calls;
    if (!g_prof.created[c]) {
        for (int k = 0; k <= kStages; ++k)
            if (cudaEventCreate(&g_prof.ev[c][k]) != cudaSuccess) { g_prof.on = false; return; }
        g_prof.created[c] = true;
    }
    cudaEventRecord(g_prof.ev[c][stage], st);
    if (stage == kStages) ++g_prof.calls;
}
}  // namespace

int current_device()
{
    int dev = 0;
    return cudaGetDevice(&dev) == cudaSuccess ? dev : 0;
}

int sm_count()
{
    static std::atomic<int> cached[kMaxDevices];
    const int dev = current_device();
    const bool slot = dev >= 0 && dev < kMaxDevices;
    int n = slot ? cached[dev].load(std::memory_order_relaxed) : 0;
    if (n == 0) {
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) return 148;
        if (slot) cached[dev].store(n, std::memory_order_relaxed);
    }
    return n;
}

namespace {

// ---------------------------------------------------------------------------------------------
// camera basis (readings R1, R2), double on the host, rounded once to fp32
// ---------------------------------------------------------------------------------------------
int make_camera(const splotch_camera *c, CameraConst *o)
{
    if (!c || c->width <= 0 || c->height <= 0 || c->width > kMaxImage || c->height > kMaxImage) return SPLOTCH_ERR_INVALID_ARG;
    const double fov = (double)c->fov_deg;
    if (!(fov > 0.0) || !(fov < 180.0)) return SPLOTCH_ERR_INVALID_ARG;
    double e[3], f[3], u[3];
    for (int k = 0; k < 3; ++k) {
        e[k] = (double)c->eye[k];
        f[k] = (double)c->lookat[k] - e[k];
        u[k] = (double)c->up[k];
        if (!isfinite(e[k]) || !isfinite(f[k]) || !isfinite(u[k])) return SPLOTCH_ERR_INVALID_ARG;
    }
    const double fn = sqrt(f[0] * f[0] + f[1] * f[1] + f[2] * f[2]);
    if (!(fn > 0.0)) return SPLOTCH_ERR_INVALID_ARG;
    for (int k = 0; k < 3; ++k) f[k] /= fn;
    double r[3] = { f[1] * u[2] - f[2] * u[1], f[2] * u[0] - f[0] * u[2], f[0] * u[1] - f[1] * u[0] };
    const double rn = sqrt(r[0] * r[0] + r[1] * r[1] + r[2] * r[2]);
    if (!(rn > 0.0)) return SPLOTCH_ERR_INVALID_ARG;     // up parallel to the view direction
    for (int k = 0; k < 3; ++k) r[k] /= rn;
    const double v[3] = { r[1] * f[2] - r[2] * f[1], r[2] * f[0] - r[0] * f[2], r[0] * f[1] - r[1] * f[0] };
    const double pi = 3.14159265358979323846;
    const double F = (0.5 * (double)c->width) / tan(0.5 * fov * pi / 180.0);
    o->ex = c->eye[0]; o->ey = c->eye[1]; o->ez = c->eye[2];
    o->rx = (float)r[0]; o->ry = (float)r[1]; o->rz = (float)r[2];
    o->ux = (float)v[0]; o->uy = (float)v[1]; o->uz = (float)v[2];
    o->fx = (float)f[0]; o->fy = (float)f[1]; o->fz = (float)f[2];
    o->F = (float)F;
    o->cx = (float)(0.5 * (double)c->width);
    o->cy = (float)(0.5 * (double)c->height);
    o->Wf = (float)c->width; o->Hf = (float)c->height;
    o->W = c->width; o->H = c->height;
    return SPLOTCH_OK;
}

int make_render_const(const splotch_camera *cam, const splotch_colormap *cm, const splotch_params *p, int bin_shift,
                      RenderConst *o)
{
    if (!p) return SPLOTCH_ERR_INVALID_ARG;
    if (p->mode != SPLOTCH_ADDITIVE && p->mode != SPLOTCH_ABSORB) return SPLOTCH_ERR_INVALID_ARG;
    if (!(p->support_f > 0.0f) || !isfinite(p->support_f) || !(p->z_near >= 0.0f) || !isfinite(p->z_near))
        return SPLOTCH_ERR_INVALID_ARG;
    for (int k = 0; k < 4; ++k) { o->brightness[k] = p->brightness[k]; o->abs_brightness[k] = p->abs_brightness[k]; }
    o->support_f = p->support_f;
    o->z_near = p->z_near;
    o->thr = (float)exp(-(double)p->support_f * (double)p->support_f);
    if (!(o->thr >= 1.17549435e-38f)) o->thr = 1.17549435e-38f;   // beyond f ~ 9.3 fp32 weights underflow anyway; keeps thr / gy > 0
    o->n_entries = cm ? cm->n_entries : 2;
    o->n_types = cm ? cm->n_types : 1;
    o->mode = p->mode;
    o->bin_shift = bin_shift;
    const int bs = 1 << bin_shift;
    o->nbx = (cam->width + bs - 1) >> bin_shift;
    o->nby = (cam->height + bs - 1) >> bin_shift;
    if (o->nbx > kMaxBinsPerAxis || o->nby > kMaxBinsPerAxis) return SPLOTCH_ERR_LIMIT;
    return SPLOTCH_OK;
}

// vector colouring (reading R19) ignores the tables: they may then be NULL (the struct still carries n_types)
int check_colormap(const splotch_colormap *cm, int mode, bool vector_colouring = false)
{
    if (!cm) return SPLOTCH_ERR_INVALID_ARG;
    if (cm->n_types < 1 || cm->n_types > SPLOTCH_MAX_TYPES) return SPLOTCH_ERR_INVALID_ARG;
    if (vector_colouring) return SPLOTCH_OK;
    if (!cm->emission || cm->n_entries < 2) return SPLOTCH_ERR_INVALID_ARG;
    if (mode == SPLOTCH_ABSORB && !cm->absorption) return SPLOTCH_ERR_INVALID_ARG;
    return SPLOTCH_OK;
}

int check_particles(const splotch_particles *p, int64_t n)
{
    if (n < 0) return SPLOTCH_ERR_INVALID_ARG;
    if (n >= (1ll << 31)) return SPLOTCH_ERR_LIMIT;
    if (n > 0 && (!p || !p->x || !p->y || !p->z || !p->r || !p->I)) return SPLOTCH_ERR_INVALID_ARG;
    if (n > 0 && p->vr && (!p->vg || !p->vb)) return SPLOTCH_ERR_INVALID_ARG;
    if (n > 0 && !p->vr && !p->colval) return SPLOTCH_ERR_INVALID_ARG;
    return SPLOTCH_OK;
}

int bits_for(int n_bins)
{
    int b = 1;
    while ((1 << b) < n_bins) ++b;
    return b;
}

// ---------------------------------------------------------------------------------------------
// workspace layout
// ---------------------------------------------------------------------------------------------
struct Layout {
    uint64_t head, records, bin_count, bin_cursor, bin_offset, unit_prefix, scan_scratch, list, bin_diff, bin_diff_bytes, binsw;
    // absorb mode
    uint64_t zkeys, ids, zkeys_tmp, ids_tmp, sort_scratch, pair_count, pair_offset, pair_bin, pair_id, pair_bin_tmp,
        partials;
    uint64_t total;
};

Layout make_layout(int64_t n, int nbx, int nby, int mode, uint64_t max_pairs, bool want_partials)
{
    const int n_bins = nbx * nby;
    Layout L;
    memset(&L, 0, sizeof(L));
    uint64_t off = 0;
    auto take = [&](uint64_t bytes) {
        const uint64_t at = off;
        off += align_up(bytes > 0 ? bytes : 1, 256);
        return at;
    };
    const uint64_t nn = (uint64_t)(n > 0 ? n : 1);
    L.head = take(256);
    L.records = take(nn * (mode == SPLOTCH_ABSORB ? sizeof(SplatAbs) : sizeof(SplatAdd)));
    L.bin_diff_bytes = (uint64_t)(nbx + 1) * (uint64_t)(nby + 1) * 4;
    L.bin_diff = take(L.bin_diff_bytes);
    if (mode != SPLOTCH_ABSORB) L.binsw = take(nn * 4);      // read by the additive scatter only; absorb lists come from the records
    L.bin_count = take((uint64_t)n_bins * 4);
    L.bin_cursor = take((uint64_t)n_bins * 4);
    L.bin_offset = take((uint64_t)(n_bins + 1) * 8);
    L.unit_prefix = take((uint64_t)(n_bins + 1) * 4);
    L.scan_scratch = take(scan_scratch_bytes((int64_t)(nn > (uint64_t)n_bins ? nn : (uint64_t)n_bins)));
    L.list = take(max_pairs * 4);
    if (mode == SPLOTCH_ABSORB) {
        L.zkeys = take(nn * 4);
        L.ids = take(nn * 4);
        L.zkeys_tmp = take(nn * 4);
        L.ids_tmp = take(nn * 4);
        const uint64_t s1 = sort_scratch_bytes((int64_t)nn), s2 = sort_scratch_bytes((int64_t)(max_pairs ? max_pairs : 1));
        L.sort_scratch = take(s1 > s2 ? s1 : s2);
        L.pair_count = take(nn * 4);
        L.pair_offset = take((nn + 1) * 8);
        L.pair_bin = take(max_pairs * 4);
        L.pair_id = take(max_pairs * 4);
        L.pair_bin_tmp = take(max_pairs * 4);
        if (want_partials) {
            const uint64_t max_units = max_pairs / kChunkAbs + (uint64_t)n_bins + 1;
            L.partials = take(max_units * 6ull * kBlockPx * kBlockPx * 4ull);
        }
    }
    L.total = off;
    return L;
}

struct Ctx {
    CameraConst cam;
    RenderConst rc;
    Layout L;
    char *ws;
    cudaStream_t st;
    int n_bins;
    template <typename T> T *at(uint64_t off) const { return reinterpret_cast<T *>(ws + off); }
    WorkHead *head() const { return at<WorkHead>(L.head); }
};

int setup(const splotch_particles *particles, int64_t n, const splotch_camera *camera, const splotch_colormap *cm,
          const splotch_params *params, int bin_shift, void *workspace, uint64_t workspace_bytes, uint64_t max_pairs,
          bool want_partials, void *stream, Ctx *c)
{
    int rc = check_particles(particles, n);
    if (rc) return rc;
    rc = make_camera(camera, &c->cam);
    if (rc) return rc;
    if (!params) return SPLOTCH_ERR_INVALID_ARG;
    rc = check_colormap(cm, params->mode, n > 0 && particles && particles->vr);
    if (rc) return rc;
    rc = make_render_const(camera, cm, params, bin_shift, &c->rc);
    if (rc) return rc;
    if (max_pairs >= (1ull << 32)) return SPLOTCH_ERR_LIMIT;
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 255u)) return SPLOTCH_ERR_INVALID_ARG;
    c->n_bins = c->rc.nbx * c->rc.nby;
    c->L = make_layout(n, c->rc.nbx, c->rc.nby, params->mode, max_pairs, want_partials);
    if (workspace_bytes < c->L.total) return SPLOTCH_ERR_WORKSPACE;
    c->ws = reinterpret_cast<char *>(workspace);
    c->st = reinterpret_cast<cudaStream_t>(stream);
    return SPLOTCH_OK;
}

// K1 + bin counts + offsets + units: everything up to (not including) the list
int run_front(const Ctx &c, const splotch_particles *particles, int64_t n, const splotch_colormap *cm,
              uint64_t max_pairs, uint32_t chunk, const DebugProjectOut *dbg, bool profiled = false)
{
    SPLOTCH_CUDA_TRY(cudaMemsetAsync(c.ws + c.L.head, 0, 256, c.st));
    SPLOTCH_CUDA_TRY(cudaMemsetAsync(c.ws + c.L.bin_diff, 0, (size_t)c.L.bin_diff_bytes, c.st));
    SPLOTCH_CUDA_TRY(cudaMemsetAsync(c.ws + c.L.bin_count, 0, (size_t)c.n_bins * 4, c.st));
    SPLOTCH_CUDA_TRY(cudaMemsetAsync(c.ws + c.L.bin_cursor, 0, (size_t)c.n_bins * 4, c.st));
    ParticlePtrs pp = { nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr };
    if (n > 0) pp = { particles->x, particles->y, particles->z, particles->r, particles->I, particles->colval, particles->type,
                      particles->vr, particles->vg, particles->vb };
    int rc = launch_project(pp, n, c.cam, c.rc, cm->emission, cm->absorption, c.ws + c.L.records,
                            c.at<int>(c.L.bin_diff), c.rc.mode == SPLOTCH_ABSORB ? nullptr : c.at<uint32_t>(c.L.binsw),
                            c.rc.mode == SPLOTCH_ABSORB ? c.at<uint32_t>(c.L.zkeys) : nullptr, c.head(), dbg, c.st);
    if (rc) return rc;
    rc = launch_bins_from_diff(c.at<int>(c.L.bin_diff), c.rc, c.at<uint32_t>(c.L.bin_count), c.st);
    if (rc) return rc;
    if (profiled) prof_mark(1, c.st);
    rc = launch_scan_u32_u64(c.at<uint32_t>(c.L.bin_count), c.at<uint64_t>(c.L.bin_offset), c.n_bins,
                             c.ws + c.L.scan_scratch, c.st);
    if (rc) return rc;
    return launch_finish_offsets(c.at<uint32_t>(c.L.bin_count), c.at<uint64_t>(c.L.bin_offset), c.n_bins, max_pairs, chunk,
                                 c.at<uint32_t>(c.L.unit_prefix), c.head(), c.st);
}

// the per-bin lists: additive = unordered scatter; absorb = depth sort, ordered expansion, stable
// split by bin.  *list_out points at the final list inside the workspace.
int run_lists(const Ctx &c, int64_t n, uint64_t max_pairs, uint32_t **list_out)
{
    const int rec_bytes = c.rc.mode == SPLOTCH_ABSORB ? (int)sizeof(SplatAbs) : (int)sizeof(SplatAdd);
    *list_out = c.at<uint32_t>(c.L.list);
    if (n <= 0 || max_pairs == 0) return SPLOTCH_OK;
    if (c.rc.mode == SPLOTCH_ADDITIVE)
        return launch_scatter(c.at<uint32_t>(c.L.binsw), n, c.rc, c.at<uint64_t>(c.L.bin_offset),
                              c.at<uint32_t>(c.L.bin_cursor), c.at<uint32_t>(c.L.list), max_pairs, c.head(), c.st);
    // a7: order the particles by (depth key, index): stable LSD sort of the keys with iota values
    int rc = launch_iota(c.at<uint32_t>(c.L.ids), n, c.st);
    if (rc) return rc;
    bool in_tmp = false;
    rc = launch_sort_pairs(c.at<uint32_t>(c.L.zkeys), c.at<uint32_t>(c.L.ids), c.at<uint32_t>(c.L.zkeys_tmp),
                           c.at<uint32_t>(c.L.ids_tmp), n, nullptr, 32, c.ws + c.L.sort_scratch, c.st, &in_tmp, &c.head()->status);
    if (rc) return rc;
    const uint32_t *sorted = in_tmp ? c.at<uint32_t>(c.L.ids_tmp) : c.at<uint32_t>(c.L.ids);
    rc = launch_pair_counts(c.ws + c.L.records, rec_bytes, sorted, n, c.at<uint32_t>(c.L.pair_count), c.st);
    if (rc) return rc;
    rc = launch_scan_u32_u64(c.at<uint32_t>(c.L.pair_count), c.at<uint64_t>(c.L.pair_offset), n, c.ws + c.L.scan_scratch, c.st);
    if (rc) return rc;
    rc = launch_expand_pairs(c.ws + c.L.records, rec_bytes, sorted, n, c.at<uint64_t>(c.L.pair_offset), c.rc,
                             c.at<uint32_t>(c.L.pair_bin), c.at<uint32_t>(c.L.pair_id), max_pairs, c.head(), c.st);
    if (rc) return rc;
    // stable split by bin keeps the depth order inside every bin; the pair count lives on the device
    rc = launch_sort_pairs(c.at<uint32_t>(c.L.pair_bin), c.at<uint32_t>(c.L.pair_id), c.at<uint32_t>(c.L.pair_bin_tmp),
                           c.at<uint32_t>(c.L.list), (int64_t)max_pairs, &c.head()->pairs, bits_for(c.n_bins),
                           c.ws + c.L.sort_scratch, c.st, &in_tmp, &c.head()->status);
    if (rc) return rc;
    *list_out = in_tmp ? c.at<uint32_t>(c.L.list) : c.at<uint32_t>(c.L.pair_id);
    return SPLOTCH_OK;
}

__global__ void copy_members_kernel(const uint32_t *__restrict__ src, uint32_t *__restrict__ dst,
                                    const WorkHead *head, unsigned long long cap)
{
    const unsigned long long D = head->pairs;
    if (head->status != 0 || D > cap) return;
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < D; i += stride) dst[i] = src[i];
}

__global__ void zero_if_failed_kernel(float *out, long long n, const WorkHead *head)
{
    if (head->status == 0) return;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) out[i] = 0.0f;
}

}  // namespace
}  // namespace splotch

using namespace splotch;

extern "C" {

int splotch_version(void) { return 100; }

const char *splotch_status_string(int status)
{
    switch (status) {
    case SPLOTCH_OK: return "ok";
    case SPLOTCH_ERR_INVALID_ARG: return "invalid argument";
    case SPLOTCH_ERR_WORKSPACE: return "workspace too small or pair count above max_pairs";
    case SPLOTCH_ERR_CUDA: return "CUDA error (see splotch_last_cuda_error)";
    case SPLOTCH_ERR_LIMIT: return "size above a library limit";
    default: return "unknown status";
    }
}

int splotch_last_cuda_error(void) { return g_last_cuda_error; }

int splotch_workspace_bytes(int64_t n, const splotch_camera *camera, const splotch_params *params, uint64_t max_pairs,
                            uint64_t *bytes)
{
    if (!bytes || !params || n < 0) return SPLOTCH_ERR_INVALID_ARG;
    CameraConst cam;
    int rc = make_camera(camera, &cam);
    if (rc) return rc;
    RenderConst r;
    rc = make_render_const(camera, nullptr, params, kBlockShift, &r);
    if (rc) return rc;
    if (max_pairs >= (1ull << 32)) return SPLOTCH_ERR_LIMIT;
    *bytes = make_layout(n, r.nbx, r.nby, params->mode, max_pairs, true).total;
    return SPLOTCH_OK;
}

int splotch_debug_workspace_bytes(int64_t n, const splotch_camera *camera, const splotch_params *params, int32_t bin_shift,
                                  uint64_t max_members, uint64_t *bytes)
{
    if (!bytes || !params || n < 0 || bin_shift < 2 || bin_shift > 10) return SPLOTCH_ERR_INVALID_ARG;
    CameraConst cam;
    int rc = make_camera(camera, &cam);
    if (rc) return rc;
    RenderConst r;
    rc = make_render_const(camera, nullptr, params, bin_shift, &r);
    if (rc) return rc;
    if (max_members >= (1ull << 32)) return SPLOTCH_ERR_LIMIT;
    *bytes = make_layout(n, r.nbx, r.nby, params->mode, max_members, false).total;
    return SPLOTCH_OK;
}

int splotch_render(const splotch_particles *particles, int64_t n, const splotch_camera *camera,
                   const splotch_colormap *colormap, const splotch_params *params, float *out_rgb, void *workspace,
                   uint64_t workspace_bytes, uint64_t max_pairs, void *stream)
{
    if (!out_rgb) return SPLOTCH_ERR_INVALID_ARG;
    Ctx c;
    int rc = setup(particles, n, camera, colormap, params, kBlockShift, workspace, workspace_bytes, max_pairs, true, stream, &c);
    if (rc) return rc;
    const bool absorb = c.rc.mode == SPLOTCH_ABSORB;
    const int64_t n_values = (int64_t)c.cam.W * c.cam.H * 3;
    prof_mark(0, c.st);
    rc = run_front(c, particles, n, colormap, max_pairs, absorb ? kChunkAbs : kChunkAdd, nullptr, true);
    if (rc) return rc;
    prof_mark(2, c.st);
    uint32_t *list = nullptr;
    rc = run_lists(c, n, max_pairs, &list);
    if (rc) return rc;
    if (!absorb) SPLOTCH_CUDA_TRY(cudaMemsetAsync(out_rgb, 0, (size_t)n_values * 4, c.st));
    prof_mark(3, c.st);
    if (absorb) prof_mark(4, c.st);
    if (!absorb) {
        const int mma_on = (params->flags & SPLOTCH_NO_TENSOR) ? 0 : (params->flags & SPLOTCH_FORCE_TENSOR) ? 1 : 2;
        if (mma_on) {
            rc = launch_raster_additive_mma(c.at<SplatAdd>(c.L.records), list, c.at<uint64_t>(c.L.bin_offset),
                                            c.at<uint32_t>(c.L.unit_prefix), c.rc, c.cam, out_rgb, c.head(), mma_on, c.st);
            if (rc) return rc;
        }
        prof_mark(4, c.st);
        rc = launch_raster_additive(c.at<SplatAdd>(c.L.records), list, c.at<uint64_t>(c.L.bin_offset),
                                    c.at<uint32_t>(c.L.unit_prefix), c.rc, c.cam, out_rgb, c.head(), mma_on, c.st);
        if (rc) return rc;
        prof_mark(5, c.st);
        if (!(params->flags & SPLOTCH_RAW_SUM)) {
            rc = launch_normalize(out_rgb, out_rgb, n_values, c.st);
            if (rc) return rc;
        }
    } else {
        rc = launch_raster_absorb(c.at<SplatAbs>(c.L.records), list, c.at<uint64_t>(c.L.bin_offset),
                                  c.at<uint32_t>(c.L.unit_prefix), c.rc, c.cam, c.at<float>(c.L.partials), c.head(), c.st);
        if (rc) return rc;
        prof_mark(5, c.st);
        rc = launch_merge_absorb(c.at<float>(c.L.partials), c.at<uint32_t>(c.L.unit_prefix), c.rc, c.cam, out_rgb, c.head(), c.st);
        if (rc) return rc;
    }
    zero_if_failed_kernel<<<sm_count() * 4, 256, 0, c.st>>>(out_rgb, (long long)n_values, c.head());
    SPLOTCH_LAUNCH_CHECK();
    prof_mark(kStages, c.st);
    return SPLOTCH_OK;
}

namespace splotch { namespace {
__global__ void copy_frame_status_kernel(const WorkHead *head, uint64_t *dst)
{
    dst[0] = (uint64_t)(int64_t)head->status;
    dst[1] = head->visible;
    dst[2] = head->pairs;
    dst[3] = 0ull;
}
} }

int splotch_render_batch(const splotch_particles *particles, int64_t n, const splotch_camera *cameras, int32_t n_cameras,
                         const splotch_colormap *colormap, const splotch_params *params, float *out_rgb,
                         uint64_t *frame_status, void *workspace, uint64_t workspace_bytes, uint64_t max_pairs, void *stream)
{
    if (!cameras || n_cameras < 0 || (n_cameras > 0 && !out_rgb)) return SPLOTCH_ERR_INVALID_ARG;
    if (frame_status && (reinterpret_cast<uintptr_t>(frame_status) & 7u)) return SPLOTCH_ERR_INVALID_ARG;
    // validate everything for every camera before enqueueing anything
    for (int32_t k = 0; k < n_cameras; ++k) {
        if (cameras[k].width != cameras[0].width || cameras[k].height != cameras[0].height) return SPLOTCH_ERR_INVALID_ARG;
        Ctx c;
        const int rc = setup(particles, n, &cameras[k], colormap, params, kBlockShift, workspace, workspace_bytes, max_pairs,
                             true, stream, &c);
        if (rc) return rc;
    }
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    for (int32_t k = 0; k < n_cameras; ++k) {
        const size_t frame = (size_t)cameras[k].width * cameras[k].height * 3;
        const int rc = splotch_render(particles, n, &cameras[k], colormap, params, out_rgb + (size_t)k * frame, workspace,
                                      workspace_bytes, max_pairs, stream);
        if (rc) return rc;
        if (frame_status) {
            copy_frame_status_kernel<<<1, 1, 0, st>>>(reinterpret_cast<const WorkHead *>(workspace), frame_status + 4 * (size_t)k);
            SPLOTCH_LAUNCH_CHECK();
        }
    }
    return SPLOTCH_OK;
}

int splotch_profile_enable(int on)
{
    std::lock_guard<std::mutex> lock(g_prof_mutex);
    g_prof.on = on != 0;
    g_prof.calls = 0;
    return SPLOTCH_OK;
}

int splotch_profile_read(double *stage_ms, int64_t *calls)
{
    if (!stage_ms) return SPLOTCH_ERR_INVALID_ARG;
    std::lock_guard<std::mutex> lock(g_prof_mutex);
    for (int k = 0; k < kStages; ++k) stage_ms[k] = 0.0;
    const int n = g_prof.calls;
    if (calls) *calls = n;
    if (n == 0) return SPLOTCH_OK;
    SPLOTCH_CUDA_TRY(cudaEventSynchronize(g_prof.ev[n - 1][kStages]));
    for (int c = 0; c < n; ++c)
        for (int k = 0; k < kStages; ++k) {
            float ms = 0.f;
            SPLOTCH_CUDA_TRY(cudaEventElapsedTime(&ms, g_prof.ev[c][k], g_prof.ev[c][k + 1]));
            stage_ms[k] += (double)ms / n;
        }
    return SPLOTCH_OK;
}

unsigned long long splotch_launch_count(void) { return g_launch_count.load(std::memory_order_relaxed); }

int splotch_workspace_status(const void *workspace, void *stream, int32_t *status, uint64_t *visible, uint64_t *pairs)
{
    if (!workspace) return SPLOTCH_ERR_INVALID_ARG;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    WorkHead h;
    SPLOTCH_CUDA_TRY(cudaMemcpyAsync(&h, workspace, sizeof(h), cudaMemcpyDeviceToHost, st));
    SPLOTCH_CUDA_TRY(cudaStreamSynchronize(st));
    if (status) *status = h.status;
    if (visible) *visible = h.visible;
    if (pairs) *pairs = h.pairs;
    return SPLOTCH_OK;
}

int splotch_count_pairs(const splotch_particles *particles, int64_t n, const splotch_camera *camera,
                        const splotch_colormap *colormap, const splotch_params *params, void *workspace,
                        uint64_t workspace_bytes, uint64_t *pairs_host, uint64_t *visible_host, void *stream)
{
    Ctx c;
    int rc = setup(particles, n, camera, colormap, params, kBlockShift, workspace, workspace_bytes, 0, false, stream, &c);
    if (rc) return rc;
    rc = run_front(c, particles, n, colormap, ~0ull, kChunkAdd, nullptr);
    if (rc) return rc;
    return splotch_workspace_status(workspace, stream, nullptr, visible_host, pairs_host);
}

int splotch_field_range(const float *values, int64_t n, int32_t log_scale, float *range, void *stream)
{
    if (n < 0 || !range || (n > 0 && !values)) return SPLOTCH_ERR_INVALID_ARG;
    return launch_field_range(values, n, log_scale != 0, range, reinterpret_cast<cudaStream_t>(stream));
}

int splotch_field_normalize(const float *values, int64_t n, int32_t log_scale, const float *range, float *out, void *stream)
{
    if (n < 0 || !range || (n > 0 && (!values || !out))) return SPLOTCH_ERR_INVALID_ARG;
    return launch_field_normalize(values, n, log_scale != 0, range, out, reinterpret_cast<cudaStream_t>(stream));
}

int splotch_tonemap_rgb8(const float *rgb, int64_t n_values, float gamma, uint8_t *out, void *stream)
{
    if (n_values < 0 || !(gamma > 0.0f) || (n_values > 0 && (!rgb || !out))) return SPLOTCH_ERR_INVALID_ARG;
    return launch_tonemap_rgb8(rgb, n_values, gamma, out, reinterpret_cast<cudaStream_t>(stream));
}

int splotch_normalize(const float *S, float *out, int64_t n_values, void *stream)
{
    if (n_values < 0 || (n_values > 0 && (!S || !out))) return SPLOTCH_ERR_INVALID_ARG;
    return launch_normalize(S, out, n_values, reinterpret_cast<cudaStream_t>(stream));
}

// ---------------------------------------------------------------------------------------------
// host-buffer variant (end-to-end measurement, bench.py "e2e")
// ---------------------------------------------------------------------------------------------
namespace {
struct HostLayout { uint64_t part[6], type, lutE, lutA, image, inner, total; };

HostLayout make_host_layout(int64_t n, const splotch_camera *camera, const splotch_colormap *cm, bool has_type,
                            uint64_t inner_bytes)
{
    HostLayout H;
    uint64_t off = 0;
    auto take = [&](uint64_t bytes) { const uint64_t at = off; off += align_up(bytes > 0 ? bytes : 1, 256); return at; };
    const uint64_t nn = (uint64_t)(n > 0 ? n : 1);
    H.inner = take(inner_bytes);
    for (int k = 0; k < 6; ++k) H.part[k] = take(nn * 4);
    H.type = take(has_type ? nn : 1);
    const uint64_t lut = (uint64_t)cm->n_types * cm->n_entries * 3 * 4;
    H.lutE = take(lut);
    H.lutA = take(lut);
    H.image = take((uint64_t)camera->width * camera->height * 12);
    H.total = off;
    return H;
}
}  // namespace

int splotch_workspace_bytes_host(int64_t n, const splotch_camera *camera, const splotch_colormap *colormap_host,
                                 const splotch_params *params, uint64_t max_pairs, uint64_t *bytes)
{
    if (!bytes || !colormap_host) return SPLOTCH_ERR_INVALID_ARG;
    uint64_t inner = 0;
    int rc = splotch_workspace_bytes(n, camera, params, max_pairs, &inner);
    if (rc) return rc;
    rc = check_colormap(colormap_host, params->mode);
    if (rc) return rc;
    *bytes = make_host_layout(n, camera, colormap_host, true, inner).total;
    return SPLOTCH_OK;
}

int splotch_render_host_async(const splotch_particles *ph, int64_t n, const splotch_camera *camera,
                              const splotch_colormap *cmh, const splotch_params *params, float *out_rgb_host,
                              void *workspace, uint64_t workspace_bytes, uint64_t max_pairs, void *stream)
{
    if (!out_rgb_host || !workspace || !params) return SPLOTCH_ERR_INVALID_ARG;
    if (ph && (ph->vr || !ph->colval) && n > 0) return SPLOTCH_ERR_INVALID_ARG;     // host path: scalar colouring only
    int rc = check_particles(ph, n);
    if (rc) return rc;
    rc = check_colormap(cmh, params->mode);
    if (rc) return rc;
    uint64_t inner = 0;
    rc = splotch_workspace_bytes(n, camera, params, max_pairs, &inner);
    if (rc) return rc;
    const HostLayout H = make_host_layout(n, camera, cmh, true, inner);
    if (workspace_bytes < H.total) return SPLOTCH_ERR_WORKSPACE;
    char *ws = reinterpret_cast<char *>(workspace);
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    const float *src[6] = { ph ? ph->x : nullptr, ph ? ph->y : nullptr, ph ? ph->z : nullptr,
                            ph ? ph->r : nullptr, ph ? ph->I : nullptr, ph ? ph->colval : nullptr };
    if (n > 0) {
        for (int k = 0; k < 6; ++k)
            SPLOTCH_CUDA_TRY(cudaMemcpyAsync(ws + H.part[k], src[k], (size_t)n * 4, cudaMemcpyHostToDevice, st));
        if (ph->type) SPLOTCH_CUDA_TRY(cudaMemcpyAsync(ws + H.type, ph->type, (size_t)n, cudaMemcpyHostToDevice, st));
    }
    const size_t lut = (size_t)cmh->n_types * cmh->n_entries * 3 * 4;
    SPLOTCH_CUDA_TRY(cudaMemcpyAsync(ws + H.lutE, cmh->emission, lut, cudaMemcpyHostToDevice, st));
    if (cmh->absorption) SPLOTCH_CUDA_TRY(cudaMemcpyAsync(ws + H.lutA, cmh->absorption, lut, cudaMemcpyHostToDevice, st));
    splotch_particles pd = { reinterpret_cast<float *>(ws + H.part[0]), reinterpret_cast<float *>(ws + H.part[1]),
                             reinterpret_cast<float *>(ws + H.part[2]), reinterpret_cast<float *>(ws + H.part[3]),
                             reinterpret_cast<float *>(ws + H.part[4]), reinterpret_cast<float *>(ws + H.part[5]),
                             (ph && ph->type) ? reinterpret_cast<uint8_t *>(ws + H.type) : nullptr };
    splotch_colormap cmd = { reinterpret_cast<float *>(ws + H.lutE),
                             cmh->absorption ? reinterpret_cast<float *>(ws + H.lutA) : nullptr, cmh->n_entries, cmh->n_types };
    float *img = reinterpret_cast<float *>(ws + H.image);
    rc = splotch_render(&pd, n, camera, &cmd, params, img, ws + H.inner, inner, max_pairs, stream);
    if (rc) return rc;
    SPLOTCH_CUDA_TRY(cudaMemcpyAsync(out_rgb_host, img, (size_t)camera->width * camera->height * 12, cudaMemcpyDeviceToHost, st));
    return SPLOTCH_OK;
}

int splotch_render_host(const splotch_particles *ph, int64_t n, const splotch_camera *camera,
                        const splotch_colormap *cmh, const splotch_params *params, float *out_rgb_host,
                        void *workspace, uint64_t workspace_bytes, uint64_t max_pairs, void *stream)
{
    int rc = splotch_render_host_async(ph, n, camera, cmh, params, out_rgb_host, workspace, workspace_bytes, max_pairs, stream);
    if (rc) return rc;
    int32_t status = SPLOTCH_OK;       // the status head sits at the start of the workspace in both layouts
    rc = splotch_workspace_status(workspace, stream, &status, nullptr, nullptr);
    return rc ? rc : status;
}

// ---------------------------------------------------------------------------------------------
// test-only exports
// ---------------------------------------------------------------------------------------------
int splotch_debug_project(const splotch_particles *particles, int64_t n, const splotch_camera *camera,
                          const splotch_colormap *colormap, const splotch_params *params, void *workspace,
                          uint64_t workspace_bytes, float *sx, float *sy, float *sigma_s, float *R, uint32_t *zkey,
                          int32_t *pix_bbox, uint8_t *visible, void *stream)
{
    Ctx c;
    int rc = setup(particles, n, camera, colormap, params, kBlockShift, workspace, workspace_bytes, 0, false, stream, &c);
    if (rc) return rc;
    if (pix_bbox && (reinterpret_cast<uintptr_t>(pix_bbox) & 15u)) return SPLOTCH_ERR_INVALID_ARG;
    DebugProjectOut d = { sx, sy, sigma_s, R, zkey, pix_bbox, visible };
    return run_front(c, particles, n, colormap, ~0ull, kChunkAdd, &d);
}

int splotch_debug_bins(const splotch_particles *particles, int64_t n, const splotch_camera *camera,
                       const splotch_colormap *colormap, const splotch_params *params, void *workspace,
                       uint64_t workspace_bytes, int32_t bin_shift, uint32_t *tile_count, uint64_t *tile_offset,
                       uint32_t *member_ids, uint64_t max_members, void *stream)
{
    if (bin_shift < 2 || bin_shift > 10 || !tile_count || !tile_offset) return SPLOTCH_ERR_INVALID_ARG;
    Ctx c;
    int rc = setup(particles, n, camera, colormap, params, bin_shift, workspace, workspace_bytes, max_members, false, stream, &c);
    if (rc) return rc;
    rc = run_front(c, particles, n, colormap, member_ids ? max_members : ~0ull, kChunkAdd, nullptr);
    if (rc) return rc;
    SPLOTCH_CUDA_TRY(cudaMemcpyAsync(tile_count, c.ws + c.L.bin_count, (size_t)c.n_bins * 4, cudaMemcpyDeviceToDevice, c.st));
    SPLOTCH_CUDA_TRY(cudaMemcpyAsync(tile_offset, c.ws + c.L.bin_offset, (size_t)(c.n_bins + 1) * 8, cudaMemcpyDeviceToDevice, c.st));
    if (member_ids && max_members > 0) {
        uint32_t *list = nullptr;
        rc = run_lists(c, n, max_members, &list);
        if (rc) return rc;
        copy_members_kernel<<<sm_count() * 4, 256, 0, c.st>>>(list, member_ids, c.head(), (unsigned long long)max_members);
        SPLOTCH_LAUNCH_CHECK();
    }
    return SPLOTCH_OK;
}

int splotch_debug_stats(const splotch_particles *particles, int64_t n, const splotch_camera *camera,
                        const splotch_colormap *colormap, const splotch_params *params, void *workspace,
                        uint64_t workspace_bytes, int32_t bin_shift, uint64_t *visible_host, uint64_t *pairs_host,
                        uint64_t *updates_host, void *stream)
{
    if (bin_shift < 2 || bin_shift > 10) return SPLOTCH_ERR_INVALID_ARG;
    Ctx c;
    int rc = setup(particles, n, camera, colormap, params, bin_shift, workspace, workspace_bytes, 0, false, stream, &c);
    if (rc) return rc;
    rc = run_front(c, particles, n, colormap, ~0ull, kChunkAdd, nullptr);
    if (rc) return rc;
    const int rec_bytes = c.rc.mode == SPLOTCH_ABSORB ? (int)sizeof(SplatAbs) : (int)sizeof(SplatAdd);
    rc = launch_count_updates(c.ws + c.L.records, rec_bytes, n, c.cam, c.rc.thr, c.head(), c.st);
    if (rc) return rc;
    WorkHead h;
    SPLOTCH_CUDA_TRY(cudaMemcpyAsync(&h, c.ws + c.L.head, sizeof(h), cudaMemcpyDeviceToHost, c.st));
    SPLOTCH_CUDA_TRY(cudaStreamSynchronize(c.st));
    if (visible_host) *visible_host = h.visible;
    if (pairs_host) *pairs_host = h.pairs;
    if (updates_host) *updates_host = h.updates;
    return SPLOTCH_OK;
}

int splotch_debug_tensor_stats(const splotch_particles *particles, int64_t n, const splotch_camera *camera,
                               const splotch_colormap *colormap, const splotch_params *params, void *workspace,
                               uint64_t workspace_bytes, uint64_t *updates_tensor_host, int32_t *tensor_on_host,
                               float *share_host, void *stream)
{
    if (!params || params->mode != SPLOTCH_ADDITIVE) return SPLOTCH_ERR_INVALID_ARG;
    Ctx c;
    int rc = setup(particles, n, camera, colormap, params, kBlockShift, workspace, workspace_bytes, 0, false, stream, &c);
    if (rc) return rc;
    rc = run_front(c, particles, n, colormap, ~0ull, kChunkAdd, nullptr);
    if (rc) return rc;
    rc = launch_count_tensor_updates(c.at<SplatAdd>(c.L.records), n, c.rc, c.cam, c.head(), c.st);
    if (rc) return rc;
    WorkHead h;
    SPLOTCH_CUDA_TRY(cudaMemcpyAsync(&h, c.ws + c.L.head, sizeof(h), cudaMemcpyDeviceToHost, c.st));
    SPLOTCH_CUDA_TRY(cudaStreamSynchronize(c.st));
    if (updates_tensor_host) *updates_tensor_host = h.updates_tensor;
    if (tensor_on_host) *tensor_on_host = (int32_t)h.tensor_on;
    if (share_host) *share_host = h.area_total > 0.0f ? h.area_tensor / h.area_total : 0.0f;
    return SPLOTCH_OK;
}

int splotch_debug_scan(const uint32_t *in, uint64_t *out, int64_t n, void *scratch, uint64_t scratch_bytes, void *stream)
{
    if (n < 0 || !out || (n > 0 && !in) || !scratch) return SPLOTCH_ERR_INVALID_ARG;
    if (scratch_bytes < scan_scratch_bytes(n)) return SPLOTCH_ERR_WORKSPACE;
    return launch_scan_u32_u64(in, out, n, scratch, reinterpret_cast<cudaStream_t>(stream));
}

uint64_t splotch_sort_scratch_bytes(int64_t n) { return sort_scratch_bytes(n > 0 ? n : 1); }

int splotch_debug_sort_pairs(uint32_t *keys, uint32_t *vals, uint32_t *keys_tmp, uint32_t *vals_tmp, int64_t n,
                             int32_t key_bits, void *scratch, uint64_t scratch_bytes, void *stream)
{
    if (n < 0 || key_bits < 1 || key_bits > 32) return SPLOTCH_ERR_INVALID_ARG;
    if (n == 0) return SPLOTCH_OK;
    if (!keys || !vals || !keys_tmp || !vals_tmp || !scratch) return SPLOTCH_ERR_INVALID_ARG;
    if (scratch_bytes < sort_scratch_bytes(n)) return SPLOTCH_ERR_WORKSPACE;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    bool in_tmp = false;
    int rc = launch_sort_pairs(keys, vals, keys_tmp, vals_tmp, n, nullptr, key_bits, scratch, st, &in_tmp);
    if (rc) return rc;
    if (in_tmp) {
        SPLOTCH_CUDA_TRY(cudaMemcpyAsync(keys, keys_tmp, (size_t)n * 4, cudaMemcpyDeviceToDevice, st));
        SPLOTCH_CUDA_TRY(cudaMemcpyAsync(vals, vals_tmp, (size_t)n * 4, cudaMemcpyDeviceToDevice, st));
    }
    return SPLOTCH_OK;
}

}  // extern "C"
