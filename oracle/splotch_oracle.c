/*
 * splotch_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, double-precision CPU statement of what the Splotch render path computes,
 * written from the paper (/root/reference/PAPER.md, arxiv 1004.1302) and from the readings
 * R1..R15 of SURVEY.md section 8(c) / DESIGN.md "Readings".  It shares no code, header, table
 * or helper with the CUDA library under paper_1004_1302_b200/csrc and neither includes the
 * other.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may call it.
 *
 * Two references live here (SURVEY.md 8(c) "Two references"):
 *
 *   1. The PIXEL ORACLE (orc_splat_table, orc_render): double precision everywhere, the
 *      definitions written out with no blocking, fusion or reordering.
 *        - density of one particle      rho_p(r) = rho_0p exp(-r^2/sigma_p^2), zero beyond
 *          f sigma_p; rays farther than f sigma_p are unaffected       PAPER.md:69 (sec. 2)
 *        - R, G, B independent
 *        - dI/dx = (E_p - A_p I) rho_p(x)                               PAPER.md:73 (Eq. 1)
 *        - E_p = A_p recommended / necessary for the parallel code
 *        - scalar -> colour through a look-up table; optical depth
 *          modulated by another scalar
 *        - "transformation into screen coordinates, assigning of
 *          colours and rendering"
 *
 *   2. The CANONICAL FP32 PROJECTOR / BINNER (orc_project_f32, orc_bins): a fixed sequence of
 *      IEEE binary32 operations that defines every integer the CUDA path must reproduce
 *      bit-exactly (visible set, pixel bounding box, bin membership, counts, offsets, depth
 *      key).  Compiled with -ffp-contract=off; fused operations are written as fmaf().
 *
 * Parity pins (tests/test_oracle_*.py): P1..P12 of SURVEY.md 8(c) -- the analytic Gaussian
 * line integral, the closed-form flux of a splat, energy conservation, permutation
 * invariance, brute-force RK4 integration of Eq. (1) on tiny inputs, absorb == additive when
 * A == E, front-to-back == back-to-front, camera conventions, scale invariance, LUT nodes,
 * tie order; P17 per-type table offset and per-type brightness / abs_brightness (two types
 * with different tables, expected values written by hand from the inputs); P18 the region-of-
 * interest path (off-origin ROI == hand-evaluated single-splat closed form at the ROI's pixel
 * centres, and == the crop of the full frame bit for bit, both modes).  Conventions the paper leaves open (f = 3 default, rho_0 = I, z_near, fov axis,
 * image orientation, slab reading under overlap) are "parity unpinned" by the paper: they
 * are pinned only by DESIGN.md.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_OK 0
#define ORC_ERR_ARG (-1)
#define ORC_ERR_MEM (-2)
#define ORC_MAX_TYPES 4

/* cam[10] = eye(3), lookat(3), up(3), fov_deg -- the same float values the C ABI receives */

/* ---------------------------------------------------------------------------------------
 * O1 camera basis (reading R1, R2): fwd = normalise(lookat - eye); right = normalise(fwd x up);
 * upv = right x fwd; F = (W/2) / tan(fov/2), fov the full horizontal angle.
 * ------------------------------------------------------------------------------------- */
int orc_camera_basis(const float *cam, int32_t W, int32_t H, double *right, double *upv, double *fwd,
                     double *F)
{
    double e[3], l[3], u[3];
    for (int k = 0; k < 3; ++k) { e[k] = cam[k]; l[k] = cam[3 + k]; u[k] = cam[6 + k]; }
    double fov = cam[9];
    if (W <= 0 || H <= 0 || !(fov > 0.0) || !(fov < 180.0)) return ORC_ERR_ARG;
    double f[3] = { l[0] - e[0], l[1] - e[1], l[2] - e[2] };
    double fn = sqrt(f[0] * f[0] + f[1] * f[1] + f[2] * f[2]);
    if (!(fn > 0.0)) return ORC_ERR_ARG;
    for (int k = 0; k < 3; ++k) f[k] /= fn;
    double r[3] = { f[1] * u[2] - f[2] * u[1], f[2] * u[0] - f[0] * u[2], f[0] * u[1] - f[1] * u[0] };
    double rn = sqrt(r[0] * r[0] + r[1] * r[1] + r[2] * r[2]);
    if (!(rn > 0.0)) return ORC_ERR_ARG;
    for (int k = 0; k < 3; ++k) r[k] /= rn;
    double v[3] = { r[1] * f[2] - r[2] * f[1], r[2] * f[0] - r[0] * f[2], r[0] * f[1] - r[1] * f[0] };
    for (int k = 0; k < 3; ++k) { right[k] = r[k]; upv[k] = v[k]; fwd[k] = f[k]; }
    const double pi = 3.14159265358979323846;
    *F = (0.5 * (double)W) / tan(0.5 * fov * pi / 180.0);
    return ORC_OK;
}

static int finite6(float a, float b, float c, float d, float e, float f)
{
    return isfinite(a) && isfinite(b) && isfinite(c) && isfinite(d) && isfinite(e) && isfinite(f);
}

/* ---------------------------------------------------------------------------------------
 * Canonical fp32 projector (SURVEY.md 8(c) "Canonical fp32 sequence", DESIGN.md "Canonical
 * sequence").  Every operation is one correctly rounded binary32 operation.
 *   visible[p] = 1 iff all six fields finite, r > 0, type < n_types, zc > z_near, ss > 0,
 *                R finite and the pixel box is non-empty.
 *   bbox[4p..] = i0, i1, j0, j1 (inclusive pixel box; column i, row j; row 0 = top)
 *   zkey[p]    = bit pattern of zc (positive floats order as unsigned integers), R11.
 * Outputs for culled particles: visible 0, everything else 0.
 * ------------------------------------------------------------------------------------- */
int orc_project_f32(int64_t n, const float *x, const float *y, const float *z, const float *r,
                    const float *I, const float *colval, const uint8_t *type, int32_t n_types,
                    const float *cam, int32_t W, int32_t H, float support_f, float z_near,
                    float *sx, float *sy, float *ss, float *R, uint32_t *zkey, int32_t *bbox,
                    uint8_t *visible)
{
    double rt[3], uv[3], fw[3], Fd;
    int rc = orc_camera_basis(cam, W, H, rt, uv, fw, &Fd);
    if (rc) return rc;
    const float rx = (float)rt[0], ry = (float)rt[1], rz = (float)rt[2];
    const float ux = (float)uv[0], uy = (float)uv[1], uz = (float)uv[2];
    const float fx = (float)fw[0], fy = (float)fw[1], fz = (float)fw[2];
    const float ex = cam[0], ey = cam[1], ez = cam[2];
    const float F = (float)Fd;
    const float cx = (float)(0.5 * (double)W), cy = (float)(0.5 * (double)H);
    const float Wf = (float)W, Hf = (float)H;
#pragma omp parallel for schedule(static)
    for (int64_t p = 0; p < n; ++p) {
        sx[p] = sy[p] = ss[p] = R[p] = 0.0f; zkey[p] = 0u; visible[p] = 0;
        bbox[4 * p] = bbox[4 * p + 1] = bbox[4 * p + 2] = bbox[4 * p + 3] = 0;
        int ty = type ? (int)type[p] : 0;
        if (!finite6(x[p], y[p], z[p], r[p], I[p], colval[p]) || !(r[p] > 0.0f) || ty >= n_types) continue;
        float dx = x[p] - ex, dy = y[p] - ey, dz = z[p] - ez;
        float xc = fmaf(dz, rz, fmaf(dy, ry, dx * rx));
        float yc = fmaf(dz, uz, fmaf(dy, uy, dx * ux));
        float zc = fmaf(dz, fz, fmaf(dy, fy, dx * fx));
        if (!(zc > z_near)) continue;
        float q = F / zc;
        float psx = fmaf(xc, q, cx);
        float psy = fmaf(-yc, q, cy);
        float pss = r[p] * q;
        float pR = support_f * pss;
        if (!(pss > 0.0f) || !isfinite(pR)) continue;   /* degenerate footprint: culled (R6) */
        /* pixel (i, j) has its centre at (i + 1/2, j + 1/2): covered candidates satisfy
           sx - R <= i + 1/2 <= sx + R */
        float i0f = fminf(fmaxf(ceilf((psx - pR) - 0.5f), 0.0f), Wf);
        float i1f = fmaxf(fminf(floorf((psx + pR) - 0.5f), Wf - 1.0f), -1.0f);
        float j0f = fminf(fmaxf(ceilf((psy - pR) - 0.5f), 0.0f), Hf);
        float j1f = fmaxf(fminf(floorf((psy + pR) - 0.5f), Hf - 1.0f), -1.0f);
        if (!(i0f <= i1f) || !(j0f <= j1f)) continue;
        sx[p] = psx; sy[p] = psy; ss[p] = pss; R[p] = pR;
        uint32_t kb; memcpy(&kb, &zc, 4); zkey[p] = kb;
        bbox[4 * p] = (int32_t)i0f; bbox[4 * p + 1] = (int32_t)i1f;
        bbox[4 * p + 2] = (int32_t)j0f; bbox[4 * p + 3] = (int32_t)j1f;
        visible[p] = 1;
    }
    return ORC_OK;
}

/* ---------------------------------------------------------------------------------------
 * Depth order R11: ascending (zkey, particle index) over the visible particles.
 * order[0..V) receives particle indices, nearest first.  Returns V.
 * ------------------------------------------------------------------------------------- */
typedef struct { uint32_t key; uint32_t pad; int64_t idx; } orc_keyidx;

static int cmp_keyidx(const void *a, const void *b)
{
    const orc_keyidx *p = (const orc_keyidx *)a, *q = (const orc_keyidx *)b;
    if (p->key != q->key) return p->key < q->key ? -1 : 1;
    if (p->idx != q->idx) return p->idx < q->idx ? -1 : 1;
    return 0;
}

int64_t orc_depth_order(int64_t n, const uint32_t *zkey, const uint8_t *visible, int64_t *order)
{
    int64_t V = 0;
    for (int64_t p = 0; p < n; ++p) V += visible[p] ? 1 : 0;
    orc_keyidx *a = (orc_keyidx *)malloc((size_t)(V > 0 ? V : 1) * sizeof(orc_keyidx));
    if (!a) return ORC_ERR_MEM;
    int64_t k = 0;
    for (int64_t p = 0; p < n; ++p)
        if (visible[p]) { a[k].key = zkey[p]; a[k].pad = 0; a[k].idx = p; ++k; }
    qsort(a, (size_t)V, sizeof(orc_keyidx), cmp_keyidx);
    for (k = 0; k < V; ++k) order[k] = a[k].idx;
    free(a);
    return V;
}

/* ---------------------------------------------------------------------------------------
 * Canonical binner (B-rules): a visible splat belongs to EVERY bin of its bin bounding box
 * (i0 >> shift .. i1 >> shift) x (j0 >> shift .. j1 >> shift); bin index = by * nbx + bx with
 * nbx = ceil(W / 2^shift).  Pass 1 (members == NULL) fills counts[T] and offsets[T+1]
 * (exclusive prefix sum, 64-bit); pass 2 (members != NULL, offsets from pass 1) fills the
 * member lists.  Particles are visited in `order[0..n_order)` if order != NULL (absorb mode:
 * the depth order), else in index order over all n.
 * ------------------------------------------------------------------------------------- */
int orc_bins(int64_t n, const int32_t *bbox, const uint8_t *visible, const int64_t *order,
             int64_t n_order, int32_t shift, int32_t W, int32_t H, uint32_t *counts,
             uint64_t *offsets, uint32_t *members)
{
    const int32_t bs = 1 << shift;
    const int64_t nbx = (W + bs - 1) >> shift, nby = (H + bs - 1) >> shift, T = nbx * nby;
    const int64_t m = order ? n_order : n;
    if (!members) {
        memset(counts, 0, (size_t)T * sizeof(uint32_t));
        for (int64_t k = 0; k < m; ++k) {
            int64_t p = order ? order[k] : k;
            if (!visible[p]) continue;
            const int32_t *b = bbox + 4 * p;
            for (int32_t by = b[2] >> shift; by <= (b[3] >> shift); ++by)
                for (int32_t bx = b[0] >> shift; bx <= (b[1] >> shift); ++bx)
                    counts[by * nbx + bx] += 1u;
        }
        uint64_t acc = 0;
        for (int64_t t = 0; t < T; ++t) { offsets[t] = acc; acc += counts[t]; }
        offsets[T] = acc;
        return ORC_OK;
    }
    uint64_t *cur = (uint64_t *)malloc((size_t)T * sizeof(uint64_t));
    if (!cur) return ORC_ERR_MEM;
    memcpy(cur, offsets, (size_t)T * sizeof(uint64_t));
    for (int64_t k = 0; k < m; ++k) {
        int64_t p = order ? order[k] : k;
        if (!visible[p]) continue;
        const int32_t *b = bbox + 4 * p;
        for (int32_t by = b[2] >> shift; by <= (b[3] >> shift); ++by)
            for (int32_t bx = b[0] >> shift; bx <= (b[1] >> shift); ++bx)
                members[cur[by * nbx + bx]++] = (uint32_t)p;
    }
    free(cur);
    return ORC_OK;
}

/* ---------------------------------------------------------------------------------------
 * O5 colour (reading R7): piece-wise linear look-up between n_entries equally spaced nodes on
 * [0, 1]; colval clamped to [0, 1].  tab = n_types x n_entries x 3 (RGB interleaved).
 * ------------------------------------------------------------------------------------- */
static void lut_sample(const float *tab, int32_t n_entries, int32_t type, double v, double *rgb)
{
    double c = v < 0.0 ? 0.0 : (v > 1.0 ? 1.0 : v);
    double u = c * (double)(n_entries - 1);
    int64_t k = (int64_t)floor(u);
    if (k > n_entries - 2) k = n_entries - 2;
    double t = u - (double)k;
    const float *e0 = tab + ((int64_t)type * n_entries + k) * 3, *e1 = e0 + 3;
    for (int c3 = 0; c3 < 3; ++c3) rgb[c3] = (1.0 - t) * (double)e0[c3] + t * (double)e1[c3];
}

/* one row of the splat table, all double */
typedef struct {
    double sx, sy, sigma, R, tau0;   /* O4 screen position, sigma_s, R = f sigma_s; O6 peak column I r sqrt(pi) */
    double E[3], A[3];               /* O5 */
} orc_splat;

/* ---------------------------------------------------------------------------------------
 * Stage 1 of the pixel oracle: O2..O6 per particle, in double.
 *   O2 d = p - eye; xc = d.right, yc = d.upv, zc = d.fwd
 *   O3 cull: non-finite field, r <= 0, bad type, zc <= z_near.  The near-plane decision is
 *      taken on the canonical fp32 zc (`near_ok`, from orc_project_f32) so that both sides
 *      decide this one integer in the same precision; everything else here is double.
 *   O4 sx = W/2 + F xc/zc; sy = H/2 - F yc/zc; sigma_s = F r / zc; R = f sigma_s
 *   O6 tau0 = I r sqrt(pi)  (line integral of rho_0 exp(-s^2/sigma^2), rho_0 = I, sigma = r)
 * table = n x 11 doubles (sx, sy, sigma, R, tau0, E rgb, A rgb); ok[p] = 1 if not culled.
 * ------------------------------------------------------------------------------------- */
int orc_splat_table(int64_t n, const float *x, const float *y, const float *z, const float *r,
                    const float *I, const float *colval, const uint8_t *type, const float *cam,
                    int32_t W, int32_t H, const float *lutE, const float *lutA, int32_t n_entries,
                    int32_t n_types, const float *brightness, const float *abs_brightness,
                    int32_t mode, float support_f, float z_near, double *table, uint8_t *ok)
{
    double rt[3], uv[3], fw[3], F;
    int rc = orc_camera_basis(cam, W, H, rt, uv, fw, &F);
    if (rc) return rc;
    if (n_entries < 2 || n_types < 1 || n_types > ORC_MAX_TYPES || !(support_f > 0.0f) || !lutE) return ORC_ERR_ARG;
    if (mode == 1 && !lutA) return ORC_ERR_ARG;
    /* canonical fp32 basis for the near-plane decision */
    const float fxf = (float)fw[0], fyf = (float)fw[1], fzf = (float)fw[2];
    const double sqrt_pi = 1.77245385090551602730;
#pragma omp parallel for schedule(static)
    for (int64_t p = 0; p < n; ++p) {
        double *t = table + 11 * p;
        for (int k = 0; k < 11; ++k) t[k] = 0.0;
        ok[p] = 0;
        int ty = type ? (int)type[p] : 0;
        if (!finite6(x[p], y[p], z[p], r[p], I[p], colval[p]) || !(r[p] > 0.0f) || ty >= n_types) continue;
        {   /* near plane in canonical fp32 */
            float dxf = x[p] - cam[0], dyf = y[p] - cam[1], dzf = z[p] - cam[2];
            float zcf = fmaf(dzf, fzf, fmaf(dyf, fyf, dxf * fxf));
            if (!(zcf > z_near)) continue;
        }
        double d[3] = { (double)x[p] - (double)cam[0], (double)y[p] - (double)cam[1], (double)z[p] - (double)cam[2] };
        double xc = d[0] * rt[0] + d[1] * rt[1] + d[2] * rt[2];
        double yc = d[0] * uv[0] + d[1] * uv[1] + d[2] * uv[2];
        double zc = d[0] * fw[0] + d[1] * fw[1] + d[2] * fw[2];
        if (!(zc > 0.0)) continue;
        t[0] = 0.5 * (double)W + F * xc / zc;
        t[1] = 0.5 * (double)H - F * yc / zc;
        t[2] = F * (double)r[p] / zc;
        t[3] = (double)support_f * t[2];
        t[4] = (double)I[p] * (double)r[p] * sqrt_pi;
        double le[3], la[3];
        lut_sample(lutE, n_entries, ty, (double)colval[p], le);
        for (int c = 0; c < 3; ++c) t[5 + c] = (double)brightness[ty] * le[c];
        if (mode == 1) {
            lut_sample(lutA, n_entries, ty, (double)colval[p], la);
            for (int c = 0; c < 3; ++c) t[8 + c] = (double)abs_brightness[ty] * la[c];
        } else {
            for (int c = 0; c < 3; ++c) t[8 + c] = t[5 + c];   /* A == E */
        }
        ok[p] = 1;
    }
    return ORC_OK;
}

/* ---------------------------------------------------------------------------------------
 * Stage 2 of the pixel oracle: O6..O8 on the pixel rectangle roi = {x0, y0, x1, y1}
 * (columns x0..x1-1, rows y0..y1-1), out = (y1-y0) x (x1-x0) x 3 doubles, row 0 = top.
 *
 *   O6  tau_p(q) = tau0 exp(-d^2 / sigma_s^2) if d^2 <= R^2 else 0, q the pixel centre
 *       (i + 1/2, j + 1/2): truncation by impact parameter, R9.
 *   O7  additive (mode 0): S_c = sum_p E_pc tau_p; out_c = 1 - exp(-S_c), or S_c when `raw`.
 *       Exact solution of Eq. (1) with A = E: J = 1 - I obeys dJ/dx = -J sum_p E_p rho_p.
 *   O8  absorb (mode 1): particles in depth order (zkey, index), visited from the FARTHEST to
 *       the nearest (the direction Eq. (1) propagates).  Across one particle, with E_p, A_p
 *       constant, Eq. (1) integrates to
 *           I_c <- I_c exp(-u_c) + E_pc tau_p phi(u_c),  u_c = A_pc tau_p,
 *           phi(u) = (1 - exp(-u)) / u, phi(0) = 1            (slab reading R10, R15)
 *       The slab solution of Eq. (1) holds for either sign of u; negative I, E or A are
 *       unphysical but "used as given" (reading R20), so phi is evaluated for u < 0 as well.
 *
 * `seq[0..m)` lists the particles to visit: index order (additive) or depth order nearest
 * first (absorb; visited backwards).  Rows are split into bands over the OpenMP threads;
 * inside a band particles are visited strictly in sequence, so every pixel sees the
 * defined order.
 * ------------------------------------------------------------------------------------- */
static void render_rows(const double *table, const int64_t *seq, int64_t m, int32_t mode,
                        const int32_t *roi, int32_t jb0, int32_t jb1, double *out)
{
    const int32_t x0 = roi[0], y0 = roi[1], x1 = roi[2];
    const int64_t rw = x1 - x0;
    for (int64_t kk = 0; kk < m; ++kk) {
        int64_t k = (mode == 1) ? (m - 1 - kk) : kk;          /* absorb: far -> near */
        const double *t = table + 11 * seq[k];
        const double sx = t[0], sy = t[1], sg = t[2], R = t[3], tau0 = t[4];
        const double R2 = R * R, inv_s2 = 1.0 / (sg * sg);
        double jl = floor(sy - R - 1.0), jh = ceil(sy + R + 1.0);
        double il = floor(sx - R - 1.0), ih = ceil(sx + R + 1.0);
        if (jh < (double)jb0 || jl > (double)(jb1 - 1) || ih < (double)x0 || il > (double)(x1 - 1)) continue;
        int32_t j0 = jl < (double)jb0 ? jb0 : (int32_t)jl, j1 = jh > (double)(jb1 - 1) ? jb1 - 1 : (int32_t)jh;
        int32_t i0 = il < (double)x0 ? x0 : (int32_t)il, i1 = ih > (double)(x1 - 1) ? x1 - 1 : (int32_t)ih;
        for (int32_t j = j0; j <= j1; ++j) {
            double dy = ((double)j + 0.5) - sy;
            for (int32_t i = i0; i <= i1; ++i) {
                double dx = ((double)i + 0.5) - sx;
                double d2 = dx * dx + dy * dy;
                if (!(d2 <= R2)) continue;
                double tau = tau0 * exp(-d2 * inv_s2);
                double *px = out + ((int64_t)(j - y0) * rw + (i - x0)) * 3;
                if (mode == 0) {
                    for (int c = 0; c < 3; ++c) px[c] += t[5 + c] * tau;
                } else {
                    for (int c = 0; c < 3; ++c) {
                        double u = t[8 + c] * tau;
                        double phi = (u != 0.0) ? (-expm1(-u) / u) : 1.0;   /* either sign of u: reading R20 */
                        px[c] = px[c] * exp(-u) + t[5 + c] * tau * phi;
                    }
                }
            }
        }
    }
}

int orc_render_table(const double *table, const int64_t *seq, int64_t m, int32_t mode, int32_t raw,
                     const int32_t *roi, double *out, int32_t *threads_used)
{
    const int32_t x0 = roi[0], y0 = roi[1], x1 = roi[2], y1 = roi[3];
    if (x1 <= x0 || y1 <= y0) return ORC_ERR_ARG;
    const int64_t rw = x1 - x0, rh = y1 - y0;
    memset(out, 0, (size_t)(rw * rh * 3) * sizeof(double));
    int nth = 1;
#ifdef _OPENMP
    nth = omp_get_max_threads();
#endif
    /* more bands than threads, handed out dynamically: dense rows do not serialise the run */
    int64_t nb = (int64_t)nth * 4;
    if (nb > rh) nb = rh;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t b = 0; b < nb; ++b) {
        int32_t jb0 = y0 + (int32_t)((rh * b) / nb), jb1 = y0 + (int32_t)((rh * (b + 1)) / nb);
        if (jb1 > jb0) render_rows(table, seq, m, mode, roi, jb0, jb1, out);
    }
    if (mode == 0 && !raw) {
        for (int64_t k = 0; k < rw * rh * 3; ++k) out[k] = -expm1(-out[k]);   /* 1 - exp(-S) */
    }
    if (threads_used) *threads_used = nth;
    return ORC_OK;
}

/* ---------------------------------------------------------------------------------------
 * The whole path in one call: stage 1, (absorb) depth order, stage 2 on `roi`.
 * Particles whose disc cannot reach the roi are dropped before stage 2 (they contribute 0).
 * ------------------------------------------------------------------------------------- */
int orc_render(int64_t n, const float *x, const float *y, const float *z, const float *r,
               const float *I, const float *colval, const uint8_t *type, const float *cam,
               int32_t W, int32_t H, const float *lutE, const float *lutA, int32_t n_entries,
               int32_t n_types, const float *brightness, const float *abs_brightness, int32_t mode,
               float support_f, float z_near, int32_t raw, const int32_t *roi, double *out,
               int32_t *threads_used)
{
    if (n < 0 || (mode != 0 && mode != 1)) return ORC_ERR_ARG;
    double *table = (double *)malloc((size_t)(n > 0 ? n : 1) * 11 * sizeof(double));
    uint8_t *ok = (uint8_t *)malloc((size_t)(n > 0 ? n : 1));
    int64_t *seq = (int64_t *)malloc((size_t)(n > 0 ? n : 1) * sizeof(int64_t));
    if (!table || !ok || !seq) { free(table); free(ok); free(seq); return ORC_ERR_MEM; }
    int rc = orc_splat_table(n, x, y, z, r, I, colval, type, cam, W, H, lutE, lutA, n_entries, n_types,
                             brightness, abs_brightness, mode, support_f, z_near, table, ok);
    int64_t m = 0;
    if (rc == ORC_OK) {
        /* keep particles whose disc (plus one pixel of slack) touches the roi */
        for (int64_t p = 0; p < n; ++p) {
            if (!ok[p]) continue;
            const double *t = table + 11 * p;
            if (t[0] + t[3] + 1.0 < (double)roi[0] || t[0] - t[3] - 1.0 > (double)roi[2] ||
                t[1] + t[3] + 1.0 < (double)roi[1] || t[1] - t[3] - 1.0 > (double)roi[3]) { ok[p] = 0; continue; }
            seq[m++] = p;
        }
        if (mode == 1) {
            /* R11: canonical fp32 depth key, ties by particle index */
            float *f4 = (float *)malloc((size_t)(n > 0 ? n : 1) * 4 * sizeof(float));
            uint32_t *zk = (uint32_t *)malloc((size_t)(n > 0 ? n : 1) * sizeof(uint32_t));
            int32_t *bb = (int32_t *)malloc((size_t)(n > 0 ? n : 1) * 4 * sizeof(int32_t));
            uint8_t *vis = (uint8_t *)malloc((size_t)(n > 0 ? n : 1));
            if (!f4 || !zk || !bb || !vis) rc = ORC_ERR_MEM;
            else {
                rc = orc_project_f32(n, x, y, z, r, I, colval, type, n_types, cam, W, H, support_f, z_near,
                                     f4, f4 + n, f4 + 2 * n, f4 + 3 * n, zk, bb, vis);
                if (rc == ORC_OK) {
                    /* order the kept set; the key of a kept particle is its canonical zc even if
                       the canonical box test dropped it */
                    for (int64_t p = 0; p < n; ++p) {
                        if (ok[p] && !vis[p]) {
                            double rt[3], uv[3], fw[3], Fd;
                            orc_camera_basis(cam, W, H, rt, uv, fw, &Fd);
                            float dxf = x[p] - cam[0], dyf = y[p] - cam[1], dzf = z[p] - cam[2];
                            float zcf = fmaf(dzf, (float)fw[2], fmaf(dyf, (float)fw[1], dxf * (float)fw[0]));
                            memcpy(&zk[p], &zcf, 4);
                        }
                    }
                    int64_t V = orc_depth_order(n, zk, ok, seq);
                    if (V < 0) rc = (int)V; else m = V;
                }
            }
            free(f4); free(zk); free(bb); free(vis);
        }
    }
    if (rc == ORC_OK) rc = orc_render_table(table, seq, m, mode, raw, roi, out, threads_used);
    free(table); free(ok); free(seq);
    return rc;
}

int orc_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
