/* vr_oracle.c -- CPU ORACLE, TEST INFRASTRUCTURE ONLY (see vr_oracle.h).
 *
 * Step-by-step restatement of the ray-casting path, PAPER.md:58-62 (Sec. 3.1
 * steps 1-5), in the order and notation of DESIGN.md Sec. 3 (S1..S13).
 * No blocking, no fusion, no reordering: one pixel at a time, one sample at a
 * time.  Every floating-point op is IEEE-754 binary32, round to nearest even;
 * fmaf() is the only fused op.  Build: gcc -std=c99 -O2 -ffp-contract=off
 * -fno-fast-math (oracle/build.py) so the compiler fuses / reassociates nothing.
 */
#include "vr_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    const float* V;        /* the cube as one array V[z][y][x], or NULL when it lives in bricks */
    const float* const* bricks;   /* S10 brick store: brick (bx,by,bz) at bricks[bx + nb0*(by + nb1*bz)] */
    int B;                 /* edge of the stored bricks in cells */
    int nb[3];             /* bricks per axis */
    int n[3];              /* nx, ny, nz */
    const float* lut;      /* n_lut * 4, straight (non-premultiplied) colours */
    float* alpha_tab;      /* EA: opacity-corrected alpha; MIP: raw alpha */
    int n_lut;
    float vmin, vmax, scale;
    float step, tau;
    int mode;
} vro_scene;

/* ---- R23: anisotropic voxel spacing (two sky axes and a frequency axis -- different units) -----
 * World space = voxel index x spacing; the camera, the step and the opacity per unit length live in
 * world space.  The ray is generated there (S1, S2: unit direction), then mapped into index space by
 * o_i = o * (1/s), d_i = d * (1/s) (one binary32 division 1/s per axis, one multiplication per
 * component); the parameter t stays the world-space distance, so S3-S6 run unchanged on (o_i, d_i).
 * Spacing (1, 1, 1) -- the default -- leaves every bit as it was (no multiplication is made).
 * Set before a render; not thread safe against a render in flight. */
static int vro_aniso = 0;
static float vro_inv_sp[3] = {1.0f, 1.0f, 1.0f};

int vro_set_voxel_spacing(const float s[3])
{
    int c;
    if (!s) return 1;
    for (c = 0; c < 3; ++c) if (!(s[c] > 0.0f) || !isfinite(s[c])) return 1;
    vro_aniso = !(s[0] == 1.0f && s[1] == 1.0f && s[2] == 1.0f);
    for (c = 0; c < 3; ++c) vro_inv_sp[c] = 1.0f / s[c];
    return 0;
}

static void vro_make_ray_world(const vro_camera* cam, int W, int H, int i, int j, float o[3], float d[3]);

/* ---- S1 + S2 (+ R23): pixel (i, j) -> ray origin o and direction d in index space ---- */
static void vro_make_ray(const vro_camera* cam, int W, int H, int i, int j,
                         float o[3], float d[3])
{
    int c;
    vro_make_ray_world(cam, W, H, i, j, o, d);
    if (vro_aniso)
        for (c = 0; c < 3; ++c) { o[c] = o[c] * vro_inv_sp[c]; d[c] = d[c] * vro_inv_sp[c]; }
}

/* ---- S1 + S2: pixel (i, j) -> ray origin o, unit direction d (world space) ------------- */
static void vro_make_ray_world(const vro_camera* cam, int W, int H, int i, int j,
                         float o[3], float d[3])
{
    /* S1: pixel centres, row 0 at the top */
    float ax = (float)(2 * i + 1) / (float)W - 1.0f;
    float ay = 1.0f - (float)(2 * j + 1) / (float)H;
    float asp = (float)W / (float)H;
    float sx = ax * asp;
    float sy = ay;
    int c;
    if (cam->projection == 0) {
        /* S2 perspective */
        float a = sx * cam->tan_half_fovy;
        float b = sy * cam->tan_half_fovy;
        float D[3], len;
        for (c = 0; c < 3; ++c)
            D[c] = fmaf(b, cam->up[c], fmaf(a, cam->right[c], cam->forward[c]));
        len = sqrtf(fmaf(D[2], D[2], fmaf(D[1], D[1], D[0] * D[0])));
        for (c = 0; c < 3; ++c) {
            d[c] = D[c] / len;
            o[c] = cam->eye[c];
        }
    } else {
        /* S2 orthographic */
        float a = sx * cam->ortho_half_height;
        float b = sy * cam->ortho_half_height;
        for (c = 0; c < 3; ++c) {
            o[c] = fmaf(b, cam->up[c], fmaf(a, cam->right[c], cam->eye[c]));
            d[c] = cam->forward[c];
        }
    }
}

/* ---- S3: slab test against [0, n-1]^3; returns 1 on hit ------------------ */
static int vro_clip(const int n[3], const float o[3], const float d[3],
                    float* tn_out, float* tf_out)
{
    float tn = 0.0f;           /* eye inside the box starts at 0 */
    float tf = INFINITY;
    int c;
    for (c = 0; c < 3; ++c) {
        float hi = (float)(n[c] - 1);
        if (d[c] == 0.0f) {
            if (o[c] < 0.0f || o[c] > hi) return 0;
        } else {
            float inv = 1.0f / d[c];
            float t0 = (0.0f - o[c]) * inv;
            float t1 = (hi - o[c]) * inv;
            float tlo = fminf(t0, t1);
            float thi = fmaxf(t0, t1);
            tn = fmaxf(tn, tlo);
            tf = fminf(tf, thi);
        }
    }
    *tn_out = tn;
    *tf_out = tf;
    return tn < tf;
}

/* ---- S4: position of sample k (midpoint rule, never t += step) ----------- */
static float vro_sample_t(int k, float step, float tn)
{
    return fmaf((float)k + 0.5f, step, tn);
}

static void vro_sample_pos(const int n[3], const float o[3], const float d[3],
                           float t, float p[3])
{
    int c;
    for (c = 0; c < 3; ++c) {
        float hi = (float)(n[c] - 1);
        float pc = fmaf(t, d[c], o[c]);
        p[c] = fminf(fmaxf(pc, 0.0f), hi);
    }
}

/* ---- S5: cell index and weights ----------------------------------------- */
static void vro_cell(const int n[3], const float p[3], int ic[3], float w[3])
{
    int c;
    for (c = 0; c < 3; ++c) {
        int i = (int)floorf(p[c]);
        if (i > n[c] - 2) i = n[c] - 2;
        ic[c] = i;
        w[c] = p[c] - (float)i;
    }
}

/* ---- S6: trilinear, x then y then z -------------------------------------- */
static float vro_lerp(float a, float b, float w)
{
    return fmaf(w, b - a, a);
}

/* Voxel (x, y, z) of the cube.  One array: V[(z*ny + y)*nx + x].  Brick store
 * (S10, "partitioned into a set of smaller sub-cubes"): brick b holds
 * the voxels [B*b, min(B*b+B, n-1)] per axis, dense, x fastest; voxel x is read
 * from brick min(x / B, nb-1), so the last voxel of an axis comes from the ghost
 * layer of the last brick. */
static float vro_voxel(const vro_scene* s, int x, int y, int z)
{
    if (s->V) {
        return s->V[((size_t)z * (size_t)s->n[1] + (size_t)y) * (size_t)s->n[0] + (size_t)x];
    } else {
        int g[3], b[3], l[3], e[3], c;
        g[0] = x; g[1] = y; g[2] = z;
        for (c = 0; c < 3; ++c) {
            int hi;
            b[c] = g[c] / s->B;
            if (b[c] > s->nb[c] - 1) b[c] = s->nb[c] - 1;
            l[c] = g[c] - s->B * b[c];
            hi = s->B * b[c] + s->B;
            if (hi > s->n[c] - 1) hi = s->n[c] - 1;
            e[c] = hi - s->B * b[c] + 1;           /* voxels the brick stores on this axis */
        }
        return s->bricks[(size_t)b[0] + (size_t)s->nb[0] * ((size_t)b[1] + (size_t)s->nb[1] * (size_t)b[2])]
                        [((size_t)l[2] * (size_t)e[1] + (size_t)l[1]) * (size_t)e[0] + (size_t)l[0]];
    }
}

static float vro_trilinear(const vro_scene* s, const int ic[3], const float w[3])
{
    int x = ic[0], y = ic[1], z = ic[2];
    float V000 = vro_voxel(s, x, y, z),         V100 = vro_voxel(s, x + 1, y, z);
    float V010 = vro_voxel(s, x, y + 1, z),     V110 = vro_voxel(s, x + 1, y + 1, z);
    float V001 = vro_voxel(s, x, y, z + 1),     V101 = vro_voxel(s, x + 1, y, z + 1);
    float V011 = vro_voxel(s, x, y + 1, z + 1), V111 = vro_voxel(s, x + 1, y + 1, z + 1);
    float c00 = vro_lerp(V000, V100, w[0]);
    float c10 = vro_lerp(V010, V110, w[0]);
    float c01 = vro_lerp(V001, V101, w[0]);
    float c11 = vro_lerp(V011, V111, w[0]);
    float c0 = vro_lerp(c00, c10, w[1]);
    float c1 = vro_lerp(c01, c11, w[1]);
    return vro_lerp(c0, c1, w[2]);
}

/* ---- S7: classification --------------------------------------------------- */
static float vro_lut_scale(int n_lut, float vmin, float vmax)
{
    return (float)((double)(n_lut - 1) / ((double)vmax - (double)vmin));
}

static void vro_classify(const float* lut, const float* alpha_tab, int n_lut,
                         float vmin, float scale, float v, float rgba[4])
{
    float xi = (v - vmin) * scale;
    int q, ch;
    float g;
    xi = fminf(fmaxf(xi, 0.0f), (float)(n_lut - 1));
    q = (int)xi;
    if (q > n_lut - 2) q = n_lut - 2;
    g = xi - (float)q;
    for (ch = 0; ch < 3; ++ch) {
        float l0 = lut[4 * q + ch], l1 = lut[4 * (q + 1) + ch];
        rgba[ch] = fmaf(g, l1 - l0, l0);
    }
    rgba[3] = fmaf(g, alpha_tab[q + 1] - alpha_tab[q], alpha_tab[q]);
}

void vro_opacity_correct(const float* lut_rgba, int n, float step, float* alpha_out)
{
    int i;
    for (i = 0; i < n; ++i) {
        double a = (double)lut_rgba[4 * i + 3];
        if (a < 0.0) a = 0.0;
        if (a > 1.0) a = 1.0;
        alpha_out[i] = (float)(1.0 - pow(1.0 - a, (double)step));
    }
}

static int vro_scene_init(vro_scene* s, const float* V, int nx, int ny, int nz,
                          const float* lut, int n_lut, float vmin, float vmax,
                          float step, int mode, float tau)
{
    int i;
    if (!V || !lut || nx < 2 || ny < 2 || nz < 2 || n_lut < 2) return 1;
    if (!(step > 0.0f) || !isfinite(step) || !(vmax > vmin)) return 1;
    /* S4 needs the sample index k and k + 0.5 exact in binary32: refuse steps that put more than 2^22 samples
       on the longest chord (argument validation only; no arithmetic of the method changes) */
    if (!(sqrt((double)nx * nx + (double)ny * ny + (double)nz * nz) / (double)step < 4194304.0)) return 1;
    s->V = V; s->bricks = NULL; s->B = 0; s->nb[0] = s->nb[1] = s->nb[2] = 0;
    s->n[0] = nx; s->n[1] = ny; s->n[2] = nz;
    s->lut = lut; s->n_lut = n_lut; s->vmin = vmin; s->vmax = vmax;
    s->scale = vro_lut_scale(n_lut, vmin, vmax);
    s->step = step; s->mode = mode; s->tau = tau;
    s->alpha_tab = (float*)malloc(sizeof(float) * (size_t)n_lut);
    if (!s->alpha_tab) return 2;
    if (mode == VRO_MODE_EA) vro_opacity_correct(lut, n_lut, step, s->alpha_tab);
    else for (i = 0; i < n_lut; ++i) s->alpha_tab[i] = lut[4 * i + 3];
    return 0;
}

/* brick ownership, S10: brick b owns cells [B*b, min(B*b+B, n-1)) per axis */
static int vro_cell_in_brick(const int ic[3], int B, const int b[3])
{
    int c;
    for (c = 0; c < 3; ++c)
        if (ic[c] / B != b[c]) return 0;
    return 1;
}

/* ---- S4-S9 along one ray; brick == NULL means "all samples".
 * EA state (C, A) and MIP state m are carried in and out so that the same
 * routine serves the unbricked render (start from 0) and S12 / S13. -------- */
static void vro_march(const vro_scene* s, const float o[3], const float d[3],
                      float tn, float tf, int B, const int* brick,
                      float C[3], float* A, float* m,
                      unsigned long long* n_eval, unsigned long long* n_nominal)
{
    int k;
    if (s->mode == VRO_MODE_EA && *A >= s->tau) return;   /* S12: saturated carry-in */
    for (k = 0; ; ++k) {
        float t = vro_sample_t(k, s->step, tn);
        float p[3], w[3], v;
        int ic[3];
        if (!(t < tf)) break;
        if (n_nominal) ++*n_nominal;
        vro_sample_pos(s->n, o, d, t, p);
        vro_cell(s->n, p, ic, w);
        if (brick && !vro_cell_in_brick(ic, B, brick)) continue;
        v = vro_trilinear(s, ic, w);
        ++*n_eval;
        if (s->mode == VRO_MODE_EA) {
            /* S7 + S8 */
            float rgba[4], tr, wgt;
            int ch;
            vro_classify(s->lut, s->alpha_tab, s->n_lut, s->vmin, s->scale, v, rgba);
            tr = 1.0f - *A;
            wgt = tr * rgba[3];
            for (ch = 0; ch < 3; ++ch) C[ch] = fmaf(wgt, rgba[ch], C[ch]);
            *A = *A + wgt;
            if (*A >= s->tau) break;      /* early ray termination */
        } else {
            /* S9 */
            *m = fmaxf(*m, v);
        }
    }
}

/* S9 output stage: LUT colour of the maximum (uncorrected LUT), alpha = 1 */
static void vro_mip_output(const vro_scene* s, float m, float out[4])
{
    if (m == -INFINITY) {
        out[0] = out[1] = out[2] = out[3] = 0.0f;
    } else {
        float rgba[4];
        vro_classify(s->lut, s->alpha_tab, s->n_lut, s->vmin, s->scale, m, rgba);
        out[0] = rgba[0]; out[1] = rgba[1]; out[2] = rgba[2]; out[3] = 1.0f;
    }
}

static void vro_one_pixel(const vro_scene* s, const vro_camera* cam, int W, int H,
                          int i, int j, float out[4], float* aux,
                          unsigned long long cnt[3])
{
    float o[3], d[3], tn, tf;
    float C[3] = {0.0f, 0.0f, 0.0f}, A = 0.0f, m = -INFINITY;
    vro_make_ray(cam, W, H, i, j, o, d);
    if (!vro_clip(s->n, o, d, &tn, &tf)) {
        out[0] = out[1] = out[2] = out[3] = 0.0f;
        if (aux) *aux = -INFINITY;
        return;
    }
    cnt[0] += 1;
    vro_march(s, o, d, tn, tf, 0, NULL, C, &A, &m, &cnt[1], &cnt[2]);
    if (s->mode == VRO_MODE_EA) {
        out[0] = C[0]; out[1] = C[1]; out[2] = C[2]; out[3] = A;
        if (aux) *aux = -INFINITY;
    } else {
        vro_mip_output(s, m, out);
        if (aux) *aux = m;
    }
}

static int vro_threads(int nthreads)
{
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_num_procs();
    return nthreads;
#else
    (void)nthreads;
    return 1;
#endif
}

int vro_render_pixels(const float* V, int nx, int ny, int nz,
                      const float* lut_rgba, int n_lut, float vmin, float vmax,
                      const vro_camera* cam, int W, int H, float step, int mode,
                      float tau, const int* ij, long npix,
                      float* out_rgba, float* out_aux,
                      unsigned long long* counters, int nthreads)
{
    vro_scene s;
    unsigned long long c0 = 0, c1 = 0, c2 = 0;
    long q;
    int rc = vro_scene_init(&s, V, nx, ny, nz, lut_rgba, n_lut, vmin, vmax, step, mode, tau);
    if (rc) return rc;
    if (!cam || !ij || !out_rgba || W < 1 || H < 1) { free(s.alpha_tab); return 1; }
    nthreads = vro_threads(nthreads);
#pragma omp parallel for schedule(dynamic, 64) num_threads(nthreads) reduction(+ : c0, c1, c2)
    for (q = 0; q < npix; ++q) {
        unsigned long long cnt[3] = {0, 0, 0};
        vro_one_pixel(&s, cam, W, H, ij[2 * q], ij[2 * q + 1], out_rgba + 4 * q,
                      out_aux ? out_aux + q : NULL, cnt);
        c0 += cnt[0]; c1 += cnt[1]; c2 += cnt[2];
    }
    if (counters) { counters[0] = c0; counters[1] = c1; counters[2] = c2; }
    free(s.alpha_tab);
    return 0;
}

/* The same pixels with the cube read from its brick store (the out-of-core cube of
 * BASELINE.json configs[3] never exists as one array): identical op sequence, only
 * vro_voxel() differs. */
int vro_render_pixels_bricks(const float* const* bricks, int B, int nx, int ny, int nz,
                             const float* lut_rgba, int n_lut, float vmin, float vmax,
                             const vro_camera* cam, int W, int H, float step, int mode,
                             float tau, const int* ij, long npix,
                             float* out_rgba, float* out_aux,
                             unsigned long long* counters, int nthreads)
{
    vro_scene s;
    unsigned long long c0 = 0, c1 = 0, c2 = 0;
    long q;
    int rc;
    if (!bricks || B < 1) return 1;
    rc = vro_scene_init(&s, bricks[0], nx, ny, nz, lut_rgba, n_lut, vmin, vmax, step, mode, tau);
    if (rc) return rc;
    if (!cam || !ij || !out_rgba || W < 1 || H < 1) { free(s.alpha_tab); return 1; }
    s.V = NULL; s.bricks = bricks; s.B = B;
    s.nb[0] = (nx - 1 + B - 1) / B; s.nb[1] = (ny - 1 + B - 1) / B; s.nb[2] = (nz - 1 + B - 1) / B;
    nthreads = vro_threads(nthreads);
#pragma omp parallel for schedule(dynamic, 64) num_threads(nthreads) reduction(+ : c0, c1, c2)
    for (q = 0; q < npix; ++q) {
        unsigned long long cnt[3] = {0, 0, 0};
        vro_one_pixel(&s, cam, W, H, ij[2 * q], ij[2 * q + 1], out_rgba + 4 * q,
                      out_aux ? out_aux + q : NULL, cnt);
        c0 += cnt[0]; c1 += cnt[1]; c2 += cnt[2];
    }
    if (counters) { counters[0] = c0; counters[1] = c1; counters[2] = c2; }
    free(s.alpha_tab);
    return 0;
}

int vro_render(const float* V, int nx, int ny, int nz,
               const float* lut_rgba, int n_lut, float vmin, float vmax,
               const vro_camera* cam, int W, int H, float step, int mode,
               float tau, float* out_rgba, float* out_aux,
               unsigned long long* counters, int nthreads)
{
    vro_scene s;
    unsigned long long c0 = 0, c1 = 0, c2 = 0;
    int j;
    int rc = vro_scene_init(&s, V, nx, ny, nz, lut_rgba, n_lut, vmin, vmax, step, mode, tau);
    if (rc) return rc;
    if (!cam || !out_rgba || W < 1 || H < 1) { free(s.alpha_tab); return 1; }
    nthreads = vro_threads(nthreads);
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads) reduction(+ : c0, c1, c2)
    for (j = 0; j < H; ++j) {
        int i;
        for (i = 0; i < W; ++i) {
            unsigned long long cnt[3] = {0, 0, 0};
            size_t q = (size_t)j * (size_t)W + (size_t)i;
            vro_one_pixel(&s, cam, W, H, i, j, out_rgba + 4 * q,
                          out_aux ? out_aux + q : NULL, cnt);
            c0 += cnt[0]; c1 += cnt[1]; c2 += cnt[2];
        }
    }
    if (counters) { counters[0] = c0; counters[1] = c1; counters[2] = c2; }
    free(s.alpha_tab);
    return 0;
}

/* ---- W1: a K x L display wall (design objective 5, "tiled display") ----------
 * The wall shows ONE image of W x H pixels: tile (a, b) -- column a from the left, row b from
 * the top -- shows the camera's off-axis sub-frustum through the rectangle
 * [a/K, (a+1)/K] x [b/L, (b+1)/L] of the image plane, sampled at w x h = W/K x H/L pixel centres
 * which are the frame's own: local pixel (i', j') of the tile is pixel (a*w + i', b*h + j') of
 * the frame (S1 with the frame's W and H).  Each tile has its own buffer. */
int vro_render_wall(const float* V, int nx, int ny, int nz,
                    const float* lut_rgba, int n_lut, float vmin, float vmax,
                    const vro_camera* cam, int W, int H, int K, int L, float step, int mode,
                    float tau, float* const* outs_rgba, float* const* outs_aux,
                    unsigned long long* counters, int nthreads)
{
    vro_scene s;
    unsigned long long c0 = 0, c1 = 0, c2 = 0;
    int row, w, h;
    int rc = vro_scene_init(&s, V, nx, ny, nz, lut_rgba, n_lut, vmin, vmax, step, mode, tau);
    if (rc) return rc;
    if (!cam || !outs_rgba || W < 1 || H < 1 || K < 1 || L < 1 || W % K != 0 || H % L != 0) { free(s.alpha_tab); return 1; }
    w = W / K; h = H / L;
    nthreads = vro_threads(nthreads);
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads) reduction(+ : c0, c1, c2)
    for (row = 0; row < L * h; ++row) {
        const int b = row / h, jl = row % h;
        int a, il;
        for (a = 0; a < K; ++a) {
            float* out = outs_rgba[b * K + a];
            float* aux = outs_aux ? outs_aux[b * K + a] : NULL;
            for (il = 0; il < w; ++il) {
                unsigned long long cnt[3] = {0, 0, 0};
                const size_t q = (size_t)jl * (size_t)w + (size_t)il;
                vro_one_pixel(&s, cam, W, H, a * w + il, b * h + jl, out + 4 * q, aux ? aux + q : NULL, cnt);
                c0 += cnt[0]; c1 += cnt[1]; c2 += cnt[2];
            }
        }
    }
    if (counters) { counters[0] = c0; counters[1] = c1; counters[2] = c2; }
    free(s.alpha_tab);
    return 0;
}

/* ---- R17b: blanked voxels --------------------------------------------------------------------
 * Radio cubes mark masked channels and pixels with NaN (PAPER.md:9 names the low signal-to-noise data
 * this renderer is for; the paper does not say what to do with blanks).  Reading: before anything
 * else, every non-finite voxel (NaN, +inf, -inf) is replaced by one caller-chosen finite value
 * (typically vmin, which a transfer function maps to nothing); the render is that of the cube so
 * blanked.  In place; returns the number of voxels replaced. */
long vro_blank_nonfinite(float* V, long n, float value)
{
    long q, count = 0;
    for (q = 0; q < n; ++q)
        if (!isfinite(V[q])) { V[q] = value; ++count; }
    return count;
}

/* ---- S11: view order ------------------------------------------------------ */
static int vro_nbricks(int n, int B) { return (n - 1 + B - 1) / B; }   /* over cells */

typedef struct { int key; int idx; } vro_keyed;

static int vro_keyed_cmp(const void* a, const void* b)
{
    const vro_keyed* x = (const vro_keyed*)a;
    const vro_keyed* y = (const vro_keyed*)b;
    if (x->key != y->key) return x->key < y->key ? -1 : 1;
    return x->idx < y->idx ? -1 : (x->idx > y->idx ? 1 : 0);
}

int vro_brick_order(int nx, int ny, int nz, int B, const vro_camera* cam,
                    int* order_out, int* keys_out)
{
    int nb[3], b[3], c, q = 0, total;
    vro_keyed* ks;
    if (nx < 2 || ny < 2 || nz < 2 || B < 1 || !cam || !order_out) return 1;
    nb[0] = vro_nbricks(nx, B); nb[1] = vro_nbricks(ny, B); nb[2] = vro_nbricks(nz, B);
    total = nb[0] * nb[1] * nb[2];
    ks = (vro_keyed*)malloc(sizeof(vro_keyed) * (size_t)total);
    if (!ks) return 2;
    for (b[2] = 0; b[2] < nb[2]; ++b[2])
        for (b[1] = 0; b[1] < nb[1]; ++b[1])
            for (b[0] = 0; b[0] < nb[0]; ++b[0]) {
                int key = 0;
                for (c = 0; c < 3; ++c) {
                    if (cam->projection == 0) {
                        /* perspective: |b_c - floor(eye_c / B)|, unclamped */
                        /* (R23: the eye in index space) */
                        float e = vro_aniso ? cam->eye[c] * vro_inv_sp[c] : cam->eye[c];
                        int ie = (int)floorf(e / (float)B);
                        key += abs(b[c] - ie);
                    } else {
                        /* orthographic: sgn(d_c) * b_c */
                        float dc = cam->forward[c];
                        int sg = (dc > 0.0f) - (dc < 0.0f);
                        key += sg * b[c];
                    }
                }
                ks[q].key = key;
                ks[q].idx = b[0] + nb[0] * (b[1] + nb[1] * b[2]);
                ++q;
            }
    qsort(ks, (size_t)total, sizeof(vro_keyed), vro_keyed_cmp);
    for (q = 0; q < total; ++q) {
        order_out[q] = ks[q].idx;
        if (keys_out) keys_out[q] = ks[q].key;
    }
    free(ks);
    return 0;
}

/* ---- S10, S12, S13: brick-by-brick render --------------------------------- */
/* brick_samples (may be NULL): samples evaluated inside each brick, by linear brick index.  Reading C1
 * of DESIGN.md (PAPER.md:9 "larger than GPU memory", :67): a sub-cube is NEEDED for a frame iff at least
 * one sample is evaluated in it -- some ray reaches it unsaturated (S12) and has a sample there; a
 * renderer that leaves the others out (does not even fetch them) produces the same image bit for bit. */
static int vro_bricked_impl(const float* V, int nx, int ny, int nz, int B, int compositor,
                            const float* lut_rgba, int n_lut, float vmin, float vmax,
                            const vro_camera* cam, int W, int H, float step, int mode,
                            float tau, float* out_rgba, float* out_aux,
                            unsigned long long* counters, unsigned long long* brick_samples, int nthreads)
{
    vro_scene s;
    unsigned long long c0 = 0, c1 = 0;
    int nb[3], total, ob, j, rc;
    int* order;
    float* M;          /* running MIP maximum per pixel */
    size_t npx;
    rc = vro_scene_init(&s, V, nx, ny, nz, lut_rgba, n_lut, vmin, vmax, step, mode, tau);
    if (rc) return rc;
    if (!cam || !out_rgba || W < 1 || H < 1 || B < 1) { free(s.alpha_tab); return 1; }
    nb[0] = vro_nbricks(nx, B); nb[1] = vro_nbricks(ny, B); nb[2] = vro_nbricks(nz, B);
    total = nb[0] * nb[1] * nb[2];
    npx = (size_t)W * (size_t)H;
    order = (int*)malloc(sizeof(int) * (size_t)total);
    M = (float*)malloc(sizeof(float) * npx);
    if (!order || !M) { free(order); free(M); free(s.alpha_tab); return 2; }
    vro_brick_order(nx, ny, nz, B, cam, order, NULL);
    nthreads = vro_threads(nthreads);

    /* running image R = 0, running maximum = -inf */
    memset(out_rgba, 0, sizeof(float) * 4 * npx);
    { size_t q; for (q = 0; q < npx; ++q) M[q] = -INFINITY; }

    for (ob = 0; ob < total; ++ob) {
        int brick[3];
        brick[0] = order[ob] % nb[0];
        brick[1] = (order[ob] / nb[0]) % nb[1];
        brick[2] = order[ob] / (nb[0] * nb[1]);
        const unsigned long long before = c1;
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads) reduction(+ : c0, c1)
        for (j = 0; j < H; ++j) {
            int i;
            for (i = 0; i < W; ++i) {
                size_t q = (size_t)j * (size_t)W + (size_t)i;
                float o[3], d[3], tn, tf;
                float* R = out_rgba + 4 * q;
                unsigned long long ne = 0;
                vro_make_ray(cam, W, H, i, j, o, d);
                if (!vro_clip(s.n, o, d, &tn, &tf)) continue;
                if (ob == 0) c0 += 1;
                if (!compositor) {
                    /* S12 fused: continue the ray from the carried-in state */
                    float A = R[3];
                    vro_march(&s, o, d, tn, tf, B, brick, R, &A, &M[q], &ne, NULL);
                    R[3] = A;
                } else {
                    /* S13: partial image of this brick from (0, 0), then over / max */
                    float P[3] = {0.0f, 0.0f, 0.0f}, PA = 0.0f, pm = -INFINITY;
                    vro_march(&s, o, d, tn, tf, B, brick, P, &PA, &pm, &ne, NULL);
                    if (mode == VRO_MODE_EA) {
                        float tr = 1.0f - R[3];
                        int ch;
                        for (ch = 0; ch < 3; ++ch) R[ch] = fmaf(tr, P[ch], R[ch]);
                        R[3] = fmaf(tr, PA, R[3]);
                    } else {
                        M[q] = fmaxf(M[q], pm);
                    }
                }
                c1 += ne;
            }
        }
        if (brick_samples) brick_samples[order[ob]] = c1 - before;
    }
    if (mode == VRO_MODE_MIP) {
        /* the transfer function is applied once, after the maxima are combined
         * (reading A14 of "reapplies the same transfer function") */
        size_t q;
        for (q = 0; q < npx; ++q) {
            vro_mip_output(&s, M[q], out_rgba + 4 * q);
            if (out_aux) out_aux[q] = M[q];
        }
    } else if (out_aux) {
        size_t q;
        for (q = 0; q < npx; ++q) out_aux[q] = -INFINITY;
    }
    if (counters) { counters[0] = c0; counters[1] = c1; counters[2] = 0; }
    free(order); free(M); free(s.alpha_tab);
    return 0;
}

int vro_render_bricked(const float* V, int nx, int ny, int nz, int B, int compositor,
                       const float* lut_rgba, int n_lut, float vmin, float vmax,
                       const vro_camera* cam, int W, int H, float step, int mode,
                       float tau, float* out_rgba, float* out_aux,
                       unsigned long long* counters, int nthreads)
{
    return vro_bricked_impl(V, nx, ny, nz, B, compositor, lut_rgba, n_lut, vmin, vmax, cam, W, H, step, mode, tau,
                            out_rgba, out_aux, counters, NULL, nthreads);
}

int vro_render_bricked_needed(const float* V, int nx, int ny, int nz, int B,
                              const float* lut_rgba, int n_lut, float vmin, float vmax,
                              const vro_camera* cam, int W, int H, float step, int mode,
                              float tau, float* out_rgba, float* out_aux,
                              unsigned long long* counters, unsigned long long* brick_samples, int nthreads)
{
    if (!brick_samples) return 1;
    return vro_bricked_impl(V, nx, ny, nz, B, 0, lut_rgba, n_lut, vmin, vmax, cam, W, H, step, mode, tau,
                            out_rgba, out_aux, counters, brick_samples, nthreads);
}

/* ---- A2: per-brick min / max, plain definition ---------------------------- */
int vro_brick_minmax(const float* V, int nx, int ny, int nz, int B,
                     float* mn_out, float* mx_out)
{
    int nb[3], b[3];
    if (!V || nx < 2 || ny < 2 || nz < 2 || B < 1 || !mn_out || !mx_out) return 1;
    nb[0] = vro_nbricks(nx, B); nb[1] = vro_nbricks(ny, B); nb[2] = vro_nbricks(nz, B);
    for (b[2] = 0; b[2] < nb[2]; ++b[2])
        for (b[1] = 0; b[1] < nb[1]; ++b[1])
            for (b[0] = 0; b[0] < nb[0]; ++b[0]) {
                int x0 = B * b[0] - 1, x1 = B * b[0] + B + 1;
                int y0 = B * b[1] - 1, y1 = B * b[1] + B + 1;
                int z0 = B * b[2] - 1, z1 = B * b[2] + B + 1;
                int x, y, z;
                float mn = INFINITY, mx = -INFINITY;
                if (x0 < 0) x0 = 0;
                if (y0 < 0) y0 = 0;
                if (z0 < 0) z0 = 0;
                if (x1 > nx - 1) x1 = nx - 1;
                if (y1 > ny - 1) y1 = ny - 1;
                if (z1 > nz - 1) z1 = nz - 1;
                for (z = z0; z <= z1; ++z)
                    for (y = y0; y <= y1; ++y)
                        for (x = x0; x <= x1; ++x) {
                            float v = V[((size_t)z * (size_t)ny + (size_t)y) * (size_t)nx + (size_t)x];
                            mn = fminf(mn, v);
                            mx = fmaxf(mx, v);
                        }
                {
                    size_t bi = (size_t)b[0] + (size_t)nb[0] * ((size_t)b[1] + (size_t)nb[1] * (size_t)b[2]);
                    mn_out[bi] = mn;
                    mx_out[bi] = mx;
                }
            }
    return 0;
}

/* ---- single-point entry points for the pins ------------------------------- */
float vro_sample_at(const float* V, int nx, int ny, int nz, float px, float py, float pz)
{
    vro_scene s;
    int ic[3];
    float p[3], w[3];
    memset(&s, 0, sizeof(s));
    s.V = V; s.n[0] = nx; s.n[1] = ny; s.n[2] = nz;
    p[0] = px; p[1] = py; p[2] = pz;
    vro_cell(s.n, p, ic, w);
    return vro_trilinear(&s, ic, w);
}

void vro_classify_at(const float* lut_rgba, const float* alpha_tab, int n_lut,
                     float vmin, float vmax, float v, float* rgba_out)
{
    vro_classify(lut_rgba, alpha_tab, n_lut, vmin, vro_lut_scale(n_lut, vmin, vmax), v, rgba_out);
}
