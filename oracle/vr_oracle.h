/* vr_oracle.h -- CPU ORACLE, TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, obviously-correct C99 restatement of the hot path of
 * Hassan, Fluke & Barnes, "GPU-Based Volume Rendering of Noisy Multi-Spectral
 * Astronomical Data" (Sec. 3.1 steps 1-5): per-pixel ray casting
 * of a spectral cube into RGBA through a transfer function, sub-cube
 * partitioning, and view-ordered integration of the partial images.
 *
 * The paper gives no formulae; every numerical definition is the reading listed
 * in DESIGN.md Sec. 3 (S1..S13, taken from SURVEY.md Sec. 8(c).2).  Precision is
 * IEEE-754 binary32 because BASELINE.json north_star fixes it ("fp32 trilinear
 * interpolation", "exactly for MIP values when fp32 interpolation is used").
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call this.  It shares no code, header, table or
 * helper with the CUDA path under paper_1001_2049_b200/.
 *
 * Pins (tests/test_oracle_pins.py): constant cube closed form, ERT integer
 * closed form, linear ramp exactness, single bright voxel under MIP, float64
 * NumPy/SciPy brute force on tiny cubes, bricked == unbricked, invariants; the
 * aspect convention of S1 on non-square frames; the display wall (W1) against an
 * independent float64 off-axis sub-frustum; the needed-brick counts (C1) against
 * the ERT closed form and a float64 binning; voxel spacing (R23) against a
 * stretched-chord closed form, a stretched footprint and float64 brute force;
 * blanking (R17b) against a hand-made cube.  Unpinned: nothing -- the
 * handedness of the camera basis is the caller's input, not a choice made here.
 */
#ifndef VR_ORACLE_H
#define VR_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
    float eye[3], right[3], up[3], forward[3];
    int   projection;         /* 0 = perspective, 1 = orthographic */
    float tan_half_fovy;      /* perspective */
    float ortho_half_height;  /* orthographic: half image height in voxels */
} vro_camera;

enum { VRO_MODE_EA = 0, VRO_MODE_MIP = 1 };

/* counters[0] = rays that hit the box (tn < tf), counters[1] = samples evaluated
 * (S4-S6 executed), counters[2] = nominal samples (all k with t_k < tf, no ERT). */

/* R23: voxel spacing s = (sx, sy, sz) > 0 of the cubes rendered from now on; world space = voxel index
 * x spacing, and cameras, the step and the LUT's opacity per unit length are world-space quantities.  (1, 1, 1) is
 * the default and changes nothing.  Returns non-zero on an invalid spacing. */
int vro_set_voxel_spacing(const float s[3]);

/* R17b: every non-finite voxel (NaN, +-inf = blanked) of V[0..n) becomes `value`, in place; returns how
 * many were replaced.  A cube is rendered as the cube so blanked. */
long vro_blank_nonfinite(float* V, long n, float value);

/* S7 (host part): opacity-corrected alpha table, alpha'_i = 1-(1-alpha_i)^step. */
void vro_opacity_correct(const float* lut_rgba, int n, float step, float* alpha_out);

/* S1-S9 for an explicit list of pixels (ij = npix pairs (i, j)); out = npix*4
 * floats, aux = npix floats or NULL (MIP raw maximum). */
int vro_render_pixels(const float* V, int nx, int ny, int nz,
                      const float* lut_rgba, int n_lut, float vmin, float vmax,
                      const vro_camera* cam, int W, int H, float step, int mode,
                      float tau, const int* ij, long npix,
                      float* out_rgba, float* out_aux,
                      unsigned long long* counters, int nthreads);

/* vro_render_pixels with the cube given as its S10 brick store instead of one
 * array: bricks[bx + nbx*(by + nby*bz)] points at the dense float32 voxels
 * [B*b, min(B*b+B, n-1)] of brick b (x fastest; one ghost layer on the high side),
 * nb = ceil((n-1)/B) per axis.  Same arithmetic, only the voxel fetch differs. */
int vro_render_pixels_bricks(const float* const* bricks, int B, int nx, int ny, int nz,
                             const float* lut_rgba, int n_lut, float vmin, float vmax,
                             const vro_camera* cam, int W, int H, float step, int mode,
                             float tau, const int* ij, long npix,
                             float* out_rgba, float* out_aux,
                             unsigned long long* counters, int nthreads);

/* S1-S9 for the full W x H frame (row 0 = top). */
int vro_render(const float* V, int nx, int ny, int nz,
               const float* lut_rgba, int n_lut, float vmin, float vmax,
               const vro_camera* cam, int W, int H, float step, int mode,
               float tau, float* out_rgba, float* out_aux,
               unsigned long long* counters, int nthreads);

/* W1 ("tiled display"): the frame as a K x L display wall.  Tile (a, b), column a
 * from the left and row b from the top, gets its own buffers outs_rgba[b*K + a] (w*h*4 floats,
 * w = W/K, h = H/L; W % K == 0 and H % L == 0) and outs_aux[b*K + a] (w*h floats; outs_aux may be
 * NULL): the camera's off-axis sub-frustum through that rectangle of the image plane, sampled
 * at the frame's own pixel centres. */
int vro_render_wall(const float* V, int nx, int ny, int nz,
                    const float* lut_rgba, int n_lut, float vmin, float vmax,
                    const vro_camera* cam, int W, int H, int K, int L, float step, int mode,
                    float tau, float* const* outs_rgba, float* const* outs_aux,
                    unsigned long long* counters, int nthreads);

/* S10-S13: the same frame rendered brick by brick (bricks of B^3 cells) in S11
 * view order.  compositor = 0: fused carry-in (S12); 1: per-brick partial images
 * combined with over / max (S13). */
int vro_render_bricked(const float* V, int nx, int ny, int nz, int B, int compositor,
                       const float* lut_rgba, int n_lut, float vmin, float vmax,
                       const vro_camera* cam, int W, int H, float step, int mode,
                       float tau, float* out_rgba, float* out_aux,
                       unsigned long long* counters, int nthreads);

/* vro_render_bricked in fused mode (S12) that also reports brick_samples[nbx*nby*nbz]: the samples
 * evaluated inside each brick (linear brick index).  Reading C1: a sub-cube is
 * needed for a frame iff that count is > 0; leaving the others out changes no pixel. */
int vro_render_bricked_needed(const float* V, int nx, int ny, int nz, int B,
                              const float* lut_rgba, int n_lut, float vmin, float vmax,
                              const vro_camera* cam, int W, int H, float step, int mode,
                              float tau, float* out_rgba, float* out_aux,
                              unsigned long long* counters, unsigned long long* brick_samples, int nthreads);

/* S11: bricks in front-to-back order; order_out has nbx*nby*nbz linear brick
 * indices (bx + nbx*(by + nby*bz)), keys_out the wavefront key of each. */
int vro_brick_order(int nx, int ny, int nz, int B, const vro_camera* cam,
                    int* order_out, int* keys_out);

/* A2: plain min / max of every brick over voxels
 * [max(B*b-1,0), min(B*b+B+1, n-1)] per axis (S9b). */
int vro_brick_minmax(const float* V, int nx, int ny, int nz, int B,
                     float* mn_out, float* mx_out);

/* S5-S6 at one position (already inside the box); for the ramp / scipy pins. */
float vro_sample_at(const float* V, int nx, int ny, int nz, float px, float py, float pz);

/* S7 at one value: rgba from the LUT (alpha from alpha_tab). */
void vro_classify_at(const float* lut_rgba, const float* alpha_tab, int n_lut,
                     float vmin, float vmax, float v, float* rgba_out);

#ifdef __cplusplus
}
#endif
#endif
