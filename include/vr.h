/* vr.h -- C ABI of the B200 spectral-cube ray caster (libvr.so).
 *
 * C99, no C++ types, no exceptions cross this boundary.  The operations are the
 * per-frame pipeline of Hassan, Fluke & Barnes, PAPER.md:56-63 (Sec. 3.1):
 *   step 1  "the spectral data cube is partitioned into a set of smaller
 *           sub-cubes"                          -> vr_volume_create / vr_volume_upload_bricks
 *   step 3  "ray-tracing volume rendering to map each output pixel into a color
 *           plus alpha transparency channel (RGBA) based on a preselected
 *           transfer function"                  -> vr_set_transfer_function / vr_render
 *   steps 4-5 "N images with the same resolution as the output screen" combined
 *           by the scene integration module     -> inside vr_render (streamed volumes)
 * The paper gives no formulae; the numerical definition of every step (S1..S13)
 * is DESIGN.md Sec. 3 (from SURVEY.md Sec. 8(c).2 and BASELINE.json north_star).
 *
 * World space = voxel index space (x the voxel spacing of VR_OPT_SPACING_*, 1 by default): voxel
 * (x, y, z) = (RA, Dec, frequency) sits at coordinate (x, y, z); the cube occupies [0, n-1]^3 (node centred).  Volumes are
 * float32, V[z][y][x], x fastest ("a stack of images").
 *
 * Every call returns a vr_status; on failure vr_last_error() holds a message
 * (thread local).  Nothing aborts, nothing throws.  There is NO CPU fallback:
 * every entry point that touches voxels runs CUDA kernels on the device.
 */
#ifndef VR_H
#define VR_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct vr_volume vr_volume;   /* opaque handle */

typedef enum {
    VR_OK = 0,
    VR_ERR_INVALID_ARG = 1,   /* null pointer, dims < 2, step <= 0, non-finite or so small that the longest chord of
                                 the cube would hold 2^22 samples or more (the sample index must stay exact in
                                 binary32, S4), vmax <= vmin, ... */
    VR_ERR_STATE = 2,         /* render before upload / before a transfer function was set */
    VR_ERR_UNSUPPORTED = 3,
    VR_ERR_OOM_HOST = 4,
    VR_ERR_OOM_DEVICE = 5,    /* d_storage too small, or a small device table could not be allocated */
    VR_ERR_CUDA = 6           /* any CUDA runtime error; message = cudaGetErrorString */
} vr_status;

typedef enum { VR_MODE_EA = 0,      /* emission-absorption, front to back (S7, S8) */
               VR_MODE_MIP = 1      /* maximum intensity projection (S9) */ } vr_mode;
typedef enum { VR_PROJ_PERSPECTIVE = 0, VR_PROJ_ORTHO = 1 } vr_proj;

/* Device layout of the voxels (north_star: "3D-blocked layout or CUDA 3D texture").
 * VR_LAYOUT_LINEAR: float32 V[z][y][x] in caller-owned d_storage; the kernels read it
 *   with 8 scalar loads per sample.
 * VR_LAYOUT_TEX: library-owned 2D-layered CUDA arrays (one layer per z, block-linear),
 *   read with two 4-texel gathers per sample (raw fp32 texels, no hardware filtering,
 *   so results are bit-identical to VR_LAYOUT_LINEAR).  One array holds 2048 layers; a
 *   resident cube with more channels is cut along z into up to 8 arrays that share one
 *   layer with their neighbour (nz <= 16377; configs[4]'s 8192 channels take 5).
 *   Streamed: host_brick + 1 <= 2048.  d_storage may be NULL. */
typedef enum { VR_LAYOUT_LINEAR = 0, VR_LAYOUT_TEX = 1 } vr_layout;

/* Camera (S1, S2).  All float32, voxel-index world space.  right / up / forward
 * must be orthonormal; the library uses them exactly as given and does NOT
 * renormalise.  Pixel (i, j) looks along forward + sx*right + sy*up with
 * sx = ((2i+1)/W - 1) * W/H, sy = 1 - (2j+1)/H: column i grows towards +right,
 * row j = 0 is the top (+up). */
typedef struct {
    float eye[3], right[3], up[3], forward[3];
    int   projection;         /* vr_proj */
    float tan_half_fovy;      /* perspective: tan(fovy / 2) */
    float ortho_half_height;  /* orthographic: half the image height, in voxels */
} vr_camera;

/* Volume description.
 * Resident volume (host_brick = 0): d_storage holds the whole cube in the
 *   library's device layout; ask vr_volume_storage_bytes() how much to allocate.
 * Streamed volume (host_brick = B > 0, the out-of-core path): the cube lives in
 *   caller-owned PINNED host memory as bricks of B^3 cells (each brick stores the
 *   voxels [B*b, min(B*b+B, n-1)] per axis, i.e. one ghost layer on the high
 *   side, dense rows); d_storage is a pool of >= 2 device slots of
 *   vr_volume_slot_bytes() each, through which bricks are streamed on a private
 *   copy stream overlapped with ray casting (S10-S12).
 * d_storage is caller-owned device memory (e.g. a torch tensor), 256-byte
 * aligned, and must outlive the handle. */
typedef struct {
    int    nx, ny, nz;        /* RA, Dec, frequency extents in voxels; each >= 2 */
    int    host_brick;        /* 0 = resident; else streamed brick edge in cells (e.g. 512) */
    int    mm_brick;          /* edge of the min/max bricks in cells; 0 = default 64 */
    int    device;            /* CUDA device ordinal */
    void*  d_storage;         /* device pointer, caller owned */
    size_t d_storage_bytes;
    int    layout;            /* vr_layout */
    int    n_slots;           /* streamed + VR_LAYOUT_TEX: number of device slots (>= 2); else ignored */
} vr_volume_desc;

/* Option keys for vr_set_option. */
enum {
    VR_OPT_ERT_TAU = 0,       /* early-ray-termination threshold tau (default 0.99; > 1 disables) */
    VR_OPT_SKIP = 1,          /* 1 = exact empty-space skipping from the min/max table (default 0) */
    VR_OPT_KERNEL = 2,        /* resident ray caster: 0 or 1 = direct kernel (global / texture loads per sample, default),
                                 2 = beam kernel (voxel boxes staged in shared memory, EA skipping by whole slabs, no MIP
                                 skipping; EXPERIMENTAL: verified on the host
                                 against the oracle, not yet run on hardware) or VR_ERR_UNSUPPORTED at
                                 vr_render; same pixels */
    VR_OPT_COUNT = 3,         /* 1 = count rays / samples into vr_stats (slower; default 0) */
    VR_OPT_COMPOSITOR = 4,    /* streamed volumes: 0 = fused carry-in (S12, default), 1 = partial images + over (S13) */
    VR_OPT_STREAM_CULL = 5,   /* streamed volumes, fused mode: 1 = bricks that no ray can still draw from are neither fetched nor
                                 ray cast (default 0): EA -- every ray that can sample the brick has reached tau, or the
                                 transfer function is zero over the brick's whole value range; MIP -- the brick's maximum
                                 cannot raise any of those rays' running maxima.  The brick's value range is measured
                                 on the device the first time it is fetched.  Decided wavefront by wavefront from the
                                 running image (one host synchronisation per wavefront).  Same pixels (reading C1). */
    VR_OPT_BEAM_STAGE = 6,    /* beam kernel: bytes of the shared-memory stage of one CTA (multiple of 16 in [4096, 196608]);
                                 0 (default) = chosen per frame from the camera: 16 KiB for dense views up to 64 KiB
                                 for sparse ones (csrc/vr_beam_plan.h: auto_stage_bytes) */
    VR_OPT_BEAM_PAD = 7,      /* beam kernel: 1 = pad the box strides against bank conflicts (default), 0 = dense */
    VR_OPT_BEAM_STAGES = 8,   /* beam kernel: 1 = one stage, copy and march alternate (default); 2 = two stages, the next
                                 slab's box is copied while this one is marched (twice the shared memory per CTA) */
    VR_OPT_BEAM_BULK = 9,     /* beam kernel: 0 = a box is copied by 16-byte cp.async, one per thread and chunk (default);
                                 1 = by cp.async.bulk, one per x row, completion counted on an mbarrier */
    VR_OPT_PIPELINE = 10,     /* direct kernel (resident cubes, streamed bricks, parts of a cube; not the skipping loop): samples a
                                 thread keeps in flight -- their voxel loads are issued before the first of them is
                                 consumed: 1, 2 or 4; 0 (default) = chosen per frame from the camera: 4 for sparse views
                                 (at most one sample per voxel: every sample is a trip to HBM), else 1.  Same pixels. */
    VR_OPT_TILE_ORDER = 11,   /* direct kernel: order in which CTAs take the 16 x 8-pixel tiles: 0 = row-major (default),
                                 1 = supertiles of 8 x 8 tiles.  Same pixels. */
    VR_OPT_STREAM_CACHE = 12,  /* streamed volumes: 1 (default) = the device slots keep their bricks from frame to frame and a
                                 brick that is still resident is not fetched again (give the volume as many slots as
                                 HBM allows: an orbit re-uses most bricks); 0 = every needed brick crosses the host
                                 link every frame.  Registered bricks must not change (register them again if they do). */
    VR_OPT_MM_BRICK = 13,     /* resident volumes: edge of the min/max bricks in cells (a power of two; vr_volume_desc::mm_brick
                                 sets the first value, default 64).  PAPER.md:9 "special attention to data with low
                                 signal to noise ratio": on noise a 64^3 brick always holds a 4.5-sigma voxel and is
                                 never skippable, an 8^3 brick often is (MIP: its maximum is below the ray's running
                                 maximum).  Edges <= 16 get a second, coarse table of 8 x the edge that is tested
                                 first, so that large empty regions are still crossed in one step.  Same pixels. */
    VR_OPT_SPACING_X = 14,    /* R23 (two sky axes and a frequency axis, different units): world units per voxel */
    VR_OPT_SPACING_Y = 15,    /* along x, y, z (default 1).  World space = voxel index x spacing: the camera, `step` and the */
    VR_OPT_SPACING_Z = 16,    /* transfer function's opacity per unit length are world-space quantities; a ray is generated in
                                 world space and mapped into index space by one multiplication per component.  With
                                 spacing (1, 1, 1) no bit changes.  Not with the beam kernel. */
    VR_OPT_BLANK_VALUE = 17,  /* R17b (real radio cubes mark masked channels and pixels with NaN): a finite value =
                                 every non-finite voxel (NaN, +-inf) is replaced by it as it arrives on the device
                                 (resident: vr_volume_upload_bricks, boxes uploaded from now on; streamed: every
                                 brick as it lands in a slot); NaN (default) = off: cubes must then be finite.
                                 VR_LAYOUT_LINEAR only. */
    VR_OPT_REUSE = 18         /* direct kernel, resident cubes, skipping off: 2 = a thread keeps the eight voxels of its last cell in
                                 registers and fetches only when the sample's cell changes (dense views with short
                                 steps: a third to three quarters of the samples), 1 = never, 0 (default) = when the view is
                                 dense (VR_OPT_PIPELINE's automatic choice took depth 1) and step <= 0.6.  Same pixels. */
};

/* Per-brick outcome of the last streamed frame (vr_get_brick_flags). */
enum {
    VR_BRICK_OUTSIDE = 1,     /* outside the view frustum */
    VR_BRICK_EMPTY = 2,       /* VR_OPT_STREAM_CULL, EA: transfer function zero over its value range */
    VR_BRICK_CULLED = 3,      /* VR_OPT_STREAM_CULL: no ray could still draw from it */
    VR_BRICK_STREAMED = 4,    /* fetched over the host link and ray cast */
    VR_BRICK_CACHED = 5       /* found in a device slot and ray cast */
};

typedef struct {
    unsigned long long rays_hit;        /* rays with tn < tf           (VR_OPT_COUNT) */
    unsigned long long samples;         /* samples evaluated (S4-S6)   (VR_OPT_COUNT) */
    unsigned long long bricks_total;    /* streamed: bricks of the cube */
    unsigned long long bricks_streamed; /* streamed: bricks copied host -> device in the last frame */
    unsigned long long bricks_skippable;/* resident: min/max bricks whose EA skip bit is set */
    unsigned long long h2d_bytes;       /* streamed: bytes copied host -> device in the last frame */
    unsigned long long mm_bricks;       /* number of min/max bricks */
    unsigned long long bricks_cached;   /* streamed: bricks of the last frame found in a device slot (VR_OPT_STREAM_CACHE) */
    unsigned long long bricks_culled;   /* streamed: bricks of the last frame no ray could still draw from (VR_OPT_STREAM_CULL) */
    unsigned long long bricks_empty;    /* streamed: bricks of the last frame the transfer function is zero on (VR_OPT_STREAM_CULL) */
    unsigned long long fetches;         /* samples whose eight voxels were fetched (VR_OPT_COUNT): = samples, less with VR_OPT_REUSE */
    double             frame_ms;        /* streamed: device time of the last frame on the render stream */
    double             h2d_ms;          /* streamed: sum of the durations of the last frame's brick copies */
    double             h2d_gbs;         /* streamed: h2d_bytes / h2d_ms */
    double             overlap_ratio;   /* streamed: h2d_ms / frame_ms (1 = the host link was busy for the whole frame) */
    int                n_slots;         /* streamed: device slots in use */
    int                kernel;          /* kernel of the last frame: 1 = direct, 2 = beam, 3 = direct with pipelined loads
                                           (VR_OPT_PIPELINE), 4 = direct with cell reuse (VR_OPT_REUSE) */
    int                beam_stage_bytes;/* beam kernel: shared-memory stage of the last frame (chosen per frame when
                                           VR_OPT_BEAM_STAGE is 0) */
    int                pipeline_depth;  /* samples in flight per thread in the last frame (1 unless kernel == 3) */
    int                timing_valid;    /* streamed: 1 once the four timing fields hold the last frame's values */
    int                reserved;
} vr_stats;

/* Bytes of d_storage a resident volume needs / bytes of one slot of a streamed
 * volume.  VR_LAYOUT_TEX needs no d_storage: both return 0 for it.  0 on invalid
 * dims too. */
size_t vr_volume_storage_bytes(const vr_volume_desc* desc);
size_t vr_volume_slot_bytes(const vr_volume_desc* desc);

/* Creates a handle.  Allocates small library-owned tables (min/max, LUT, skip
 * bits), a private copy stream and events, and -- for VR_LAYOUT_TEX only -- the
 * CUDA array(s) that hold the voxels.  *out is NULL on failure. */
vr_status vr_volume_create(const vr_volume_desc* desc, vr_volume** out);

/* PAPER.md:58-62 (Sec. 3.1 steps 1-5, the paper's own architecture: one sub-cube and one partial image per GPU,
 * combined by the scene-integration step) -- SURVEY 8(f)2, sort-last rendering.  A handle for the PART of the cube
 * `whole` (a resident description: nx, ny, nz = the whole cube) that holds the voxels [origin, origin + dims) and
 * owns the cells [origin, origin + dims - 1) per axis (S10: parts that tile the cube share one voxel layer with
 * their neighbour).  d_storage of `whole` holds the PART (dims[0]*dims[1]*dims[2] float32 for VR_LAYOUT_LINEAR).
 * vr_volume_upload_bricks takes boxes in the cube's coordinates.  vr_render on a part gives the PARTIAL image of its
 * cells, from zero (S13): EA premultiplied (C, A); MIP the raw maximum in channel 0 (-inf where the part has no
 * sample) -- combine partial images in view order with vr_composite, then vr_mip_finish (MIP).  No skipping, no aux,
 * direct kernel. */
vr_status vr_volume_create_part(const vr_volume_desc* whole, const int origin[3], const int dims[3], vr_volume** out);

/* PAPER.md:62 (Sec. 3.1 step 5, "scene integration"), S13: running = running OVER partial (EA, front to back: the
 * partial image lies behind everything composited so far) or max (MIP, raw maxima in channel 0), pixel by pixel.
 * Both DEVICE pointers to W*H*4 float32.  The first partial image is composited onto zeros (EA) / onto the image
 * vr_render gives for a part that has no sample (MIP: -inf in channel 0). */
vr_status vr_composite(float* running_rgba, const float* partial_rgba, int width, int height, int mode, void* stream);

/* PAPER.md:62 "reapplies the same transfer function" (reading R14): the combined raw maxima (channel 0 of running)
 * -> LUT colour, alpha 1 (0 where no sample), with `vol`'s transfer function; aux (if set) receives the maxima. */
vr_status vr_mip_finish(vr_volume* vol, float* running_rgba, int width, int height, void* stream);

/* Frees what vr_volume_create allocated (never d_storage or caller bricks);
 * synchronises the private copy stream first.  NULL is allowed. */
void vr_volume_destroy(vr_volume* vol);

/* PAPER.md:58 (Sec. 3.1 step 1).  n boxes of voxels: box q covers voxels
 * origin[q] .. origin[q]+dims[q]-1 (x, y, z order) and ptrs[q] points at
 * dims[q][0]*dims[q][1]*dims[q][2] float32, x fastest, dense.
 * Resident: copies every box into the device layout on `stream` (asynchronous;
 *   host pointers should be pinned to overlap) and marks the min/max table stale;
 *   boxes may be any partition of the cube, or a single box = the whole cube.
 *   ptrs_are_device = 1 means device pointers (a box equal to d_storage itself is
 *   accepted as "already in place").
 * Streamed: registers the pointers (no copy); the boxes must be exactly the
 *   bricks described at vr_volume_desc (any order), in pinned host memory that
 *   outlives the handle; ptrs_are_device must be 0.
 * stream: cudaStream_t as void* (NULL = legacy default stream). */
vr_status vr_volume_upload_bricks(vr_volume* vol, int n, const int (*origin)[3],
                                  const int (*dims)[3], const float* const* ptrs,
                                  int ptrs_are_device, void* stream);

/* PAPER.md:60 "preselected transfer function" (S7).  lut_rgba: HOST pointer to
 * n_entries*4 float32, straight (non-premultiplied) colours and opacity per
 * unit length (1 voxel); node i sits at value vmin + i*(vmax-vmin)/(n_entries-1);
 * lookups are linear between nodes and clamped.  Copied; 2 <= n_entries <= 4096. */
vr_status vr_set_transfer_function(vr_volume* vol, const float* lut_rgba, int n_entries,
                                   float vmin, float vmax);

/* PAPER.md:9 "control the volume rendering process": the knobs of the render that are not part of
 * the camera or the transfer function (keys above).  VR_ERR_INVALID_ARG for an unknown key or a
 * value outside its range, VR_ERR_UNSUPPORTED for an option the volume's kind does not have. */
vr_status vr_set_option(vr_volume* vol, int key, double value);

/* Optional second output of the next renders: d_aux = device float32 W*H (MIP:
 * raw maximum per pixel, -inf where the ray has no sample; EA: -inf).  NULL
 * switches it off. */
vr_status vr_set_aux_output(vr_volume* vol, float* d_aux);

/* PAPER.md:60-62 (Sec. 3.1 steps 3-5).  Renders one frame into out_rgba: DEVICE
 * pointer to width*height*4 float32, out_rgba[(j*W+i)*4+c], row 0 = top,
 * premultiplied colour, no background, no gamma; a ray that misses the cube
 * gives (0,0,0,0).  step: sample spacing along the ray in voxels (> 0).
 * Resident volume: enqueues kernels on `stream` and returns without
 * synchronising.  Streamed volume: enqueues brick copies on the private copy
 * stream and per-brick kernels on `stream`, ordered by events; out_rgba is
 * complete once `stream` is. */
vr_status vr_render(vr_volume* vol, const vr_camera* cam, int width, int height,
                    float step, int mode, float* out_rgba, void* stream);

/* PAPER.md:25 (design objective 5, "tiled display"), reading W1 of DESIGN.md: the same frame delivered
 * as a K x L display wall in ONE launch.  Tile (a, b) -- column a from the left, row b from the top --
 * is the camera's off-axis sub-frustum through the rectangle [a/K, (a+1)/K] x [b/L, (b+1)/L] of the
 * image plane, sampled at the frame's own pixel centres: its pixels are bit for bit the pixels
 * [a*w, (a+1)*w) x [b*h, (b+1)*h) of vr_render's width x height frame (w = width/K, h = height/L).
 * outs: HOST array of K*L DEVICE pointers, outs[b*K + a] = w*h*4 float32 of tile (a, b), each dense.
 * width % K == 0, height % L == 0, K*L <= 64.  Resident volumes, direct kernel, no aux output. */
vr_status vr_render_wall(vr_volume* vol, const vr_camera* cam, int width, int height, int K, int L,
                         float step, int mode, float* const* outs, void* stream);

/* PAPER.md:24 (design objective 4, "minimum user intervention"): measures the variants of the direct
 * kernel on ONE representative frame of the caller's -- plain, VR_OPT_PIPELINE 2 and 4, VR_OPT_REUSE on, each under
 * VR_OPT_TILE_ORDER 0 and 1, each rendered three times into out_rgba (device, width*height*4 float32, left holding
 * a valid frame), timed with events on `stream` -- and sets the three options to the fastest combination, also
 * returned through pipeline_out / tile_order_out / reuse_out (each may be NULL).  All variants give the same pixels.
 * Synchronises `stream`.  Resident whole cubes only. */
vr_status vr_autotune(vr_volume* vol, const vr_camera* cam, int width, int height, float step, int mode,
                      float* out_rgba, void* stream, int* pipeline_out, int* tile_order_out, int* reuse_out);

/* Same frame delivered to HOST memory: renders into d_staging (device,
 * width*height*4 float32, caller owned) and copies to h_out_rgba (pinned host
 * memory for an asynchronous copy) on `stream`. */
vr_status vr_render_host(vr_volume* vol, const vr_camera* cam, int width, int height,
                         float step, int mode, float* d_staging, float* h_out_rgba,
                         void* stream);

/* A2: the per-brick min / max table (brick b covers voxels
 * [max(B*b-1,0), min(B*b+B+1, n-1)] per axis, B = mm_brick).  Computes it on the
 * device if stale, then copies nbx*nby*nbz floats each to the HOST arrays
 * (brick index bx + nbx*(by + nby*bz)); synchronises `stream`.  Resident only. */
vr_status vr_get_minmax(vr_volume* vol, float* h_min, float* h_max, void* stream);

/* PAPER.md:9 (the user "controls" and therefore observes the process): counters of the last frame
 * (synchronises the device if VR_OPT_COUNT is on; waits for the last streamed frame to read its timing). */
vr_status vr_get_stats(vr_volume* vol, vr_stats* out);

/* Streamed volumes: what happened to each brick in the last frame -- flags_out has one VR_BRICK_* value per
 * brick (linear brick index bx + nbx*(by + nby*bz)), 0 for bricks of a volume that has not rendered yet. */
vr_status vr_get_brick_flags(vr_volume* vol, int* flags_out);

/* Front-to-back order (S11) of the streamed bricks for a camera: order_out has
 * one linear brick index per brick, keys_out (may be NULL) its wavefront key.
 * Host-only logic; works for resident volumes too when brick_edge > 0 is given. */
vr_status vr_brick_order(const vr_volume_desc* desc, int brick_edge, const vr_camera* cam,
                         int* order_out, int* keys_out);

/* Diagnostic of the beam kernel (VR_OPT_KERNEL = 2), host-only logic, needs no GPU and renders nothing:
 * the slabs that the CTA of pixel tile (tile_i, tile_j) -- 16 x 8 pixels, first pixel (16*tile_i,
 * 8*tile_j) -- marches through and the voxel box it stages for each, computed by the very functions
 * thread 0 of the kernel runs (csrc/vr_beam_plan.h).  Needs nx % 4 == 0 like the kernel.
 * stage_bytes <= 0 takes the per-frame choice of VR_OPT_BEAM_STAGE = 0, pad_mode < 0 the default of VR_OPT_BEAM_PAD.
 * slabs_out: max_slabs records of 16 ints {kind (1 = staged box, 2 = direct global loads), first cell
 * of the slab, depth in cells, box origin x y z, box extent x y z, shared-memory stride x y z (floats),
 * floats of the stage spanned, largest corner index allowed, 16-byte chunks per x row, depth set used};
 * info_out: 10 ints {slab axis, 1 if marched towards +axis, first cell, last cell, number of slabs (may
 * exceed max_slabs), 1 if the whole tile is direct, rays of the tile that hit the cube, bytes of the
 * stage, fast (stride 1) axis, pad mode}.  Tests use it to check that every sample finds its eight
 * voxels inside the box of its slab. */
vr_status vr_beam_plan(const vr_volume_desc* desc, const vr_camera* cam, int width, int height,
                       int tile_i, int tile_j, int stage_bytes, int pad_mode, int max_slabs,
                       int* slabs_out, int* info_out);

/* Page-locked host memory for streamed bricks (A12): bricks must be pinned for the
 * copy engine to overlap with rendering, and generic pinned allocators round sizes
 * up (a 513^3 brick is 515 MiB).  *out is NULL on failure (VR_ERR_OOM_HOST).
 * vr_host_free accepts NULL. */
vr_status vr_host_alloc(size_t bytes, void** out);
void      vr_host_free(void* p);

const char* vr_last_error(void);

/* Library version string, e.g. "vr-b200 0.1 (sm_100a)". */
const char* vr_version(void);

#ifdef __cplusplus
}
#endif
#endif /* VR_H */
