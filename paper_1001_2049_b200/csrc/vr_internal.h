// vr_internal.h -- structs shared by the host API (vr_api.cu) and the kernels
// (vr_kernels.cu).  Not part of the public boundary (include/vr.h).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/vr.h"

// Kernel launch and dynamic shared memory, spelled so that tests/hostemu (a host emulation of the CUDA subset used
// here, test infrastructure only) can compile these sources with a plain C++ compiler.  VR_HOSTEMU is never defined
// in the product build.
#ifdef VR_HOSTEMU
#define VR_LAUNCH(kern, grid, block, smem, stream, ...) emu::launch(kern, grid, block, smem, stream, __VA_ARGS__)
#define VR_DYN_SHARED(T, name) T* name = reinterpret_cast<T*>(emu::dyn_smem())
#else
#define VR_LAUNCH(kern, grid, block, smem, stream, ...) kern<<<(grid), (block), (smem), (stream)>>>(__VA_ARGS__)
#define VR_DYN_SHARED(T, name) extern __shared__ __align__(16) T name[]
#endif

namespace vr {

constexpr int kTileW = 16;        // pixels per CTA tile in x (2 warps of 8)
constexpr int kTileH = 8;         // pixels per CTA tile in y (2 warps of 4)
constexpr int kThreads = 128;     // 4 warps, each an 8 x 4 pixel footprint
constexpr int kMaxLut = 4096;

// VR_LAYOUT_TEX: a 2D-layered array holds at most 2048 layers, so a resident cube with more channels is cut along z
// into chunks of `chunk_step` + 1 layers that overlap by one layer: chunk c holds layers [c * chunk_step,
// c * chunk_step + chunk_step], and a sample whose cell has z index iz finds both of its layers (iz, iz + 1) in chunk
// iz / chunk_step.  configs[4] (8192 channels) takes 5 chunks.
constexpr int kMaxTexChunks = 8;

// One box of voxels in device memory: the whole resident cube (origin 0) or one
// streamed brick in a slot.  `base` is pre-offset so that the voxel with GLOBAL
// index (x, y, z) is base[(z*sz) + (y*sy) + x].
struct VoxelBox {
    const float* base;
    long long sy, sz;             // strides in elements
    // VR_LAYOUT_TEX: 2D-layered arrays, texel (u, v, layer l) of chunk c = voxel (u + org[0], v + org[1],
    // l + c * chunk_step + org[2]); gx = 1 - org[0], gy = 1 - org[1] (exact small integers): the gather at
    // ((float)ix + gx, (float)iy + gy) sits on the corner shared by texels ix..ix+1, iy..iy+1
    cudaTextureObject_t tex[kMaxTexChunks];
    int   n_chunks;               // 1: everything is in tex[0]
    int   chunk_step;             // layers from one chunk's first layer to the next one's
    unsigned int chunk_magic;     // beam::magic_of(chunk_step): layer / chunk_step = umulhi(layer, chunk_magic)
    float gx, gy;
    int   org_z;
};

// W1 ("tiled display"): a frame delivered as wall_k x wall_l tiles, each into its own buffer
constexpr int kMaxWallTiles = 64;

// Everything a ray needs (S1-S9).  Passed as __grid_constant__.
struct FrameParams {
    float eye[3], right[3], up[3], fwd[3];
    int   projection;
    float th, hh;                 // tan_half_fovy, ortho_half_height
    // R23: anisotropic voxel spacing.  aniso != 0: the world-space ray (o, d) becomes (o * inv_sp, d * inv_sp) in
    // index space, t stays world distance; aniso == 0 (also the value of a zeroed struct): nothing is multiplied
    int   aniso;
    float inv_sp[3];
    int   W, H;
    float step, inv_step, tau;
    int   n[3];
    VoxelBox vol;
    // classification (S7): lut[q] = (r, g, b, alpha'), lut[n_lut + q] = lut[q+1] - lut[q]
    const float4* lut;
    int   n_lut;
    float vmin, scale;
    // output
    float4* out;
    float*  aux;
    // display wall (vr_render_wall): wall_k > 0 -> pixel (i, j) of the frame goes to pixel (i % wall_w, j % wall_h) of
    // wall_out[(j / wall_h) * wall_k + i / wall_w] instead of out[j * W + i]
    int     wall_k, wall_l, wall_w, wall_h;
    float4* wall_out[kMaxWallTiles];
    // pixel rectangle rendered by this launch and its tiling
    int   x0, y0, x1, y1;
    int   tiles_x, tiles_y;
    int   tile_order;             // dev::tile_of_block: 0 = row-major, 1 = 8 x 8 supertiles (direct and pipelined kernels)
    // empty-space skipping over min/max bricks of edge 2^mm_shift cells (A10)
    const float2*  minmax;
    const uint8_t* skip;
    int   nb[3];
    int   mm_shift;
    // optional coarse level over the same cube (bricks 8 x the edge): tested first, so that large empty regions are
    // crossed in one step; mm2_shift == 0: none
    const float2*  minmax2;
    const uint8_t* skip2;
    int   nb2[3];
    int   mm2_shift;
    // streamed brick (S10, S12): cells owned [clo, chi) per axis
    int   clo[3], chi[3];
    int   fresh;                  // 1: start from zero and write every pixel (partial image, S13)
    unsigned long long* counters; // [0] rays hit, [1] samples evaluated, [2] samples whose eight voxels were fetched (cell-reuse kernel)
};

// kernel parameters live in the 4 KiB constant parameter space (the beam kernel passes BeamParams besides)
static_assert(sizeof(FrameParams) <= 3072, "FrameParams must leave room in the kernel parameter space");

// Beam kernel (vr_beam.cu): a tile's rays are marched in slabs along their dominant axis and the
// voxel box of every slab is staged in shared memory.  Depth set s, slab axis a: a slab holds
// depth[s][a] cells (depth + 1 voxel planes) along a; set 0 is tried first, then the thinner ones.
constexpr int kBeamSets = 4;
struct BeamParams {
    int depth[kBeamSets][3];
    int stage_bytes;              // bytes of one shared-memory stage (multiple of 16)
    int n_stages;                 // 1: copy | march alternate (2 barriers per slab); 2: the next box is copied while
                                  // this one is marched (1 barrier per slab, twice the shared memory)
    int pad_mode;                 // 0 = dense strides, 1 = strides padded against bank conflicts
    int bulk;                     // 1: x rows of a box are copied by cp.async.bulk (one instruction per row, completion
                                  // counted on an mbarrier) instead of per-thread 16-byte cp.async; x slabs are unaffected
    int use_skip;                 // 1 (EA only): slabs whose min/max bricks are all skippable are neither copied nor sampled (A10)
    // EA classification shortcuts, both exact (vr_beam_plan.h: lut_is_grey, lut_zero_bits):
    const float4* lut_grey;       // r = g = b in every LUT entry: table of (grey, alpha', d grey, d alpha'), else null
    int zero_skip;                // 1: zero_bits is in use
    unsigned int zero_bits[32];   // bit q set: alpha'[q] = alpha'[q+1] = 0, a sample in LUT cell q adds exactly nothing
};

struct MinMaxParams {
    VoxelBox vol;
    int tex;                      // 1: read through vol.tex
    int n[3];
    int nb[3];
    int B;
    float2* out;
};

// coarse table from the fine one: brick b of edge 8 B = the 8 x 8 x 8 fine bricks it holds (their voxel ranges with
// the one-voxel ring add up to exactly the coarse brick's)
struct CoarseParams {
    const float2* fine;
    int nb[3];                    // fine grid
    float2* coarse;
    int nb2[3];                   // coarse grid
};

struct SkipParams {
    const float2* minmax;
    int n_bricks;
    const int* nz_prefix;         // nz_prefix[i] = number of entries j < i with alpha'_j != 0
    int n_lut;
    float vmin, scale;
    uint8_t* skip;
    unsigned int* n_skippable;
};

// launchers (vr_kernels.cu)
cudaError_t launch_raycast(const FrameParams& P, int mode, bool skip, bool count, bool brick,
                           bool tex, cudaStream_t stream);
cudaError_t launch_raycast_pipe(const FrameParams& P, int mode, bool count, bool brick, bool tex, int depth, cudaStream_t stream);
cudaError_t launch_raycast_reuse(const FrameParams& P, int mode, bool count, bool tex, cudaStream_t stream);
cudaError_t launch_raycast_beam(const FrameParams& P, const BeamParams& B, int mode, bool count,
                                cudaStream_t stream);
cudaError_t beam_fault_flag(unsigned int* flag);
cudaError_t launch_minmax(const MinMaxParams& P, cudaStream_t stream);
cudaError_t launch_coarse_minmax(const CoarseParams& P, cudaStream_t stream);
cudaError_t launch_skipbits(const SkipParams& P, cudaStream_t stream);
// min / max of a streamed brick as it sits in its slot (dense dims[0] x dims[1] x dims[2] voxels from first_voxel, or
// the texels [0, dims) of the slot's layered array) folded into out[0], out[1]
cudaError_t launch_brick_range(const float* first_voxel, cudaTextureObject_t tex, bool is_tex, const int dims[3],
                               float* out, cudaStream_t stream);
cudaError_t launch_cull_reduce(const FrameParams& P, int mode, float* out, cudaStream_t stream);
cudaError_t launch_blank(float* p, const int dims[3], long long sy, long long sz, float value, cudaStream_t stream);
cudaError_t launch_mip_init(float4* out, int W, int H, cudaStream_t stream);
cudaError_t launch_fill(float* p, size_t n, float value, cudaStream_t stream);
cudaError_t launch_mip_finish(const FrameParams& P, cudaStream_t stream);
cudaError_t launch_composite(float4* running, const float4* partial, int W, int x0, int y0,
                             int x1, int y1, int mode, cudaStream_t stream);

}  // namespace vr
