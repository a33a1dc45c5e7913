// vr_beam_plan.h -- the geometry of the beam kernel (vr_beam.cu), host + device.
//
// Which slab axis a tile marches along, which cells of that axis its rays cross, and which
// box of voxels covers everything the tile's rays can sample inside one slab.  The producer
// warp of raycast_beam_kernel runs exactly these functions; vr_beam_plan() (vr_api.cu) runs
// them on the host so that the coverage property -- every sample of every ray of the tile finds
// its eight voxels inside the box of its slab -- can be tested without a GPU.
// None of this touches pixel values: a wrong box would read wrong voxels, a right box reads
// the same voxels as the direct kernel.
#pragma once

#include "vr_device.cuh"

#ifdef __CUDA_ARCH__
#define VR_FLOOR_I(x) __float2int_rd(x)
#else
#define VR_FLOOR_I(x) ((int)floorf(x))
#endif

namespace vr {
namespace beam {

using dev::Ray;

struct SlabBox {
    int kind;                  // 1 = box staged in shared memory, 2 = direct (global loads)
    int depth;                 // cells of the slab along the slab axis
    int clo;                   // first cell of the slab
    int org[3];                // voxel index of box element 0
    int dim[3];                // box extents in voxels
    int map_index;             // index into BeamParams::maps
    unsigned int bytes;        // box bytes = TMA transaction size
};

// Ladder and depth sets of the TMA boxes (see BeamParams).  Returns the number of maps.
__host__ __device__ inline int default_ladder(BeamParams& B)
{
    B.lx0 = 12; B.lxs = 8; B.nlx = 8;        // 12 .. 68 voxels along x (never a multiple of 16: shared-memory banks)
    B.ly0 = 5;  B.lys = 4; B.nly = 16;       // 5 .. 65 voxels along y / z
    B.stage_bytes = 24576;
    const int depth[kBeamSets][3] = {{11, 8, 8}, {3, 4, 4}};   // x slabs: depth + 1 is a multiple of 4 (16-byte rows)
    int n_maps = 0;
    for (int s = 0; s < kBeamSets; ++s)
        for (int a = 0; a < 3; ++a) {
            B.depth[s][a] = depth[s][a];
            B.map_base[s][a] = n_maps;
            n_maps += (a == 0 ? B.nly : B.nlx) * B.nly;
        }
    return n_maps;
}

// Unnormalised direction of the ray through the centre of the tile whose first pixel is
// (tile_x, tile_y): its dominant axis is the slab axis of the whole tile.
__host__ __device__ inline void tile_centre_direction(const FrameParams& P, int tile_x, int tile_y, float D[3])
{
    D[0] = P.fwd[0]; D[1] = P.fwd[1]; D[2] = P.fwd[2];
    if (P.projection == VR_PROJ_PERSPECTIVE) {
        const float a = ((float)(2 * tile_x + kTileW) / (float)P.W - 1.0f) * ((float)P.W / (float)P.H) * P.th;
        const float b = (1.0f - (float)(2 * tile_y + kTileH) / (float)P.H) * P.th;
        for (int c = 0; c < 3; ++c) D[c] = P.fwd[c] + a * P.right[c] + b * P.up[c];
    }
}

__host__ __device__ inline int dominant_axis(const float D[3])
{
    const float m0 = fabsf(D[0]), m1 = fabsf(D[1]), m2 = fabsf(D[2]);
    if (m0 >= m1 && m0 >= m2) return 0;
    return m1 >= m2 ? 1 : 2;
}

// A ray fits the tile's slab march when it advances along the slab axis in the tile's sense
// and not too obliquely (boxes grow with the slope).
__host__ __device__ inline bool ray_is_bad(const float d[3], int AX, bool pos)
{
    return ((d[AX] > 0.0f) != pos) || fabsf(d[AX]) < 0.25f;
}

// Cells [ca, cb] of the slab axis that the samples of a clipped ray can fall into: positions are
// monotone in t (correctly rounded fma), every sample has tn <= t_k < tf.
__host__ __device__ inline void ray_cell_range(const FrameParams& P, const Ray& r, int AX, int& ca, int& cb)
{
    const float ha = (float)(P.n[AX] - 1);
    const float pa = fminf(fmaxf(VR_FMA(r.tn, r.d[AX], r.o[AX]), 0.0f), ha);
    const float pb = fminf(fmaxf(VR_FMA(r.tf, r.d[AX], r.o[AX]), 0.0f), ha);
    ca = min(VR_FLOOR_I(fminf(pa, pb)), P.n[AX] - 2);
    cb = min(VR_FLOOR_I(fmaxf(pa, pb)), P.n[AX] - 2);
}

// Span {umin, umax, vmin, vmax} of one corner line of the tile between the planes that bound the
// cells [clo, clo + D) of the slab axis, clamped to the cube like the sample positions are.
// inv_a = 1 / d[AX].  (U, V) = the two other axes in ascending order.
__host__ __device__ inline void corner_span(const Ray& c, float inv_a, int AX, int clo, int D, const int n[3], float span[4])
{
    const int U = AX == 0 ? 1 : 0, V = AX == 2 ? 1 : 2;
    const float su = c.d[U] * inv_a, sv = c.d[V] * inv_a;
    const float hu = (float)(n[U] - 1), hv = (float)(n[V] - 1);
    const float a0 = (float)max(clo, 0) - c.o[AX];
    const float a1 = (float)min(clo + D, n[AX] - 1) - c.o[AX];
    const float u0 = fminf(fmaxf(c.o[U] + a0 * su, 0.0f), hu), u1 = fminf(fmaxf(c.o[U] + a1 * su, 0.0f), hu);
    const float v0 = fminf(fmaxf(c.o[V] + a0 * sv, 0.0f), hv), v1 = fminf(fmaxf(c.o[V] + a1 * sv, 0.0f), hv);
    span[0] = fminf(u0, u1); span[1] = fmaxf(u0, u1);
    span[2] = fminf(v0, v1); span[3] = fmaxf(v0, v1);
}

// The ladder box of depth set s that covers the span (already reduced over the four corners) with
// a quarter-voxel margin, plus the far corner of the last cell.  False when no entry fits a stage.
__host__ __device__ inline bool choose_box(const BeamParams& B, int s, int AX, int clo, const float span[4], SlabBox& out)
{
    const int U = AX == 0 ? 1 : 0, V = AX == 2 ? 1 : 2;
    const int D = B.depth[s][AX];
    const int lo_u = VR_FLOOR_I(span[0] - 0.25f), need_u = VR_FLOOR_I(span[1] + 0.25f) + 2 - lo_u;
    const int lo_v = VR_FLOOR_I(span[2] - 0.25f), need_v = VR_FLOOR_I(span[3] + 0.25f) + 2 - lo_v;
    const int u0l = U == 0 ? B.lx0 : B.ly0, usl = U == 0 ? B.lxs : B.lys, unl = U == 0 ? B.nlx : B.nly;
    const int iu = max(0, (need_u - u0l + usl - 1) / usl);
    const int iv = max(0, (need_v - B.ly0 + B.lys - 1) / B.lys);
    const int size_u = u0l + usl * iu, size_v = B.ly0 + B.lys * iv;
    const unsigned int nbytes = (unsigned int)size_u * (unsigned int)size_v * (unsigned int)(D + 1) * 4u;
    if (iu >= unl || iv >= B.nly || nbytes > (unsigned int)B.stage_bytes) return false;
    out.kind = 1;
    out.depth = D;
    out.clo = clo;
    out.org[AX] = clo; out.org[U] = lo_u; out.org[V] = lo_v;
    out.dim[AX] = D + 1; out.dim[U] = size_u; out.dim[V] = size_v;
    out.map_index = B.map_base[s][AX] + iu * B.nly + iv;
    out.bytes = nbytes;
    return true;
}

}  // namespace beam
}  // namespace vr
