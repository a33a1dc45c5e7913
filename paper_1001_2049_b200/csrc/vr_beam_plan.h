// vr_beam_plan.h -- the geometry of the beam kernel (vr_beam.cu), host + device.
//
// Which slab axis a 16 x 8 pixel tile marches along, which cells of that axis its rays cross,
// and which box of voxels covers everything the tile's rays can sample inside one slab, with the
// shared-memory strides the box is stored with.  Thread 0 of raycast_beam_kernel runs exactly
// these functions; vr_beam_plan() (vr_api.cu) and the host harness tests/beam_harness.cu run
// them on the host, so the coverage property -- every sample of every ray of the tile finds its
// eight voxels inside the box of its slab -- is tested without a GPU.
// None of this touches pixel values: a wrong box would read wrong voxels, a right box reads
// the same voxels as the direct kernel.
#pragma once

#include "vr_device.cuh"

#include <cstring>

#ifdef __CUDA_ARCH__
#define VR_FLOOR_I(x) __float2int_rd(x)
#else
#define VR_FLOOR_I(x) ((int)floorf(x))
#endif

namespace vr {
namespace beam {

using dev::Ray;

// One slab of a tile's march and the staged box that serves it.
struct Slab {
    int kind;                  // 0 = end of the beam, 1 = box staged in shared memory, 2 = direct (global loads),
                               // 3 = empty: every min/max brick its samples can fall into is skippable (A10)
    int set;                   // depth set the slab was planned with (kBeamSets for a direct slab)
    int clo, depth;            // the slab owns cells [clo, clo + depth) of the slab axis
    int org[3];                // voxel index of box element (0, 0, 0)
    int dim[3];                // box extents in voxels; fast axis x: org[0] and dim[0] are multiples of 4 (16-byte chunks)
    int str[3];                // shared-memory strides in floats; str[fast axis] == 1
    int floats;                // floats of the stage the box spans
    int lim;                   // largest index a sample may use for its corner 000 (defensive clamp)
    int cx;                    // 16-byte chunks read per x row
    int interior;              // 1: the box touches no face of the cube (voxels 1 .. n - 2 on every axis)
    int xoff;                  // x slabs: elements of the first chunk that precede org[0] (0 when x is the fast axis)
    unsigned int mg0, mg1;     // magic_of() the two divisors of the copy loop (see copy_box)
    float lo_f, hi_f;          // (float)clo, (float)(clo + depth)
    float of[3];               // (float)org
    float fsm, fss;            // (float)str[middle axis], (float)str[slab axis]
};

// What a tile's threads share (shared memory on the device).
struct TileGeom {
    float co[4][3], cd[4][3];  // origin and unit direction of the four corner rays of the tile
    float su[4], sv[4];        // their slopes d[U] / d[AX], d[V] / d[AX] (corner_slopes)
    int AX;                    // slab axis = dominant axis of the tile's central ray
    int FAST;                  // axis stored with stride 1 in shared memory
    int pos;                   // 1: the march goes towards +AX
    int cmin, cmax;            // cells of AX that the samples of the tile's rays fall into
    int flags;                 // != 0: some ray does not fit the slab march -> the whole tile is direct
    int alive;                 // warps that still have unfinished rays
};

// Depth sets: deep slabs first, thinner ones when the deep box does not fit the stage (sparse views).
__host__ __device__ inline void default_params(BeamParams& B)
{
    const int depth[kBeamSets][3] = {{12, 8, 8}, {4, 4, 4}, {2, 2, 2}, {1, 1, 1}};
    for (int s = 0; s < kBeamSets; ++s)
        for (int a = 0; a < 3; ++a) B.depth[s][a] = depth[s][a];
    B.stage_bytes = 32768;
    B.n_stages = 1;
    B.pad_mode = 1;
    B.bulk = 0;
    B.use_skip = 0;
    B.lut_grey = nullptr;
    B.zero_skip = 0;
    for (int q = 0; q < 32; ++q) B.zero_bits[q] = 0u;
}

// ---- exact shortcuts of the EA classification (S7, S8), decided on the host from the table the
// kernels read: tab[4q..] = (r, g, b, alpha') of entry q, tab[4(n+q)..] = entry q+1 minus entry q.

// r, g and b are the same bits in every entry: the three colour channels of a ray then go through
// the same operations on the same values, so one channel is computed and stored three times.
inline bool lut_is_grey(const float* tab, int n)
{
    for (int q = 0; q < 2 * n; ++q)
        if (std::memcmp(tab + 4 * q, tab + 4 * q + 1, sizeof(float)) != 0 ||
            std::memcmp(tab + 4 * q, tab + 4 * q + 2, sizeof(float)) != 0)
            return false;
    return true;
}

// out[4q..] = (grey, alpha', d grey, d alpha') of entry q: one 16-byte read per sample instead of two
inline void lut_grey_table(const float* tab, int n, float* out)
{
    for (int q = 0; q < n; ++q) {
        out[4 * q + 0] = tab[4 * q + 0];
        out[4 * q + 1] = tab[4 * q + 3];
        out[4 * q + 2] = tab[4 * (n + q) + 0];
        out[4 * q + 3] = tab[4 * (n + q) + 3];
    }
}

// Bit q (q <= n - 2, n <= 1024) is set when alpha'[q] and alpha'[q+1] are both +0: the interpolated
// alpha of a sample in LUT cell q is then fma(g, 0, 0) = 0, its weight 0, and fma(0, rgb, C) = C,
// A + 0 = A: the sample leaves the ray exactly as it found it and need not be classified.
// Returns the number of bits set.
inline int lut_zero_bits(const float* tab, int n, unsigned int bits[32])
{
    for (int w = 0; w < 32; ++w) bits[w] = 0u;
    if (n > 1024) return 0;
    int count = 0;
    const float zero = 0.0f;
    for (int q = 0; q + 1 < n; ++q)
        if (std::memcmp(&tab[4 * q + 3], &zero, sizeof(float)) == 0 &&
            std::memcmp(&tab[4 * (q + 1) + 3], &zero, sizeof(float)) == 0) {
            bits[q >> 5] |= 1u << (q & 31);
            ++count;
        }
    return count;
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

// Slab axis, marching sense and fast axis of a tile.  The fast axis is x (16-byte copies of x rows)
// unless x is the slab axis: then it is the axis the image's `right` vector runs along, so that the
// eight pixels of a warp row read consecutive shared-memory words.
__host__ __device__ inline void tile_axes(const FrameParams& P, int tile_x, int tile_y, TileGeom& G)
{
    float D[3];
    tile_centre_direction(P, tile_x, tile_y, D);
    G.AX = dominant_axis(D);
    G.pos = D[G.AX] > 0.0f ? 1 : 0;
    G.FAST = 0;
    if (G.AX == 0) G.FAST = fabsf(P.right[2]) >= fabsf(P.right[1]) ? 2 : 1;
}

// component a of a 3-vector without dynamic indexing (keeps rays in registers on the device)
__host__ __device__ __forceinline__ float pick(const float v[3], int a)
{
    return a == 0 ? v[0] : (a == 1 ? v[1] : v[2]);
}

__host__ __device__ __forceinline__ int pick(const int v[3], int a)
{
    return a == 0 ? v[0] : (a == 1 ? v[1] : v[2]);
}

// A ray fits the tile's slab march when it advances along the slab axis in the tile's sense
// and not too obliquely (boxes grow with the slope).
__host__ __device__ inline bool ray_is_bad(const float d[3], int AX, bool pos)
{
    const float da = pick(d, AX);
    return ((da > 0.0f) != pos) || fabsf(da) < 0.25f;
}

// Cells [ca, cb] of the slab axis that the samples of a clipped ray can fall into: positions are
// monotone in t (correctly rounded fma), every sample has tn <= t_k < tf.
__host__ __device__ inline void ray_cell_range(const FrameParams& P, const Ray& r, int AX, int& ca, int& cb)
{
    const int na = pick(P.n, AX);
    const float ha = (float)(na - 1), da = pick(r.d, AX), oa = pick(r.o, AX);
    const float pa = fminf(fmaxf(VR_FMA(r.tn, da, oa), 0.0f), ha);
    const float pb = fminf(fmaxf(VR_FMA(r.tf, da, oa), 0.0f), ha);
    ca = min(VR_FLOOR_I(fminf(pa, pb)), na - 2);
    cb = min(VR_FLOOR_I(fmaxf(pa, pb)), na - 2);
}

// Slopes of the four corner lines against the slab axis, once per tile (G.AX and the corner rays set).
// A tile with a corner ray that does not fit the march (ray_is_bad) is direct and never uses them.
__host__ __device__ inline void corner_slopes(TileGeom& G)
{
    const int U = G.AX == 0 ? 1 : 0, V = G.AX == 2 ? 1 : 2;
    for (int q = 0; q < 4; ++q) {
        const float da = pick(G.cd[q], G.AX);
        const float inv_a = da != 0.0f ? 1.0f / da : 0.0f;
        G.su[q] = pick(G.cd[q], U) * inv_a;
        G.sv[q] = pick(G.cd[q], V) * inv_a;
    }
}

// Span {umin, umax, vmin, vmax} of one corner line of the tile between the planes that bound the
// cells [clo, clo + D) of the slab axis, clamped to the cube like the sample positions are.
// (U, V) = the two other axes in ascending order.  Positions on a plane of constant slab
// coordinate are a linear-fractional function of the pixel coordinates, so over the tile their
// extremes sit at its four corners; inside the slab a position lies between its two plane points.
template <int AX>
__host__ __device__ inline void corner_span(const float o[3], float su, float sv, int clo, int D, const int n[3],
                                            float span[4])
{
    constexpr int U = AX == 0 ? 1 : 0, V = AX == 2 ? 1 : 2;
    const float hu = (float)(n[U] - 1), hv = (float)(n[V] - 1);
    const float a0 = (float)max(clo, 0) - o[AX];
    const float a1 = (float)min(clo + D, n[AX] - 1) - o[AX];
    const float u0 = fminf(fmaxf(o[U] + a0 * su, 0.0f), hu), u1 = fminf(fmaxf(o[U] + a1 * su, 0.0f), hu);
    const float v0 = fminf(fmaxf(o[V] + a0 * sv, 0.0f), hv), v1 = fminf(fmaxf(o[V] + a1 * sv, 0.0f), hv);
    span[0] = fminf(u0, u1); span[1] = fmaxf(u0, u1);
    span[2] = fminf(v0, v1); span[3] = fmaxf(v0, v1);
}

// e / d for e * d < 2^32 is umulhi(e, 2^32 / d + 1); d == 1 has no 32-bit magic number and is coded as 0
__host__ __device__ inline unsigned int magic_of(unsigned int d)
{
    // 0xffffffff / d + 1 = floor(2^32 / d) + 1, or exactly 2^32 / d when d is a power of two: both divide exactly
    return d <= 1u ? 0u : 0xffffffffu / d + 1u;
}

// smallest v >= w with v % mod == rem
__host__ __device__ inline int pad_to(int w, int mod, int rem)
{
    const int r = ((rem - w) % mod + mod) % mod;
    return w + r;
}

// The box of voxels that covers the span (already reduced over the four corners) with a
// quarter-voxel margin plus the far corner of the last cell, its x range widened to 16-byte chunks,
// and the strides it is stored with.  False when it does not fit the stage.
//   fast axis x (y and z slabs): rows of x are copied as 16-byte chunks, so every stride is a multiple
//     of 4 floats; pad_mode 1 makes the row stride = 8 mod 16 so that the four pixel rows of a warp's
//     8 x 4 footprint fall into four different groups of 8 banks.
//   fast axis y or z (x slabs): voxels are stored one by one (transposed), strides are free; the
//     stride of x is made = 2 mod 8 so that the transposing stores of copy_box spread over all banks.
template <int AX, int FAST>
__host__ __device__ inline bool choose_box(const BeamParams& B, const int n[3], int clo, int depth,
                                           const float span[4], Slab& out)
{
    constexpr int U = AX == 0 ? 1 : 0, V = AX == 2 ? 1 : 2;
    int lo[3], hi[3];
    lo[AX] = clo;
    hi[AX] = min(clo + depth, n[AX] - 1);
    lo[U] = max(VR_FLOOR_I(span[0] - 0.25f), 0);
    hi[U] = min(VR_FLOOR_I(span[1] + 0.25f) + 1, n[U] - 1);
    lo[V] = max(VR_FLOOR_I(span[2] - 0.25f), 0);
    hi[V] = min(VR_FLOOR_I(span[3] + 0.25f) + 1, n[V] - 1);
    // x rows are read as aligned 16-byte chunks (n[0] % 4 == 0: the widened row stays inside the cube).
    // Fast axis x: the whole chunks are stored.  x slabs: only the voxels [clo, hi] are stored, the
    // copy drops the xoff + ... elements of the first and last chunk that lie outside.
    const int x_al = lo[0] & ~3;
    const int cx = (hi[0] - x_al + 4) >> 2;
    const int xoff = FAST == 0 ? 0 : lo[0] - x_al;
    if (FAST == 0) lo[0] = x_al;
    int dim[3];
    for (int c = 0; c < 3; ++c) dim[c] = hi[c] - lo[c] + 1;
    if (FAST == 0) dim[0] = 4 * cx;
    if (dim[0] < 1 || dim[1] < 1 || dim[2] < 1) return false;
    constexpr int f = FAST, s = AX, m = 3 - f - s;
    int str[3];
    str[f] = 1;
    str[m] = B.pad_mode ? pad_to(dim[f], 16, 8) : dim[f];
    str[s] = str[m] * dim[m];
    if (FAST != 0 && B.pad_mode) str[s] = pad_to(str[s], 8, 2);
    const long long floats = (long long)str[s] * dim[s];
    if (floats * 4 > (long long)B.stage_bytes) return false;
    out.kind = 1;
    out.clo = clo;
    out.depth = depth;
    for (int c = 0; c < 3; ++c) { out.org[c] = lo[c]; out.dim[c] = dim[c]; out.str[c] = str[c]; out.of[c] = (float)lo[c]; }
    out.floats = (int)floats;
    out.lim = (B.stage_bytes >> 2) - 1 - (str[0] + str[1] + str[2]);
    out.cx = cx;
    out.xoff = xoff;
    out.interior = 1;
    for (int c = 0; c < 3; ++c)
        if (lo[c] < 1 || lo[c] + dim[c] - 1 > n[c] - 2) out.interior = 0;
    // copy loop divisors: fast axis x: e -> (chunk, row) by cx, row -> (m, s) by dim[m];
    //                     else:        e -> (chunk, rest) by cx, rest -> (f, m) by dim[f]
    const unsigned int d0 = (unsigned int)out.cx, d1 = (unsigned int)(FAST == 0 ? dim[m] : dim[f]);
    out.mg0 = magic_of(d0);
    out.mg1 = magic_of(d1);
    out.lo_f = (float)clo;
    out.hi_f = (float)(clo + depth);
    out.fsm = (float)str[m];
    out.fss = (float)str[s];
    return true;
}

__host__ __device__ inline void clear_slab(Slab& s)
{
    s.kind = 0; s.set = kBeamSets; s.clo = 0; s.depth = 0; s.floats = 0; s.lim = 0; s.cx = 1; s.xoff = 0; s.interior = 0; s.mg0 = s.mg1 = 0;
    s.lo_f = s.hi_f = 0.0f; s.fsm = s.fss = 0.0f;
    for (int c = 0; c < 3; ++c) { s.org[c] = 0; s.dim[c] = 0; s.str[c] = 0; s.of[c] = 0.0f; }
}

// The next slab of the tile's march, starting at cell `cursor` (which it advances past the slab).
// Precondition: the march is not over (cmin <= cursor <= cmax).
template <int AX, int FAST>
__host__ __device__ inline void plan_slab(const int n[3], const BeamParams& B, const TileGeom& G, int& cursor, Slab& out)
{
    clear_slab(out);
    if (G.flags) {                                         // one direct slab over the whole range
        out.kind = 2;
        out.clo = G.cmin;
        out.depth = G.cmax - G.cmin + 1;
        out.lo_f = (float)out.clo;
        out.hi_f = (float)(out.clo + out.depth);
        cursor = G.pos ? G.cmax + 1 : G.cmin - 1;
        return;
    }
    for (int s = 0; s <= kBeamSets; ++s) {
        const int D = B.depth[s < kBeamSets ? s : 0][AX];
        const int clo = G.pos ? cursor : max(cursor - D + 1, 0);
        const int depth = G.pos ? D : cursor - clo + 1;
        bool ok = false;
        if (s < kBeamSets) {
            float span[4] = {VR_INF, -VR_INF, VR_INF, -VR_INF};
            for (int q = 0; q < 4; ++q) {
                float sp[4];
                corner_span<AX>(G.co[q], G.su[q], G.sv[q], clo, depth, n, sp);
                span[0] = fminf(span[0], sp[0]); span[1] = fmaxf(span[1], sp[1]);
                span[2] = fminf(span[2], sp[2]); span[3] = fmaxf(span[3], sp[3]);
            }
            ok = choose_box<AX, FAST>(B, n, clo, depth, span, out);
        } else {                                           // no set fits the stage: this slab is sampled with global loads
            out.kind = 2;
            out.clo = clo;
            out.depth = depth;
            out.lo_f = (float)clo;
            out.hi_f = (float)(clo + depth);
            ok = true;
        }
        if (ok) {
            out.set = s;
            cursor = G.pos ? clo + depth : clo - 1;
            return;
        }
    }
}

// A10 at slab granularity (EA): every sample of a staged slab has its cell inside the slab's box, so if every
// min/max brick (edge 2^mm_shift cells, S9b) that holds a cell of the box has its skip byte set, every
// sample of the slab has alpha' = 0 and leaves its ray exactly as it found it: the slab is neither copied nor sampled.
template <int AX>
__host__ __device__ inline bool slab_is_empty(const FrameParams& P, const Slab& s)
{
    int b0[3], b1[3];
    for (int c = 0; c < 3; ++c) {
        const int lo = c == AX ? s.clo : s.org[c];
        int hi = c == AX ? s.clo + s.depth - 1 : s.org[c] + s.dim[c] - 2;
        hi = min(max(hi, lo), P.n[c] - 2);
        b0[c] = lo >> P.mm_shift;
        b1[c] = min(hi >> P.mm_shift, P.nb[c] - 1);
    }
    for (int z = b0[2]; z <= b1[2]; ++z)
        for (int y = b0[1]; y <= b1[1]; ++y)
            for (int x = b0[0]; x <= b1[0]; ++x)
                if (!P.skip[x + P.nb[0] * (y + P.nb[1] * z)]) return false;
    return true;
}

// plan_slab, then the empty-slab test when skipping is on
template <int AX, int FAST>
__host__ __device__ inline void plan_next(const FrameParams& P, const BeamParams& B, const TileGeom& G, int& cursor, Slab& out)
{
    plan_slab<AX, FAST>(P.n, B, G, cursor, out);
    if (B.use_skip && out.kind == 1 && slab_is_empty<AX>(P, out)) out.kind = 3;
}

// plan_slab for the axes stored in G (host callers)
inline void plan_slab_any(const int n[3], const BeamParams& B, const TileGeom& G, int& cursor, Slab& out)
{
    if (G.AX == 2)        plan_slab<2, 0>(n, B, G, cursor, out);
    else if (G.AX == 1)   plan_slab<1, 0>(n, B, G, cursor, out);
    else if (G.FAST == 2) plan_slab<0, 2>(n, B, G, cursor, out);
    else                  plan_slab<0, 1>(n, B, G, cursor, out);
}

// The prologue of raycast_beam_kernel for one tile, on the host: axes, corner rays, cell range and
// flags of the tile whose first pixel is (tile_x, tile_y).  Returns the rays that hit the cube.
inline int tile_geometry(const FrameParams& P, int tile_x, int tile_y, TileGeom& G)
{
    tile_axes(P, tile_x, tile_y, G);
    const bool pos = G.pos != 0;
    G.cmin = 0x7fffffff; G.cmax = -1; G.flags = 0; G.alive = 0;
    int hits = 0;
    for (int q = 0; q < kTileW * kTileH; ++q) {
        const int lx = q % kTileW, ly = q / kTileW;
        const int i = tile_x + lx, j = tile_y + ly;
        Ray r;
        dev::make_ray(P, i, j, r);
        if ((lx == 0 || lx == kTileW - 1) && (ly == 0 || ly == kTileH - 1)) {
            const int cq = (lx ? 1 : 0) + (ly ? 2 : 0);
            for (int c = 0; c < 3; ++c) { G.co[cq][c] = r.o[c]; G.cd[cq][c] = r.d[c]; }
            if (ray_is_bad(r.d, G.AX, pos)) G.flags |= 1;
        }
        if (i >= P.x1 || j >= P.y1) continue;
        if (!dev::clip_ray(P, r)) continue;
        int ca, cb;
        ray_cell_range(P, r, G.AX, ca, cb);
        G.cmin = ca < G.cmin ? ca : G.cmin;
        G.cmax = cb > G.cmax ? cb : G.cmax;
        if (ray_is_bad(r.d, G.AX, pos)) G.flags |= 1;
        ++hits;
    }
    G.alive = hits ? 1 : 0;
    corner_slopes(G);
    return hits;
}

// Stage size for a frame (VR_OPT_BEAM_STAGE = 0): the smallest candidate with which at least 90 % of
// the slabs probed -- five positions along the march of 3 x 3 tiles spread over the frame -- are staged
// with one of the two deepest sets (4 cells or more); failing that, with one of the three deepest;
// failing that, the largest candidate.
// Dense views (a pixel per voxel or finer) need small boxes and get the small stage, which lets more
// CTAs share an SM; sparse views (configs[2] at 1080p: two voxels per pixel) need the room.
inline int auto_stage_bytes(const FrameParams& P, BeamParams B)
{
    static const int cand[5] = {16384, 24576, 32768, 49152, 65536};
    TileGeom G[9];
    bool use[9];
    for (int q = 0; q < 9; ++q) {
        const int tx = (P.tiles_x * (2 * (q % 3) + 1)) / 6, ty = (P.tiles_y * (2 * (q / 3) + 1)) / 6;
        const int hits = tile_geometry(P, P.x0 + tx * kTileW, P.y0 + ty * kTileH, G[q]);
        use[q] = hits > 0 && !G[q].flags;
    }
    for (int pass = 0; pass < 2; ++pass)
        for (int ci = 0; ci < 5; ++ci) {
            B.stage_bytes = cand[ci];
            int total = 0, good = 0;
            for (int q = 0; q < 9; ++q) {
                if (!use[q]) continue;
                for (int k = 0; k < 5; ++k) {
                    int cursor = G[q].cmin + (int)(((long long)(G[q].cmax - G[q].cmin) * k) / 4);
                    Slab sl;
                    plan_slab_any(P.n, B, G[q], cursor, sl);
                    ++total;
                    if (sl.kind == 1 && sl.set <= pass + 1) ++good;
                }
            }
            if (total == 0) return cand[0];
            if (10 * good >= 9 * total) return cand[ci];
        }
    return cand[4];
}

__host__ __device__ inline bool march_over(const TileGeom& G, int cursor)
{
    return G.pos ? cursor > G.cmax : cursor < G.cmin;
}

}  // namespace beam
}  // namespace vr
