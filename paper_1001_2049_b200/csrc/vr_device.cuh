// vr_device.cuh -- device functions shared by the ray-casting kernels (vr_kernels.cu, vr_beam.cu):
// the per-ray and per-sample steps S1-S7 of the numerical contract.
// Every floating-point op is IEEE-754 binary32 round-to-nearest; the translation units are
// compiled with -fmad=false and every fused multiply-add is an explicit __fmaf_rn.
#pragma once

#include "vr_internal.h"

#include <math_constants.h>

#include <cmath>

// make_ray / clip_ray also run on the host (vr_beam_plan, a diagnostic that needs no GPU):
// same op sequence, correctly rounded either way (the host side is built with -ffp-contract=off)
#ifdef __CUDA_ARCH__
#define VR_FMA(a, b, c) __fmaf_rn((a), (b), (c))
#define VR_SQRT(x) __fsqrt_rn(x)
#define VR_DIV(a, b) __fdiv_rn((a), (b))
#define VR_INF CUDART_INF_F
#else
#define VR_FMA(a, b, c) fmaf((a), (b), (c))
#define VR_SQRT(x) sqrtf(x)
#define VR_DIV(a, b) ((a) / (b))
#define VR_INF INFINITY
#endif

namespace vr {
namespace dev {

struct Ray {
    float o[3], d[3], inv[3];
    float tn, tf;
};

// Which 16 x 8-pixel tile a CTA renders (VR_OPT_TILE_ORDER, FrameParams::tile_order).
//   0: row-major -- CTA b renders tile (b % tiles_x, b / tiles_x);
//   1: supertiles of 8 x 8 tiles, row-major inside a supertile and from supertile to supertile, so that the CTAs
//      resident at one time cover a compact patch of the image (neighbouring beams share voxels in L2) instead of a
//      band as wide as the frame; the grid is padded to whole supertiles and CTAs past the edge exit at once.
__host__ __device__ __forceinline__ int grid_blocks(const FrameParams& P)
{
    if (P.tile_order == 0) return P.tiles_x * P.tiles_y;
    return ((P.tiles_x + 7) >> 3) * ((P.tiles_y + 7) >> 3) * 64;
}
__host__ __device__ __forceinline__ bool tile_of_block(const FrameParams& P, int b, int& tx, int& ty)
{
    if (P.tile_order == 0) {
        tx = b % P.tiles_x;
        ty = b / P.tiles_x;
        return true;
    }
    const int nsx = (P.tiles_x + 7) >> 3;
    const int st = b >> 6, r = b & 63;
    tx = (st % nsx) * 8 + (r & 7);
    ty = (st / nsx) * 8 + (r >> 3);
    return tx < P.tiles_x && ty < P.tiles_y;
}

// min / max of floats through integer atomics (any finite value or infinity; the cell starts at +inf / -inf):
// non-negative floats order like their bit patterns as signed ints, negative ones in reverse as unsigned ints
__device__ __forceinline__ void atomic_min_float(float* addr, float v)
{
    if (v >= 0.0f) atomicMin(reinterpret_cast<int*>(addr), __float_as_int(v));
    else atomicMax(reinterpret_cast<unsigned int*>(addr), __float_as_uint(v));
}
__device__ __forceinline__ void atomic_max_float(float* addr, float v)
{
    if (v >= 0.0f) atomicMax(reinterpret_cast<int*>(addr), __float_as_int(v));
    else atomicMin(reinterpret_cast<unsigned int*>(addr), __float_as_uint(v));
}

// A11: where pixel (i, j) of the frame is stored -- the frame buffer, or the buffer of its display-wall tile (W1)
__device__ __forceinline__ float4* pixel_ptr(const FrameParams& P, int i, int j)
{
    if (P.wall_k == 0) return P.out + ((size_t)j * (size_t)P.W + (size_t)i);
    const int a = i / P.wall_w, b = j / P.wall_h;
    return P.wall_out[b * P.wall_k + a] + ((size_t)(j - b * P.wall_h) * (size_t)P.wall_w + (size_t)(i - a * P.wall_w));
}

// S1 + S2 (+ R23): pixel (i, j) -> origin and direction in index space (unit direction when the spacing is 1)
__host__ __device__ __forceinline__ void make_ray(const FrameParams& P, int i, int j, Ray& r)
{
    const float ax = (float)(2 * i + 1) / (float)P.W - 1.0f;
    const float ay = 1.0f - (float)(2 * j + 1) / (float)P.H;
    const float asp = (float)P.W / (float)P.H;
    const float sx = ax * asp;
    const float sy = ay;
    if (P.projection == VR_PROJ_PERSPECTIVE) {
        const float a = sx * P.th;
        const float b = sy * P.th;
        float D[3];
#pragma unroll
        for (int c = 0; c < 3; ++c)
            D[c] = VR_FMA(b, P.up[c], VR_FMA(a, P.right[c], P.fwd[c]));
        const float len = VR_SQRT(VR_FMA(D[2], D[2], VR_FMA(D[1], D[1], D[0] * D[0])));
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            r.d[c] = VR_DIV(D[c], len);
            r.o[c] = P.eye[c];
        }
    } else {
        const float a = sx * P.hh;
        const float b = sy * P.hh;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            r.o[c] = VR_FMA(b, P.up[c], VR_FMA(a, P.right[c], P.eye[c]));
            r.d[c] = P.fwd[c];
        }
    }
    if (P.aniso) {                // R23: world space -> index space
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            r.o[c] = r.o[c] * P.inv_sp[c];
            r.d[c] = r.d[c] * P.inv_sp[c];
        }
    }
}

// S3: slabs against [0, n-1]^3
__host__ __device__ __forceinline__ bool clip_ray(const FrameParams& P, Ray& r)
{
    float tn = 0.0f, tf = VR_INF;
    bool hit = true;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const float hi = (float)(P.n[c] - 1);
        if (r.d[c] == 0.0f) {
            r.inv[c] = 0.0f;
            if (r.o[c] < 0.0f || r.o[c] > hi) hit = false;
        } else {
            const float inv = VR_DIV(1.0f, r.d[c]);
            r.inv[c] = inv;
            const float t0 = (0.0f - r.o[c]) * inv;
            const float t1 = (hi - r.o[c]) * inv;
            tn = fmaxf(tn, fminf(t0, t1));
            tf = fminf(tf, fmaxf(t0, t1));
        }
    }
    r.tn = tn;
    r.tf = tf;
    return hit && (tn < tf);
}

// conservative k-range of the samples that can lie in the streamed brick (S10):
// the exact membership test on the integer cell index decides, this only bounds k
__device__ __forceinline__ bool brick_k_range(const FrameParams& P, const Ray& r, int& k_lo, int& k_hi)
{
    float ta = r.tn, tb = r.tf;
    bool any = true;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const float lo = (float)(P.clo[c] - 1), hi = (float)(P.chi[c] + 1);
        if (r.d[c] == 0.0f) {
            if (r.o[c] < lo || r.o[c] > hi) any = false;
        } else {
            const float t0 = (lo - r.o[c]) * r.inv[c];
            const float t1 = (hi - r.o[c]) * r.inv[c];
            ta = fmaxf(ta, fminf(t0, t1));
            tb = fminf(tb, fmaxf(t0, t1));
        }
    }
    if (!any || !(ta <= tb)) return false;
    const float a = (ta - r.tn) * P.inv_step;
    const float b = (tb - r.tn) * P.inv_step;
    k_lo = max(0, __float2int_rd(fminf(a, 1.0e9f)) - 2);
    k_hi = __float2int_ru(fminf(b, 1.0e9f)) + 2;
    return true;
}

// S4 + S5: position, cell, weights of the sample at parameter t
__device__ __forceinline__ void locate(const FrameParams& P, const Ray& r, float t,
                                       int ic[3], float w[3])
{
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        float p = __fmaf_rn(t, r.d[c], r.o[c]);
        p = fminf(fmaxf(p, 0.0f), (float)(P.n[c] - 1));
        const int i = min(__float2int_rd(p), P.n[c] - 2);
        ic[c] = i;
        w[c] = p - (float)i;
    }
}

__device__ __forceinline__ float lerp1(float a, float b, float w)
{
    return __fmaf_rn(w, b - a, a);
}

// VR_LAYOUT_TEX: the 2 x 2 texels around the corner (x, y) of layer `layer`, raw fp32 (no filtering).
// tld4 returns them counter-clockwise from the lower-left of the footprint:
// .x = (i, j+1), .y = (i+1, j+1), .z = (i+1, j), .w = (i, j)
__device__ __forceinline__ float4 gather4(cudaTextureObject_t tex, int layer, float x, float y)
{
#ifdef VR_HOSTEMU
    return emu::tld4_a2d(tex, layer, x, y);          // tests/hostemu: the instruction by its definition
#else
    float4 r;
    asm volatile("tld4.r.a2d.v4.f32.f32 {%0,%1,%2,%3}, [%4, {%5,%6,%7,%8}];"
                 : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w)
                 : "l"(tex), "r"(layer), "f"(x), "f"(y), "f"(0.0f));
    return r;
#endif
}

// VR_LAYOUT_TEX with more than one z chunk (VoxelBox): the array that holds layers `layer` and `layer` + 1 of the
// box, and `layer` made relative to it.  `layer` <= (layers of the box) - 2, or - 1 when only that layer is read.
__device__ __forceinline__ cudaTextureObject_t tex_chunk(const VoxelBox& vol, int& layer)
{
    if (vol.n_chunks <= 1) return vol.tex[0];
    // (magic 0 codes chunk_step == 1, which has no 32-bit magic number)
    const int q = vol.chunk_magic ? (int)__umulhi((unsigned int)layer, vol.chunk_magic) : layer;
    const int c = min(q, vol.n_chunks - 1);
    layer -= c * vol.chunk_step;
    return vol.tex[c];
}

// Where the kernels read voxels from (template argument TEX of the ray casters): a linear array, ONE layered CUDA array
// (the texture handle is uniform over the warp and feeds the gathers from a uniform register), or a cube cut into z
// chunks (the handle differs from lane to lane: an extra lookup per sample and a loop over the distinct handles around
// each gather, which only cubes with more than 2048 channels pay)
enum { VR_SRC_LINEAR = 0, VR_SRC_TEX = 1, VR_SRC_TEX_CHUNKS = 2 };

// The eight voxels of cell `ic`: v[0..7] = V000 V100 V010 V110 V001 V101 V011 V111 (offsets dx, dy, dz)
template <int TEX>
__device__ __forceinline__ void fetch8(const VoxelBox& vol, const int ic[3], float v[8])
{
    if (TEX) {
        const float gx = (float)ic[0] + vol.gx, gy = (float)ic[1] + vol.gy;
        int layer = ic[2] - vol.org_z;
        float4 a, b;
        if (TEX == VR_SRC_TEX) {
            a = gather4(vol.tex[0], layer, gx, gy);
            b = gather4(vol.tex[0], layer + 1, gx, gy);
        } else {
            const cudaTextureObject_t tex = tex_chunk(vol, layer);
            a = gather4(tex, layer, gx, gy);
            b = gather4(tex, layer + 1, gx, gy);
        }
        v[0] = a.w; v[1] = a.z; v[2] = a.x; v[3] = a.y;
        v[4] = b.w; v[5] = b.z; v[6] = b.x; v[7] = b.y;
    } else {
        const float* p0 = vol.base + ((long long)ic[2] * vol.sz + (long long)ic[1] * vol.sy + ic[0]);
        const float* p1 = p0 + vol.sy;
        const float* p2 = p0 + vol.sz;
        const float* p3 = p2 + vol.sy;
        v[0] = __ldg(p0); v[1] = __ldg(p0 + 1);
        v[2] = __ldg(p1); v[3] = __ldg(p1 + 1);
        v[4] = __ldg(p2); v[5] = __ldg(p2 + 1);
        v[6] = __ldg(p3); v[7] = __ldg(p3 + 1);
    }
}

// S6: trilinear, x then y then z
__device__ __forceinline__ float lerp8(const float v[8], const float w[3])
{
    const float c00 = lerp1(v[0], v[1], w[0]);
    const float c10 = lerp1(v[2], v[3], w[0]);
    const float c01 = lerp1(v[4], v[5], w[0]);
    const float c11 = lerp1(v[6], v[7], w[0]);
    const float c0 = lerp1(c00, c10, w[1]);
    const float c1 = lerp1(c01, c11, w[1]);
    return lerp1(c0, c1, w[2]);
}

template <int TEX>
__device__ __forceinline__ float trilinear(const VoxelBox& vol, const int ic[3], const float w[3])
{
    float v[8];
    fetch8<TEX>(vol, ic, v);
    return lerp8(v, w);
}

// S7: value -> LUT cell q and fraction g
__device__ __forceinline__ void lut_coord(const FrameParams& P, float v, int& q, float& g)
{
    float xi = (v - P.vmin) * P.scale;
    xi = fminf(fmaxf(xi, 0.0f), (float)(P.n_lut - 1));
    q = min(__float2int_rz(xi), P.n_lut - 2);
    g = xi - (float)q;
}

__device__ __forceinline__ float4 classify(const FrameParams& P, const float4* s_lut, float v)
{
    int q;
    float g;
    lut_coord(P, v, q, g);
    const float4 b = s_lut[q];
    const float4 d = s_lut[P.n_lut + q];
    return make_float4(__fmaf_rn(g, d.x, b.x), __fmaf_rn(g, d.y, b.y), __fmaf_rn(g, d.z, b.z),
                       __fmaf_rn(g, d.w, b.w));
}

}  // namespace dev
}  // namespace vr
