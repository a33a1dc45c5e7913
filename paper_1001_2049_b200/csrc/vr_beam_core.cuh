// vr_beam_core.cuh -- the per-thread phases of the beam kernel (vr_beam.cu), host + device.
//
// A CTA of raycast_beam_kernel alternates two phases separated by __syncthreads():
//   copy_box : every thread copies its share of the slab's voxel box into the shared-memory stage,
//   march    : every thread marches its own ray through the slab, sample by sample, in the order and
//              with the exact binary32 op sequence of the numerical contract (DESIGN.md Sec. 3,
//              S4-S9); only the place the eight voxels of a sample are read from differs from
//              raycast_kernel, so the image is bitwise the same.
// Both phases are plain functions of (thread id, slab record, stage pointer).  They compile for the
// host as well: tests/beam_harness.cu runs the same code thread after thread against a host array
// and checks every index it forms, so the addressing is verified without a GPU.  Only the memory
// instructions differ per side and sit behind the VR_* macros below.
#pragma once

#include "vr_beam_plan.h"

#include <cstring>

#ifdef __CUDA_ARCH__
// floor(p) for 0 <= p < 2^23 without a conversion: the round-down add leaves floor(p) + 2^23 exactly
#define VR_FLOORF(p) (__fadd_rd((p), 8388608.0f) - 8388608.0f)
#define VR_F2I(x) __float2int_rn(x)
#define VR_F2I_RZ(x) __float2int_rz(x)
#define VR_LDG(p) __ldg(p)
#define VR_LDG4(p) __ldg(reinterpret_cast<const float4*>(p))
#define VR_UMULHI(a, b) __umulhi((a), (b))
#ifdef VR_HOSTEMU   // tests/hostemu: no PTX; the copy lands at once
#define VR_CP16(dst, src) std::memcpy((dst), (src), 16)
#else
#define VR_CP16(dst, src)                                                                                   \
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(dst)), \
                 "l"(src) : "memory")
#endif
// Blackwell's packed binary32 pairs (FFMA2 / FADD2: two IEEE operations per instruction, each rounded
// exactly like the scalar one): component-wise fma, add, and floor by the same 2^23 round-down add
#define VR_FMA2(a, b, c) __ffma2_rn((a), (b), (c))
#define VR_ADD2(a, b) __fadd2_rn((a), (b))
#define VR_FLOOR2(p) __fadd2_rn(__fadd2_rd((p), make_float2(8388608.0f, 8388608.0f)), make_float2(-8388608.0f, -8388608.0f))
#else
#define VR_FMA2(a, b, c) make_float2(fmaf((a).x, (b).x, (c).x), fmaf((a).y, (b).y, (c).y))
#define VR_ADD2(a, b) make_float2((a).x + (b).x, (a).y + (b).y)
#define VR_FLOOR2(p) make_float2(floorf((p).x), floorf((p).y))
#define VR_FLOORF(p) floorf(p)
#define VR_F2I(x) ((int)(x))
#define VR_F2I_RZ(x) ((int)(x))
#define VR_LDG(p) (*(p))
#define VR_LDG4(p) (*reinterpret_cast<const float4*>(p))
#define VR_UMULHI(a, b) ((unsigned int)(((unsigned long long)(a) * (unsigned long long)(b)) >> 32))
#define VR_CP16(dst, src) std::memcpy((dst), (src), 16)
#endif

// 1: the sample loop uses the packed pair operations where two independent operations of the contract
// line up (positions, floors, weights, the lerps); 0: one scalar instruction per operation.  Same values.
#ifndef VR_BEAM_PACKED
#define VR_BEAM_PACKED 1
#endif

// hooks of the host harness: every stage index formed by march / copy_box, every global element read
#ifndef VR_BEAM_TRACE_READ
#define VR_BEAM_TRACE_READ(idx, lim)
#endif
#ifndef VR_BEAM_TRACE_WRITE
#define VR_BEAM_TRACE_WRITE(idx, count)
#endif
#ifndef VR_BEAM_TRACE_GLOBAL
#define VR_BEAM_TRACE_GLOBAL(x, y, z, count)
#endif
#ifndef VR_BEAM_TRACE_LUT
#define VR_BEAM_TRACE_LUT(q)
#endif

namespace vr {
namespace beam {

struct RayState {
    float kh;                  // k + 0.5 of the next sample (exact: k < 2^22)
    float C0, C1, C2, A, m;
};

__host__ __device__ __forceinline__ float2 neg2(float2 a) { return make_float2(-a.x, -a.y); }

// S7: same op sequence as dev::classify
__host__ __device__ __forceinline__ float4 classify_hd(const FrameParams& P, const float4* lut, float v)
{
    float xi = (v - P.vmin) * P.scale;
    xi = fminf(fmaxf(xi, 0.0f), (float)(P.n_lut - 1));
    const int q = min(VR_F2I_RZ(xi), P.n_lut - 2);
    const float g = xi - (float)q;
    const float4 b = lut[q];
    const float4 d = lut[P.n_lut + q];
    return make_float4(VR_FMA(g, d.x, b.x), VR_FMA(g, d.y, b.y), VR_FMA(g, d.z, b.z), VR_FMA(g, d.w, b.w));
}

// S7 + S8 for one interpolated value v.  Returns true when the ray terminates (A >= tau).
//   zbits (or null): LUT cells whose two alpha' entries are 0 -- the sample changes nothing (lut_zero_bits);
//   GREY: `lut` is the table of lut_grey_table, only C0 is accumulated (the caller copies it to C1, C2).
template <bool GREY>
__host__ __device__ __forceinline__ bool ea_step(const FrameParams& P, const float4* lut, const unsigned int* zbits,
                                                 float v, RayState& S)
{
    float xi = (v - P.vmin) * P.scale;
    xi = fminf(fmaxf(xi, 0.0f), (float)(P.n_lut - 1));
    const int q = min(VR_F2I_RZ(xi), P.n_lut - 2);
    if (zbits && ((zbits[q >> 5] >> (q & 31)) & 1u)) { VR_BEAM_TRACE_LUT(-1); return false; }
    VR_BEAM_TRACE_LUT(q);
    const float g = xi - (float)q;
    const float tr = 1.0f - S.A;
#if VR_BEAM_PACKED
    // the same operations two to an instruction; A + wgt is written fma(wgt, 1, A): one rounding of the same sum
    const float2 gg = make_float2(g, g);
    if (GREY) {
        const float4 t = lut[q];
        const float2 ga = VR_FMA2(gg, make_float2(t.z, t.w), make_float2(t.x, t.y));        // (grey, alpha)
        const float wgt = tr * ga.y;
        const float2 ca = VR_FMA2(make_float2(wgt, wgt), make_float2(ga.x, 1.0f), make_float2(S.C0, S.A));
        S.C0 = ca.x;
        S.A = ca.y;
    } else {
        const float4 b = lut[q];
        const float4 d = lut[P.n_lut + q];
        const float2 rg = VR_FMA2(gg, make_float2(d.x, d.y), make_float2(b.x, b.y));
        const float2 ba = VR_FMA2(gg, make_float2(d.z, d.w), make_float2(b.z, b.w));
        const float wgt = tr * ba.y;
        const float2 ww = make_float2(wgt, wgt);
        const float2 c01 = VR_FMA2(ww, rg, make_float2(S.C0, S.C1));
        const float2 c2a = VR_FMA2(ww, make_float2(ba.x, 1.0f), make_float2(S.C2, S.A));
        S.C0 = c01.x; S.C1 = c01.y; S.C2 = c2a.x; S.A = c2a.y;
    }
#else
    if (GREY) {
        const float4 t = lut[q];
        const float grey = VR_FMA(g, t.z, t.x);
        const float alpha = VR_FMA(g, t.w, t.y);
        const float wgt = tr * alpha;
        S.C0 = VR_FMA(wgt, grey, S.C0);
        S.A = S.A + wgt;
    } else {
        const float4 b = lut[q];
        const float4 d = lut[P.n_lut + q];
        const float wgt = tr * VR_FMA(g, d.w, b.w);
        S.C0 = VR_FMA(wgt, VR_FMA(g, d.x, b.x), S.C0);
        S.C1 = VR_FMA(wgt, VR_FMA(g, d.y, b.y), S.C1);
        S.C2 = VR_FMA(wgt, VR_FMA(g, d.z, b.z), S.C2);
        S.A = S.A + wgt;
    }
#endif
    return S.A >= P.tau;
}

__host__ __device__ __forceinline__ float lerp_hd(float a, float b, float w)
{
    return VR_FMA(w, b - a, a);
}

// S4-S9 over the samples of this ray that fall into the slab `si`.  Returns false when the ray is
// finished (left the cube, or early ray termination), true when its next sample belongs to another
// slab.  SMEM: the eight voxels come from the staged box `s_box`, else from global memory.
// EA: lut / zbits / GREY as in ea_step.
// INTERIOR (staged slabs only): the slab's box touches no face of the cube (Slab::interior), so for every sample that
// belongs to the slab the six clamps of S4 and the three min(cell, n - 2) of S5 are identities and are left out; a
// sample whose unclamped cell along the slab axis falls outside the slab falls outside it clamped too.
template <int MODE, bool COUNT, int AX, int FAST, bool SMEM, bool GREY, bool INTERIOR>
__host__ __device__ __forceinline__ bool march(const FrameParams& P, const Ray& r, const float4* lut,
                                               const unsigned int* zbits, const Slab& si, const float* s_box,
                                               RayState& S, unsigned int& n_eval)
{
    constexpr int M = 3 - FAST - AX;
    const float hx = (float)(P.n[0] - 1), hy = (float)(P.n[1] - 1), hz = (float)(P.n[2] - 1);
    const float mx = (float)(P.n[0] - 2), my = (float)(P.n[1] - 2), mz = (float)(P.n[2] - 2);
    const float lo_f = si.lo_f, hi_f = si.hi_f;
    const float of0 = si.of[0], of1 = si.of[1], of2 = si.of[2];
    const float fsm = si.fsm, fss = si.fss;
    const int lim = si.lim;
    // offset of the +1 neighbour along each axis
    const int ox = FAST == 0 ? 1 : (M == 0 ? si.str[M] : si.str[AX]);
    const int oy = FAST == 1 ? 1 : (M == 1 ? si.str[M] : si.str[AX]);
    const int oz = FAST == 2 ? 1 : (M == 2 ? si.str[M] : si.str[AX]);
    for (;;) {
        const float t = VR_FMA(S.kh, P.step, r.tn);
        if (!(t < r.tf)) return false;
        // S4, S5: fminf on the float floor equals min on the integer cell
#if VR_BEAM_PACKED
        const float2 pxy0 = VR_FMA2(make_float2(t, t), make_float2(r.d[0], r.d[1]), make_float2(r.o[0], r.o[1]));
        const float pz0 = VR_FMA(t, r.d[2], r.o[2]);
        const float px = INTERIOR ? pxy0.x : fminf(fmaxf(pxy0.x, 0.0f), hx);
        const float py = INTERIOR ? pxy0.y : fminf(fmaxf(pxy0.y, 0.0f), hy);
        const float pz = INTERIOR ? pz0 : fminf(fmaxf(pz0, 0.0f), hz);
        const float2 pxy = make_float2(px, py);
        const float2 fl = VR_FLOOR2(pxy);
        const float fz0 = VR_FLOORF(pz);
        const float fx = INTERIOR ? fl.x : fminf(fl.x, mx);
        const float fy = INTERIOR ? fl.y : fminf(fl.y, my);
        const float fz = INTERIOR ? fz0 : fminf(fz0, mz);
#else
        const float px0 = VR_FMA(t, r.d[0], r.o[0]), py0 = VR_FMA(t, r.d[1], r.o[1]), pz0 = VR_FMA(t, r.d[2], r.o[2]);
        const float px = INTERIOR ? px0 : fminf(fmaxf(px0, 0.0f), hx);
        const float py = INTERIOR ? py0 : fminf(fmaxf(py0, 0.0f), hy);
        const float pz = INTERIOR ? pz0 : fminf(fmaxf(pz0, 0.0f), hz);
        const float fx0 = VR_FLOORF(px), fy0 = VR_FLOORF(py), fz0 = VR_FLOORF(pz);
        const float fx = INTERIOR ? fx0 : fminf(fx0, mx);
        const float fy = INTERIOR ? fy0 : fminf(fy0, my);
        const float fz = INTERIOR ? fz0 : fminf(fz0, mz);
#endif
        const float fa = AX == 0 ? fx : (AX == 1 ? fy : fz);
        if (!(fa >= lo_f && fa < hi_f)) return true;
#if VR_BEAM_PACKED
        const float2 fxy = make_float2(fx, fy);
        const float2 wxy = VR_ADD2(pxy, neg2(fxy));
        const float wx = wxy.x, wy = wxy.y, wz = pz - fz;
#else
        const float wx = px - fx, wy = py - fy, wz = pz - fz;
#endif

        float v000, v100, v010, v110, v001, v101, v011, v111;
        if (SMEM) {
#if VR_BEAM_PACKED
            const float2 rxy = VR_ADD2(fxy, make_float2(-of0, -of1));
            const float rx = rxy.x, ry = rxy.y, rz = fz - of2;
#else
            const float rx = fx - of0, ry = fy - of1, rz = fz - of2;
#endif
            const float rf = FAST == 0 ? rx : (FAST == 1 ? ry : rz);
            const float rm = M == 0 ? rx : (M == 1 ? ry : rz);
            const float rs = AX == 0 ? rx : (AX == 1 ? ry : rz);
            int idx = VR_F2I(VR_FMA(rs, fss, VR_FMA(rm, fsm, rf)));
            VR_BEAM_TRACE_READ(idx, lim);
            idx = min(max(idx, 0), lim);                 // never leaves the stage, whatever the plan
            const float* q = s_box + idx;
            v000 = q[0];       v100 = q[ox];           v010 = q[oy];      v110 = q[ox + oy];
            v001 = q[oz];      v101 = q[oz + ox];      v011 = q[oz + oy]; v111 = q[oz + oy + ox];
        } else {
            const float* p0 = P.vol.base + ((long long)(int)fz * P.vol.sz + (long long)(int)fy * P.vol.sy + (int)fx);
            const float* p1 = p0 + P.vol.sy;
            const float* p2 = p0 + P.vol.sz;
            const float* p3 = p2 + P.vol.sy;
            v000 = VR_LDG(p0); v100 = VR_LDG(p0 + 1); v010 = VR_LDG(p1); v110 = VR_LDG(p1 + 1);
            v001 = VR_LDG(p2); v101 = VR_LDG(p2 + 1); v011 = VR_LDG(p3); v111 = VR_LDG(p3 + 1);
        }
        // S6
#if VR_BEAM_PACKED
        // pairs over z: (c00, c01) and (c10, c11) by x, then (c0, c1) by y -- each lane of a pair is the
        // contract's lerp(a, b, w) = fma(w, b - a, a)
        const float2 a0 = make_float2(v000, v001), b0 = make_float2(v100, v101);
        const float2 a1 = make_float2(v010, v011), b1 = make_float2(v110, v111);
        const float2 wxx = make_float2(wx, wx), wyy = make_float2(wy, wy);
        const float2 c0x = VR_FMA2(wxx, VR_ADD2(b0, neg2(a0)), a0);       // (c00, c01)
        const float2 c1x = VR_FMA2(wxx, VR_ADD2(b1, neg2(a1)), a1);       // (c10, c11)
        const float2 cy = VR_FMA2(wyy, VR_ADD2(c1x, neg2(c0x)), c0x);      // (c0, c1)
        const float v = lerp_hd(cy.x, cy.y, wz);
#else
        const float c00 = lerp_hd(v000, v100, wx);
        const float c10 = lerp_hd(v010, v110, wx);
        const float c01 = lerp_hd(v001, v101, wx);
        const float c11 = lerp_hd(v011, v111, wx);
        const float c0 = lerp_hd(c00, c10, wy);
        const float c1 = lerp_hd(c01, c11, wy);
        const float v = lerp_hd(c0, c1, wz);
#endif
        if (COUNT) ++n_eval;
        S.kh += 1.0f;
        if (MODE == VR_MODE_EA) {
            if (ea_step<GREY>(P, lut, zbits, v, S)) return false;   // S7, S8
        } else {
            S.m = fmaxf(S.m, v);                                  // S9
        }
    }
}

// An empty slab (Slab::kind 3): the ray steps over its samples without evaluating them -- only the cell along the
// slab axis is formed, to find the first sample that belongs to another slab.  Same return value as march().
template <int AX>
__host__ __device__ __forceinline__ bool march_empty(const FrameParams& P, const Ray& r, const Slab& si, RayState& S)
{
    const float ha = (float)(P.n[AX] - 1), ma = (float)(P.n[AX] - 2);
    const float da = r.d[AX], oa = r.o[AX];
    const float lo_f = si.lo_f, hi_f = si.hi_f;
    for (;;) {
        const float t = VR_FMA(S.kh, P.step, r.tn);
        if (!(t < r.tf)) return false;
        const float pa = fminf(fmaxf(VR_FMA(t, da, oa), 0.0f), ha);
        const float fa = fminf(VR_FLOORF(pa), ma);
        if (!(fa >= lo_f && fa < hi_f)) return true;
        S.kh += 1.0f;
    }
}

// e / d with the magic number of d (magic_of in vr_beam_plan.h; 0 codes d == 1)
__host__ __device__ __forceinline__ unsigned int div_magic(unsigned int e, unsigned int mg)
{
    return mg ? VR_UMULHI(e, mg) : e;
}

// One thread's share of the copy of the slab's box into the stage.
//   FAST == 0: an x row of the box is cx 16-byte chunks; chunk e of the box -> (chunk of row, row),
//     row -> (index along the middle axis, index along the slab axis); one cp.async each.
//   FAST != 0 (x is the slab axis): chunk e -> (chunk of the x row, rest), rest -> (index along the
//     fast axis, index along the middle axis); one 16-byte load, up to four transposing 4-byte stores
//     (the elements of the aligned chunks that lie outside the slab's x range are dropped).
// Consecutive threads take consecutive chunks: global reads are coalesced 16-byte pieces, and the
// shared-memory writes of a warp fall into different banks (strides from choose_box).
template <int AX, int FAST>
__host__ __device__ __forceinline__ void copy_box(const VoxelBox& vol, const Slab& si, float* s_stage, int tid,
                                                  int nthreads)
{
    constexpr int f = FAST, s = AX, m = 3 - f - s;
    const unsigned int cx = (unsigned int)si.cx;
    const unsigned int mg0 = si.mg0, mg1 = si.mg1;
    if (FAST == 0) {
        const unsigned int dm = (unsigned int)si.dim[m];
        const unsigned int total = cx * dm * (unsigned int)si.dim[s];
        const int sm = si.str[m], ss = si.str[s];
        for (unsigned int e = (unsigned int)tid; e < total; e += (unsigned int)nthreads) {
            const unsigned int row = div_magic(e, mg0), c = e - row * cx;
            const unsigned int is = div_magic(row, mg1), im = row - is * dm;
            int v[3];
            v[0] = si.org[0] + 4 * (int)c;
            v[m] = si.org[m] + (int)im;
            v[s] = si.org[s] + (int)is;
            const float* src = vol.base + ((long long)v[2] * vol.sz + (long long)v[1] * vol.sy + v[0]);
            const int d = (int)is * ss + (int)im * sm + 4 * (int)c;
            VR_BEAM_TRACE_GLOBAL(v[0], v[1], v[2], 4);
            VR_BEAM_TRACE_WRITE(d, 4);
            VR_CP16(s_stage + d, src);
        }
    } else {
        const unsigned int df = (unsigned int)si.dim[f];
        const unsigned int total = cx * df * (unsigned int)si.dim[m];
        const int sm = si.str[m], s0 = si.str[0], xoff = si.xoff, dx = si.dim[0];
#pragma unroll 4
        for (unsigned int e = (unsigned int)tid; e < total; e += (unsigned int)nthreads) {
            const unsigned int rest = div_magic(e, mg0), c = e - rest * cx;
            const unsigned int im = div_magic(rest, mg1), jf = rest - im * df;
            int v[3];
            v[0] = si.org[0] - xoff + 4 * (int)c;
            v[f] = si.org[f] + (int)jf;
            v[m] = si.org[m] + (int)im;
            const float* src = vol.base + ((long long)v[2] * vol.sz + (long long)v[1] * vol.sy + v[0]);
            VR_BEAM_TRACE_GLOBAL(v[0], v[1], v[2], 4);
            const float4 q = VR_LDG4(src);
            const float qv[4] = {q.x, q.y, q.z, q.w};
            const int xr = 4 * (int)c - xoff;                // box x index of the chunk's first element
            const int d = xr * s0 + (int)im * sm + (int)jf;
#pragma unroll
            for (int k = 0; k < 4; ++k)
                if (xr + k >= 0 && xr + k < dx) {
                    VR_BEAM_TRACE_WRITE(d + k * s0, 1);
                    s_stage[d + k * s0] = qv[k];
                }
        }
    }
}

// The same copy for fast axis x with bulk copies: one thread copies a whole x row of the box (cx 16-byte chunks,
// contiguous in the cube and in the stage) with one cp.async.bulk; row e -> (index along the middle axis, index
// along the slab axis).  cx.bulk_row counts the bytes on the mbarrier `bar` (vr_beam_cta.cuh).
template <int AX, class CTX>
__host__ __device__ __forceinline__ void copy_rows(const VoxelBox& vol, const Slab& si, float* s_stage, int tid,
                                                   int nthreads, CTX& cx, unsigned long long* bar)
{
    constexpr int s = AX, m = 3 - s;                     // fast axis 0
    const unsigned int dm = (unsigned int)si.dim[m];
    const unsigned int rows = dm * (unsigned int)si.dim[s];
    const unsigned int mg1 = si.mg1;
    const int sm = si.str[m], ss = si.str[s];
    const unsigned int bytes = 16u * (unsigned int)si.cx;
    for (unsigned int e = (unsigned int)tid; e < rows; e += (unsigned int)nthreads) {
        const unsigned int is = div_magic(e, mg1), im = e - is * dm;
        int v[3];
        v[0] = si.org[0];
        v[m] = si.org[m] + (int)im;
        v[s] = si.org[s] + (int)is;
        const float* src = vol.base + ((long long)v[2] * vol.sz + (long long)v[1] * vol.sy + v[0]);
        const int d = (int)is * ss + (int)im * sm;
        VR_BEAM_TRACE_GLOBAL(v[0], v[1], v[2], 4 * si.cx);
        VR_BEAM_TRACE_WRITE(d, 4 * si.cx);
        cx.bulk_row(bar, s_stage + d, src, bytes);
    }
}

// A11: the pixel of a finished ray
template <int MODE>
__host__ __device__ __forceinline__ void finish_pixel(const FrameParams& P, const float4* lut, const RayState& S,
                                                      size_t pix)
{
    float4 o;
    if (MODE == VR_MODE_EA) {
        o = make_float4(S.C0, S.C1, S.C2, S.A);
        if (P.aux) P.aux[pix] = -VR_INF;
    } else {
        if (S.m == -VR_INF) {
            o = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        } else {
            const float4 cl = classify_hd(P, lut, S.m);
            o = make_float4(cl.x, cl.y, cl.z, 1.0f);
        }
        if (P.aux) P.aux[pix] = S.m;
    }
    P.out[pix] = o;
}

}  // namespace beam
}  // namespace vr
