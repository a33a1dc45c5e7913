// vr_kernels.cu -- sm_100a kernels of the spectral-cube ray caster.
//
// Per-pixel ray casting (Sec. 3.1 step 3) with the numerical
// contract of DESIGN.md Sec. 3: every floating-point op below is IEEE-754
// binary32 round-to-nearest; the file is compiled with -fmad=false so nothing
// is contracted, and every fused multiply-add is an explicit __fmaf_rn.
// No fast-math, no approximate division, no flush-to-zero.
#include "vr_device.cuh"

#include <algorithm>

namespace vr {

namespace {

using namespace dev;

// A10: is the min/max brick of edge 2^shift that owns cell `ic` skippable for this ray?  EA: its skip byte (alpha' = 0
// over its guarded value range); MIP: its guarded maximum cannot raise the running maximum m (S9b)
template <int MODE>
__device__ __forceinline__ bool brick_is_empty(const uint8_t* skip, const float2* minmax, const int nb[3], int shift,
                                               const int ic[3], float m)
{
    const int bi = (ic[0] >> shift) + nb[0] * ((ic[1] >> shift) + nb[1] * (ic[2] >> shift));
    if (MODE == VR_MODE_EA) return skip[bi] != 0;
    const float2 mm = minmax[bi];
    const float guard = fmaxf(fabsf(mm.x), fabsf(mm.y)) * 9.5367431640625e-07f;
    return (mm.y + guard) <= m;
}

// parameter at which the ray leaves that brick (its faces clipped to the cube)
__device__ __forceinline__ float brick_exit(const FrameParams& P, const Ray& r, const int ic[3], int shift)
{
    float t_exit = r.tf;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        if (r.d[c] != 0.0f) {
            const int b = ic[c] >> shift;
            const int face = (r.d[c] > 0.0f) ? min((b + 1) << shift, P.n[c] - 1) : (b << shift);
            t_exit = fminf(t_exit, ((float)face - r.o[c]) * r.inv[c]);
        }
    }
    return t_exit;
}

template <int MODE, bool SKIP, bool COUNT, bool BRICK, int TEX>
__global__ void __launch_bounds__(kThreads)
raycast_kernel(const __grid_constant__ FrameParams P)
{
    // EA classifies every sample: the LUT (values, then forward differences) lives in shared memory.  MIP classifies
    // once per pixel, at the end: it reads the two entries it needs from global memory and the CTA starts at once.
    VR_DYN_SHARED(float4, s_dyn_lut);
    const float4* s_lut = P.lut;
    if (MODE == VR_MODE_EA) {
        for (int q = threadIdx.x; q < 2 * P.n_lut; q += kThreads) s_dyn_lut[q] = P.lut[q];
        __syncthreads();
        s_lut = s_dyn_lut;
    }

    int tx, ty;
    if (!tile_of_block(P, (int)blockIdx.x, tx, ty)) return;       // padding of the supertile order (no barrier follows)
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int i = P.x0 + tx * kTileW + (warp & 1) * 8 + (lane & 7);
    const int j = P.y0 + ty * kTileH + (warp >> 1) * 4 + (lane >> 3);
    const bool inside = (i < P.x1) && (j < P.y1);

    unsigned int n_eval = 0, n_hit = 0;
    if (inside) {
        Ray r;
        make_ray(P, i, j, r);
        const bool hit = clip_ray(P, r);
        const size_t pix = (size_t)j * (size_t)P.W + (size_t)i;

        float C0 = 0.0f, C1 = 0.0f, C2 = 0.0f, A = 0.0f;
        float m = -CUDART_INF_F;
        int k = 0, k_end = 0x7fffffff;
        bool live = hit;
        if (BRICK && hit) {
            live = brick_k_range(P, r, k, k_end);
            if (live && !P.fresh) {
                const float4 R = P.out[pix];           // carried-in state (S12)
                if (MODE == VR_MODE_EA) {
                    C0 = R.x; C1 = R.y; C2 = R.z; A = R.w;
                    if (A >= P.tau) live = false;
                } else {
                    m = R.x;
                }
            }
        }
        if (COUNT && hit && !BRICK) n_hit = 1;     // streamed frames do not count rays

        if (live) {
            while (k <= k_end) {
                float t = __fmaf_rn((float)k + 0.5f, P.step, r.tn);
                if (!(t < r.tf)) break;
                int k_stop = k + 1;
                if (SKIP) {
                    // which min/max brick holds sample k, and until which k does the ray stay in it; the coarse level
                    // (if any) first: an empty coarse brick is crossed in one step
                    int ic[3];
                    float w[3];
                    locate(P, r, t, ic, w);
                    bool empty = false;
                    float t_exit = r.tf;
                    if (P.mm2_shift) {
                        empty = brick_is_empty<MODE>(P.skip2, P.minmax2, P.nb2, P.mm2_shift, ic, m);
                        if (empty) t_exit = brick_exit(P, r, ic, P.mm2_shift);
                    }
                    if (!empty) {
                        empty = brick_is_empty<MODE>(P.skip, P.minmax, P.nb, P.mm_shift, ic, m);
                        t_exit = brick_exit(P, r, ic, P.mm_shift);
                    }
                    // all samples k' < k_stop lie at least one step before the exit face
                    const float x = (t_exit - r.tn) * P.inv_step - 0.5f;
                    k_stop = max(k + 1, __float2int_rd(fminf(x, 1.0e9f)));
                    if (empty) { k = k_stop; continue; }
                }
                // samples k .. k_stop-1
                bool done = false;
                for (;;) {
                    int ic[3];
                    float w[3];
                    locate(P, r, t, ic, w);
                    bool mine = true;
                    if (BRICK) {
                        mine = ic[0] >= P.clo[0] && ic[0] < P.chi[0] && ic[1] >= P.clo[1] &&
                               ic[1] < P.chi[1] && ic[2] >= P.clo[2] && ic[2] < P.chi[2];
                    }
                    if (mine) {
                        const float v = trilinear<TEX>(P.vol, ic, w);
                        if (COUNT) ++n_eval;
                        if (MODE == VR_MODE_EA) {
                            const float4 cl = classify(P, s_lut, v);
                            const float tr = 1.0f - A;
                            const float wgt = tr * cl.w;
                            C0 = __fmaf_rn(wgt, cl.x, C0);
                            C1 = __fmaf_rn(wgt, cl.y, C1);
                            C2 = __fmaf_rn(wgt, cl.z, C2);
                            A = A + wgt;
                            if (A >= P.tau) { done = true; break; }
                        } else {
                            m = fmaxf(m, v);
                        }
                    }
                    ++k;
                    if (SKIP) { if (k >= k_stop) break; } else { if (k > k_end) break; }
                    t = __fmaf_rn((float)k + 0.5f, P.step, r.tn);
                    if (!(t < r.tf)) { done = true; break; }
                }
                if (done) break;
            }
        }

        // A11: one float4 per pixel
        if (!BRICK) {
            float4 o;
            if (MODE == VR_MODE_EA) {
                o = make_float4(C0, C1, C2, A);
                if (P.aux) P.aux[pix] = -CUDART_INF_F;
            } else {
                if (m == -CUDART_INF_F) {
                    o = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
                } else {
                    const float4 cl = classify(P, s_lut, m);
                    o = make_float4(cl.x, cl.y, cl.z, 1.0f);
                }
                if (P.aux) P.aux[pix] = m;
            }
            *pixel_ptr(P, i, j) = o;
        } else if (live || P.fresh) {
            // running image: EA (C, A); MIP (m, 0, 0, 0) until vr::launch_mip_finish
            P.out[pix] = (MODE == VR_MODE_EA) ? make_float4(C0, C1, C2, A)
                                              : make_float4(m, 0.0f, 0.0f, 0.0f);
        }
    }

    if (COUNT) {
#pragma unroll
        for (int s = 16; s > 0; s >>= 1) {
            n_eval += __shfl_xor_sync(0xffffffffu, n_eval, s);
            n_hit += __shfl_xor_sync(0xffffffffu, n_hit, s);
        }
        if (lane == 0) {
            if (n_hit) atomicAdd(&P.counters[0], (unsigned long long)n_hit);
            if (n_eval) atomicAdd(&P.counters[1], (unsigned long long)n_eval);
        }
    }
}

// A2: min / max of one brick over voxels [B*b-1, B*b+B+1] (clipped), one CTA per brick
__global__ void __launch_bounds__(256) minmax_kernel(const __grid_constant__ MinMaxParams P)
{
    const int bi = blockIdx.x;
    const int b0 = bi % P.nb[0], b1 = (bi / P.nb[0]) % P.nb[1], b2 = bi / (P.nb[0] * P.nb[1]);
    const int x0 = max(P.B * b0 - 1, 0), x1 = min(P.B * b0 + P.B + 1, P.n[0] - 1);
    const int y0 = max(P.B * b1 - 1, 0), y1 = min(P.B * b1 + P.B + 1, P.n[1] - 1);
    const int z0 = max(P.B * b2 - 1, 0), z1 = min(P.B * b2 + P.B + 1, P.n[2] - 1);
    const int ny = y1 - y0 + 1, nz = z1 - z0 + 1;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float mn = CUDART_INF_F, mx = -CUDART_INF_F;
    for (int row = warp; row < ny * nz; row += 8) {
        const int y = y0 + row % ny, z = z0 + row / ny;
        const float* p = P.vol.base + ((long long)z * P.vol.sz + (long long)y * P.vol.sy);
        for (int x = x0 + lane; x <= x1; x += 32) {
            const float v = __ldg(p + x);
            mn = fminf(mn, v);
            mx = fmaxf(mx, v);
        }
    }
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) {
        mn = fminf(mn, __shfl_xor_sync(0xffffffffu, mn, s));
        mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, s));
    }
    __shared__ float s_mn[8], s_mx[8];
    if (lane == 0) { s_mn[warp] = mn; s_mx[warp] = mx; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int q = 1; q < 8; ++q) { mn = fminf(mn, s_mn[q]); mx = fmaxf(mx, s_mx[q]); }
        P.out[bi] = make_float2(mn, mx);
    }
}

// A2, rows read as aligned 16-byte pieces (x extent a multiple of 4, base 16-byte aligned): a brick's rows start one
// voxel before a multiple of the brick edge, so each row is widened to whole float4s and the elements outside
// [x0, x1] are masked.  One warp per row (at most 18 pieces of a 66-voxel row), no division in the loop, four rows
// in flight per warp.  Same set of voxels as minmax_kernel, and min / max do not depend on the order.
__global__ void __launch_bounds__(256, 6) minmax_vec_kernel(const __grid_constant__ MinMaxParams P)
{
    const int bi = blockIdx.x;
    const int b0 = bi % P.nb[0], b1 = (bi / P.nb[0]) % P.nb[1], b2 = bi / (P.nb[0] * P.nb[1]);
    const int x0 = max(P.B * b0 - 1, 0), x1 = min(P.B * b0 + P.B + 1, P.n[0] - 1);
    const int y0 = max(P.B * b1 - 1, 0), y1 = min(P.B * b1 + P.B + 1, P.n[1] - 1);
    const int z0 = max(P.B * b2 - 1, 0), z1 = min(P.B * b2 + P.B + 1, P.n[2] - 1);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int xa = x0 & ~3;                                  // first piece of a row
    const int pieces = (x1 >> 2) - (xa >> 2) + 1;            // x1 | 3 <= n[0] - 1 because n[0] % 4 == 0
    float mn = CUDART_INF_F, mx = -CUDART_INF_F;
    for (int z = z0; z <= z1; ++z) {
        const float* pz = P.vol.base + (long long)z * P.vol.sz;
#pragma unroll 4
        for (int y = y0 + warp; y <= y1; y += 8) {
            const float* p = pz + (long long)y * P.vol.sy;
            for (int c = lane; c < pieces; c += 32) {        // more than 32 pieces only for bricks wider than 124 voxels
                const int x = xa + 4 * c;
                const float4 v = __ldg(reinterpret_cast<const float4*>(p + x));
                if (x >= x0) { mn = fminf(mn, v.x); mx = fmaxf(mx, v.x); }
                if (x + 1 >= x0 && x + 1 <= x1) { mn = fminf(mn, v.y); mx = fmaxf(mx, v.y); }
                if (x + 2 >= x0 && x + 2 <= x1) { mn = fminf(mn, v.z); mx = fmaxf(mx, v.z); }
                if (x + 3 <= x1) { mn = fminf(mn, v.w); mx = fmaxf(mx, v.w); }
            }
        }
    }
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) {
        mn = fminf(mn, __shfl_xor_sync(0xffffffffu, mn, s));
        mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, s));
    }
    __shared__ float s_mn[8], s_mx[8];
    if (lane == 0) { s_mn[warp] = mn; s_mx[warp] = mx; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int q = 1; q < 8; ++q) { mn = fminf(mn, s_mn[q]); mx = fmaxf(mx, s_mx[q]); }
        P.out[bi] = make_float2(mn, mx);
    }
}

// A2 for VR_LAYOUT_TEX: same table, voxels read as 2 x 2 gathers (components outside the
// brick's voxel range are masked, so the result equals the plain definition exactly)
__global__ void __launch_bounds__(256) minmax_tex_kernel(const __grid_constant__ MinMaxParams P)
{
    const int bi = blockIdx.x;
    const int b0 = bi % P.nb[0], b1 = (bi / P.nb[0]) % P.nb[1], b2 = bi / (P.nb[0] * P.nb[1]);
    const int x0 = max(P.B * b0 - 1, 0), x1 = min(P.B * b0 + P.B + 1, P.n[0] - 1);
    const int y0 = max(P.B * b1 - 1, 0), y1 = min(P.B * b1 + P.B + 1, P.n[1] - 1);
    const int z0 = max(P.B * b2 - 1, 0), z1 = min(P.B * b2 + P.B + 1, P.n[2] - 1);
    const int fx = (x1 - x0 + 2) >> 1, fy = (y1 - y0 + 2) >> 1, nz = z1 - z0 + 1;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float mn = CUDART_INF_F, mx = -CUDART_INF_F;
    for (int q = threadIdx.x; q < fx * fy * nz; q += 256) {
        const int a = q % fx, b = (q / fx) % fy, z = z0 + q / (fx * fy);
        const int x = x0 + 2 * a, y = y0 + 2 * b;
        int layer = z;
        const cudaTextureObject_t tex = tex_chunk(P.vol, layer);      // the last layer of the cube lies in the last chunk
        const float4 g = gather4(tex, layer, (float)x + 1.0f, (float)y + 1.0f);
        const bool xin = x + 1 <= x1, yin = y + 1 <= y1;
        mn = fminf(mn, g.w); mx = fmaxf(mx, g.w);
        if (xin) { mn = fminf(mn, g.z); mx = fmaxf(mx, g.z); }
        if (yin) { mn = fminf(mn, g.x); mx = fmaxf(mx, g.x); }
        if (xin && yin) { mn = fminf(mn, g.y); mx = fmaxf(mx, g.y); }
    }
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) {
        mn = fminf(mn, __shfl_xor_sync(0xffffffffu, mn, s));
        mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, s));
    }
    __shared__ float s_mn[8], s_mx[8];
    if (lane == 0) { s_mn[warp] = mn; s_mx[warp] = mx; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int q = 1; q < 8; ++q) { mn = fminf(mn, s_mn[q]); mx = fmaxf(mx, s_mx[q]); }
        P.out[bi] = make_float2(mn, mx);
    }
}

// A2, coarse level: min / max over the 8 x 8 x 8 fine bricks of every coarse brick
__global__ void coarse_minmax_kernel(const __grid_constant__ CoarseParams P)
{
    const int bi = blockIdx.x * blockDim.x + threadIdx.x;
    if (bi >= P.nb2[0] * P.nb2[1] * P.nb2[2]) return;
    const int c0 = bi % P.nb2[0], c1 = (bi / P.nb2[0]) % P.nb2[1], c2 = bi / (P.nb2[0] * P.nb2[1]);
    float mn = CUDART_INF_F, mx = -CUDART_INF_F;
    for (int z = 8 * c2; z < min(8 * c2 + 8, P.nb[2]); ++z)
        for (int y = 8 * c1; y < min(8 * c1 + 8, P.nb[1]); ++y)
            for (int x = 8 * c0; x < min(8 * c0 + 8, P.nb[0]); ++x) {
                const float2 f = P.fine[x + P.nb[0] * (y + P.nb[1] * z)];
                mn = fminf(mn, f.x);
                mx = fmaxf(mx, f.y);
            }
    P.coarse[bi] = make_float2(mn, mx);
}

// A3 / A10: EA skip byte of every min/max brick: 1 iff alpha' = 0 over the whole
// guarded value range of the brick (so every sample in it contributes exactly 0)
__global__ void skipbits_kernel(const __grid_constant__ SkipParams P)
{
    const int bi = blockIdx.x * blockDim.x + threadIdx.x;
    if (bi >= P.n_bricks) return;
    const float2 mm = P.minmax[bi];
    const float guard = fmaxf(fabsf(mm.x), fabsf(mm.y)) * 9.5367431640625e-07f;   // 2^-20
    const float lo = mm.x - guard, hi = mm.y + guard;
    const float top = (float)(P.n_lut - 1);
    const float xlo = fminf(fmaxf((lo - P.vmin) * P.scale, 0.0f), top);
    const float xhi = fminf(fmaxf((hi - P.vmin) * P.scale, 0.0f), top);
    const int qlo = max(min(__float2int_rz(xlo), P.n_lut - 2) - 1, 0);
    const int qhi = min(min(__float2int_rz(xhi), P.n_lut - 2) + 2, P.n_lut - 1);
    const bool empty = (P.nz_prefix[qhi + 1] - P.nz_prefix[qlo]) == 0;
    P.skip[bi] = empty ? 1 : 0;
    if (empty && P.n_skippable) atomicAdd(P.n_skippable, 1u);
}

// A2 for a streamed brick: min / max over all voxels of the brick as it sits in its slot (the brick stores exactly
// the voxels its own samples read, S10), folded into out[0] = min, out[1] = max, which start at +inf / -inf
__global__ void __launch_bounds__(256) brick_range_kernel(const float* vox, size_t n, float* out)
{
    float mn = CUDART_INF_F, mx = -CUDART_INF_F;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < n; q += (size_t)gridDim.x * blockDim.x) {
        const float v = __ldg(vox + q);
        mn = fminf(mn, v);
        mx = fmaxf(mx, v);
    }
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) {
        mn = fminf(mn, __shfl_xor_sync(0xffffffffu, mn, s));
        mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, s));
    }
    if ((threadIdx.x & 31) == 0 && mn <= mx) {
        atomic_min_float(out, mn);
        atomic_max_float(out + 1, mx);
    }
}

// Same through a slot's layered array (VR_LAYOUT_TEX): one texel per thread and step
__global__ void __launch_bounds__(256) brick_range_tex_kernel(cudaTextureObject_t tex, int dx, int dy, int dz, float* out)
{
    float mn = CUDART_INF_F, mx = -CUDART_INF_F;
    const size_t n = (size_t)dx * dy * dz;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < n; q += (size_t)gridDim.x * blockDim.x) {
        const int x = (int)(q % (size_t)dx), y = (int)((q / (size_t)dx) % (size_t)dy), z = (int)(q / ((size_t)dx * dy));
        const float v = gather4(tex, z, (float)x + 1.0f, (float)y + 1.0f).w;     // .w = texel (x, y)
        mn = fminf(mn, v);
        mx = fmaxf(mx, v);
    }
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) {
        mn = fminf(mn, __shfl_xor_sync(0xffffffffu, mn, s));
        mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, s));
    }
    if ((threadIdx.x & 31) == 0 && mn <= mx) {
        atomic_min_float(out, mn);
        atomic_max_float(out + 1, mx);
    }
}

// Saturation culling of the out-of-core path (reading C1): the smallest running value -- opacity A (EA) or maximum m
// (MIP) -- over the pixels of the brick's screen rectangle whose rays can have a sample in the brick (the same
// conservative k-range the brick's own ray segment starts from).  out starts at +inf: no such pixel leaves it there.
__global__ void __launch_bounds__(256) cull_reduce_kernel(const __grid_constant__ FrameParams P, int mode, float* out)
{
    const int i = P.x0 + blockIdx.x * 32 + (threadIdx.x & 31);
    const int j = P.y0 + blockIdx.y * 8 + (threadIdx.x >> 5);
    float val = CUDART_INF_F;
    if (i < P.x1 && j < P.y1) {
        Ray r;
        make_ray(P, i, j, r);
        int k_lo, k_hi;
        if (clip_ray(P, r) && brick_k_range(P, r, k_lo, k_hi)) {
            const float4 R = P.out[(size_t)j * (size_t)P.W + (size_t)i];
            val = mode == VR_MODE_EA ? R.w : R.x;
        }
    }
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) val = fminf(val, __shfl_xor_sync(0xffffffffu, val, s));
    if ((threadIdx.x & 31) == 0 && val < CUDART_INF_F) atomic_min_float(out, val);
}

// R17b: blanked voxels.  Every non-finite voxel (NaN, +-inf: how radio cubes mark masked channels and pixels) of the box
// [0, dx) x [0, dy) x [0, dz) at `p` (row pitch sy, slice pitch sz, in elements) becomes `value`
__global__ void __launch_bounds__(256) blank_kernel(float* p, int dx, int dy, int dz, long long sy, long long sz, float value)
{
    const size_t n = (size_t)dx * dy * dz;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < n; q += (size_t)gridDim.x * blockDim.x) {
        const int x = (int)(q % (size_t)dx), y = (int)((q / (size_t)dx) % (size_t)dy), z = (int)(q / ((size_t)dx * dy));
        float* a = p + ((long long)z * sz + (long long)y * sy + x);
        const float v = *a;
        if (!(fabsf(v) <= 3.402823466e+38f)) *a = value;        // NaN fails every comparison, inf the bound
    }
}

__global__ void fill_kernel(float* p, size_t n, float value)
{
    const size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q < n) p[q] = value;
}

__global__ void mip_init_kernel(float4* out, size_t n)
{
    const size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q < n) out[q] = make_float4(-CUDART_INF_F, 0.0f, 0.0f, 0.0f);
}

// streamed MIP: running maximum (in .x) -> LUT colour, once, after all bricks
// (reading A14 of PAPER.md:62 "reapplies the same transfer function")
__global__ void mip_finish_kernel(const __grid_constant__ FrameParams P)
{
    VR_DYN_SHARED(float4, s_lut);
    for (int q = threadIdx.x; q < 2 * P.n_lut; q += blockDim.x) s_lut[q] = P.lut[q];
    __syncthreads();
    const size_t n = (size_t)P.W * (size_t)P.H;
    for (size_t pix = (size_t)blockIdx.x * blockDim.x + threadIdx.x; pix < n;
         pix += (size_t)gridDim.x * blockDim.x) {
        const float m = P.out[pix].x;
        float4 o = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        if (m != -CUDART_INF_F) {
            const float4 cl = classify(P, s_lut, m);
            o = make_float4(cl.x, cl.y, cl.z, 1.0f);
        }
        P.out[pix] = o;
        if (P.aux) P.aux[pix] = m;
    }
}

// S13: running = running over partial (EA) / max (MIP, raw maxima in .x)
__global__ void composite_kernel(float4* running, const float4* partial, int W, int x0, int y0,
                                 int x1, int y1, int mode)
{
    const int i = x0 + blockIdx.x * blockDim.x + threadIdx.x;
    const int j = y0 + blockIdx.y * blockDim.y + threadIdx.y;
    if (i >= x1 || j >= y1) return;
    const size_t pix = (size_t)j * (size_t)W + (size_t)i;
    float4 R = running[pix];
    const float4 Pp = partial[pix];
    if (mode == VR_MODE_EA) {
        const float tr = 1.0f - R.w;
        R.x = __fmaf_rn(tr, Pp.x, R.x);
        R.y = __fmaf_rn(tr, Pp.y, R.y);
        R.z = __fmaf_rn(tr, Pp.z, R.z);
        R.w = __fmaf_rn(tr, Pp.w, R.w);
    } else {
        R.x = fmaxf(R.x, Pp.x);
    }
    running[pix] = R;
}

template <int MODE, bool SKIP, bool COUNT, bool BRICK, int TEX>
cudaError_t launch_one(const FrameParams& P, cudaStream_t stream)
{
    const size_t smem = MODE == VR_MODE_EA ? (size_t)2 * P.n_lut * sizeof(float4) : 0;      // MIP keeps the LUT in global memory
    auto kern = raycast_kernel<MODE, SKIP, COUNT, BRICK, TEX>;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    const int blocks = grid_blocks(P);
    if (blocks <= 0) return cudaSuccess;
    VR_LAUNCH(kern, blocks, kThreads, smem, stream, P);
    return cudaGetLastError();
}

template <int MODE, int TEX>
cudaError_t launch_mode(const FrameParams& P, bool skip, bool count, bool brick, cudaStream_t s)
{
    if (brick) {
        constexpr int T = TEX == VR_SRC_TEX_CHUNKS ? VR_SRC_TEX : TEX;      // (never reached with chunks: launch_raycast)
        return count ? launch_one<MODE, false, true, true, T>(P, s) : launch_one<MODE, false, false, true, T>(P, s);
    }
    if (skip) return count ? launch_one<MODE, true, true, false, TEX>(P, s) : launch_one<MODE, true, false, false, TEX>(P, s);
    return count ? launch_one<MODE, false, true, false, TEX>(P, s) : launch_one<MODE, false, false, false, TEX>(P, s);
}

}  // namespace

cudaError_t launch_raycast(const FrameParams& P, int mode, bool skip, bool count, bool brick,
                           bool tex, cudaStream_t stream)
{
    const int src = tex ? (P.vol.n_chunks > 1 ? VR_SRC_TEX_CHUNKS : VR_SRC_TEX) : VR_SRC_LINEAR;
    if (src == VR_SRC_TEX_CHUNKS) {
        if (brick) return cudaErrorInvalidValue;             // slots and parts hold one array each (vr_api.cu sees to it)
        return mode == VR_MODE_EA ? launch_mode<VR_MODE_EA, VR_SRC_TEX_CHUNKS>(P, skip, count, false, stream)
                                  : launch_mode<VR_MODE_MIP, VR_SRC_TEX_CHUNKS>(P, skip, count, false, stream);
    }
    if (src == VR_SRC_TEX)
        return mode == VR_MODE_EA ? launch_mode<VR_MODE_EA, VR_SRC_TEX>(P, skip, count, brick, stream)
                                  : launch_mode<VR_MODE_MIP, VR_SRC_TEX>(P, skip, count, brick, stream);
    return mode == VR_MODE_EA ? launch_mode<VR_MODE_EA, VR_SRC_LINEAR>(P, skip, count, brick, stream)
                              : launch_mode<VR_MODE_MIP, VR_SRC_LINEAR>(P, skip, count, brick, stream);
}

cudaError_t launch_minmax(const MinMaxParams& P, cudaStream_t stream)
{
    const int nbricks = P.nb[0] * P.nb[1] * P.nb[2];
    const bool vec = P.n[0] % 4 == 0 && P.vol.sy % 4 == 0 && P.vol.sz % 4 == 0 && ((uintptr_t)P.vol.base & 15u) == 0;
    if (P.tex) VR_LAUNCH(minmax_tex_kernel, nbricks, 256, 0, stream, P);
    else if (vec) VR_LAUNCH(minmax_vec_kernel, nbricks, 256, 0, stream, P);
    else VR_LAUNCH(minmax_kernel, nbricks, 256, 0, stream, P);
    return cudaGetLastError();
}

cudaError_t launch_coarse_minmax(const CoarseParams& P, cudaStream_t stream)
{
    const int n = P.nb2[0] * P.nb2[1] * P.nb2[2];
    VR_LAUNCH(coarse_minmax_kernel, (n + 127) / 128, 128, 0, stream, P);
    return cudaGetLastError();
}

cudaError_t launch_skipbits(const SkipParams& P, cudaStream_t stream)
{
    VR_LAUNCH(skipbits_kernel, (P.n_bricks + 127) / 128, 128, 0, stream, P);
    return cudaGetLastError();
}

cudaError_t launch_brick_range(const float* first_voxel, cudaTextureObject_t tex, bool is_tex, const int dims[3],
                               float* out, cudaStream_t stream)
{
    const size_t n = (size_t)dims[0] * dims[1] * dims[2];
    const unsigned int blocks = (unsigned int)std::min<size_t>((n + 1023) / 1024, 148 * 16);
    if (is_tex) VR_LAUNCH(brick_range_tex_kernel, blocks, 256, 0, stream, tex, dims[0], dims[1], dims[2], out);
    else VR_LAUNCH(brick_range_kernel, blocks, 256, 0, stream, first_voxel, n, out);
    return cudaGetLastError();
}

cudaError_t launch_cull_reduce(const FrameParams& P, int mode, float* out, cudaStream_t stream)
{
    if (P.x1 <= P.x0 || P.y1 <= P.y0) return cudaSuccess;
    dim3 grd((P.x1 - P.x0 + 31) / 32, (P.y1 - P.y0 + 7) / 8);
    VR_LAUNCH(cull_reduce_kernel, grd, 256, 0, stream, P, mode, out);
    return cudaGetLastError();
}

cudaError_t launch_blank(float* p, const int dims[3], long long sy, long long sz, float value, cudaStream_t stream)
{
    const size_t n = (size_t)dims[0] * dims[1] * dims[2];
    if (n == 0) return cudaSuccess;
    const unsigned int blocks = (unsigned int)std::min<size_t>((n + 1023) / 1024, 148 * 16);
    VR_LAUNCH(blank_kernel, blocks, 256, 0, stream, p, dims[0], dims[1], dims[2], sy, sz, value);
    return cudaGetLastError();
}

cudaError_t launch_mip_init(float4* out, int W, int H, cudaStream_t stream)
{
    const size_t n = (size_t)W * (size_t)H;
    VR_LAUNCH(mip_init_kernel, (unsigned)((n + 255) / 256), 256, 0, stream, out, n);
    return cudaGetLastError();
}

cudaError_t launch_fill(float* p, size_t n, float value, cudaStream_t stream)
{
    if (n == 0) return cudaSuccess;
    VR_LAUNCH(fill_kernel, (unsigned)((n + 255) / 256), 256, 0, stream, p, n, value);
    return cudaGetLastError();
}

cudaError_t launch_mip_finish(const FrameParams& P, cudaStream_t stream)
{
    const size_t smem = (size_t)2 * P.n_lut * sizeof(float4);
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(mip_finish_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    VR_LAUNCH(mip_finish_kernel, 148 * 4, 256, smem, stream, P);
    return cudaGetLastError();
}

cudaError_t launch_composite(float4* running, const float4* partial, int W, int x0, int y0,
                             int x1, int y1, int mode, cudaStream_t stream)
{
    if (x1 <= x0 || y1 <= y0) return cudaSuccess;
    dim3 blk(32, 8), grd((x1 - x0 + 31) / 32, (y1 - y0 + 7) / 8);
    VR_LAUNCH(composite_kernel, grd, blk, 0, stream, running, partial, W, x0, y0, x1, y1, mode);
    return cudaGetLastError();
}

}  // namespace vr
