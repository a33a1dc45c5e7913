// vr_beam.cu -- the beam ray caster: TMA-staged voxel boxes in shared memory (sm_100a).
//
// One CTA = one 16 x 8 pixel tile = a thin beam of rays.  The beam is marched in slabs along
// the dominant axis of its central ray.  For every slab a producer warp computes the box of
// voxels the beam can touch (from the four corner rays of the tile), and one
// cp.async.bulk.tensor.3d (TMA) brings that box into a shared-memory stage while the four
// consumer warps sample the previous stage.  Each consumer thread still marches its own ray,
// sample by sample, in the order and with the exact binary32 op sequence of the numerical
// contract (S1-S9): the staging changes where the eight voxels of a sample
// are read from, never what is computed, so the image is bitwise the image of raycast_kernel.
//
// A slab whose box does not fit a stage (or a tile whose rays do not share a dominant axis)
// is sampled with plain global loads by the same code ("direct" stages).
#include "vr_beam_plan.h"

#include <cuda.h>

namespace vr {

namespace {

using namespace dev;

constexpr int kStages = 2;
constexpr int kBeamThreads = kThreads + 32;      // 4 consumer warps + 1 producer warp
constexpr float kMagic = 8388608.0f;             // 2^23: floor(p) = (p +_rd 2^23) - 2^23 for 0 <= p < 2^23

struct __align__(16) StageInfo {
    int   kind;                // 0 = end of beam, 1 = box in shared memory, 2 = direct (global loads)
    float depth;               // cells of this slab along the slab axis
    int   isy, isz;            // box strides in elements
    float o[3];                // voxel index of box element 0 (o[slab axis] = first cell of the slab)
    float fsy;                 // (float)isy
    float fsz;                 // (float)isz
    int   pad[3];
};

__device__ __forceinline__ uint32_t smem_u32(const void* p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}

__device__ __forceinline__ void mbar_init(uint64_t* b, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}

__device__ __forceinline__ void mbar_arrive(uint64_t* b)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}

__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* b, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}

__device__ __forceinline__ void mbar_wait(uint64_t* b, uint32_t parity)
{
    const uint32_t a = smem_u32(b);
    uint32_t ok;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                     "selp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(a), "r"(parity) : "memory");
    } while (!ok);
}

// A tensor map that lives in global memory and was written by the host (cudaMemcpy) must be
// acquired through the tensormap proxy by the thread that is going to use it (CUDA programming
// guide, "passing a tensor map through global memory"): system scope, 128 bytes.
__device__ __forceinline__ void tensormap_acquire(const void* map)
{
    asm volatile("fence.proxy.tensormap::generic.acquire.sys [%0], 128;" ::"l"(map) : "memory");
}

// one 3-D box of the cube -> shared memory, completion counted in bytes on `bar`
__device__ __forceinline__ void tma_load_box(uint32_t dst, const void* map, int x, int y, int z, uint64_t* bar)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes "
                 "[%0], [%1, {%2, %3, %4}], [%5];"
                 ::"r"(dst), "l"(map), "r"(x), "r"(y), "r"(z), "r"(smem_u32(bar)) : "memory");
}

struct RayState {
    float kh;                  // k + 0.5 of the next sample (exact: k < 2^22)
    float C0, C1, C2, A, m;
};

// S4-S9 over the samples of this ray that fall into the current slab.  Returns false when the
// ray is finished (left the cube, or early ray termination), true when its next sample belongs
// to a later slab.
template <int MODE, bool COUNT, int AX, bool SMEM>
__device__ __forceinline__ bool march(const FrameParams& P, const Ray& r, const float4* s_lut,
                                      const StageInfo& si, const float* s_box, RayState& S,
                                      unsigned int& n_eval)
{
    const float hx = (float)(P.n[0] - 1), hy = (float)(P.n[1] - 1), hz = (float)(P.n[2] - 1);
    const float mx = (float)(P.n[0] - 2), my = (float)(P.n[1] - 2), mz = (float)(P.n[2] - 2);
    for (;;) {
        const float t = __fmaf_rn(S.kh, P.step, r.tn);
        if (!(t < r.tf)) return false;
        // S4, S5: floor without a conversion; fminf on the float equals min on the integer
        const float px = fminf(fmaxf(__fmaf_rn(t, r.d[0], r.o[0]), 0.0f), hx);
        const float py = fminf(fmaxf(__fmaf_rn(t, r.d[1], r.o[1]), 0.0f), hy);
        const float pz = fminf(fmaxf(__fmaf_rn(t, r.d[2], r.o[2]), 0.0f), hz);
        const float fx = fminf(__fadd_rd(px, kMagic) - kMagic, mx);
        const float fy = fminf(__fadd_rd(py, kMagic) - kMagic, my);
        const float fz = fminf(__fadd_rd(pz, kMagic) - kMagic, mz);
        const float rx = fx - si.o[0], ry = fy - si.o[1], rz = fz - si.o[2];
        const float ra = AX == 0 ? rx : (AX == 1 ? ry : rz);
        if (!(ra >= 0.0f && ra < si.depth)) return true;
        const float wx = px - fx, wy = py - fy, wz = pz - fz;

        float v000, v100, v010, v110, v001, v101, v011, v111;
        if (SMEM) {
            const int idx = __float2int_rn(__fmaf_rn(rz, si.fsz, __fmaf_rn(ry, si.fsy, rx)));
            const float* q0 = s_box + idx;
            const float* q1 = q0 + si.isy;
            const float* q2 = q0 + si.isz;
            const float* q3 = q2 + si.isy;
            v000 = q0[0]; v100 = q0[1]; v010 = q1[0]; v110 = q1[1];
            v001 = q2[0]; v101 = q2[1]; v011 = q3[0]; v111 = q3[1];
        } else {
            const float* p0 = P.vol.base + ((long long)(int)fz * P.vol.sz + (long long)(int)fy * P.vol.sy + (int)fx);
            const float* p1 = p0 + P.vol.sy;
            const float* p2 = p0 + P.vol.sz;
            const float* p3 = p2 + P.vol.sy;
            v000 = __ldg(p0); v100 = __ldg(p0 + 1); v010 = __ldg(p1); v110 = __ldg(p1 + 1);
            v001 = __ldg(p2); v101 = __ldg(p2 + 1); v011 = __ldg(p3); v111 = __ldg(p3 + 1);
        }
        // S6
        const float c00 = lerp1(v000, v100, wx);
        const float c10 = lerp1(v010, v110, wx);
        const float c01 = lerp1(v001, v101, wx);
        const float c11 = lerp1(v011, v111, wx);
        const float c0 = lerp1(c00, c10, wy);
        const float c1 = lerp1(c01, c11, wy);
        const float v = lerp1(c0, c1, wz);
        if (COUNT) ++n_eval;
        S.kh += 1.0f;
        if (MODE == VR_MODE_EA) {
            const float4 cl = classify(P, s_lut, v);            // S7
            const float tr = 1.0f - S.A;                        // S8
            const float wgt = tr * cl.w;
            S.C0 = __fmaf_rn(wgt, cl.x, S.C0);
            S.C1 = __fmaf_rn(wgt, cl.y, S.C1);
            S.C2 = __fmaf_rn(wgt, cl.z, S.C2);
            S.A = S.A + wgt;
            if (S.A >= P.tau) return false;
        } else {
            S.m = fmaxf(S.m, v);                                 // S9
        }
    }
}

struct BeamShared {
    uint64_t  full[kStages], empty[kStages];
    StageInfo info[kStages];
    int cmin, cmax, flags, alive;      // cell range of the beam along the slab axis; alive = warps with live rays
};

template <int MODE, bool COUNT, int AX>
__device__ __forceinline__ void beam_body(const FrameParams& P, const BeamParams& B, BeamShared& sh,
                                          const float4* s_lut, float* s_stage, int tile_x, int tile_y, bool pos)
{
    constexpr int U = AX == 0 ? 1 : 0, V = AX == 2 ? 1 : 2;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int stage_floats = B.stage_bytes >> 2;

    Ray r;
    bool hit = false, inside = false;
    int i = 0, j = 0;
    if (warp < 4) {
        i = tile_x + (warp & 1) * 8 + (lane & 7);
        j = tile_y + (warp >> 1) * 4 + (lane >> 3);
        inside = (i < P.x1) && (j < P.y1);
        int ca = 0x7fffffff, cb = -1;
        bool bad = false;
        if (inside) {
            make_ray(P, i, j, r);
            hit = clip_ray(P, r);
        }
        if (hit) {
            beam::ray_cell_range(P, r, AX, ca, cb);
            bad = beam::ray_is_bad(r.d, AX, pos);
        }
        const int wmin = __reduce_min_sync(0xffffffffu, ca);
        const int wmax = __reduce_max_sync(0xffffffffu, cb);
        const bool any = __any_sync(0xffffffffu, hit);
        const bool anybad = __any_sync(0xffffffffu, bad);
        if (lane == 0) {
            if (any) { atomicMin(&sh.cmin, wmin); atomicMax(&sh.cmax, wmax); atomicAdd(&sh.alive, 1); }
            if (anybad) atomicOr(&sh.flags, 1);
        }
    }
    __syncthreads();

    if (warp == 4) {
        // ---- producer: one box per slab, from the four corner rays of the tile --------------------
        Ray c;
        make_ray(P, tile_x + (lane & 1) * (kTileW - 1), tile_y + ((lane >> 1) & 1) * (kTileH - 1), c);
        const bool cbad = beam::ray_is_bad(c.d, AX, pos);
        const bool all_direct = (sh.flags != 0) || __any_sync(0xffffffffu, cbad);
        const float inv_a = cbad ? 0.0f : 1.0f / c.d[AX];
        const int cmin = sh.cmin, cmax = sh.cmax;
        const bool none = sh.alive == 0;
        int cursor = pos ? cmin : cmax;              // next cell to cover
        const uint32_t stage_addr = smem_u32(s_stage);
        const void* acquired = nullptr;              // last tensor map this thread fenced
        for (uint32_t it = 0;; ++it) {
            const int buf = it % kStages;
            if (it >= kStages) mbar_wait(&sh.empty[buf], ((it / kStages) - 1) & 1);
            const bool end = none || (pos ? cursor > cmax : cursor < cmin) || (*(volatile int*)&sh.alive == 0);
            if (end) {
                if (lane == 0) { sh.info[buf].kind = 0; mbar_arrive(&sh.full[buf]); }
                break;
            }
            beam::SlabBox box;
            box.kind = 2; box.depth = 0; box.clo = 0; box.map_index = 0; box.bytes = 0;
            box.org[0] = box.org[1] = box.org[2] = 0;
            box.dim[0] = box.dim[1] = box.dim[2] = 0;
            if (all_direct) {
                cursor = pos ? cmax + 1 : cmin - 1;
            } else {
                bool staged = false;
#pragma unroll
                for (int s = 0; s < kBeamSets && !staged; ++s) {
                    const int D = B.depth[s][AX];
                    const int clo = pos ? cursor : cursor - D + 1;
                    float span[4];
                    beam::corner_span(c, inv_a, AX, clo, D, P.n, span);
#pragma unroll
                    for (int x = 1; x <= 2; x <<= 1) {
                        span[0] = fminf(span[0], __shfl_xor_sync(0xffffffffu, span[0], x));
                        span[1] = fmaxf(span[1], __shfl_xor_sync(0xffffffffu, span[1], x));
                        span[2] = fminf(span[2], __shfl_xor_sync(0xffffffffu, span[2], x));
                        span[3] = fmaxf(span[3], __shfl_xor_sync(0xffffffffu, span[3], x));
                    }
                    staged = beam::choose_box(B, s, AX, clo, span, box);
                }
                if (!staged) {                           // this slab is sampled with global loads
                    box.kind = 2;
                    box.depth = B.depth[0][AX];
                    box.clo = pos ? cursor : cursor - box.depth + 1;
                }
                cursor = pos ? box.clo + box.depth : box.clo - 1;
            }
            StageInfo si;
            si.kind = box.kind;
            si.pad[0] = si.pad[1] = si.pad[2] = 0;
            if (all_direct) {
                si.depth = 3.0e7f; si.isy = 0; si.isz = 0; si.fsy = si.fsz = 0.0f;
                si.o[0] = si.o[1] = si.o[2] = 0.0f;
            } else {
                si.depth = (float)box.depth;
                si.isy = box.dim[0]; si.isz = box.dim[0] * box.dim[1];
                si.fsy = (float)si.isy; si.fsz = (float)si.isz;
                si.o[0] = (float)box.org[0]; si.o[1] = (float)box.org[1]; si.o[2] = (float)box.org[2];
                si.o[AX] = (float)box.clo;
            }
            const void* map = (const char*)B.maps + 128 * (size_t)box.map_index;
            const uint32_t bytes = box.bytes;
            const int* org = box.org;
            if (lane == 0) {
                sh.info[buf] = si;
                if (si.kind == 1) {
                    if (map != acquired) { tensormap_acquire(map); acquired = map; }
                    mbar_arrive_expect_tx(&sh.full[buf], bytes);
                    tma_load_box(stage_addr + (uint32_t)buf * (uint32_t)B.stage_bytes, map, org[0], org[1], org[2], &sh.full[buf]);
                } else {
                    mbar_arrive(&sh.full[buf]);
                }
            }
            __syncwarp();
        }
        return;
    }

    // ---- consumers: every thread marches its own ray through the staged slabs ---------------------
    RayState S;
    S.kh = 0.5f; S.C0 = S.C1 = S.C2 = S.A = 0.0f; S.m = -CUDART_INF_F;
    unsigned int n_eval = 0;
    bool active = hit;
    bool warp_alive = __any_sync(0xffffffffu, hit);
    for (uint32_t it = 0;; ++it) {
        const int buf = it % kStages;
        mbar_wait(&sh.full[buf], (it / kStages) & 1);
        const StageInfo si = sh.info[buf];
        if (si.kind == 0) break;
        if (warp_alive) {
            if (active) {
                if (si.kind == 1) active = march<MODE, COUNT, AX, true>(P, r, s_lut, si, s_stage + buf * stage_floats, S, n_eval);
                else active = march<MODE, COUNT, AX, false>(P, r, s_lut, si, nullptr, S, n_eval);
            }
            if (!__any_sync(0xffffffffu, active)) {
                warp_alive = false;
                if (lane == 0) atomicSub(&sh.alive, 1);
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&sh.empty[buf]);
    }

    // A11: one float4 per pixel
    if (inside) {
        const size_t pix = (size_t)j * (size_t)P.W + (size_t)i;
        float4 o;
        if (MODE == VR_MODE_EA) {
            o = make_float4(S.C0, S.C1, S.C2, S.A);
            if (P.aux) P.aux[pix] = -CUDART_INF_F;
        } else {
            if (S.m == -CUDART_INF_F) {
                o = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
            } else {
                const float4 cl = classify(P, s_lut, S.m);
                o = make_float4(cl.x, cl.y, cl.z, 1.0f);
            }
            if (P.aux) P.aux[pix] = S.m;
        }
        P.out[pix] = o;
    }
    if (COUNT) {
        unsigned int n_hit = hit ? 1u : 0u;
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

template <int MODE, bool COUNT>
__global__ void __launch_bounds__(kBeamThreads)
raycast_beam_kernel(const __grid_constant__ FrameParams P, const __grid_constant__ BeamParams B)
{
    extern __shared__ __align__(128) unsigned char s_dyn[];
    __shared__ BeamShared sh;
    float4* s_lut = reinterpret_cast<float4*>(s_dyn);
    for (int q = threadIdx.x; q < 2 * P.n_lut; q += kBeamThreads) s_lut[q] = P.lut[q];
    const uint32_t dyn = smem_u32(s_dyn);
    const uint32_t stage_off = ((dyn + 2u * (uint32_t)P.n_lut * 16u + 127u) & ~127u) - dyn;
    float* s_stage = reinterpret_cast<float*>(s_dyn + stage_off);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < kStages; ++s) {
            mbar_init(&sh.full[s], 1);
            mbar_init(&sh.empty[s], 4);
        }
        sh.cmin = 0x7fffffff; sh.cmax = -1; sh.flags = 0; sh.alive = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int tile = blockIdx.x;
    const int tile_x = P.x0 + (tile % P.tiles_x) * kTileW;
    const int tile_y = P.y0 + (tile / P.tiles_x) * kTileH;
    // slab axis = dominant axis of the tile's central ray (uniform over the CTA)
    float D[3];
    beam::tile_centre_direction(P, tile_x, tile_y, D);
    const int ax = beam::dominant_axis(D);
    if (ax == 0)      beam_body<MODE, COUNT, 0>(P, B, sh, s_lut, s_stage, tile_x, tile_y, D[0] > 0.0f);
    else if (ax == 1) beam_body<MODE, COUNT, 1>(P, B, sh, s_lut, s_stage, tile_x, tile_y, D[1] > 0.0f);
    else              beam_body<MODE, COUNT, 2>(P, B, sh, s_lut, s_stage, tile_x, tile_y, D[2] > 0.0f);
}

template <int MODE, bool COUNT>
cudaError_t launch_beam(const FrameParams& P, const BeamParams& B, cudaStream_t stream)
{
    const size_t smem = (size_t)2 * P.n_lut * sizeof(float4) + 128 + (size_t)kStages * B.stage_bytes;
    auto kern = raycast_beam_kernel<MODE, COUNT>;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    const int tiles = P.tiles_x * P.tiles_y;
    if (tiles <= 0) return cudaSuccess;
    kern<<<tiles, kBeamThreads, smem, stream>>>(P, B);
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_raycast_beam(const FrameParams& P, const BeamParams& B, int mode, bool count, cudaStream_t stream)
{
    if (mode == VR_MODE_EA)
        return count ? launch_beam<VR_MODE_EA, true>(P, B, stream) : launch_beam<VR_MODE_EA, false>(P, B, stream);
    return count ? launch_beam<VR_MODE_MIP, true>(P, B, stream) : launch_beam<VR_MODE_MIP, false>(P, B, stream);
}

}  // namespace vr
