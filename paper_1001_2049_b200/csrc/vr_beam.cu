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
#include "vr_device.cuh"

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
            const float ha = (float)(P.n[AX] - 1);
            const float pa = fminf(fmaxf(__fmaf_rn(r.tn, r.d[AX], r.o[AX]), 0.0f), ha);
            const float pb = fminf(fmaxf(__fmaf_rn(r.tf, r.d[AX], r.o[AX]), 0.0f), ha);
            ca = min(__float2int_rd(fminf(pa, pb)), P.n[AX] - 2);
            cb = min(__float2int_rd(fmaxf(pa, pb)), P.n[AX] - 2);
            bad = ((r.d[AX] > 0.0f) != pos) || fabsf(r.d[AX]) < 0.25f;
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
        const bool cbad = ((c.d[AX] > 0.0f) != pos) || fabsf(c.d[AX]) < 0.25f;
        const bool all_direct = (sh.flags != 0) || __any_sync(0xffffffffu, cbad);
        const float inv_a = cbad ? 0.0f : 1.0f / c.d[AX];
        const float su = c.d[U] * inv_a, sv = c.d[V] * inv_a;
        const float hu = (float)(P.n[U] - 1), hv = (float)(P.n[V] - 1);
        const int cmin = sh.cmin, cmax = sh.cmax;
        const bool none = sh.alive == 0;
        int cursor = pos ? cmin : cmax;              // next cell to cover
        const uint32_t stage_addr = smem_u32(s_stage);
        for (uint32_t it = 0;; ++it) {
            const int buf = it % kStages;
            if (it >= kStages) mbar_wait(&sh.empty[buf], ((it / kStages) - 1) & 1);
            const bool end = none || (pos ? cursor > cmax : cursor < cmin) || (*(volatile int*)&sh.alive == 0);
            if (end) {
                if (lane == 0) { sh.info[buf].kind = 0; mbar_arrive(&sh.full[buf]); }
                break;
            }
            StageInfo si;
            si.kind = 2; si.depth = 3.0e7f; si.isy = 0; si.isz = 0;
            si.o[0] = si.o[1] = si.o[2] = 0.0f; si.fsy = si.fsz = 0.0f;
            si.pad[0] = si.pad[1] = si.pad[2] = 0;
            const void* map = nullptr;
            int org[3] = {0, 0, 0};
            uint32_t bytes = 0;
            if (all_direct) {
                cursor = pos ? cmax + 1 : cmin - 1;
            } else {
                int D = B.depth[0][AX], clo = 0;
                bool staged = false;
#pragma unroll
                for (int s = 0; s < kBeamSets && !staged; ++s) {
                    D = B.depth[s][AX];
                    clo = pos ? cursor : cursor - D + 1;
                    const float a0 = (float)max(clo, 0) - c.o[AX];
                    const float a1 = (float)min(clo + D, P.n[AX] - 1) - c.o[AX];
                    const float u0 = fminf(fmaxf(c.o[U] + a0 * su, 0.0f), hu), u1 = fminf(fmaxf(c.o[U] + a1 * su, 0.0f), hu);
                    const float v0 = fminf(fmaxf(c.o[V] + a0 * sv, 0.0f), hv), v1 = fminf(fmaxf(c.o[V] + a1 * sv, 0.0f), hv);
                    float umin = fminf(u0, u1), umax = fmaxf(u0, u1), vmin = fminf(v0, v1), vmax = fmaxf(v0, v1);
#pragma unroll
                    for (int x = 1; x <= 2; x <<= 1) {
                        umin = fminf(umin, __shfl_xor_sync(0xffffffffu, umin, x));
                        umax = fmaxf(umax, __shfl_xor_sync(0xffffffffu, umax, x));
                        vmin = fminf(vmin, __shfl_xor_sync(0xffffffffu, vmin, x));
                        vmax = fmaxf(vmax, __shfl_xor_sync(0xffffffffu, vmax, x));
                    }
                    const int lo_u = __float2int_rd(umin - 0.25f), need_u = __float2int_rd(umax + 0.25f) + 2 - lo_u;
                    const int lo_v = __float2int_rd(vmin - 0.25f), need_v = __float2int_rd(vmax + 0.25f) + 2 - lo_v;
                    const int u0l = U == 0 ? B.lx0 : B.ly0, usl = U == 0 ? B.lxs : B.lys, unl = U == 0 ? B.nlx : B.nly;
                    const int iu = max(0, (need_u - u0l + usl - 1) / usl);
                    const int iv = max(0, (need_v - B.ly0 + B.lys - 1) / B.lys);
                    const int size_u = u0l + usl * iu, size_v = B.ly0 + B.lys * iv;
                    const uint32_t nbytes = (uint32_t)size_u * (uint32_t)size_v * (uint32_t)(D + 1) * 4u;
                    if (iu < unl && iv < B.nly && nbytes <= (uint32_t)B.stage_bytes) {
                        staged = true;
                        bytes = nbytes;
                        int box[3];
                        box[AX] = D + 1; box[U] = size_u; box[V] = size_v;
                        org[AX] = clo; org[U] = lo_u; org[V] = lo_v;
                        si.kind = 1;
                        si.isy = box[0]; si.isz = box[0] * box[1];
                        si.fsy = (float)si.isy; si.fsz = (float)si.isz;
                        map = (const char*)B.maps + 128 * (size_t)(B.map_base[s][AX] + iu * B.nly + iv);
                    }
                }
                si.depth = (float)D;
                si.o[0] = (float)org[0]; si.o[1] = (float)org[1]; si.o[2] = (float)org[2];
                si.o[AX] = (float)clo;
                cursor = pos ? clo + D : clo - 1;
            }
            if (lane == 0) {
                sh.info[buf] = si;
                if (si.kind == 1) {
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
    float D[3] = {P.fwd[0], P.fwd[1], P.fwd[2]};
    if (P.projection == VR_PROJ_PERSPECTIVE) {
        const float a = ((float)(2 * tile_x + kTileW) / (float)P.W - 1.0f) * ((float)P.W / (float)P.H) * P.th;
        const float b = (1.0f - (float)(2 * tile_y + kTileH) / (float)P.H) * P.th;
#pragma unroll
        for (int c = 0; c < 3; ++c) D[c] = P.fwd[c] + a * P.right[c] + b * P.up[c];
    }
    const float m0 = fabsf(D[0]), m1 = fabsf(D[1]), m2 = fabsf(D[2]);
    if (m0 >= m1 && m0 >= m2) beam_body<MODE, COUNT, 0>(P, B, sh, s_lut, s_stage, tile_x, tile_y, D[0] > 0.0f);
    else if (m1 >= m2)        beam_body<MODE, COUNT, 1>(P, B, sh, s_lut, s_stage, tile_x, tile_y, D[1] > 0.0f);
    else                      beam_body<MODE, COUNT, 2>(P, B, sh, s_lut, s_stage, tile_x, tile_y, D[2] > 0.0f);
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
