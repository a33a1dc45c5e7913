// vr_pipe.cu -- variants of the direct ray caster (sm_100a): voxel loads software-pipelined (raycast_pipe_kernel), and
// the voxels of the last cell kept in registers (raycast_reuse_kernel, further down).
//
// raycast_kernel (vr_kernels.cu) has one sample in flight per thread: the loop forms a position, issues the eight
// voxel loads (two tld4 gathers on VR_LAYOUT_TEX) and stalls on them at the first lerp.  Where consecutive samples of
// a ray and neighbouring rays of a warp touch voxels nobody has fetched before -- sparse views: configs[2] at 1080p has
// 2.1 voxels between pixels and one voxel between samples, 0.25 samples per voxel -- every sample is an HBM round trip
// and the SM holds only (resident warps x 1) of them: 101 Gsamples/s on configs[2] against 199 on configs[1] with the
// same instructions (profiles/r01c_bench_lines.md), DRAM, L2 and TEX all far from busy.  This kernel keeps U samples
// per thread in flight: positions and loads of samples k .. k+U-1 are issued back to back, then the samples are
// consumed in order with exactly the op sequence of the contract (S4-S9), so the image is bitwise the same; loads
// issued for samples past an early termination are never used (their addresses are valid: positions are clamped).
// Every path but the skipping loop: resident cubes, streamed bricks, parts of a cube (VR_OPT_PIPELINE).
#include "vr_device.cuh"

namespace vr {

namespace {

using namespace dev;

// BRICK: the ray segment inside one streamed brick / one part of a cube (S10, S12, S13) -- the same carry-in, k-range,
// membership test on the integer cell index and carry-out as raycast_kernel<..., BRICK = true>; loads are issued only
// for the samples the brick owns.
template <int MODE, bool COUNT, int TEX, int U, bool BRICK>
__global__ void __launch_bounds__(kThreads)
raycast_pipe_kernel(const __grid_constant__ FrameParams P)
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
    if (!tile_of_block(P, (int)blockIdx.x, tx, ty)) return;  // padding of the supertile order (no barrier follows)
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
        int k0 = 0, k_end = 0x7fffffff;
        bool live = hit;
        if (BRICK && hit) {
            live = brick_k_range(P, r, k0, k_end);
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
            bool done = false;
            for (int k = k0; !done; k += U) {
                float v[U][8], w[U][3];
                bool valid[U], mine[U];
                // issue: positions and loads of samples k .. k + U - 1 (those inside the chord and the k-range)
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    const float t = __fmaf_rn((float)(k + u) + 0.5f, P.step, r.tn);
                    valid[u] = (t < r.tf) && (!BRICK || k + u <= k_end);
                    mine[u] = false;
                    if (valid[u]) {
                        int ic[3];
                        locate(P, r, t, ic, w[u]);
                        mine[u] = !BRICK || (ic[0] >= P.clo[0] && ic[0] < P.chi[0] && ic[1] >= P.clo[1] &&
                                             ic[1] < P.chi[1] && ic[2] >= P.clo[2] && ic[2] < P.chi[2]);
                        if (mine[u]) fetch8<TEX>(P.vol, ic, v[u]);
                    }
                }
                // consume, in order
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    if (done) break;
                    if (!valid[u]) { done = true; break; }
                    if (!mine[u]) continue;
                    const float val = lerp8(v[u], w[u]);
                    if (COUNT) ++n_eval;
                    if (MODE == VR_MODE_EA) {
                        const float4 cl = classify(P, s_lut, val);
                        const float tr = 1.0f - A;
                        const float wgt = tr * cl.w;
                        C0 = __fmaf_rn(wgt, cl.x, C0);
                        C1 = __fmaf_rn(wgt, cl.y, C1);
                        C2 = __fmaf_rn(wgt, cl.z, C2);
                        A = A + wgt;
                        if (A >= P.tau) done = true;
                    } else {
                        m = fmaxf(m, val);
                    }
                }
            }
        }
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
            P.out[pix] = (MODE == VR_MODE_EA) ? make_float4(C0, C1, C2, A) : make_float4(m, 0.0f, 0.0f, 0.0f);
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

// The direct kernel with the eight voxels of the last cell kept in registers (VR_OPT_REUSE).  Dense views with short
// steps -- configs[1] at step 0.5, configs[4] at 0.25 -- find a third to three quarters of their samples in the cell of
// the sample before; such a sample needs no load at all, and the stage that limits the direct kernel there is the
// write-back of the gathers' results (l1tex__tex_writeback_active 93 - 97 %, profiles/r01b_*).  Same voxels, same op
// sequence per sample: bitwise the same image.  Resident cubes, no skipping.
template <int MODE, bool COUNT, int TEX>
__global__ void __launch_bounds__(kThreads)
raycast_reuse_kernel(const __grid_constant__ FrameParams P)
{
    VR_DYN_SHARED(float4, s_dyn_lut);
    const float4* s_lut = P.lut;
    if (MODE == VR_MODE_EA) {
        for (int q = threadIdx.x; q < 2 * P.n_lut; q += kThreads) s_dyn_lut[q] = P.lut[q];
        __syncthreads();
        s_lut = s_dyn_lut;
    }
    int tx, ty;
    if (!tile_of_block(P, (int)blockIdx.x, tx, ty)) return;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int i = P.x0 + tx * kTileW + (warp & 1) * 8 + (lane & 7);
    const int j = P.y0 + ty * kTileH + (warp >> 1) * 4 + (lane >> 3);
    const bool inside = (i < P.x1) && (j < P.y1);

    unsigned int n_eval = 0, n_hit = 0, n_fetch = 0;
    if (inside) {
        Ray r;
        make_ray(P, i, j, r);
        const bool hit = clip_ray(P, r);
        const size_t pix = (size_t)j * (size_t)P.W + (size_t)i;
        float C0 = 0.0f, C1 = 0.0f, C2 = 0.0f, A = 0.0f;
        float m = -CUDART_INF_F;
        if (COUNT && hit) n_hit = 1;
        if (hit) {
            int pc0 = -1, pc1 = -1, pc2 = -1;           // cell whose voxels v[] holds (no cell has a negative index)
            float v[8];
            for (int k = 0;; ++k) {
                const float t = __fmaf_rn((float)k + 0.5f, P.step, r.tn);
                if (!(t < r.tf)) break;
                int ic[3];
                float w[3];
                locate(P, r, t, ic, w);
                if (ic[0] != pc0 || ic[1] != pc1 || ic[2] != pc2) {
                    fetch8<TEX>(P.vol, ic, v);
                    pc0 = ic[0]; pc1 = ic[1]; pc2 = ic[2];
                    if (COUNT) ++n_fetch;
                }
                const float val = lerp8(v, w);
                if (COUNT) ++n_eval;
                if (MODE == VR_MODE_EA) {
                    const float4 cl = classify(P, s_lut, val);
                    const float tr = 1.0f - A;
                    const float wgt = tr * cl.w;
                    C0 = __fmaf_rn(wgt, cl.x, C0);
                    C1 = __fmaf_rn(wgt, cl.y, C1);
                    C2 = __fmaf_rn(wgt, cl.z, C2);
                    A = A + wgt;
                    if (A >= P.tau) break;
                } else {
                    m = fmaxf(m, val);
                }
            }
        }
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
    }
    if (COUNT) {
#pragma unroll
        for (int s = 16; s > 0; s >>= 1) {
            n_eval += __shfl_xor_sync(0xffffffffu, n_eval, s);
            n_hit += __shfl_xor_sync(0xffffffffu, n_hit, s);
            n_fetch += __shfl_xor_sync(0xffffffffu, n_fetch, s);
        }
        if (lane == 0) {
            if (n_hit) atomicAdd(&P.counters[0], (unsigned long long)n_hit);
            if (n_eval) atomicAdd(&P.counters[1], (unsigned long long)n_eval);
            if (n_fetch) atomicAdd(&P.counters[2], (unsigned long long)n_fetch);
        }
    }
}

template <int MODE, bool COUNT, int TEX>
cudaError_t launch_reuse(const FrameParams& P, cudaStream_t stream)
{
    const size_t smem = MODE == VR_MODE_EA ? (size_t)2 * P.n_lut * sizeof(float4) : 0;
    auto kern = raycast_reuse_kernel<MODE, COUNT, TEX>;
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
cudaError_t launch_reuse_count(const FrameParams& P, bool count, cudaStream_t s)
{
    return count ? launch_reuse<MODE, true, TEX>(P, s) : launch_reuse<MODE, false, TEX>(P, s);
}

template <int MODE, bool COUNT, int TEX, int U, bool BRICK>
cudaError_t launch_pipe(const FrameParams& P, cudaStream_t stream)
{
    const size_t smem = MODE == VR_MODE_EA ? (size_t)2 * P.n_lut * sizeof(float4) : 0;      // MIP keeps the LUT in global memory
    auto kern = raycast_pipe_kernel<MODE, COUNT, TEX, U, BRICK>;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    const int blocks = grid_blocks(P);
    if (blocks <= 0) return cudaSuccess;
    VR_LAUNCH(kern, blocks, kThreads, smem, stream, P);
    return cudaGetLastError();
}

template <int MODE, int TEX, bool BRICK>
cudaError_t launch_depth(const FrameParams& P, bool count, int depth, cudaStream_t s)
{
    if (depth >= 4) return count ? launch_pipe<MODE, true, TEX, 4, BRICK>(P, s) : launch_pipe<MODE, false, TEX, 4, BRICK>(P, s);
    return count ? launch_pipe<MODE, true, TEX, 2, BRICK>(P, s) : launch_pipe<MODE, false, TEX, 2, BRICK>(P, s);
}

template <int MODE, int TEX>
cudaError_t launch_brick(const FrameParams& P, bool count, bool brick, int depth, cudaStream_t s)
{
    constexpr int T = TEX == VR_SRC_TEX_CHUNKS ? VR_SRC_TEX : TEX;          // bricks and parts hold one array each
    return brick ? launch_depth<MODE, T, true>(P, count, depth, s) : launch_depth<MODE, TEX, false>(P, count, depth, s);
}

}  // namespace

cudaError_t launch_raycast_reuse(const FrameParams& P, int mode, bool count, bool tex, cudaStream_t stream)
{
    const int src = tex ? (P.vol.n_chunks > 1 ? VR_SRC_TEX_CHUNKS : VR_SRC_TEX) : VR_SRC_LINEAR;
    if (src == VR_SRC_TEX_CHUNKS)
        return mode == VR_MODE_EA ? launch_reuse_count<VR_MODE_EA, VR_SRC_TEX_CHUNKS>(P, count, stream)
                                  : launch_reuse_count<VR_MODE_MIP, VR_SRC_TEX_CHUNKS>(P, count, stream);
    if (src == VR_SRC_TEX)
        return mode == VR_MODE_EA ? launch_reuse_count<VR_MODE_EA, VR_SRC_TEX>(P, count, stream)
                                  : launch_reuse_count<VR_MODE_MIP, VR_SRC_TEX>(P, count, stream);
    return mode == VR_MODE_EA ? launch_reuse_count<VR_MODE_EA, VR_SRC_LINEAR>(P, count, stream)
                              : launch_reuse_count<VR_MODE_MIP, VR_SRC_LINEAR>(P, count, stream);
}

cudaError_t launch_raycast_pipe(const FrameParams& P, int mode, bool count, bool brick, bool tex, int depth, cudaStream_t stream)
{
    const int src = tex ? (P.vol.n_chunks > 1 ? VR_SRC_TEX_CHUNKS : VR_SRC_TEX) : VR_SRC_LINEAR;
    if (src == VR_SRC_TEX_CHUNKS) {
        if (brick) return cudaErrorInvalidValue;
        return mode == VR_MODE_EA ? launch_brick<VR_MODE_EA, VR_SRC_TEX_CHUNKS>(P, count, false, depth, stream)
                                  : launch_brick<VR_MODE_MIP, VR_SRC_TEX_CHUNKS>(P, count, false, depth, stream);
    }
    if (src == VR_SRC_TEX)
        return mode == VR_MODE_EA ? launch_brick<VR_MODE_EA, VR_SRC_TEX>(P, count, brick, depth, stream)
                                  : launch_brick<VR_MODE_MIP, VR_SRC_TEX>(P, count, brick, depth, stream);
    return mode == VR_MODE_EA ? launch_brick<VR_MODE_EA, VR_SRC_LINEAR>(P, count, brick, depth, stream)
                              : launch_brick<VR_MODE_MIP, VR_SRC_LINEAR>(P, count, brick, depth, stream);
}

}  // namespace vr
