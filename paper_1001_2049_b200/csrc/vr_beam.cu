// vr_beam.cu -- the beam ray caster: voxel boxes staged in shared memory (sm_100a).
//
// One CTA = one 16 x 8 pixel tile = a thin beam of rays.  The beam is marched in slabs along the
// dominant axis of its central ray.  For every slab, thread 0 bounds the voxels the beam can touch
// from the four corner rays of the tile (vr_beam_plan.h), all threads copy that box into the
// shared-memory stage (16-byte cp.async of x rows; a transposing copy when x is the slab axis),
// and then every thread marches its own ray through the slab reading its eight voxels per sample
// from shared memory (vr_beam_core.cuh): one box element is fetched from L2 once per CTA instead
// of once per sample that touches it.  The stage is single-buffered and small, so that several
// CTAs share an SM and one CTA's copy overlaps the marching of the others.
//
// A slab whose box does not fit the stage (or a tile whose rays do not share a dominant axis) is
// sampled with plain global loads by the same code ("direct" slabs).
//
// The per-thread phases are host + device functions; tests/beam_harness.cu runs them on the host
// against the oracle.  This file only adds what needs a GPU: barriers, warp votes, cp.async.
#include "vr_beam_core.cuh"

namespace vr {

namespace {

using namespace dev;

struct BeamShared {
    beam::TileGeom G;
    beam::Slab slab[2];
};

// The slab loop of one CTA.  Two barriers per slab: box copied and next slab planned | box read.
template <int MODE, bool COUNT, int AX, int FAST>
__device__ __forceinline__ void beam_loop(const FrameParams& P, const BeamParams& B, BeamShared& sh,
                                          const float4* lut, float* s_stage, const Ray& r, bool hit,
                                          beam::RayState& S, unsigned int& n_eval)
{
    const int lane = threadIdx.x & 31;
    bool active = hit;
    bool warp_alive = __any_sync(0xffffffffu, hit);
    int cursor = 0;                                      // thread 0: next cell of the slab axis to cover
    if (threadIdx.x == 0) {
        beam::corner_slopes(sh.G);
        cursor = sh.G.pos ? sh.G.cmin : sh.G.cmax;
        if (sh.G.alive == 0 || beam::march_over(sh.G, cursor)) sh.slab[0].kind = 0;
        else beam::plan_slab<AX, FAST>(P.n, B, sh.G, cursor, sh.slab[0]);
    }
    __syncthreads();
    for (int cur = 0;; cur ^= 1) {
        const beam::Slab& si = sh.slab[cur];
        const int kind = si.kind;
        if (kind == 0) break;
        if (kind == 1) {
            beam::copy_box<AX, FAST>(P.vol, si, s_stage, (int)threadIdx.x, kThreads);
            if (FAST == 0) asm volatile("cp.async.commit_group;\n\tcp.async.wait_group 0;" ::: "memory");
        }
        if (threadIdx.x == 0) {
            beam::Slab& nx = sh.slab[cur ^ 1];
            if (beam::march_over(sh.G, cursor) || *(volatile int*)&sh.G.alive == 0) nx.kind = 0;
            else beam::plan_slab<AX, FAST>(P.n, B, sh.G, cursor, nx);
        }
        __syncthreads();                                 // the box is in the stage, the next slab is planned
        if (active) {
            if (kind == 1) active = beam::march<MODE, COUNT, AX, FAST, true>(P, r, lut, si, s_stage, S, n_eval);
            else active = beam::march<MODE, COUNT, AX, FAST, false>(P, r, lut, si, nullptr, S, n_eval);
        }
        if (warp_alive && !__any_sync(0xffffffffu, active)) {
            warp_alive = false;
            if (lane == 0) atomicSub(&sh.G.alive, 1);
        }
        __syncthreads();                                 // everyone is done with the stage and with slab[cur]
    }
}

template <int MODE, bool COUNT>
__global__ void __launch_bounds__(kThreads)
raycast_beam_kernel(const __grid_constant__ FrameParams P, const __grid_constant__ BeamParams B)
{
    extern __shared__ __align__(16) unsigned char s_dyn[];
    __shared__ BeamShared sh;
    // EA classifies every sample: LUT (values, then forward differences) in shared memory ahead of the
    // stage.  MIP classifies once per pixel: it reads the LUT from global memory and keeps the room.
    const float4* lut = P.lut;
    float* s_stage = reinterpret_cast<float*>(s_dyn);
    if (MODE == VR_MODE_EA) {
        float4* s_lut = reinterpret_cast<float4*>(s_dyn);
        for (int q = threadIdx.x; q < 2 * P.n_lut; q += kThreads) s_lut[q] = P.lut[q];
        lut = s_lut;
        s_stage = reinterpret_cast<float*>(s_lut + 2 * P.n_lut);
    }
    if (threadIdx.x == 0) {
        sh.G.cmin = 0x7fffffff; sh.G.cmax = -1; sh.G.flags = 0; sh.G.alive = 0;
    }
    __syncthreads();

    const int tile = blockIdx.x;
    const int tile_x = P.x0 + (tile % P.tiles_x) * kTileW;
    const int tile_y = P.y0 + (tile / P.tiles_x) * kTileH;
    beam::TileGeom ax;                                   // AX, pos, FAST: uniform over the CTA, from P alone
    beam::tile_axes(P, tile_x, tile_y, ax);
    const int AX = ax.AX, FAST = ax.FAST;
    const bool pos = ax.pos != 0;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int lx = (warp & 1) * 8 + (lane & 7), ly = (warp >> 1) * 4 + (lane >> 3);
    const int i = tile_x + lx, j = tile_y + ly;
    const bool inside = (i < P.x1) && (j < P.y1);
    Ray r;
    make_ray(P, i, j, r);                                // also for pixels past the image edge: corner rays
    if ((lx == 0 || lx == kTileW - 1) && (ly == 0 || ly == kTileH - 1)) {
        const int q = (lx ? 1 : 0) + (ly ? 2 : 0);
#pragma unroll
        for (int c = 0; c < 3; ++c) { sh.G.co[q][c] = r.o[c]; sh.G.cd[q][c] = r.d[c]; }
        if (beam::ray_is_bad(r.d, AX, pos)) atomicOr(&sh.G.flags, 1);
    }
    if (threadIdx.x == 0) { sh.G.AX = AX; sh.G.FAST = FAST; sh.G.pos = pos ? 1 : 0; }
    bool hit = false;
    {
        int ca = 0x7fffffff, cb = -1;
        bool bad = false;
        if (inside) hit = clip_ray(P, r);
        if (hit) {
            beam::ray_cell_range(P, r, AX, ca, cb);
            bad = beam::ray_is_bad(r.d, AX, pos);
        }
        const int wmin = __reduce_min_sync(0xffffffffu, ca);
        const int wmax = __reduce_max_sync(0xffffffffu, cb);
        const bool any = __any_sync(0xffffffffu, hit);
        const bool anybad = __any_sync(0xffffffffu, bad);
        if (lane == 0) {
            if (any) { atomicMin(&sh.G.cmin, wmin); atomicMax(&sh.G.cmax, wmax); atomicAdd(&sh.G.alive, 1); }
            if (anybad) atomicOr(&sh.G.flags, 1);
        }
    }
    __syncthreads();

    beam::RayState S;
    S.kh = 0.5f; S.C0 = S.C1 = S.C2 = S.A = 0.0f; S.m = -CUDART_INF_F;
    unsigned int n_eval = 0;
    if (AX == 2)      beam_loop<MODE, COUNT, 2, 0>(P, B, sh, lut, s_stage, r, hit, S, n_eval);
    else if (AX == 1) beam_loop<MODE, COUNT, 1, 0>(P, B, sh, lut, s_stage, r, hit, S, n_eval);
    else if (FAST == 2) beam_loop<MODE, COUNT, 0, 2>(P, B, sh, lut, s_stage, r, hit, S, n_eval);
    else              beam_loop<MODE, COUNT, 0, 1>(P, B, sh, lut, s_stage, r, hit, S, n_eval);

    if (inside) beam::finish_pixel<MODE>(P, lut, S, (size_t)j * (size_t)P.W + (size_t)i);   // A11
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
cudaError_t launch_beam(const FrameParams& P, const BeamParams& B, cudaStream_t stream)
{
    const size_t smem = (MODE == VR_MODE_EA ? (size_t)2 * P.n_lut * sizeof(float4) : 0) + (size_t)B.stage_bytes;
    auto kern = raycast_beam_kernel<MODE, COUNT>;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    const int tiles = P.tiles_x * P.tiles_y;
    if (tiles <= 0) return cudaSuccess;
    kern<<<tiles, kThreads, smem, stream>>>(P, B);
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
