// vr_beam_cta.cuh -- the body of one CTA of the beam kernel, written against a small context
// interface so that the very same statements run on the device (vr_beam.cu: barriers, warp votes
// and shared-memory atomics are the hardware's) and on the host (tests/beam_harness.cu: 128 OS
// threads, pthread barriers, std::atomic -- under ThreadSanitizer, which sees every shared-memory
// access between two barriers).
//
// A context CTX provides:
//   int  tid() / block()                     thread index in the CTA, CTA index in the grid
//   void sync()                              __syncthreads()
//   bool any(bool)                           __any_sync(full mask, p): all 32 lanes of a warp call it together
//   int  warp_min(int) / warp_max(int)       __reduce_min_sync / __reduce_max_sync over the warp
//   unsigned warp_sum(unsigned)              sum over the warp (every lane gets it)
//   void smem_min / smem_max / smem_add / smem_or (int*, int)     atomics on shared memory
//   int  smem_peek(const int*)               volatile read of shared memory
//   void copies_done()                       cp.async.commit_group + wait_group 0 (host: nothing)
//   void bulk_init(bar) / bulk_expect(bar, bytes) / bulk_row(bar, dst, src, bytes) / bulk_wait(bar, parity)
//                                            an mbarrier with one arrival per phase: thread 0 arrives announcing the
//                                            bytes of a box, every cp.async.bulk row counts its bytes down, and
//                                            everybody waits for the phase to complete (BeamParams::bulk)
//   void count(unsigned long long*, unsigned long long)           atomicAdd on global memory
#pragma once

#include "vr_beam_core.cuh"

namespace vr {
namespace beam {

struct BeamShared {
    TileGeom G;
    Slab slab[3];                                        // one stage: [cur], [next]; two stages: a ring of three
    unsigned int zero_bits[32];                          // BeamParams::zero_bits, for per-lane indexing
    unsigned long long bar[2];                           // mbarriers of the bulk copies, one per stage
};

// Start the copy of slab `s` into `stage`: asynchronous when x is the fast axis (16-byte cp.async per thread, or bulk
// rows counted on `bar`), a synchronous transposing copy for x slabs.  finish_copy waits for what start_copy started.
template <int AX, int FAST, class CTX>
__host__ __device__ __forceinline__ void start_copy(const FrameParams& P, const BeamParams& B, const Slab& s, float* stage,
                                                    CTX& cx, unsigned long long* bar)
{
    if (FAST == 0 && B.bulk) {
        constexpr int M = 3 - AX;
        if (cx.tid() == 0) cx.bulk_expect(bar, 16u * (unsigned int)(s.cx * s.dim[M] * s.dim[AX]));
        copy_rows<AX>(P.vol, s, stage, cx.tid(), kThreads, cx, bar);
    } else {
        copy_box<AX, FAST>(P.vol, s, stage, cx.tid(), kThreads);
    }
}

// `parity`: bit b = the phase of bar[b] this thread waits for next (every completed box flips it)
template <int FAST, class CTX>
__host__ __device__ __forceinline__ void finish_copy(const BeamParams& B, CTX& cx, unsigned long long* bars, int b,
                                                     unsigned int& parity)
{
    if (FAST != 0) return;
    if (B.bulk) { cx.bulk_wait(bars + b, (parity >> b) & 1u); parity ^= 1u << b; }
    else cx.copies_done();
}

// The slab loop of one CTA.  Two barriers per slab: box copied and next slab planned | box read.
template <int MODE, bool COUNT, bool GREY, int AX, int FAST, class CTX>
__host__ __device__ __forceinline__ void beam_loop(const FrameParams& P, const BeamParams& B, BeamShared& sh, CTX& cx,
                                                   const float4* lut, float* s_stage, const Ray& r, bool hit,
                                                   RayState& S, unsigned int& n_eval)
{
    const unsigned int* zbits = (MODE == VR_MODE_EA && B.zero_skip) ? sh.zero_bits : nullptr;
    const int tid = cx.tid(), lane = tid & 31;
    bool active = hit;
    bool warp_alive = cx.any(hit);
    unsigned int parity = 0;                             // see finish_copy
    int cursor = 0;                                      // thread 0: next cell of the slab axis to cover
    if (tid == 0) {
        corner_slopes(sh.G);
        cursor = sh.G.pos ? sh.G.cmin : sh.G.cmax;
        if (sh.G.alive == 0 || march_over(sh.G, cursor)) sh.slab[0].kind = 0;
        else plan_next<AX, FAST>(P, B, sh.G, cursor, sh.slab[0]);
    }
    cx.sync();
    for (int cur = 0;; cur ^= 1) {
        const Slab& si = sh.slab[cur];
        const int kind = si.kind;
        if (kind == 0) break;
        if (kind == 1) start_copy<AX, FAST>(P, B, si, s_stage, cx, &sh.bar[0]);
        if (tid == 0) {                                  // planned while the asynchronous copies are in flight
            Slab& nx = sh.slab[cur ^ 1];
            if (march_over(sh.G, cursor) || cx.smem_peek(&sh.G.alive) == 0) nx.kind = 0;
            else plan_next<AX, FAST>(P, B, sh.G, cursor, nx);
        }
        if (kind == 1) finish_copy<FAST>(B, cx, sh.bar, 0, parity);
        cx.sync();                                       // the box is in the stage, the next slab is planned
        if (active) {
            if (kind == 3) active = march_empty<AX>(P, r, si, S);
            else if (kind == 1 && si.interior) active = march<MODE, COUNT, AX, FAST, true, GREY, true>(P, r, lut, zbits, si, s_stage, S, n_eval);
            else if (kind == 1) active = march<MODE, COUNT, AX, FAST, true, GREY, false>(P, r, lut, zbits, si, s_stage, S, n_eval);
            else active = march<MODE, COUNT, AX, FAST, false, GREY, false>(P, r, lut, zbits, si, nullptr, S, n_eval);
        }
        if (warp_alive && !cx.any(active)) {
            warp_alive = false;
            if (lane == 0) cx.smem_add(&sh.G.alive, -1);
        }
        cx.sync();                                       // everyone is done with the stage and with slab[cur]
    }
}

// The same march with two stages: the box of slab s + 1 is copied (asynchronously when x is the fast axis)
// while slab s is marched, so a CTA hides its own copy latency and needs one barrier per slab -- at twice
// the shared memory per CTA.  Slab records form a ring of three: [s] marched, [s + 1] being copied,
// [s + 2] being planned by thread 0.
template <int MODE, bool COUNT, bool GREY, int AX, int FAST, class CTX>
__host__ __device__ __forceinline__ void beam_loop2(const FrameParams& P, const BeamParams& B, BeamShared& sh, CTX& cx,
                                                    const float4* lut, float* s_stage, const Ray& r, bool hit,
                                                    RayState& S, unsigned int& n_eval)
{
    const unsigned int* zbits = (MODE == VR_MODE_EA && B.zero_skip) ? sh.zero_bits : nullptr;
    const int tid = cx.tid(), lane = tid & 31;
    const int stage_floats = B.stage_bytes >> 2;
    bool active = hit;
    bool warp_alive = cx.any(hit);
    int cursor = 0;                                      // thread 0: next cell of the slab axis to cover
    if (tid == 0) {
        corner_slopes(sh.G);
        cursor = sh.G.pos ? sh.G.cmin : sh.G.cmax;
        sh.slab[0].kind = 0;
        sh.slab[1].kind = 0;
        if (sh.G.alive != 0 && !march_over(sh.G, cursor)) {
            plan_next<AX, FAST>(P, B, sh.G, cursor, sh.slab[0]);
            if (!march_over(sh.G, cursor)) plan_next<AX, FAST>(P, B, sh.G, cursor, sh.slab[1]);
        }
    }
    cx.sync();
    unsigned int parity = 0;                             // see finish_copy
    if (sh.slab[0].kind == 1) {
        start_copy<AX, FAST>(P, B, sh.slab[0], s_stage, cx, &sh.bar[0]);
        finish_copy<FAST>(B, cx, sh.bar, 0, parity);
    }
    cx.sync();
    int cur = 0, nxt = 1, nn = 2, b = 0;
    for (;;) {
        const Slab& si = sh.slab[cur];
        const int kind = si.kind;
        if (kind == 0) break;
        const Slab& sn = sh.slab[nxt];
        const int nkind = sn.kind;
        float* buf = s_stage + b * stage_floats;
        if (nkind == 1) start_copy<AX, FAST>(P, B, sn, s_stage + (b ^ 1) * stage_floats, cx, &sh.bar[b ^ 1]);
        if (tid == 0) {
            Slab& nx = sh.slab[nn];
            if (nkind == 0 || march_over(sh.G, cursor) || cx.smem_peek(&sh.G.alive) == 0) nx.kind = 0;
            else plan_next<AX, FAST>(P, B, sh.G, cursor, nx);
        }
        if (active) {
            if (kind == 3) active = march_empty<AX>(P, r, si, S);
            else if (kind == 1 && si.interior) active = march<MODE, COUNT, AX, FAST, true, GREY, true>(P, r, lut, zbits, si, buf, S, n_eval);
            else if (kind == 1) active = march<MODE, COUNT, AX, FAST, true, GREY, false>(P, r, lut, zbits, si, buf, S, n_eval);
            else active = march<MODE, COUNT, AX, FAST, false, GREY, false>(P, r, lut, zbits, si, nullptr, S, n_eval);
        }
        if (warp_alive && !cx.any(active)) {
            warp_alive = false;
            if (lane == 0) cx.smem_add(&sh.G.alive, -1);
        }
        if (nkind == 1) finish_copy<FAST>(B, cx, sh.bar, b ^ 1, parity);
        cx.sync();                                       // slab s is done with, box s + 1 is in its stage, slab s + 2 is planned
        const int t = cur; cur = nxt; nxt = nn; nn = t;
        b ^= 1;
    }
}

// One CTA = one 16 x 8 pixel tile.  s_dyn: the dynamic shared memory (EA: LUT then NSTAGE stages; MIP: the stages).
// GREY (EA only): B.lut_grey is set and replaces the LUT in shared memory (half the size).
template <int MODE, bool COUNT, bool GREY, int NSTAGE, class CTX>
__host__ __device__ __forceinline__ void beam_cta(const FrameParams& P, const BeamParams& B, BeamShared& sh,
                                                  unsigned char* s_dyn, CTX& cx)
{
    const int tid = cx.tid();
    // EA classifies every sample: LUT (values, then forward differences) in shared memory ahead of the
    // stage.  MIP classifies once per pixel: it reads the LUT from global memory and keeps the room.
    const float4* lut = P.lut;
    float* s_stage = reinterpret_cast<float*>(s_dyn);
    if (MODE == VR_MODE_EA) {
        float4* s_lut = reinterpret_cast<float4*>(s_dyn);
        const int n_tab = GREY ? P.n_lut : 2 * P.n_lut;
        const float4* src = GREY ? B.lut_grey : P.lut;
        for (int q = tid; q < n_tab; q += kThreads) s_lut[q] = src[q];
        lut = s_lut;
        s_stage = reinterpret_cast<float*>(s_lut + n_tab);
        if (tid < 32) sh.zero_bits[tid] = B.zero_bits[tid];
    }
    if (tid == 0) {
        sh.G.cmin = 0x7fffffff; sh.G.cmax = -1; sh.G.flags = 0; sh.G.alive = 0;
        if (B.bulk) { cx.bulk_init(&sh.bar[0]); cx.bulk_init(&sh.bar[1]); }
    }
    cx.sync();

    const int tile = cx.block();
    const int tile_x = P.x0 + (tile % P.tiles_x) * kTileW;
    const int tile_y = P.y0 + (tile / P.tiles_x) * kTileH;
    TileGeom ax;                                         // AX, pos, FAST: uniform over the CTA, from P alone
    tile_axes(P, tile_x, tile_y, ax);
    const int AX = ax.AX, FAST = ax.FAST;
    const bool pos = ax.pos != 0;

    const int warp = tid >> 5, lane = tid & 31;
    const int lx = (warp & 1) * 8 + (lane & 7), ly = (warp >> 1) * 4 + (lane >> 3);
    const int i = tile_x + lx, j = tile_y + ly;
    const bool inside = (i < P.x1) && (j < P.y1);
    Ray r;
    dev::make_ray(P, i, j, r);                           // also for pixels past the image edge: corner rays
    if ((lx == 0 || lx == kTileW - 1) && (ly == 0 || ly == kTileH - 1)) {
        const int q = (lx ? 1 : 0) + (ly ? 2 : 0);
        for (int c = 0; c < 3; ++c) { sh.G.co[q][c] = r.o[c]; sh.G.cd[q][c] = r.d[c]; }
        if (ray_is_bad(r.d, AX, pos)) cx.smem_or(&sh.G.flags, 1);
    }
    if (tid == 0) { sh.G.AX = AX; sh.G.FAST = FAST; sh.G.pos = pos ? 1 : 0; }
    bool hit = false;
    {
        int ca = 0x7fffffff, cb = -1;
        bool bad = false;
        if (inside) hit = dev::clip_ray(P, r);
        if (hit) {
            ray_cell_range(P, r, AX, ca, cb);
            bad = ray_is_bad(r.d, AX, pos);
        }
        const int wmin = cx.warp_min(ca);
        const int wmax = cx.warp_max(cb);
        const bool any = cx.any(hit);
        const bool anybad = cx.any(bad);
        if (lane == 0) {
            if (any) { cx.smem_min(&sh.G.cmin, wmin); cx.smem_max(&sh.G.cmax, wmax); cx.smem_add(&sh.G.alive, 1); }
            if (anybad) cx.smem_or(&sh.G.flags, 1);
        }
    }
    cx.sync();

    RayState S;
    S.kh = 0.5f; S.C0 = S.C1 = S.C2 = S.A = 0.0f; S.m = -VR_INF;
    unsigned int n_eval = 0;
    if (NSTAGE == 1) {
        if (AX == 2)        beam_loop<MODE, COUNT, GREY, 2, 0>(P, B, sh, cx, lut, s_stage, r, hit, S, n_eval);
        else if (AX == 1)   beam_loop<MODE, COUNT, GREY, 1, 0>(P, B, sh, cx, lut, s_stage, r, hit, S, n_eval);
        else if (FAST == 2) beam_loop<MODE, COUNT, GREY, 0, 2>(P, B, sh, cx, lut, s_stage, r, hit, S, n_eval);
        else                beam_loop<MODE, COUNT, GREY, 0, 1>(P, B, sh, cx, lut, s_stage, r, hit, S, n_eval);
    } else {
        if (AX == 2)        beam_loop2<MODE, COUNT, GREY, 2, 0>(P, B, sh, cx, lut, s_stage, r, hit, S, n_eval);
        else if (AX == 1)   beam_loop2<MODE, COUNT, GREY, 1, 0>(P, B, sh, cx, lut, s_stage, r, hit, S, n_eval);
        else if (FAST == 2) beam_loop2<MODE, COUNT, GREY, 0, 2>(P, B, sh, cx, lut, s_stage, r, hit, S, n_eval);
        else                beam_loop2<MODE, COUNT, GREY, 0, 1>(P, B, sh, cx, lut, s_stage, r, hit, S, n_eval);
    }

    if (GREY) { S.C1 = S.C0; S.C2 = S.C0; }
    if (inside) finish_pixel<MODE>(P, lut, S, (size_t)j * (size_t)P.W + (size_t)i);   // A11
    if (COUNT) {
        const unsigned int w_hit = cx.warp_sum(hit ? 1u : 0u);
        const unsigned int w_eval = cx.warp_sum(n_eval);
        if (lane == 0) {
            if (w_hit) cx.count(&P.counters[0], (unsigned long long)w_hit);
            if (w_eval) cx.count(&P.counters[1], (unsigned long long)w_eval);
        }
    }
}

}  // namespace beam
}  // namespace vr
