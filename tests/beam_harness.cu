// beam_harness.cu -- TEST INFRASTRUCTURE: runs the per-thread phases of the beam kernel on the host.
//
// The beam kernel (paper_1001_2049_b200/csrc/vr_beam.cu) is written as host + device functions
// (csrc/vr_beam_plan.h: the geometry; csrc/vr_beam_core.cuh: copy_box and march) plus a thin
// device-only glue of barriers and warp votes.  This harness is the same glue for the host: it
// walks the 128 threads of every CTA through the same phases in the same order, with the stage a
// plain host array.  tests/test_beam_harness_cpu.py compares the image with the CPU oracle
// (bitwise) and reads the counters below.  What it proves without a GPU:
//   * the slab march visits exactly the samples of the numerical contract, in order;
//   * every stage index a sample forms lies inside the stage and was written by this slab's copy
//     (the stage is refilled with NaN before every copy, so a missed voxel poisons the pixel);
//   * every 16-byte copy is aligned and stays inside the cube and the stage.
// It also models shared-memory bank conflicts (32 banks x 4 bytes: wavefronts per warp-wide load)
// and counts the bytes staged per sample.  Nothing here is part of libvr.so, and vr_render never
// runs on the host.  Build: nvcc -x cu (host code only is used), see test_beam_harness_cpu.py.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>

struct HarnessTrace {
    unsigned long long bad_read = 0, bad_write = 0, bad_global = 0, misaligned = 0;
    unsigned long long chunks16 = 0, floats_written = 0;
    std::vector<int>* seq = nullptr;       // stage indices (corner 000) of the samples of the lane being marched
    std::vector<int>* seq_q = nullptr;     // LUT cells of its classified samples (-1: skipped by the zero bits)
    int stage_floats = 0;
    int n[3] = {0, 0, 0};
};
static thread_local HarnessTrace* g_tr = nullptr;

// (host + device only so that the host + device phases may call them; the bodies are host code)
static inline __host__ __device__ void tr_read(int idx, int lim)
{
#ifndef __CUDA_ARCH__
    if (idx < 0 || idx > lim) ++g_tr->bad_read;
    if (g_tr->seq) g_tr->seq->push_back(idx);
#endif
}
static inline __host__ __device__ void tr_write(int idx, int count)
{
#ifndef __CUDA_ARCH__
    if (idx < 0 || idx + count > g_tr->stage_floats) ++g_tr->bad_write;
    if (count == 4) { if (idx & 3) ++g_tr->misaligned; ++g_tr->chunks16; }
    g_tr->floats_written += (unsigned long long)count;
#endif
}
static inline __host__ __device__ void tr_global(int x, int y, int z, int count)
{
#ifndef __CUDA_ARCH__
    if (x < 0 || y < 0 || z < 0 || x + count > g_tr->n[0] || y >= g_tr->n[1] || z >= g_tr->n[2]) ++g_tr->bad_global;
    if (x & 3) ++g_tr->misaligned;
#endif
}
static inline __host__ __device__ void tr_lut(int q)
{
#ifndef __CUDA_ARCH__
    if (g_tr && g_tr->seq_q) g_tr->seq_q->push_back(q);
#endif
}
#define VR_BEAM_TRACE_LUT(q) tr_lut(q)
#define VR_BEAM_TRACE_READ(idx, lim) tr_read((idx), (lim))
#define VR_BEAM_TRACE_WRITE(idx, count) tr_write((idx), (count))
#define VR_BEAM_TRACE_GLOBAL(x, y, z, count) tr_global((x), (y), (z), (count))

#include "../paper_1001_2049_b200/csrc/vr_beam_cta.cuh"

#include <pthread.h>

namespace {

using namespace vr;

enum { ST_RAYS_HIT, ST_SAMPLES, ST_BAD_READ, ST_BAD_WRITE, ST_BAD_GLOBAL, ST_MISALIGNED, ST_SLABS_STAGED,
       ST_SLABS_DIRECT, ST_TILES, ST_TILES_DIRECT, ST_FLOATS_STAGED, ST_CHUNKS16, ST_LDS, ST_LDS_WAVEFRONTS,
       ST_SAMPLES_STAGED, ST_BOX_FLOATS, ST_LUT_LDS, ST_LUT_WAVEFRONTS, ST_LUT_SKIPPED, ST_SAMPLES_INTERIOR, ST_SLABS_EMPTY, ST_N };

struct TileStats {
    unsigned long long v[ST_N] = {0};
};

// wavefronts of one warp-wide 4-byte shared-memory load: the largest number of distinct words any bank serves
int wavefronts(const int* addr, int n_lanes)
{
    int worst = 0;
    for (int b = 0; b < 32; ++b) {
        int words[32], nw = 0;
        for (int l = 0; l < n_lanes; ++l) {
            if ((addr[l] & 31) != b) continue;
            bool seen = false;
            for (int q = 0; q < nw; ++q) seen = seen || words[q] == addr[l];
            if (!seen) words[nw++] = addr[l];
        }
        worst = nw > worst ? nw : worst;
    }
    return worst;
}

// wavefronts of one warp-wide 16-byte shared-memory load of LUT entries q[lane] (q < 0: lane inactive): the
// warp is served a quarter (8 lanes x 16 B = 128 B) at a time; within a quarter, entries that differ but share
// a 16-byte bank group (q mod 8) serialise
int lut_wavefronts(const int* q, int n_lanes)
{
    int total = 0;
    for (int ph = 0; ph < 4; ++ph) {
        int worst = 0;
        bool any = false;
        for (int g = 0; g < 8; ++g) {
            int seen[8], ns = 0;
            for (int l = ph * 8; l < ph * 8 + 8 && l < n_lanes; ++l) {
                if (q[l] < 0) continue;
                any = true;
                if ((q[l] & 7) != g) continue;
                bool dup = false;
                for (int k = 0; k < ns; ++k) dup = dup || seen[k] == q[l];
                if (!dup) seen[ns++] = q[l];
            }
            worst = ns > worst ? ns : worst;
        }
        total += any ? worst : 0;
    }
    return total;
}

template <int MODE, bool GREY, int AX, int FAST>
void run_tile(const FrameParams& P, const BeamParams& B, const float4* lut, int tile_x, int tile_y, beam::TileGeom& G,
              float* stage, HarnessTrace& tr, TileStats& st)
{
    const unsigned int* zbits = (MODE == VR_MODE_EA && B.zero_skip) ? B.zero_bits : nullptr;
    const bool pos = G.pos != 0;
    dev::Ray rays[kThreads];
    bool hit[kThreads], inside[kThreads], active[kThreads];
    beam::RayState S[kThreads];
    unsigned int n_eval[kThreads];
    int pix_i[kThreads], pix_j[kThreads];
    G.cmin = 0x7fffffff; G.cmax = -1; G.flags = 0; G.alive = 0;
    bool warp_alive[4] = {false, false, false, false};
    for (int tid = 0; tid < kThreads; ++tid) {
        const int warp = tid >> 5, lane = tid & 31;
        const int lx = (warp & 1) * 8 + (lane & 7), ly = (warp >> 1) * 4 + (lane >> 3);
        const int i = tile_x + lx, j = tile_y + ly;
        pix_i[tid] = i; pix_j[tid] = j;
        inside[tid] = (i < P.x1) && (j < P.y1);
        dev::Ray& r = rays[tid];
        dev::make_ray(P, i, j, r);
        if ((lx == 0 || lx == kTileW - 1) && (ly == 0 || ly == kTileH - 1)) {
            const int q = (lx ? 1 : 0) + (ly ? 2 : 0);
            for (int c = 0; c < 3; ++c) { G.co[q][c] = r.o[c]; G.cd[q][c] = r.d[c]; }
            if (beam::ray_is_bad(r.d, AX, pos)) G.flags |= 1;
        }
        hit[tid] = inside[tid] && dev::clip_ray(P, r);
        if (hit[tid]) {
            int ca, cb;
            beam::ray_cell_range(P, r, AX, ca, cb);
            G.cmin = ca < G.cmin ? ca : G.cmin;
            G.cmax = cb > G.cmax ? cb : G.cmax;
            if (beam::ray_is_bad(r.d, AX, pos)) G.flags |= 1;
            warp_alive[warp] = true;
            ++st.v[ST_RAYS_HIT];
        }
        active[tid] = hit[tid];
        S[tid].kh = 0.5f; S[tid].C0 = S[tid].C1 = S[tid].C2 = S[tid].A = 0.0f;
        S[tid].m = -std::numeric_limits<float>::infinity();
        n_eval[tid] = 0;
    }
    for (int w = 0; w < 4; ++w) G.alive += warp_alive[w] ? 1 : 0;
    ++st.v[ST_TILES];
    if (G.flags && G.alive) ++st.v[ST_TILES_DIRECT];

    beam::corner_slopes(G);
    beam::Slab slab[2];
    int cursor = pos ? G.cmin : G.cmax;
    if (G.alive == 0 || beam::march_over(G, cursor)) slab[0].kind = 0;
    else beam::plan_next<AX, FAST>(P, B, G, cursor, slab[0]);
    const int stage_floats = B.stage_bytes >> 2;
    std::vector<int> seq[32], seq_q[32];
    for (int cur = 0;; cur ^= 1) {
        const beam::Slab& si = slab[cur];
        const int kind = si.kind;
        if (kind == 0) break;
        if (kind == 1) {
            for (int q = 0; q < stage_floats; ++q) stage[q] = std::numeric_limits<float>::quiet_NaN();
            for (int tid = 0; tid < kThreads; ++tid) beam::copy_box<AX, FAST>(P.vol, si, stage, tid, kThreads);
            ++st.v[ST_SLABS_STAGED];
            st.v[ST_BOX_FLOATS] += (unsigned long long)si.floats;
        } else if (kind == 3) {
            ++st.v[ST_SLABS_EMPTY];
        } else {
            ++st.v[ST_SLABS_DIRECT];
        }
        {
            beam::Slab& nx = slab[cur ^ 1];
            if (beam::march_over(G, cursor) || G.alive == 0) nx.kind = 0;
            else beam::plan_next<AX, FAST>(P, B, G, cursor, nx);
        }
        constexpr int M = 3 - FAST - AX;
        const int ox = FAST == 0 ? 1 : (M == 0 ? si.str[M] : si.str[AX]);
        const int oy = FAST == 1 ? 1 : (M == 1 ? si.str[M] : si.str[AX]);
        const int oz = FAST == 2 ? 1 : (M == 2 ? si.str[M] : si.str[AX]);
        const int off[8] = {0, ox, oy, ox + oy, oz, oz + ox, oz + oy, oz + oy + ox};
        for (int w = 0; w < 4; ++w) {
            size_t longest = 0;
            for (int lane = 0; lane < 32; ++lane) {
                const int tid = w * 32 + lane;
                seq[lane].clear();
                seq_q[lane].clear();
                if (!active[tid]) continue;
                tr.seq = &seq[lane];
                tr.seq_q = &seq_q[lane];
                const unsigned int before = n_eval[tid];
                if (kind == 3)
                    active[tid] = beam::march_empty<AX>(P, rays[tid], si, S[tid]);
                else if (kind == 1)
                    active[tid] = si.interior
                        ? beam::march<MODE, true, AX, FAST, true, GREY, true>(P, rays[tid], lut, zbits, si, stage, S[tid], n_eval[tid])
                        : beam::march<MODE, true, AX, FAST, true, GREY, false>(P, rays[tid], lut, zbits, si, stage, S[tid], n_eval[tid]);
                else
                    active[tid] = beam::march<MODE, true, AX, FAST, false, GREY, false>(P, rays[tid], lut, zbits, si, nullptr, S[tid], n_eval[tid]);
                tr.seq = nullptr;
                tr.seq_q = nullptr;
                if (kind == 1) st.v[ST_SAMPLES_STAGED] += n_eval[tid] - before;
                if (kind == 1 && si.interior) st.v[ST_SAMPLES_INTERIOR] += n_eval[tid] - before;
                longest = seq[lane].size() > longest ? seq[lane].size() : longest;
            }
            // bank model: the lanes of a warp run the sample loop in lockstep, iteration by iteration
            for (size_t it = 0; it < longest; ++it) {
                for (int c = 0; c < 8; ++c) {
                    int addr[32], nl = 0;
                    for (int lane = 0; lane < 32; ++lane)
                        if (it < seq[lane].size()) {
                            int idx = seq[lane][it];
                            idx = idx < 0 ? 0 : (idx > si.lim ? si.lim : idx);
                            addr[nl++] = idx + off[c];
                        }
                    st.v[ST_LDS] += 1;
                    st.v[ST_LDS_WAVEFRONTS] += (unsigned long long)wavefronts(addr, nl);
                }
            }
            // the classification reads of the same lockstep iterations (EA): one 16-byte load per sample with a
            // grey LUT, two (value, difference: same bank groups) otherwise
            size_t longest_q = 0;
            for (int lane = 0; lane < 32; ++lane) longest_q = seq_q[lane].size() > longest_q ? seq_q[lane].size() : longest_q;
            for (size_t it = 0; it < longest_q; ++it) {
                int q[32];
                bool any_q = false;
                for (int lane = 0; lane < 32; ++lane) {
                    q[lane] = it < seq_q[lane].size() ? seq_q[lane][it] : -2;
                    if (q[lane] == -1) ++st.v[ST_LUT_SKIPPED];
                    any_q = any_q || q[lane] >= 0;
                }
                if (!any_q) continue;
                const int loads = GREY ? 1 : 2;
                st.v[ST_LUT_LDS] += (unsigned long long)loads;
                st.v[ST_LUT_WAVEFRONTS] += (unsigned long long)(loads * lut_wavefronts(q, 32));
            }
            if (warp_alive[w]) {
                bool any = false;
                for (int lane = 0; lane < 32; ++lane) any = any || active[w * 32 + lane];
                if (!any) { warp_alive[w] = false; --G.alive; }
            }
        }
    }
    for (int tid = 0; tid < kThreads; ++tid) {
        st.v[ST_SAMPLES] += n_eval[tid];
        if (GREY) { S[tid].C1 = S[tid].C0; S[tid].C2 = S[tid].C0; }
        if (inside[tid]) beam::finish_pixel<MODE>(P, P.lut, S[tid], (size_t)pix_j[tid] * (size_t)P.W + (size_t)pix_i[tid]);
    }
}

}  // namespace

namespace {

// the EA skip bytes of the min/max bricks (A10) for the next frames: set by beam_harness_set_skip, null = skipping off
const uint8_t* g_skip = nullptr;
int g_skip_nb[3] = {0, 0, 0}, g_skip_shift = 0;

struct Frame {
    std::vector<float4> tab, grey;
    FrameParams P;
    BeamParams B;
};

// FrameParams / BeamParams of a frame, all pointers host pointers.  The table the kernels read
// (opacity-corrected alpha', forward differences) is rebuilt here exactly as DESIGN.md S7 states it.
// pad_mode: -1 default, 0 / 1 = VR_OPT_BEAM_PAD; + 16 = do not use the grey-LUT table, + 32 = do not use the zero bits,
// + 64 = two stages (VR_OPT_BEAM_STAGES = 2), + 128 = bulk row copies (VR_OPT_BEAM_BULK = 1): the threaded CTA body only
bool make_frame(Frame& F, const float* vol, int nx, int ny, int nz, const vr_camera* cam, int W, int H, float step,
                const float* lut_rgba, int n_lut, float vmin, float vmax, float tau, int stage_bytes, int pad_mode,
                float* out_rgba, float* out_aux)
{
    bool use_grey = true, use_zero = true, two_stages = false, bulk = false;
    if (pad_mode >= 0) {
        use_grey = (pad_mode & 16) == 0;
        use_zero = (pad_mode & 32) == 0;
        two_stages = (pad_mode & 64) != 0;
        bulk = (pad_mode & 128) != 0;
        pad_mode &= 15;
        if (pad_mode > 1) pad_mode = -1;
    }
    if (!vol || !cam || !lut_rgba || !out_rgba || nx % 4 != 0 || ((uintptr_t)vol & 15u) != 0) return false;
    F.tab.assign((size_t)2 * n_lut, make_float4(0.f, 0.f, 0.f, 0.f));
    for (int i = 0; i < n_lut; ++i) {
        double a = (double)lut_rgba[4 * i + 3];
        a = a < 0.0 ? 0.0 : (a > 1.0 ? 1.0 : a);
        F.tab[i] = make_float4(lut_rgba[4 * i], lut_rgba[4 * i + 1], lut_rgba[4 * i + 2],
                               (float)(1.0 - std::pow(1.0 - a, (double)step)));
    }
    for (int i = 0; i + 1 < n_lut; ++i)
        F.tab[n_lut + i] = make_float4(F.tab[i + 1].x - F.tab[i].x, F.tab[i + 1].y - F.tab[i].y,
                                       F.tab[i + 1].z - F.tab[i].z, F.tab[i + 1].w - F.tab[i].w);
    FrameParams& P = F.P;
    std::memset(&P, 0, sizeof(P));
    for (int c = 0; c < 3; ++c) {
        P.eye[c] = cam->eye[c]; P.right[c] = cam->right[c];
        P.up[c] = cam->up[c];   P.fwd[c] = cam->forward[c];
    }
    P.projection = cam->projection;
    P.th = cam->tan_half_fovy;
    P.hh = cam->ortho_half_height;
    P.W = W; P.H = H;
    P.step = step;
    P.inv_step = 1.0f / step;
    P.tau = tau;
    P.n[0] = nx; P.n[1] = ny; P.n[2] = nz;
    P.vol.base = vol;
    P.vol.sy = nx;
    P.vol.sz = (long long)nx * ny;
    P.lut = F.tab.data();
    P.n_lut = n_lut;
    P.vmin = vmin;
    P.scale = (float)((double)(n_lut - 1) / ((double)vmax - (double)vmin));
    P.out = reinterpret_cast<float4*>(out_rgba);
    P.aux = out_aux;
    P.x0 = 0; P.y0 = 0; P.x1 = W; P.y1 = H;
    P.tiles_x = (W + kTileW - 1) / kTileW;
    P.tiles_y = (H + kTileH - 1) / kTileH;
    beam::default_params(F.B);
    if (stage_bytes > 0) F.B.stage_bytes = stage_bytes;
    if (pad_mode >= 0) F.B.pad_mode = pad_mode ? 1 : 0;
    F.B.n_stages = two_stages ? 2 : 1;
    F.B.bulk = bulk ? 1 : 0;
    if (g_skip) {
        P.skip = g_skip;
        for (int c = 0; c < 3; ++c) P.nb[c] = g_skip_nb[c];
        P.mm_shift = g_skip_shift;
        F.B.use_skip = 1;
    }
    // the exact EA shortcuts, decided as vr_api.cu: ensure_lut decides them
    const float* tabf = reinterpret_cast<const float*>(F.tab.data());
    if (use_grey && beam::lut_is_grey(tabf, n_lut)) {
        F.grey.assign((size_t)n_lut, make_float4(0.f, 0.f, 0.f, 0.f));
        beam::lut_grey_table(tabf, n_lut, reinterpret_cast<float*>(F.grey.data()));
        F.B.lut_grey = F.grey.data();
    }
    if (use_zero) F.B.zero_skip = beam::lut_zero_bits(tabf, n_lut, F.B.zero_bits) > 0 ? 1 : 0;
    return true;
}

}  // namespace

// stats_out: ST_N unsigned 64-bit counters in the order of the enum above.
// lut_rgba: n_lut x 4 floats as given to vr_set_transfer_function; the table the kernels read
// (opacity-corrected alpha', forward differences) is rebuilt here exactly as DESIGN.md S7 states it.
// tile_stride > 1 renders only every tile_stride-th tile in x and y (statistics on large frames).
extern "C" int beam_harness_render(const float* vol, int nx, int ny, int nz, const vr_camera* cam, int W, int H,
                                   float step, int mode, const float* lut_rgba, int n_lut, float vmin, float vmax,
                                   float tau, int stage_bytes, int pad_mode, int tile_stride, float* out_rgba,
                                   float* out_aux, unsigned long long* stats_out)
{
    Frame F;
    if (!stats_out || !make_frame(F, vol, nx, ny, nz, cam, W, H, step, lut_rgba, n_lut, vmin, vmax, tau, stage_bytes,
                                  pad_mode, out_rgba, out_aux))
        return 1;
    if (tile_stride < 1) tile_stride = 1;
    const FrameParams& P = F.P;
    const BeamParams& B = F.B;

    TileStats total;
    const int n_tiles = P.tiles_x * P.tiles_y;
#pragma omp parallel
    {
        HarnessTrace tr;
        tr.stage_floats = B.stage_bytes >> 2;
        tr.n[0] = nx; tr.n[1] = ny; tr.n[2] = nz;
        g_tr = &tr;
        TileStats st;
        // the stage, 16-byte aligned like the dynamic shared memory of the kernel
        std::vector<float4> stage_store((size_t)(B.stage_bytes >> 4) + 1);
        float* stage = reinterpret_cast<float*>(stage_store.data());
#pragma omp for schedule(dynamic, 4)
        for (int tile = 0; tile < n_tiles; ++tile) {
            const int tx = tile % P.tiles_x, ty = tile / P.tiles_x;
            if (tx % tile_stride != 0 || ty % tile_stride != 0) continue;
            const int tile_x = P.x0 + tx * kTileW, tile_y = P.y0 + ty * kTileH;
            beam::TileGeom G;
            std::memset(&G, 0, sizeof(G));
            beam::tile_axes(P, tile_x, tile_y, G);
#define RUN(MODE_, GREY_, LUT_)                                                                                    \
            do {                                                                                                   \
                if (G.AX == 2)        run_tile<MODE_, GREY_, 2, 0>(P, B, LUT_, tile_x, tile_y, G, stage, tr, st);  \
                else if (G.AX == 1)   run_tile<MODE_, GREY_, 1, 0>(P, B, LUT_, tile_x, tile_y, G, stage, tr, st);  \
                else if (G.FAST == 2) run_tile<MODE_, GREY_, 0, 2>(P, B, LUT_, tile_x, tile_y, G, stage, tr, st);  \
                else                  run_tile<MODE_, GREY_, 0, 1>(P, B, LUT_, tile_x, tile_y, G, stage, tr, st);  \
            } while (0)
            if (mode == VR_MODE_EA) {
                if (B.lut_grey) RUN(VR_MODE_EA, true, B.lut_grey); else RUN(VR_MODE_EA, false, P.lut);
            } else {
                RUN(VR_MODE_MIP, false, P.lut);
            }
#undef RUN
        }
        st.v[ST_BAD_READ] = tr.bad_read; st.v[ST_BAD_WRITE] = tr.bad_write; st.v[ST_BAD_GLOBAL] = tr.bad_global;
        st.v[ST_MISALIGNED] = tr.misaligned; st.v[ST_FLOATS_STAGED] = tr.floats_written; st.v[ST_CHUNKS16] = tr.chunks16;
#pragma omp critical
        for (int q = 0; q < ST_N; ++q) total.v[q] += st.v[q];
        g_tr = nullptr;
    }
    for (int q = 0; q < ST_N; ++q) stats_out[q] = total.v[q];
    return 0;
}

extern "C" int beam_harness_n_stats(void) { return ST_N; }

// skip: one byte per min/max brick of edge 2^shift cells, x fastest over an nbx x nby x nbz grid; null switches
// skipping off.  The array must stay alive while frames are rendered.
extern "C" void beam_harness_set_skip(const uint8_t* skip, int nbx, int nby, int nbz, int shift)
{
    g_skip = skip;
    g_skip_nb[0] = nbx; g_skip_nb[1] = nby; g_skip_nb[2] = nbz;
    g_skip_shift = shift;
}

// ---------------------------------------------------------------------------------------------------
// The CTA body itself (csrc/vr_beam_cta.cuh: beam_cta, the code raycast_beam_kernel runs), with 128 OS
// threads per CTA: __syncthreads() = a pthread barrier over the team, warp votes and reductions = a
// barrier over the 32 threads of a warp around a scratch array, shared-memory atomics = __atomic
// builtins.  The "shared memory" of the CTA is plain host memory, so ThreadSanitizer (build with
// -fsanitize=thread, see test_beam_harness_cpu.py) reports any access that two threads make without
// a barrier between them: a missing or misplaced __syncthreads() in the CTA body is a data race here.
namespace {

// An mbarrier as the CTA body uses it (one arrival per phase): the phase completes when the arrival has come and
// the announced bytes have all been counted down; a waiter for parity p goes on once the phase of parity p is over.
struct HostMbarrier {
    pthread_mutex_t mu = PTHREAD_MUTEX_INITIALIZER;
    pthread_cond_t cv = PTHREAD_COND_INITIALIZER;
    long long tx = 0;
    int pending = 1;
    unsigned int phase = 0;
    void complete_if_done() { if (pending == 0 && tx == 0) { phase ^= 1u; pending = 1; pthread_cond_broadcast(&cv); } }
};

struct Team {
    HostMbarrier hbar[2];
    pthread_barrier_t cta_bar;
    pthread_barrier_t warp_bar[kThreads / 32];
    int scratch[kThreads];
    beam::BeamShared sh;
    std::vector<float4> dyn;                 // dynamic shared memory: LUT (EA) + stage, 16-byte aligned
    const FrameParams* P = nullptr;
    const BeamParams* B = nullptr;
    int mode = 0;
    std::vector<int> tiles;                  // the tiles this team renders, one after the other
    HarnessTrace trace[kThreads];
};

struct HostCtx {
    Team* team;
    int tid_, block_;
    int tid() const { return tid_; }
    int block() const { return block_; }
    void sync() const { pthread_barrier_wait(&team->cta_bar); }
    template <class F> int warp_reduce(int v, F f) const
    {
        const int w = tid_ >> 5;
        __atomic_store_n(&team->scratch[tid_], v, __ATOMIC_RELAXED);
        pthread_barrier_wait(&team->warp_bar[w]);
        int r = __atomic_load_n(&team->scratch[w * 32], __ATOMIC_RELAXED);
        for (int l = 1; l < 32; ++l) r = f(r, __atomic_load_n(&team->scratch[w * 32 + l], __ATOMIC_RELAXED));
        pthread_barrier_wait(&team->warp_bar[w]);
        return r;
    }
    bool any(bool p) const { return warp_reduce(p ? 1 : 0, [](int a, int b) { return a | b; }) != 0; }
    int warp_min(int v) const { return warp_reduce(v, [](int a, int b) { return a < b ? a : b; }); }
    int warp_max(int v) const { return warp_reduce(v, [](int a, int b) { return a > b ? a : b; }); }
    unsigned int warp_sum(unsigned int v) const
    {
        return (unsigned int)warp_reduce((int)v, [](int a, int b) { return (int)((unsigned int)a + (unsigned int)b); });
    }
    void smem_min(int* p, int v) const
    {
        int cur = __atomic_load_n(p, __ATOMIC_RELAXED);
        while (v < cur && !__atomic_compare_exchange_n(p, &cur, v, false, __ATOMIC_RELAXED, __ATOMIC_RELAXED)) {}
    }
    void smem_max(int* p, int v) const
    {
        int cur = __atomic_load_n(p, __ATOMIC_RELAXED);
        while (v > cur && !__atomic_compare_exchange_n(p, &cur, v, false, __ATOMIC_RELAXED, __ATOMIC_RELAXED)) {}
    }
    void smem_add(int* p, int v) const { __atomic_fetch_add(p, v, __ATOMIC_RELAXED); }
    void smem_or(int* p, int v) const { __atomic_fetch_or(p, v, __ATOMIC_RELAXED); }
    int smem_peek(const int* p) const { return __atomic_load_n(p, __ATOMIC_RELAXED); }
    void copies_done() const {}
    void count(unsigned long long* p, unsigned long long v) const { __atomic_fetch_add(p, v, __ATOMIC_RELAXED); }
    HostMbarrier& mbar(unsigned long long* bar) const { return team->hbar[bar - team->sh.bar]; }
    void bulk_init(unsigned long long* bar) const
    {
        HostMbarrier& m = mbar(bar);
        pthread_mutex_lock(&m.mu); m.tx = 0; m.pending = 1; m.phase = 0; pthread_mutex_unlock(&m.mu);
    }
    void bulk_expect(unsigned long long* bar, unsigned int bytes) const
    {
        HostMbarrier& m = mbar(bar);
        pthread_mutex_lock(&m.mu); m.tx += bytes; m.pending -= 1; m.complete_if_done(); pthread_mutex_unlock(&m.mu);
    }
    void bulk_row(unsigned long long* bar, float* dst, const float* src, unsigned int bytes) const
    {
        std::memcpy(dst, src, bytes);
        HostMbarrier& m = mbar(bar);
        pthread_mutex_lock(&m.mu); m.tx -= bytes; m.complete_if_done(); pthread_mutex_unlock(&m.mu);
    }
    void bulk_wait(unsigned long long* bar, unsigned int parity) const
    {
        HostMbarrier& m = mbar(bar);
        pthread_mutex_lock(&m.mu);
        while (m.phase == parity) pthread_cond_wait(&m.cv, &m.mu);
        pthread_mutex_unlock(&m.mu);
    }
};

struct ThreadArg {
    Team* team;
    int tid;
};

void* team_thread(void* argp)
{
    ThreadArg* arg = static_cast<ThreadArg*>(argp);
    Team* team = arg->team;
    g_tr = &team->trace[arg->tid];
    unsigned char* s_dyn = reinterpret_cast<unsigned char*>(team->dyn.data());
    for (int tile : team->tiles) {
        HostCtx cx{team, arg->tid, tile};
#define CTA(MODE_, GREY_)                                                                                     \
        do {                                                                                                  \
            if (team->B->n_stages == 2)                                                                       \
                beam::beam_cta<MODE_, true, GREY_, 2>(*team->P, *team->B, team->sh, s_dyn, cx);               \
            else                                                                                              \
                beam::beam_cta<MODE_, true, GREY_, 1>(*team->P, *team->B, team->sh, s_dyn, cx);               \
        } while (0)
        if (team->mode == VR_MODE_EA && team->B->lut_grey) CTA(VR_MODE_EA, true);
        else if (team->mode == VR_MODE_EA) CTA(VR_MODE_EA, false);
        else CTA(VR_MODE_MIP, false);
#undef CTA
        cx.sync();                            // a CTA's shared memory is its own: the next tile starts afresh
    }
    g_tr = nullptr;
    return nullptr;
}

}  // namespace

// The frame rendered by beam_cta with thread teams.  stats_out: {rays hit, samples, bad reads, bad writes,
// bad global reads, misaligned copies}.  n_teams CTAs run concurrently (tiles are dealt round-robin).
extern "C" int beam_harness_render_threads(const float* vol, int nx, int ny, int nz, const vr_camera* cam, int W, int H,
                                           float step, int mode, const float* lut_rgba, int n_lut, float vmin,
                                           float vmax, float tau, int stage_bytes, int pad_mode, int n_teams,
                                           float* out_rgba, float* out_aux, unsigned long long* stats_out)
{
    Frame F;
    if (!stats_out || !make_frame(F, vol, nx, ny, nz, cam, W, H, step, lut_rgba, n_lut, vmin, vmax, tau, stage_bytes,
                                  pad_mode, out_rgba, out_aux))
        return 1;
    unsigned long long counters[2] = {0, 0};
    F.P.counters = counters;
    if (n_teams < 1) n_teams = 1;
    const int n_tiles = F.P.tiles_x * F.P.tiles_y;
    std::vector<Team> teams((size_t)n_teams);
    std::vector<ThreadArg> args((size_t)n_teams * kThreads);
    std::vector<pthread_t> threads((size_t)n_teams * kThreads);
    const size_t dyn_bytes = (size_t)2 * n_lut * sizeof(float4) + (size_t)F.B.n_stages * (size_t)F.B.stage_bytes;
    for (int t = 0; t < n_teams; ++t) {
        Team& T = teams[(size_t)t];
        pthread_barrier_init(&T.cta_bar, nullptr, kThreads);
        for (int w = 0; w < kThreads / 32; ++w) pthread_barrier_init(&T.warp_bar[w], nullptr, 32);
        T.dyn.assign(dyn_bytes / sizeof(float4) + 1, make_float4(0.f, 0.f, 0.f, 0.f));
        T.P = &F.P; T.B = &F.B; T.mode = mode;
        for (int tile = t; tile < n_tiles; tile += n_teams) T.tiles.push_back(tile);
        for (int q = 0; q < kThreads; ++q) {
            T.trace[q].stage_floats = F.B.stage_bytes >> 2;
            T.trace[q].n[0] = nx; T.trace[q].n[1] = ny; T.trace[q].n[2] = nz;
        }
    }
    pthread_attr_t attr;
    pthread_attr_init(&attr);
    pthread_attr_setstacksize(&attr, 1 << 20);
    int rc = 0;
    size_t started = 0;
    for (int t = 0; t < n_teams && !rc; ++t)
        for (int q = 0; q < kThreads && !rc; ++q) {
            args[started] = ThreadArg{&teams[(size_t)t], q};
            rc = pthread_create(&threads[started], &attr, team_thread, &args[started]);
            if (!rc) ++started;
        }
    pthread_attr_destroy(&attr);
    if (rc) return 2;                          // (a partly started team would wait for ever: not handled, tests only)
    for (size_t q = 0; q < started; ++q) pthread_join(threads[q], nullptr);
    unsigned long long bad[4] = {0, 0, 0, 0};
    for (Team& T : teams) {
        for (int q = 0; q < kThreads; ++q) {
            bad[0] += T.trace[q].bad_read; bad[1] += T.trace[q].bad_write;
            bad[2] += T.trace[q].bad_global; bad[3] += T.trace[q].misaligned;
        }
        pthread_barrier_destroy(&T.cta_bar);
        for (int w = 0; w < kThreads / 32; ++w) pthread_barrier_destroy(&T.warp_bar[w]);
    }
    stats_out[0] = counters[0]; stats_out[1] = counters[1];
    for (int q = 0; q < 4; ++q) stats_out[2 + q] = bad[q];
    return 0;
}

#ifdef BEAM_HARNESS_MAIN
// Stand-alone driver for the ThreadSanitizer build: a seeded random cube, a few small views in both
// modes, the threaded CTA body against the sequential harness above (which the Python tests hold
// against the oracle).  Exit code 0 and "beam_cta threads OK" = same pixels, no bad index; data races
// are reported by the sanitizer itself (run with TSAN_OPTIONS=halt_on_error=1 exitcode=66).
#include <cstdio>

int main()
{
    const int nx = 32, ny = 20, nz = 24, W = 48, H = 24;
    std::vector<float4> store((size_t)nx * ny * nz / 4 + 1);
    float* vol = reinterpret_cast<float*>(store.data());
    unsigned int seed = 12345u;
    for (int q = 0; q < nx * ny * nz; ++q) {
        seed = seed * 1664525u + 1013904223u;
        vol[q] = (float)(seed >> 8) * (1.0f / 16777216.0f) * 8.0f - 3.0f;
    }
    std::vector<float> lut(256 * 4);
    for (int i = 0; i < 256; ++i) {
        lut[4 * i] = lut[4 * i + 1] = lut[4 * i + 2] = (float)i / 255.0f;
        lut[4 * i + 3] = 0.05f * (float)i / 255.0f;
    }
    // perspective views from four sides (z and x slabs, both senses) and one from above (y slabs)
    const float c[3] = {(nx - 1) * 0.5f, (ny - 1) * 0.5f, (nz - 1) * 0.5f};
    const float dirs[5][3] = {{0.f, 0.f, 1.f}, {0.f, 0.f, -1.f}, {1.f, 0.f, 0.f}, {-1.f, 0.f, 0.f}, {0.f, -1.f, 0.f}};
    int failures = 0;
    for (int v = 0; v < 5; ++v)
        for (int mode = 0; mode < 2; ++mode) {
            vr_camera cam;
            std::memset(&cam, 0, sizeof(cam));
            const float* f = dirs[v];
            const float up[3] = {0.f, f[1] != 0.f ? 0.f : 1.f, f[1] != 0.f ? 1.f : 0.f};
            const float right[3] = {up[1] * f[2] - up[2] * f[1], up[2] * f[0] - up[0] * f[2], up[0] * f[1] - up[1] * f[0]};
            for (int k = 0; k < 3; ++k) {
                cam.forward[k] = f[k]; cam.up[k] = up[k]; cam.right[k] = right[k];
                cam.eye[k] = c[k] - 45.0f * f[k] + 1.7f * up[k] + 0.9f * right[k];
            }
            cam.projection = VR_PROJ_PERSPECTIVE;
            cam.tan_half_fovy = 0.45f;
            std::vector<float> a((size_t)W * H * 4), b((size_t)W * H * 4), aux_a((size_t)W * H), aux_b((size_t)W * H);
            unsigned long long sa[ST_N], sb[6];
            const int stages_flag = ((v + mode) % 2 ? 64 : 0) + (v % 2 ? 128 : 0);   // two stages / bulk row copies in turn
            if (beam_harness_render(vol, nx, ny, nz, &cam, W, H, 0.5f, mode, lut.data(), 256, -3.f, 5.f, 0.99f, 8192, 1, 1,
                                    a.data(), aux_a.data(), sa) ||
                beam_harness_render_threads(vol, nx, ny, nz, &cam, W, H, 0.5f, mode, lut.data(), 256, -3.f, 5.f, 0.99f,
                                            8192, 1 + stages_flag, 2, b.data(), aux_b.data(), sb)) {
                std::printf("view %d mode %d: harness call failed\n", v, mode);
                ++failures;
                continue;
            }
            const bool same = std::memcmp(a.data(), b.data(), a.size() * sizeof(float)) == 0 &&
                              std::memcmp(aux_a.data(), aux_b.data(), aux_a.size() * sizeof(float)) == 0;
            const bool clean = sb[2] + sb[3] + sb[4] + sb[5] == 0;
            std::printf("view %d mode %d stages %d: %llu rays, %llu samples, %s, %s\n", v, mode, (stages_flag & 64) ? 2 : 1, sb[0], sb[1],
                        same && sa[ST_SAMPLES] == sb[1] && sa[ST_RAYS_HIT] == sb[0] ? "same pixels" : "PIXELS DIFFER",
                        clean ? "indices clean" : "BAD INDEX");
            if (!same || !clean || sa[ST_SAMPLES] != sb[1] || sa[ST_RAYS_HIT] != sb[0] || sb[1] == 0) ++failures;
        }
    if (failures) { std::printf("beam_cta threads: %d FAILURES\n", failures); return 1; }
    std::printf("beam_cta threads OK\n");
    return 0;
}
#endif

// Exhaustive check of the copy loops' division by multiplication (magic_of / div_magic): every divisor a box can
// have against every chunk index a stage of 192 KiB can hold.  Returns the number of wrong quotients.
extern "C" unsigned long long beam_harness_check_div_magic(void)
{
    unsigned long long bad = 0;
    for (unsigned int d = 1; d <= 12288; ++d) {
        const unsigned int mg = vr::beam::magic_of(d);
        for (unsigned int e = 0; e < 49152; ++e)
            if (vr::beam::div_magic(e, mg) != e / d) ++bad;
    }
    return bad;
}
