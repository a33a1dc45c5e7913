// vr_api.cu -- the C ABI of include/vr.h: handles, validation, transfer-function
// setup, min/max + skip tables, and the out-of-core brick streaming scheduler.
// All voxel work runs in the kernels of vr_kernels.cu; there is no CPU fallback.
#include "vr_beam_plan.h"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#ifndef VR_HOSTEMU
#include <nvtx3/nvToolsExt.h>       // header-only; ranges show up in Nsight Systems / ncu --nvtx, cost nothing otherwise
#endif

namespace {

// NVTX range for the lifetime of the object (upload / render / brick)
struct Range {
#ifndef VR_HOSTEMU
    explicit Range(const char* name) { nvtxRangePushA(name); }
    ~Range() { nvtxRangePop(); }
#else
    explicit Range(const char*) {}
#endif
    Range(const Range&) = delete;
    Range& operator=(const Range&) = delete;
};

thread_local char g_err[512] = "";

vr_status fail(vr_status st, const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return st;
}

#define VR_CUDA(expr)                                                                     \
    do {                                                                                  \
        cudaError_t e_ = (expr);                                                          \
        if (e_ != cudaSuccess)                                                            \
            return fail(VR_ERR_CUDA, "%s failed: %s", #expr, cudaGetErrorString(e_));     \
    } while (0)

struct HostBrick {
    const float* ptr = nullptr;
    int origin[3] = {0, 0, 0};
    int dims[3] = {0, 0, 0};
};

int ceil_div(int a, int b) { return (a + b - 1) / b; }

}  // namespace

struct vr_volume {
    vr_volume_desc desc{};
    bool streamed = false;
    bool uploaded = false;
    // a PART of a larger cube (vr_volume_create_part, sort-last rendering): desc.nx/ny/nz are the part's voxels,
    // `full` the cube's, `p_org` the part's first voxel; it owns cells [p_org, p_org + dims - 1) per axis (S10)
    bool part = false;
    int full[3] = {0, 0, 0}, p_org[3] = {0, 0, 0};

    // VR_LAYOUT_TEX: library-owned 2D-layered arrays (resident: the cube; streamed: one per slot)
    bool tex = false;
    std::vector<cudaArray_t> chunk_arr;          // resident: z chunks of <= kMaxLayers layers, overlapping by one layer
    std::vector<cudaTextureObject_t> chunk_tex;
    int chunk_step = 0;                          // first layer of chunk c = c * chunk_step
    std::vector<cudaArray_t> slot_arr;
    std::vector<cudaTextureObject_t> slot_tex;

    // beam kernel (vr_beam.cu): depth sets, stage size and padding of the shared-memory boxes
    vr::BeamParams beam_params{};
    struct StageChoice { vr_camera cam; int W, H, pad_mode, stage_bytes; };
    std::vector<StageChoice> stage_cache;    // per-frame stage sizes already chosen (auto_stage_bytes), newest last

    // min/max bricks (A2) and EA skip bytes (A10)
    int mm_B = 64, mm_shift = 6;
    int nb[3] = {0, 0, 0};
    int n_mm = 0;
    float2* d_minmax = nullptr;
    uint8_t* d_skip = nullptr;
    // coarse level (bricks of 8 x the edge) when the fine bricks are small (mm_B <= 16): two-level skipping
    int mm2_shift = 0, nb2[3] = {0, 0, 0}, n_mm2 = 0;
    float2* d_minmax2 = nullptr;
    uint8_t* d_skip2 = nullptr;
    int* d_nzprefix = nullptr;
    unsigned int* d_nskip = nullptr;
    bool minmax_valid = false;
    bool skip_valid = false;

    // transfer function (A3)
    std::vector<float> lut;       // n_lut * 4, as given
    std::vector<float> h_tab;     // device table image (values, then forward differences)
    std::vector<int> h_prefix;    // running count of non-zero alpha' entries
    int n_lut = 0;
    float vmin = 0.f, vmax = 1.f, scale = 1.f;
    float4* d_lut = nullptr;      // 2 * n_lut: value table, then forward differences
    float4* d_lut_grey = nullptr; // beam kernel: n_lut entries (grey, alpha', d grey, d alpha') when r = g = b everywhere
    std::vector<float> h_grey;
    bool lut_valid = false;
    float lut_step = 0.f;

    // options
    float tau = 0.99f;
    int opt_skip = 0, opt_kernel = 0, opt_count = 0, opt_compositor = 0, opt_pipeline = 0, opt_tile_order = 0, opt_reuse = 0;
    float spacing[3] = {1.f, 1.f, 1.f};      // R23: world units per voxel (VR_OPT_SPACING_X / Y / Z)
    bool blank = false;                      // R17b: non-finite voxels become blank_value as they arrive on the device
    float blank_value = 0.f;
    float* d_aux = nullptr;
    unsigned long long* d_counters = nullptr;

    // streamed volumes (A12, A13)
    int hb = 0;
    int nhb[3] = {0, 0, 0};
    std::vector<HostBrick> bricks;
    size_t slot_bytes = 0;
    int n_slots = 0;
    cudaStream_t copy_stream = nullptr;
    std::vector<cudaEvent_t> ev_copied, ev_free;
    std::vector<char> slot_used;
    float4* d_partial = nullptr;
    size_t partial_px = 0;
    // device slots as a cache of bricks across frames (8(f)1): which brick a slot holds, when it was last used
    std::vector<int> slot_brick;                  // -1: nothing
    std::vector<unsigned long long> slot_tick;    // value of `tick` when the slot was last assigned or hit
    std::vector<unsigned long long> slot_frame;   // frame in which that was
    std::vector<int> brick_slot;                  // brick -> slot holding it, or -1
    unsigned long long tick = 0, frame_no = 0;
    int opt_cache = 1, opt_cull = 0;
    // per-brick value range (A2 for streamed bricks): computed on the device the first time a brick sits in a slot
    float2* d_brick_mm = nullptr;                 // [bricks]
    float2* h_brick_mm = nullptr;                 // pinned mirror
    std::vector<char> brick_mm_state;             // 0 unknown, 1 copy to the host mirror in flight, 2 known
    cudaEvent_t ev_frame = nullptr;               // end of the last streamed frame (brick_mm_state 1 -> 2 once it completed)
    bool mm_in_flight = false;
    // saturation culling: one reduced running value per brick of a wavefront
    float* d_cull = nullptr;
    float* h_cull = nullptr;                      // pinned
    cudaEvent_t ev_cull = nullptr;
    std::vector<int> brick_flags;                 // VR_BRICK_* of the last frame
    // timing of the last streamed frame
    std::vector<cudaEvent_t> tev;                 // pairs around every brick copy, grown on demand
    int n_tev = 0;
    cudaEvent_t ev_f0 = nullptr, ev_f1 = nullptr; // frame start / end on the render stream

    vr_stats stats{};
};

namespace {

bool valid_dims(const vr_volume_desc* d)
{
    return d && d->nx >= 2 && d->ny >= 2 && d->nz >= 2 && d->host_brick >= 0 && d->mm_brick >= 0;
}

constexpr int kMaxSlots = 1024;        // device slots of a streamed volume (a 180 GB pool holds ~330 bricks of 513^3)
constexpr int kMaxLayers = 2048;       // maxTexture2DLayered[2]
constexpr int kMaxTexExtent = 32768;   // maxTexture2DLayered[0..1]

// layers per array of a resident VR_LAYOUT_TEX cube; VR_TEX_MAX_LAYERS (>= 2) lowers it so that tests can cut small
// cubes into several chunks
int tex_max_layers()
{
    const char* e = std::getenv("VR_TEX_MAX_LAYERS");
    const int v = e ? std::atoi(e) : 0;
    return v >= 2 && v < kMaxLayers ? v : kMaxLayers;
}

// a float32 2D-layered array of w x h texels and `layers` layers, with a point-sampled,
// unnormalised, clamped texture object over it (read with tld4 gathers, never filtered)
cudaError_t make_layered(int w, int h, int layers, cudaArray_t* arr, cudaTextureObject_t* tex)
{
    const cudaChannelFormatDesc cd = cudaCreateChannelDesc<float>();
    cudaError_t e = cudaMalloc3DArray(arr, &cd, make_cudaExtent((size_t)w, (size_t)h, (size_t)layers), cudaArrayLayered);
    if (e != cudaSuccess) { *arr = nullptr; return e; }
    cudaResourceDesc rd{};
    rd.resType = cudaResourceTypeArray;
    rd.res.array.array = *arr;
    cudaTextureDesc td{};
    td.addressMode[0] = td.addressMode[1] = td.addressMode[2] = cudaAddressModeClamp;
    td.filterMode = cudaFilterModePoint;
    td.readMode = cudaReadModeElementType;
    td.normalizedCoords = 0;
    e = cudaCreateTextureObject(tex, &rd, &td, nullptr);
    if (e != cudaSuccess) { cudaFreeArray(*arr); *arr = nullptr; *tex = 0; }
    return e;
}

// one box of dense float32 voxels -> texels [pos, pos + dims) of a layered array
cudaError_t copy_box_to_array(cudaArray_t arr, const int pos[3], const int dims[3], const float* src,
                              cudaMemcpyKind kind, cudaStream_t s)
{
    cudaMemcpy3DParms p{};
    p.srcPtr = make_cudaPitchedPtr((void*)src, (size_t)dims[0] * sizeof(float), (size_t)dims[0], (size_t)dims[1]);
    p.dstArray = arr;
    p.dstPos = make_cudaPos((size_t)pos[0], (size_t)pos[1], (size_t)pos[2]);     // elements when an array takes part
    p.extent = make_cudaExtent((size_t)dims[0], (size_t)dims[1], (size_t)dims[2]);
    p.kind = kind;
    return cudaMemcpy3DAsync(&p, s);
}

size_t brick_voxels_max(const vr_volume_desc* d)
{
    const int B = d->host_brick;
    const size_t bx = (size_t)std::min(B + 1, d->nx), by = (size_t)std::min(B + 1, d->ny),
                 bz = (size_t)std::min(B + 1, d->nz);
    return bx * by * bz;
}

size_t round_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// S7 host part: alpha' = 1 - (1 - alpha)^step in double, rounded once
float corrected_alpha(float a, float step)
{
    double x = (double)a;
    x = x < 0.0 ? 0.0 : (x > 1.0 ? 1.0 : x);
    return (float)(1.0 - std::pow(1.0 - x, (double)step));
}

vr_status ensure_lut(vr_volume* v, float step, int mode, cudaStream_t s)
{
    (void)mode;   // MIP only reads the colours; they are shared with the EA table
    if (v->lut_valid && v->lut_step == step) return VR_OK;
    const int n = v->n_lut;
    std::vector<float>& tab = v->h_tab;      // kept alive in the handle: sources of async copies
    std::vector<int>& prefix = v->h_prefix;
    tab.assign((size_t)8 * n, 0.f);
    prefix.assign((size_t)n + 1, 0);
    for (int i = 0; i < n; ++i) {
        tab[4 * i + 0] = v->lut[4 * i + 0];
        tab[4 * i + 1] = v->lut[4 * i + 1];
        tab[4 * i + 2] = v->lut[4 * i + 2];
        tab[4 * i + 3] = corrected_alpha(v->lut[4 * i + 3], step);
        prefix[i + 1] = prefix[i] + (tab[4 * i + 3] != 0.0f ? 1 : 0);
    }
    for (int i = 0; i + 1 < n; ++i)
        for (int ch = 0; ch < 4; ++ch)
            tab[4 * (n + i) + ch] = tab[4 * (i + 1) + ch] - tab[4 * i + ch];   // one fp32 subtraction
    VR_CUDA(cudaMemcpyAsync(v->d_lut, tab.data(), tab.size() * sizeof(float), cudaMemcpyHostToDevice, s));
    VR_CUDA(cudaMemcpyAsync(v->d_nzprefix, prefix.data(), prefix.size() * sizeof(int), cudaMemcpyHostToDevice, s));
    // exact shortcuts of the beam kernel's EA classification (vr_beam_plan.h)
    vr::BeamParams& B = v->beam_params;
    B.lut_grey = nullptr;
    if (vr::beam::lut_is_grey(tab.data(), n)) {
        v->h_grey.assign((size_t)4 * n, 0.f);
        vr::beam::lut_grey_table(tab.data(), n, v->h_grey.data());
        VR_CUDA(cudaMemcpyAsync(v->d_lut_grey, v->h_grey.data(), v->h_grey.size() * sizeof(float), cudaMemcpyHostToDevice, s));
        B.lut_grey = v->d_lut_grey;
    }
    B.zero_skip = vr::beam::lut_zero_bits(tab.data(), n, B.zero_bits) > 0 ? 1 : 0;
    v->lut_valid = true;
    v->lut_step = step;
    v->skip_valid = false;
    return VR_OK;
}

// Flipped to true once the beam kernel has passed the GPU parity tests and beaten the direct kernel on a B200
// (validation order); until then VR_OPT_KERNEL = 0 means the direct kernel.
constexpr bool kBeamIsDefault = false;

// The beam kernel copies 16-byte chunks of x rows: rows and base must be 16-byte aligned, and its float
// floor trick and k + 0.5 counter need extents and ray lengths below 2^22.
bool beam_eligible(const vr_volume* v)
{
    const vr_volume_desc& d = v->desc;
    if (v->tex || v->streamed) return false;
    if (d.nx % 4 != 0 || ((uintptr_t)d.d_storage & 15u) != 0) return false;
    if (d.nx > (1 << 22) || d.ny > (1 << 22) || d.nz > (1 << 22)) return false;
    return true;
}

vr::VoxelBox resident_box(const vr_volume* v)
{
    vr::VoxelBox b{};
    b.base = (const float*)v->desc.d_storage;
    b.sy = v->desc.nx;
    b.sz = (long long)v->desc.nx * v->desc.ny;
    for (size_t c = 0; c < v->chunk_tex.size(); ++c) b.tex[c] = v->chunk_tex[c];
    b.n_chunks = (int)v->chunk_tex.size();
    b.chunk_step = v->chunk_step;
    b.chunk_magic = vr::beam::magic_of((unsigned int)v->chunk_step);
    b.gx = 1.0f;
    b.gy = 1.0f;
    b.org_z = 0;
    return b;
}

// (re)allocates the min/max and skip tables for bricks of edge mmB (a power of two >= 2)
cudaError_t alloc_mm_tables(vr_volume* v, int mmB)
{
    cudaFree(v->d_minmax); cudaFree(v->d_skip); cudaFree(v->d_minmax2); cudaFree(v->d_skip2);
    v->d_minmax = v->d_minmax2 = nullptr;
    v->d_skip = v->d_skip2 = nullptr;
    v->mm_B = mmB;
    v->mm_shift = 0;
    while ((1 << v->mm_shift) < mmB) ++v->mm_shift;
    const int n[3] = {v->desc.nx, v->desc.ny, v->desc.nz};
    for (int c = 0; c < 3; ++c) v->nb[c] = ceil_div(n[c] - 1, mmB);
    v->n_mm = v->nb[0] * v->nb[1] * v->nb[2];
    v->stats.mm_bricks = (unsigned long long)v->n_mm;
    v->minmax_valid = v->skip_valid = false;
    cudaError_t e = cudaMalloc((void**)&v->d_minmax, sizeof(float2) * (size_t)v->n_mm);
    if (e == cudaSuccess) e = cudaMalloc((void**)&v->d_skip, (size_t)v->n_mm);
    v->mm2_shift = 0;
    v->n_mm2 = 0;
    if (e == cudaSuccess && mmB <= 16) {
        v->mm2_shift = v->mm_shift + 3;
        for (int c = 0; c < 3; ++c) v->nb2[c] = ceil_div(v->nb[c], 8);
        v->n_mm2 = v->nb2[0] * v->nb2[1] * v->nb2[2];
        e = cudaMalloc((void**)&v->d_minmax2, sizeof(float2) * (size_t)v->n_mm2);
        if (e == cudaSuccess) e = cudaMalloc((void**)&v->d_skip2, (size_t)v->n_mm2);
    }
    return e;
}

vr_status ensure_minmax(vr_volume* v, cudaStream_t s)
{
    if (v->minmax_valid) return VR_OK;
    vr::MinMaxParams M{};
    M.vol = resident_box(v);
    M.tex = v->tex ? 1 : 0;
    M.n[0] = v->desc.nx; M.n[1] = v->desc.ny; M.n[2] = v->desc.nz;
    for (int c = 0; c < 3; ++c) M.nb[c] = v->nb[c];
    M.B = v->mm_B;
    M.out = v->d_minmax;
    VR_CUDA(vr::launch_minmax(M, s));
    if (v->mm2_shift) {
        vr::CoarseParams C{};
        C.fine = v->d_minmax;
        C.coarse = v->d_minmax2;
        for (int c = 0; c < 3; ++c) { C.nb[c] = v->nb[c]; C.nb2[c] = v->nb2[c]; }
        VR_CUDA(vr::launch_coarse_minmax(C, s));
    }
    v->minmax_valid = true;
    v->skip_valid = false;
    return VR_OK;
}

vr_status ensure_skip(vr_volume* v, cudaStream_t s)
{
    if (v->skip_valid) return VR_OK;
    VR_CUDA(cudaMemsetAsync(v->d_nskip, 0, sizeof(unsigned int), s));
    vr::SkipParams S{};
    S.minmax = v->d_minmax;
    S.n_bricks = v->n_mm;
    S.nz_prefix = v->d_nzprefix;
    S.n_lut = v->n_lut;
    S.vmin = v->vmin;
    S.scale = v->scale;
    S.skip = v->d_skip;
    S.n_skippable = v->d_nskip;
    VR_CUDA(vr::launch_skipbits(S, s));
    if (v->mm2_shift) {
        S.minmax = v->d_minmax2;
        S.n_bricks = v->n_mm2;
        S.skip = v->d_skip2;
        S.n_skippable = nullptr;          // the count reported is the fine level's
        VR_CUDA(vr::launch_skipbits(S, s));
    }
    v->skip_valid = true;
    return VR_OK;
}

void fill_frame(const vr_volume* v, const vr_camera* cam, int W, int H, float step, float4* out,
                vr::FrameParams& P)
{
    std::memset(&P, 0, sizeof(P));
    for (int c = 0; c < 3; ++c) {
        P.eye[c] = cam->eye[c]; P.right[c] = cam->right[c];
        P.up[c] = cam->up[c];   P.fwd[c] = cam->forward[c];
    }
    P.projection = cam->projection;
    P.th = cam->tan_half_fovy;
    P.hh = cam->ortho_half_height;
    P.W = W; P.H = H;
    P.aniso = !(v->spacing[0] == 1.0f && v->spacing[1] == 1.0f && v->spacing[2] == 1.0f);
    for (int c = 0; c < 3; ++c) P.inv_sp[c] = 1.0f / v->spacing[c];
    P.step = step;
    P.inv_step = 1.0f / step;
    P.tau = v->tau;
    P.n[0] = v->desc.nx; P.n[1] = v->desc.ny; P.n[2] = v->desc.nz;
    P.lut = v->d_lut;
    P.n_lut = v->n_lut;
    P.vmin = v->vmin;
    P.scale = v->scale;
    P.out = out;
    P.aux = v->d_aux;
    P.x0 = 0; P.y0 = 0; P.x1 = W; P.y1 = H;
    P.tiles_x = ceil_div(W, vr::kTileW);
    P.tiles_y = ceil_div(H, vr::kTileH);
    P.tile_order = v->opt_tile_order;
    P.minmax = v->d_minmax;
    P.skip = v->d_skip;
    for (int c = 0; c < 3; ++c) { P.nb[c] = v->nb[c]; P.nb2[c] = v->nb2[c]; }
    P.mm_shift = v->mm_shift;
    P.minmax2 = v->d_minmax2;
    P.skip2 = v->d_skip2;
    P.mm2_shift = v->mm2_shift;
    P.counters = v->d_counters;
}

// S11: wavefront key of brick b for this camera
int brick_key(const vr_camera* cam, int B, const int b[3], const float* spacing)
{
    int key = 0;
    for (int c = 0; c < 3; ++c) {
        if (cam->projection == VR_PROJ_PERSPECTIVE) {
            // (R23: the eye in index space, by the same binary32 operations as the kernels' rays)
            const bool aniso = spacing && !(spacing[0] == 1.0f && spacing[1] == 1.0f && spacing[2] == 1.0f);
            const float e = aniso ? cam->eye[c] * (1.0f / spacing[c]) : cam->eye[c];
            const int ie = (int)std::floor(e / (float)B);
            key += std::abs(b[c] - ie);
        } else {
            const float d = cam->forward[c];
            key += ((d > 0.f) - (d < 0.f)) * b[c];
        }
    }
    return key;
}

struct Keyed { int key, idx; };

void order_bricks(const int nhb[3], int B, const vr_camera* cam, std::vector<Keyed>& ks, const float* spacing = nullptr)
{
    ks.clear();
    ks.reserve((size_t)nhb[0] * nhb[1] * nhb[2]);
    int b[3];
    for (b[2] = 0; b[2] < nhb[2]; ++b[2])
        for (b[1] = 0; b[1] < nhb[1]; ++b[1])
            for (b[0] = 0; b[0] < nhb[0]; ++b[0])
                ks.push_back({brick_key(cam, B, b, spacing), b[0] + nhb[0] * (b[1] + nhb[1] * b[2])});
    std::stable_sort(ks.begin(), ks.end(), [](const Keyed& a, const Keyed& c) {
        return a.key != c.key ? a.key < c.key : a.idx < c.idx;
    });
}

// conservative screen rectangle of the position box [lo, hi] (host, double)
bool screen_bbox(const vr_camera* cam, int W, int H, const double lo_i[3], const double hi_i[3], int r[4],
                 const float* spacing = nullptr)
{
    // the box is given in voxel-index coordinates; the camera lives in world space (R23)
    double lo[3], hi[3];
    for (int c = 0; c < 3; ++c) {
        const double sp = spacing ? (double)spacing[c] : 1.0;
        lo[c] = lo_i[c] * sp;
        hi[c] = hi_i[c] * sp;
    }
    const double asp = (double)W / (double)H;
    double xmin = 1e300, xmax = -1e300, ymin = 1e300, ymax = -1e300;
    bool full = false;
    for (int q = 0; q < 8 && !full; ++q) {
        double v[3];
        for (int c = 0; c < 3; ++c) v[c] = ((q >> c) & 1 ? hi[c] : lo[c]) - (double)cam->eye[c];
        double xr = 0, yu = 0, zf = 0;
        for (int c = 0; c < 3; ++c) {
            xr += v[c] * cam->right[c]; yu += v[c] * cam->up[c]; zf += v[c] * cam->forward[c];
        }
        double sx, sy;
        if (cam->projection == VR_PROJ_PERSPECTIVE) {
            if (zf <= 1e-3) { full = true; break; }
            sx = xr / (zf * cam->tan_half_fovy);
            sy = yu / (zf * cam->tan_half_fovy);
        } else {
            sx = xr / cam->ortho_half_height;
            sy = yu / cam->ortho_half_height;
        }
        const double pi = ((sx / asp + 1.0) * W - 1.0) / 2.0;
        const double pj = ((1.0 - sy) * H - 1.0) / 2.0;
        xmin = std::min(xmin, pi); xmax = std::max(xmax, pi);
        ymin = std::min(ymin, pj); ymax = std::max(ymax, pj);
    }
    if (full) { r[0] = 0; r[1] = 0; r[2] = W; r[3] = H; return true; }
    const double x0 = std::floor(xmin) - 2.0, y0 = std::floor(ymin) - 2.0;
    const double x1 = std::ceil(xmax) + 3.0, y1 = std::ceil(ymax) + 3.0;
    r[0] = (int)std::max(0.0, std::min((double)W, x0));
    r[1] = (int)std::max(0.0, std::min((double)H, y0));
    r[2] = (int)std::max(0.0, std::min((double)W, x1));
    r[3] = (int)std::max(0.0, std::min((double)H, y1));
    return r[2] > r[0] && r[3] > r[1];
}

vr_status check_render_args(vr_volume* v, const vr_camera* cam, int W, int H, float step, int mode,
                            const float* out)
{
    if (!v || !cam || !out) return fail(VR_ERR_INVALID_ARG, "vr_render: null argument");
    if (W < 1 || H < 1 || (long long)W * H > (1ll << 31))
        return fail(VR_ERR_INVALID_ARG, "vr_render: bad image size %d x %d", W, H);
    if (!(step > 0.0f) || !std::isfinite(step))
        return fail(VR_ERR_INVALID_ARG, "vr_render: step must be finite and > 0");
    if (mode != VR_MODE_EA && mode != VR_MODE_MIP)
        return fail(VR_ERR_INVALID_ARG, "vr_render: unknown mode %d", mode);
    if (cam->projection != VR_PROJ_PERSPECTIVE && cam->projection != VR_PROJ_ORTHO)
        return fail(VR_ERR_INVALID_ARG, "vr_render: unknown projection %d", cam->projection);
    if (cam->projection == VR_PROJ_PERSPECTIVE && !(cam->tan_half_fovy > 0.0f))
        return fail(VR_ERR_INVALID_ARG, "vr_render: tan_half_fovy must be > 0");
    if (cam->projection == VR_PROJ_ORTHO && !(cam->ortho_half_height > 0.0f))
        return fail(VR_ERR_INVALID_ARG, "vr_render: ortho_half_height must be > 0");
    // the sample index k and k + 0.5 must stay exact in binary32 (S4): at most 2^22 samples on the longest chord
    const double ex = v->part ? v->full[0] : v->desc.nx, ey = v->part ? v->full[1] : v->desc.ny,
                 ez = v->part ? v->full[2] : v->desc.nz;
    const double diag = std::sqrt(ex * ex + ey * ey + ez * ez);
    if (!(diag / (double)step < 4194304.0))
        return fail(VR_ERR_INVALID_ARG, "vr_render: step %g gives more than 2^22 samples per ray on this cube", (double)step);
    if (!v->uploaded) return fail(VR_ERR_STATE, "vr_render: no voxels uploaded yet");
    if (v->n_lut < 2) return fail(VR_ERR_STATE, "vr_render: no transfer function set");
    return VR_OK;
}

// VR_OPT_PIPELINE = 0: how many samples a thread of the direct kernel keeps in flight.  Samples per voxel
// = 1 / (pitch^2 * step), pitch = voxels between neighbouring pixels at the depth of the cube's centre: at most
// one sample per voxel means nearly every sample reads voxels no other sample has touched -- a trip to HBM each --
// and the kernel is bound by how many of those an SM has in flight (vr_pipe.cu); denser views hit L1 and are bound
// by the texture / load pipe, where the extra registers buy nothing.
int auto_pipeline_depth(const vr_volume* v, const vr_camera* cam, int H, float step)
{
    double pitch;
    if (cam->projection == VR_PROJ_PERSPECTIVE) {
        double dist = 0.0;
        const double c[3] = {0.5 * ((v->part ? v->full[0] : v->desc.nx) - 1), 0.5 * ((v->part ? v->full[1] : v->desc.ny) - 1),
                             0.5 * ((v->part ? v->full[2] : v->desc.nz) - 1)};
        for (int a = 0; a < 3; ++a) dist += (c[a] - (double)cam->eye[a]) * (double)cam->forward[a];
        pitch = 2.0 * (double)cam->tan_half_fovy * std::fabs(dist) / (double)H;
    } else {
        pitch = 2.0 * (double)cam->ortho_half_height / (double)H;
    }
    const double samples_per_voxel = 1.0 / std::max(pitch * pitch * (double)step, 1e-30);
    return samples_per_voxel <= 1.0 ? 4 : 1;
}

struct Wall { int K, L; float* const* outs; };

// one brick / one part: the direct kernel, with pipelined loads when the depth says so
cudaError_t launch_brick_segment(const vr::FrameParams& P, int mode, bool count, bool tex, int depth, cudaStream_t s)
{
    if (depth > 1) return vr::launch_raycast_pipe(P, mode, count, true, tex, depth, s);
    return vr::launch_raycast(P, mode, false, count, true, tex, s);
}

vr_status render_resident(vr_volume* v, const vr_camera* cam, int W, int H, float step, int mode,
                          float* out, cudaStream_t s, const Wall* wall = nullptr)
{
    Range range(wall ? "vr_render_wall" : (mode == VR_MODE_EA ? "vr_render resident EA" : "vr_render resident MIP"));
    vr_status st = ensure_lut(v, step, mode, s);
    if (st != VR_OK) return st;
    const bool skip = v->opt_skip != 0;
    if (skip) {
        if ((st = ensure_minmax(v, s)) != VR_OK) return st;
        if ((st = ensure_skip(v, s)) != VR_OK) return st;
    }
    vr::FrameParams P;
    fill_frame(v, cam, W, H, step, (float4*)out, P);
    P.vol = resident_box(v);
    if (wall) {
        P.out = nullptr;
        P.wall_k = wall->K; P.wall_l = wall->L;
        P.wall_w = W / wall->K; P.wall_h = H / wall->L;
        for (int q = 0; q < wall->K * wall->L; ++q) P.wall_out[q] = (float4*)wall->outs[q];
    }
    if (v->opt_count) VR_CUDA(cudaMemsetAsync(v->d_counters, 0, 4 * sizeof(unsigned long long), s));
    // kernel choice (VR_OPT_KERNEL): 0 / 1 = direct kernel; 2 = beam kernel (experimental, opt-in only:
    // DESIGN.md Sec. 7) or VR_ERR_UNSUPPORTED where it cannot run
    const double diag = std::sqrt((double)P.n[0] * P.n[0] + (double)P.n[1] * P.n[1] + (double)P.n[2] * P.n[2]);
    // (empty-space skipping: the beam kernel skips whole slabs in EA; the MIP rule needs the ray's running maximum)
    const bool beam_ok = !P.aniso && beam_eligible(v) && (!skip || mode == VR_MODE_EA) && diag / (double)step < 4.0e6 && v->n_lut <= 1024 && !wall;
    if (v->opt_kernel == 2 && !beam_ok)
        return fail(VR_ERR_UNSUPPORTED, "vr_render: the beam kernel needs a resident VR_LAYOUT_LINEAR cube with nx %% 4 == 0, "
                    "no skipping in MIP mode, at most 1024 LUT entries, fewer than 4e6 samples per ray and a single frame buffer");
    // the automatic choice (0) takes the beam kernel where it can run only once kBeamIsDefault says it has been
    // validated on hardware
    if (v->opt_kernel == 2 || (v->opt_kernel == 0 && kBeamIsDefault && beam_ok)) {
        vr::BeamParams B = v->beam_params;
        B.use_skip = skip ? 1 : 0;
        if (B.stage_bytes <= 0) {
            // chosen from the camera alone: remember the last few (an orbit repeats its views)
            for (const vr_volume::StageChoice& c : v->stage_cache)
                if (c.W == W && c.H == H && c.pad_mode == B.pad_mode && std::memcmp(&c.cam, cam, sizeof(vr_camera)) == 0)
                    B.stage_bytes = c.stage_bytes;
            if (B.stage_bytes <= 0) {
                B.stage_bytes = vr::beam::auto_stage_bytes(P, B);
                if (v->stage_cache.size() >= 32) v->stage_cache.erase(v->stage_cache.begin());
                v->stage_cache.push_back({*cam, W, H, B.pad_mode, B.stage_bytes});
            }
        }
        VR_CUDA(vr::launch_raycast_beam(P, B, mode, v->opt_count != 0, s));
        v->stats.kernel = 2;
        v->stats.beam_stage_bytes = B.stage_bytes;
    } else {
        int depth = v->opt_pipeline ? v->opt_pipeline : auto_pipeline_depth(v, cam, H, step);
        if (skip) depth = 1;                  // the skipping loop walks min/max bricks sample by sample
        // VR_OPT_REUSE: dense views with short steps find most samples in the cell of the sample before (0 = automatic:
        // when the view is dense -- the pipelined kernel was not chosen -- and the step is at most 0.6 voxels)
        const bool reuse = !skip && depth == 1 && !wall &&
                           (v->opt_reuse == 2 || (v->opt_reuse == 0 && v->opt_pipeline == 0 && step <= 0.6f));
        if (reuse) {
            VR_CUDA(vr::launch_raycast_reuse(P, mode, v->opt_count != 0, v->tex, s));
            v->stats.kernel = 4;
        } else if (depth > 1) {
            VR_CUDA(vr::launch_raycast_pipe(P, mode, v->opt_count != 0, false, v->tex, depth, s));
            v->stats.kernel = 3;
        } else {
            VR_CUDA(vr::launch_raycast(P, mode, skip, v->opt_count != 0, false, v->tex, s));
            v->stats.kernel = 1;
        }
        v->stats.pipeline_depth = depth;
    }
    return VR_OK;
}

// S7 on the host: LUT cell of a value (same binary32 ops as dev::lut_coord)
int lut_cell(const vr_volume* v, float val)
{
    float xi = (val - v->vmin) * v->scale;
    xi = std::fmin(std::fmax(xi, 0.0f), (float)(v->n_lut - 1));
    return std::min((int)xi, v->n_lut - 2);
}

// EA: true iff alpha' = 0 over the whole guarded value range of the brick (the rule of skipbits_kernel, S9b):
// none of its samples can contribute, so the brick need not be fetched at all
bool brick_is_empty(const vr_volume* v, float2 mm)
{
    const float guard = std::fmax(std::fabs(mm.x), std::fabs(mm.y)) * 9.5367431640625e-07f;   // 2^-20
    const int qlo = std::max(lut_cell(v, mm.x - guard) - 1, 0);
    const int qhi = std::min(lut_cell(v, mm.y + guard) + 2, v->n_lut - 1);
    return v->h_prefix[(size_t)qhi + 1] - v->h_prefix[(size_t)qlo] == 0;
}

// Which slot takes a brick that is not resident.  Slots nothing has touched in this frame go first, the one used LAST
// in the frame before leading: with a view that changes little from frame to frame that is the brick farthest back --
// needed last, or not at all once the rays have saturated -- whereas the least recently used one is the next brick the
// frame will ask for.  When every slot has been touched in this frame the bricks pass through a ring of three.
int choose_victim(vr_volume* v)
{
    int best = -1;
    for (int q = 0; q < v->n_slots; ++q)
        if (!v->slot_used[q]) return q;
    for (int q = 0; q < v->n_slots; ++q)
        if (v->slot_frame[q] != v->frame_no && (best < 0 || v->slot_tick[q] > v->slot_tick[best])) best = q;
    if (best >= 0) return best;
    const int ring = std::min(3, v->n_slots);
    std::vector<int> idx((size_t)v->n_slots);
    for (int q = 0; q < v->n_slots; ++q) idx[(size_t)q] = q;
    std::partial_sort(idx.begin(), idx.begin() + ring, idx.end(),
                      [&](int a, int b) { return v->slot_tick[(size_t)a] > v->slot_tick[(size_t)b]; });
    return idx[(size_t)ring - 1];            // the oldest of the `ring` most recently used slots
}

cudaError_t timing_event(vr_volume* v, cudaEvent_t* out)
{
    if (v->n_tev == (int)v->tev.size()) {
        cudaEvent_t e = nullptr;
        cudaError_t err = cudaEventCreateWithFlags(&e, cudaEventDefault);
        if (err != cudaSuccess) return err;
        v->tev.push_back(e);
    }
    *out = v->tev[(size_t)v->n_tev++];
    return cudaSuccess;
}

vr_status render_streamed(vr_volume* v, const vr_camera* cam, int W, int H, float step, int mode,
                          float* out, cudaStream_t s)
{
    Range range(mode == VR_MODE_EA ? "vr_render streamed EA" : "vr_render streamed MIP");
    vr_status st = ensure_lut(v, step, mode, s);
    if (st != VR_OK) return st;
    const size_t npx = (size_t)W * (size_t)H;
    const bool comp = v->opt_compositor != 0;
    const bool cull = v->opt_cull != 0 && !comp;      // partial images start from zero: nothing saturates
    if (comp && v->partial_px < npx) {
        if (v->d_partial) VR_CUDA(cudaFree(v->d_partial));
        v->d_partial = nullptr;
        v->partial_px = 0;
        if (cudaMalloc(&v->d_partial, npx * sizeof(float4)) != cudaSuccess) {
            cudaGetLastError();
            return fail(VR_ERR_OOM_DEVICE, "vr_render: cannot allocate the partial image");
        }
        v->partial_px = npx;
    }
    // value ranges measured in earlier frames become usable once those frames have completed
    if (v->mm_in_flight && cull) {
        VR_CUDA(cudaEventSynchronize(v->ev_frame));
        for (char& c : v->brick_mm_state) if (c == 1) c = 2;
        v->mm_in_flight = false;
    }
    ++v->frame_no;
    v->n_tev = 0;
    VR_CUDA(cudaEventRecord(v->ev_f0, s));
    // running image R: EA (0,0,0,0); MIP (-inf, 0, 0, 0) until the final LUT pass
    if (mode == VR_MODE_EA) VR_CUDA(cudaMemsetAsync(out, 0, npx * sizeof(float4), s));
    else VR_CUDA(vr::launch_mip_init((float4*)out, W, H, s));
    if (v->opt_count) VR_CUDA(cudaMemsetAsync(v->d_counters, 0, 4 * sizeof(unsigned long long), s));

    std::vector<Keyed> order;
    order_bricks(v->nhb, v->hb, cam, order, v->spacing);
    const int depth = v->opt_pipeline ? v->opt_pipeline : auto_pipeline_depth(v, cam, H, step);
    v->stats.kernel = depth > 1 ? 3 : 1;
    v->stats.pipeline_depth = depth;

    vr::FrameParams P;
    fill_frame(v, cam, W, H, step, (float4*)out, P);
    v->stats.bricks_total = order.size();
    v->stats.bricks_streamed = v->stats.bricks_cached = v->stats.bricks_culled = v->stats.bricks_empty = 0;
    v->stats.h2d_bytes = 0;
    std::fill(v->brick_flags.begin(), v->brick_flags.end(), 0);
    const int n[3] = {v->desc.nx, v->desc.ny, v->desc.nz};

    struct Cand { int idx; int r[4]; int clo[3], chi[3]; };
    std::vector<Cand> wave;
    size_t pos = 0;
    while (pos < order.size()) {
        // one wavefront: the bricks of equal key (no ray crosses two of them, S11)
        const int key = order[pos].key;
        wave.clear();
        for (; pos < order.size() && order[pos].key == key; ++pos) {
            Cand c;
            c.idx = order[pos].idx;
            const int b[3] = {c.idx % v->nhb[0], (c.idx / v->nhb[0]) % v->nhb[1], c.idx / (v->nhb[0] * v->nhb[1])};
            double lo[3], hi[3];
            for (int a = 0; a < 3; ++a) {
                c.clo[a] = v->hb * b[a];
                c.chi[a] = std::min(v->hb * b[a] + v->hb, n[a] - 1);
                lo[a] = (double)c.clo[a] - 1.0;
                hi[a] = (double)c.chi[a] + 1.0;
            }
            if (!screen_bbox(cam, W, H, lo, hi, c.r, v->spacing)) { v->brick_flags[(size_t)c.idx] = VR_BRICK_OUTSIDE; continue; }
            if (cull && v->brick_mm_state[(size_t)c.idx] == 2 && mode == VR_MODE_EA &&
                brick_is_empty(v, v->h_brick_mm[c.idx])) {
                v->brick_flags[(size_t)c.idx] = VR_BRICK_EMPTY;
                ++v->stats.bricks_empty;
                continue;
            }
            wave.push_back(c);
        }
        if (wave.empty()) continue;
        if (cull) {
            // the smallest running opacity / maximum under each brick, as of everything enqueued so far
            VR_CUDA(vr::launch_fill(v->d_cull, wave.size(), INFINITY, s));
            for (size_t q = 0; q < wave.size(); ++q) {
                const Cand& c = wave[q];
                for (int a = 0; a < 3; ++a) { P.clo[a] = c.clo[a]; P.chi[a] = c.chi[a]; }
                P.x0 = c.r[0]; P.y0 = c.r[1]; P.x1 = c.r[2]; P.y1 = c.r[3];
                P.out = (float4*)out;
                VR_CUDA(vr::launch_cull_reduce(P, mode, v->d_cull + q, s));
            }
            VR_CUDA(cudaMemcpyAsync(v->h_cull, v->d_cull, wave.size() * sizeof(float), cudaMemcpyDeviceToHost, s));
            VR_CUDA(cudaEventRecord(v->ev_cull, s));
            VR_CUDA(cudaEventSynchronize(v->ev_cull));
        }
        for (size_t q = 0; q < wave.size(); ++q) {
            const Cand& c = wave[q];
            if (cull) {
                const float low = v->h_cull[q];          // +inf: no ray of the image can sample this brick
                bool needed;
                if (mode == VR_MODE_EA) {
                    needed = low < v->tau;
                } else {
                    needed = low < INFINITY;
                    if (needed && v->brick_mm_state[(size_t)c.idx] == 2) {
                        const float2 mm = v->h_brick_mm[c.idx];
                        const float guard = std::fmax(std::fabs(mm.x), std::fabs(mm.y)) * 9.5367431640625e-07f;
                        if (mm.y + guard <= low) needed = false;     // no sample of it can raise any ray's maximum (S9b)
                    }
                }
                if (!needed) {
                    v->brick_flags[(size_t)c.idx] = VR_BRICK_CULLED;
                    ++v->stats.bricks_culled;
                    continue;
                }
            }
            Range brick_range("brick");
            const HostBrick& hb = v->bricks[(size_t)c.idx];
            const size_t bytes = (size_t)hb.dims[0] * hb.dims[1] * hb.dims[2] * sizeof(float);
            int slot = v->opt_cache ? v->brick_slot[(size_t)c.idx] : -1;
            const bool hit = slot >= 0;
            if (!hit) {
                slot = choose_victim(v);
                if (v->slot_used[(size_t)slot]) VR_CUDA(cudaStreamWaitEvent(v->copy_stream, v->ev_free[(size_t)slot], 0));
                if (v->slot_brick[(size_t)slot] >= 0) v->brick_slot[(size_t)v->slot_brick[(size_t)slot]] = -1;
                v->slot_brick[(size_t)slot] = c.idx;
                v->brick_slot[(size_t)c.idx] = slot;
                cudaEvent_t t0 = nullptr, t1 = nullptr;
                VR_CUDA(timing_event(v, &t0));
                VR_CUDA(timing_event(v, &t1));
                VR_CUDA(cudaEventRecord(t0, v->copy_stream));
                if (v->tex) {
                    // the brick becomes texels [0, dims) of the slot's layered array
                    const int zero[3] = {0, 0, 0};
                    VR_CUDA(copy_box_to_array(v->slot_arr[(size_t)slot], zero, hb.dims, hb.ptr, cudaMemcpyHostToDevice, v->copy_stream));
                } else {
                    float* d_slot = (float*)((char*)v->desc.d_storage + (size_t)slot * v->slot_bytes);
                    VR_CUDA(cudaMemcpyAsync(d_slot, hb.ptr, bytes, cudaMemcpyHostToDevice, v->copy_stream));
                    if (v->blank)
                        VR_CUDA(vr::launch_blank(d_slot, hb.dims, (long long)hb.dims[0], (long long)hb.dims[0] * hb.dims[1],
                                                 v->blank_value, v->copy_stream));
                }
                VR_CUDA(cudaEventRecord(t1, v->copy_stream));
                VR_CUDA(cudaEventRecord(v->ev_copied[(size_t)slot], v->copy_stream));
                ++v->stats.bricks_streamed;
                v->stats.h2d_bytes += bytes;
                v->brick_flags[(size_t)c.idx] = VR_BRICK_STREAMED;
            } else {
                ++v->stats.bricks_cached;
                v->brick_flags[(size_t)c.idx] = VR_BRICK_CACHED;
            }
            v->slot_used[(size_t)slot] = 1;
            v->slot_tick[(size_t)slot] = ++v->tick;
            v->slot_frame[(size_t)slot] = v->frame_no;
            float* d_first = nullptr;
            if (v->tex) {
                P.vol.tex[0] = v->slot_tex[(size_t)slot];
                P.vol.n_chunks = 1;
                P.vol.gx = (float)(1 - hb.origin[0]);
                P.vol.gy = (float)(1 - hb.origin[1]);
                P.vol.org_z = hb.origin[2];
            } else {
                d_first = (float*)((char*)v->desc.d_storage + (size_t)slot * v->slot_bytes);
                // global voxel (x,y,z) -> slot[(z-oz)*sz + (y-oy)*sy + (x-ox)]
                P.vol.sy = hb.dims[0];
                P.vol.sz = (long long)hb.dims[0] * hb.dims[1];
                const long long off = (long long)hb.origin[2] * P.vol.sz + (long long)hb.origin[1] * P.vol.sy + hb.origin[0];
                P.vol.base = (const float*)((uintptr_t)d_first - (uintptr_t)(off * (long long)sizeof(float)));
            }
            VR_CUDA(cudaStreamWaitEvent(s, v->ev_copied[(size_t)slot], 0));
            if (v->brick_mm_state[(size_t)c.idx] == 0 && v->opt_cull) {
                // first time on the device: its value range, mirrored to the host for the frames to come
                float* d_mm = reinterpret_cast<float*>(v->d_brick_mm + c.idx);
                VR_CUDA(vr::launch_fill(d_mm, 1, INFINITY, s));
                VR_CUDA(vr::launch_fill(d_mm + 1, 1, -INFINITY, s));
                VR_CUDA(vr::launch_brick_range(d_first, v->tex ? v->slot_tex[(size_t)slot] : 0, v->tex, hb.dims, d_mm, s));
                VR_CUDA(cudaMemcpyAsync(v->h_brick_mm + c.idx, v->d_brick_mm + c.idx, sizeof(float2), cudaMemcpyDeviceToHost, s));
                v->brick_mm_state[(size_t)c.idx] = 1;
                v->mm_in_flight = true;
            }
            for (int a = 0; a < 3; ++a) { P.clo[a] = c.clo[a]; P.chi[a] = c.chi[a]; }
            P.x0 = c.r[0]; P.y0 = c.r[1]; P.x1 = c.r[2]; P.y1 = c.r[3];
            P.tiles_x = ceil_div(c.r[2] - c.r[0], vr::kTileW);
            P.tiles_y = ceil_div(c.r[3] - c.r[1], vr::kTileH);
            if (!comp) {
                P.out = (float4*)out;
                P.fresh = 0;
                VR_CUDA(launch_brick_segment(P, mode, v->opt_count != 0, v->tex, depth, s));
            } else {
                P.out = v->d_partial;
                P.fresh = 1;
                VR_CUDA(launch_brick_segment(P, mode, v->opt_count != 0, v->tex, depth, s));
                VR_CUDA(vr::launch_composite((float4*)out, v->d_partial, W, c.r[0], c.r[1], c.r[2], c.r[3], mode, s));
            }
            VR_CUDA(cudaEventRecord(v->ev_free[(size_t)slot], s));
        }
    }
    if (mode == VR_MODE_MIP) {
        P.out = (float4*)out;
        VR_CUDA(vr::launch_mip_finish(P, s));
    } else if (v->d_aux) {
        // EA has no raw maximum: aux = -inf, as for resident volumes
        VR_CUDA(vr::launch_fill(v->d_aux, npx, -INFINITY, s));
    }
    VR_CUDA(cudaEventRecord(v->ev_f1, s));
    VR_CUDA(cudaEventRecord(v->ev_frame, s));
    v->stats.timing_valid = 0;
    return VR_OK;
}

// A part of a cube renders the PARTIAL image of the cells it owns, from zero (S13): EA premultiplied (C, A); MIP the raw
// maximum in .x (-inf where the part has no sample), to be combined with vr_composite and finished by vr_mip_finish
vr_status render_part(vr_volume* v, const vr_camera* cam, int W, int H, float step, int mode, float* out, cudaStream_t s)
{
    if (v->opt_skip) return fail(VR_ERR_UNSUPPORTED, "vr_render: no empty-space skipping on a part of a cube");
    if (v->opt_kernel == 2) return fail(VR_ERR_UNSUPPORTED, "vr_render: the beam kernel does not render parts of a cube");
    vr_status st = ensure_lut(v, step, mode, s);
    if (st != VR_OK) return st;
    const size_t npx = (size_t)W * (size_t)H;
    if (mode == VR_MODE_EA) VR_CUDA(cudaMemsetAsync(out, 0, npx * sizeof(float4), s));
    else VR_CUDA(vr::launch_mip_init((float4*)out, W, H, s));
    if (v->opt_count) VR_CUDA(cudaMemsetAsync(v->d_counters, 0, 4 * sizeof(unsigned long long), s));
    vr::FrameParams P;
    fill_frame(v, cam, W, H, step, (float4*)out, P);
    P.vol = resident_box(v);
    const int dims[3] = {v->desc.nx, v->desc.ny, v->desc.nz};
    double lo[3], hi[3];
    for (int c = 0; c < 3; ++c) {
        P.n[c] = v->full[c];                                 // rays are clipped against the whole cube (global k, S10)
        P.clo[c] = v->p_org[c];
        P.chi[c] = std::min(v->p_org[c] + dims[c] - 1, v->full[c] - 1);
        lo[c] = (double)P.clo[c] - 1.0;
        hi[c] = (double)P.chi[c] + 1.0;
    }
    if (v->tex) {
        P.vol.gx = (float)(1 - v->p_org[0]);
        P.vol.gy = (float)(1 - v->p_org[1]);
        P.vol.org_z = v->p_org[2];
    } else {
        const long long off = (long long)v->p_org[2] * P.vol.sz + (long long)v->p_org[1] * P.vol.sy + v->p_org[0];
        P.vol.base = (const float*)((uintptr_t)P.vol.base - (uintptr_t)(off * (long long)sizeof(float)));
    }
    int r[4];
    v->stats.kernel = 1;
    v->stats.pipeline_depth = 1;
    if (!screen_bbox(cam, W, H, lo, hi, r, v->spacing)) return VR_OK;      // the part is outside the frustum: an empty partial image
    P.x0 = r[0]; P.y0 = r[1]; P.x1 = r[2]; P.y1 = r[3];
    P.tiles_x = ceil_div(r[2] - r[0], vr::kTileW);
    P.tiles_y = ceil_div(r[3] - r[1], vr::kTileH);
    P.fresh = 1;
    P.aux = nullptr;
    const int depth = v->opt_pipeline ? v->opt_pipeline : auto_pipeline_depth(v, cam, H, step);
    VR_CUDA(launch_brick_segment(P, mode, v->opt_count != 0, v->tex, depth, s));
    v->stats.kernel = depth > 1 ? 3 : 1;
    v->stats.pipeline_depth = depth;
    return VR_OK;
}

}  // namespace

extern "C" {

const char* vr_last_error(void) { return g_err; }

const char* vr_version(void) { return "vr-b200 0.1 (sm_100a)"; }

size_t vr_volume_storage_bytes(const vr_volume_desc* d)
{
    if (!valid_dims(d) || d->layout == VR_LAYOUT_TEX) return 0;
    if (d->host_brick > 0) return 2 * vr_volume_slot_bytes(d);
    return (size_t)d->nx * (size_t)d->ny * (size_t)d->nz * sizeof(float);
}

size_t vr_volume_slot_bytes(const vr_volume_desc* d)
{
    if (!valid_dims(d) || d->host_brick <= 0 || d->layout == VR_LAYOUT_TEX) return 0;
    return round_up(brick_voxels_max(d) * sizeof(float), 256);
}

vr_status vr_volume_create(const vr_volume_desc* d, vr_volume** out)
{
    if (out) *out = nullptr;
    if (!out || !d) return fail(VR_ERR_INVALID_ARG, "vr_volume_create: null argument");
    if (!valid_dims(d)) return fail(VR_ERR_INVALID_ARG, "vr_volume_create: every extent must be >= 2");
    if (d->layout != VR_LAYOUT_LINEAR && d->layout != VR_LAYOUT_TEX)
        return fail(VR_ERR_INVALID_ARG, "vr_volume_create: unknown layout %d", d->layout);
    const bool tex = d->layout == VR_LAYOUT_TEX;
    if (tex) {
        const int B1 = d->host_brick + 1;
        const int ext[3] = {d->host_brick ? std::min(B1, d->nx) : d->nx, d->host_brick ? std::min(B1, d->ny) : d->ny,
                            d->host_brick ? std::min(B1, d->nz) : d->nz};
        const int max_z = d->host_brick ? kMaxLayers : (tex_max_layers() - 1) * vr::kMaxTexChunks + 1;
        if (ext[0] > kMaxTexExtent || ext[1] > kMaxTexExtent || ext[2] > max_z)
            return fail(VR_ERR_UNSUPPORTED, "vr_volume_create: VR_LAYOUT_TEX holds at most %d x %d x %d voxels "
                        "(%d x %d x %d asked); use bricks or VR_LAYOUT_LINEAR", kMaxTexExtent, kMaxTexExtent, max_z,
                        ext[0], ext[1], ext[2]);
        if (d->host_brick && d->n_slots < 2)
            return fail(VR_ERR_INVALID_ARG, "vr_volume_create: a streamed VR_LAYOUT_TEX volume needs n_slots >= 2");
    } else {
        if (!d->d_storage) return fail(VR_ERR_INVALID_ARG, "vr_volume_create: d_storage is null");
        if (((uintptr_t)d->d_storage & 255u) != 0)
            return fail(VR_ERR_INVALID_ARG, "vr_volume_create: d_storage must be 256-byte aligned");
    }
    const int mmB = d->mm_brick ? d->mm_brick : 64;
    if (mmB < 2 || (mmB & (mmB - 1)) != 0)
        return fail(VR_ERR_INVALID_ARG, "vr_volume_create: mm_brick must be a power of two >= 2");
    const size_t need = vr_volume_storage_bytes(d);
    if (d->d_storage_bytes < need)
        return fail(VR_ERR_OOM_DEVICE, "vr_volume_create: d_storage has %zu bytes, %zu needed",
                    d->d_storage_bytes, need);
    int ndev = 0;
    VR_CUDA(cudaGetDeviceCount(&ndev));
    if (d->device < 0 || d->device >= ndev)
        return fail(VR_ERR_INVALID_ARG, "vr_volume_create: no CUDA device %d", d->device);
    VR_CUDA(cudaSetDevice(d->device));

    vr_volume* v = new (std::nothrow) vr_volume();
    if (!v) return fail(VR_ERR_OOM_HOST, "vr_volume_create: out of host memory");
    v->desc = *d;
    v->streamed = d->host_brick > 0;
    v->tex = tex;
    vr::beam::default_params(v->beam_params);
    v->beam_params.stage_bytes = 0;      // chosen per frame (auto_stage_bytes)

    cudaError_t e = alloc_mm_tables(v, mmB);
    auto alloc = [&](void** p, size_t bytes) {
        if (e == cudaSuccess) e = cudaMalloc(p, bytes);
    };
    alloc((void**)&v->d_nzprefix, sizeof(int) * (vr::kMaxLut + 1));
    alloc((void**)&v->d_nskip, sizeof(unsigned int));
    alloc((void**)&v->d_lut, sizeof(float4) * 2 * vr::kMaxLut);
    alloc((void**)&v->d_lut_grey, sizeof(float4) * vr::kMaxLut);
    alloc((void**)&v->d_counters, 4 * sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaMemset(v->d_counters, 0, 4 * sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaMemset(v->d_nskip, 0, sizeof(unsigned int));
    if (e == cudaSuccess && v->streamed) {
        v->hb = d->host_brick;
        v->nhb[0] = ceil_div(d->nx - 1, v->hb);
        v->nhb[1] = ceil_div(d->ny - 1, v->hb);
        v->nhb[2] = ceil_div(d->nz - 1, v->hb);
        v->bricks.assign((size_t)v->nhb[0] * v->nhb[1] * v->nhb[2], HostBrick());
        v->slot_bytes = tex ? round_up(brick_voxels_max(d) * sizeof(float), 256) : vr_volume_slot_bytes(d);
        v->n_slots = tex ? std::min(d->n_slots, kMaxSlots) : (int)std::min<size_t>(d->d_storage_bytes / v->slot_bytes, (size_t)kMaxSlots);
        v->stats.n_slots = v->n_slots;
        v->stats.bricks_total = v->bricks.size();
        e = cudaStreamCreateWithFlags(&v->copy_stream, cudaStreamNonBlocking);
        v->ev_copied.assign((size_t)v->n_slots, nullptr);
        v->ev_free.assign((size_t)v->n_slots, nullptr);
        v->slot_used.assign((size_t)v->n_slots, 0);
        v->slot_brick.assign((size_t)v->n_slots, -1);
        v->slot_tick.assign((size_t)v->n_slots, 0);
        v->slot_frame.assign((size_t)v->n_slots, 0);
        v->brick_slot.assign(v->bricks.size(), -1);
        v->brick_mm_state.assign(v->bricks.size(), 0);
        v->brick_flags.assign(v->bricks.size(), 0);
        if (e == cudaSuccess) e = cudaMalloc((void**)&v->d_brick_mm, sizeof(float2) * v->bricks.size());
        if (e == cudaSuccess) e = cudaHostAlloc((void**)&v->h_brick_mm, sizeof(float2) * v->bricks.size(), cudaHostAllocDefault);
        if (e == cudaSuccess) e = cudaMalloc((void**)&v->d_cull, sizeof(float) * v->bricks.size());
        if (e == cudaSuccess) e = cudaHostAlloc((void**)&v->h_cull, sizeof(float) * v->bricks.size(), cudaHostAllocDefault);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&v->ev_frame, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&v->ev_cull, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&v->ev_f0, cudaEventDefault);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&v->ev_f1, cudaEventDefault);
        for (int q = 0; q < v->n_slots && e == cudaSuccess; ++q) {
            e = cudaEventCreateWithFlags(&v->ev_copied[q], cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&v->ev_free[q], cudaEventDisableTiming);
        }
        if (tex) {
            const int B1 = v->hb + 1;
            v->slot_arr.assign((size_t)v->n_slots, nullptr);
            v->slot_tex.assign((size_t)v->n_slots, 0);
            for (int q = 0; q < v->n_slots && e == cudaSuccess; ++q)
                e = make_layered(std::min(B1, d->nx), std::min(B1, d->ny), std::min(B1, d->nz),
                                 &v->slot_arr[q], &v->slot_tex[q]);
        }
    } else if (e == cudaSuccess && tex) {
        // z chunks of at most L layers; neighbours share one layer so that every cell finds both of its layers in one
        const int L = tex_max_layers();
        v->chunk_step = d->nz <= L ? d->nz : L - 1;
        const int n_chunks = d->nz <= L ? 1 : ceil_div(d->nz - 1, L - 1);
        v->chunk_arr.assign((size_t)n_chunks, nullptr);
        v->chunk_tex.assign((size_t)n_chunks, 0);
        for (int c = 0; c < n_chunks && e == cudaSuccess; ++c)
            e = make_layered(d->nx, d->ny, std::min(v->chunk_step + 1, d->nz - c * v->chunk_step),
                             &v->chunk_arr[(size_t)c], &v->chunk_tex[(size_t)c]);
    }
    if (e != cudaSuccess) {
        const vr_status st = fail(e == cudaErrorMemoryAllocation ? VR_ERR_OOM_DEVICE : VR_ERR_CUDA,
                                  "vr_volume_create: %s", cudaGetErrorString(e));
        cudaGetLastError();
        vr_volume_destroy(v);
        return st;
    }
    *out = v;
    return VR_OK;
}

vr_status vr_volume_create_part(const vr_volume_desc* whole, const int origin[3], const int dims[3], vr_volume** out)
{
    if (out) *out = nullptr;
    if (!out || !whole || !origin || !dims) return fail(VR_ERR_INVALID_ARG, "vr_volume_create_part: null argument");
    if (!valid_dims(whole) || whole->host_brick != 0)
        return fail(VR_ERR_INVALID_ARG, "vr_volume_create_part: `whole` must describe a resident cube");
    const int N[3] = {whole->nx, whole->ny, whole->nz};
    for (int c = 0; c < 3; ++c)
        if (origin[c] < 0 || dims[c] < 2 || origin[c] + dims[c] > N[c])
            return fail(VR_ERR_INVALID_ARG, "vr_volume_create_part: the part must hold >= 2 voxels per axis inside the cube");
    if (whole->layout == VR_LAYOUT_TEX && dims[2] > tex_max_layers())
        return fail(VR_ERR_UNSUPPORTED, "vr_volume_create_part: a VR_LAYOUT_TEX part holds at most %d layers (one array); "
                    "cut the cube into more parts or use VR_LAYOUT_LINEAR", tex_max_layers());
    vr_volume_desc d = *whole;
    d.nx = dims[0]; d.ny = dims[1]; d.nz = dims[2];
    vr_volume* v = nullptr;
    vr_status st = vr_volume_create(&d, &v);
    if (st != VR_OK) return st;
    v->part = true;
    for (int c = 0; c < 3; ++c) { v->full[c] = N[c]; v->p_org[c] = origin[c]; }
    *out = v;
    return VR_OK;
}

vr_status vr_composite(float* running, const float* partial, int W, int H, int mode, void* stream)
{
    if (!running || !partial || W < 1 || H < 1 || (mode != VR_MODE_EA && mode != VR_MODE_MIP))
        return fail(VR_ERR_INVALID_ARG, "vr_composite: bad argument");
    VR_CUDA(vr::launch_composite((float4*)running, (const float4*)partial, W, 0, 0, W, H, mode, (cudaStream_t)stream));
    return VR_OK;
}

vr_status vr_mip_finish(vr_volume* v, float* running, int W, int H, void* stream)
{
    if (!v || !running || W < 1 || H < 1) return fail(VR_ERR_INVALID_ARG, "vr_mip_finish: bad argument");
    if (v->n_lut < 2) return fail(VR_ERR_STATE, "vr_mip_finish: no transfer function set");
    VR_CUDA(cudaSetDevice(v->desc.device));
    cudaStream_t s = (cudaStream_t)stream;
    vr_status st = ensure_lut(v, v->lut_valid ? v->lut_step : 1.0f, VR_MODE_MIP, s);   // MIP reads the colours only
    if (st != VR_OK) return st;
    vr::FrameParams P;
    std::memset(&P, 0, sizeof(P));
    P.W = W; P.H = H;
    P.lut = v->d_lut;
    P.n_lut = v->n_lut;
    P.vmin = v->vmin;
    P.scale = v->scale;
    P.out = (float4*)running;
    P.aux = v->d_aux;
    VR_CUDA(vr::launch_mip_finish(P, s));
    return VR_OK;
}

void vr_volume_destroy(vr_volume* v)
{
    if (!v) return;
    cudaSetDevice(v->desc.device);
    if (v->copy_stream) {
        cudaStreamSynchronize(v->copy_stream);
        cudaStreamDestroy(v->copy_stream);
    }
    for (cudaEvent_t ev : v->ev_copied) if (ev) cudaEventDestroy(ev);
    for (cudaEvent_t ev : v->ev_free) if (ev) cudaEventDestroy(ev);
    for (cudaEvent_t ev : v->tev) if (ev) cudaEventDestroy(ev);
    for (cudaEvent_t ev : {v->ev_frame, v->ev_cull, v->ev_f0, v->ev_f1}) if (ev) cudaEventDestroy(ev);
    cudaFree(v->d_brick_mm);
    cudaFree(v->d_cull);
    if (v->h_brick_mm) cudaFreeHost(v->h_brick_mm);
    if (v->h_cull) cudaFreeHost(v->h_cull);
    cudaFree(v->d_minmax);
    cudaFree(v->d_skip);
    cudaFree(v->d_minmax2);
    cudaFree(v->d_skip2);
    cudaFree(v->d_nzprefix);
    cudaFree(v->d_nskip);
    cudaFree(v->d_lut);
    cudaFree(v->d_lut_grey);
    cudaFree(v->d_counters);
    cudaFree(v->d_partial);
    for (cudaTextureObject_t t : v->chunk_tex) if (t) cudaDestroyTextureObject(t);
    for (cudaArray_t a : v->chunk_arr) if (a) cudaFreeArray(a);
    for (cudaTextureObject_t t : v->slot_tex) if (t) cudaDestroyTextureObject(t);
    for (cudaArray_t a : v->slot_arr) if (a) cudaFreeArray(a);
    delete v;
}

vr_status vr_volume_upload_bricks(vr_volume* v, int n, const int (*origin)[3], const int (*dims)[3],
                                  const float* const* ptrs, int ptrs_are_device, void* stream)
{
    if (!v || !origin || !dims || !ptrs || n < 1)
        return fail(VR_ERR_INVALID_ARG, "vr_volume_upload_bricks: null argument or n < 1");
    Range range("vr_volume_upload_bricks");
    cudaStream_t s = (cudaStream_t)stream;
    const int N[3] = {v->desc.nx, v->desc.ny, v->desc.nz};
    // a part of a cube takes boxes in the CUBE's coordinates; inside, everything is relative to the part
    std::vector<int> local;
    if (v->part) {
        local.resize((size_t)3 * n);
        for (int q = 0; q < n; ++q)
            for (int c = 0; c < 3; ++c) local[(size_t)3 * q + c] = origin[q][c] - v->p_org[c];
        origin = reinterpret_cast<const int (*)[3]>(local.data());
    }
    for (int q = 0; q < n; ++q) {
        if (!ptrs[q]) return fail(VR_ERR_INVALID_ARG, "vr_volume_upload_bricks: box %d has a null pointer", q);
        for (int c = 0; c < 3; ++c)
            if (origin[q][c] < 0 || dims[q][c] < 1 || origin[q][c] + dims[q][c] > N[c])
                return fail(VR_ERR_INVALID_ARG, "vr_volume_upload_bricks: box %d leaves the %s", q, v->part ? "part" : "cube");
    }
    VR_CUDA(cudaSetDevice(v->desc.device));
    if (v->blank && v->tex)
        return fail(VR_ERR_UNSUPPORTED, "vr_volume_upload_bricks: blanking of non-finite voxels needs VR_LAYOUT_LINEAR");
    if (v->streamed) {
        if (ptrs_are_device)
            return fail(VR_ERR_INVALID_ARG, "vr_volume_upload_bricks: streamed bricks must be host pointers");
        for (int q = 0; q < n; ++q) {
            int b[3];
            for (int c = 0; c < 3; ++c) {
                if (origin[q][c] % v->hb != 0)
                    return fail(VR_ERR_INVALID_ARG, "vr_volume_upload_bricks: box %d is not brick aligned", q);
                b[c] = origin[q][c] / v->hb;
                const int want = std::min(v->hb * b[c] + v->hb, N[c] - 1) - v->hb * b[c] + 1;
                if (b[c] >= v->nhb[c] || dims[q][c] != want)
                    return fail(VR_ERR_INVALID_ARG,
                                "vr_volume_upload_bricks: box %d must hold %d voxels on axis %d (brick + ghost layer)",
                                q, want, c);
            }
            HostBrick& hb = v->bricks[(size_t)b[0] + (size_t)v->nhb[0] * ((size_t)b[1] + (size_t)v->nhb[1] * b[2])];
            hb.ptr = ptrs[q];
            for (int c = 0; c < 3; ++c) { hb.origin[c] = origin[q][c]; hb.dims[c] = dims[q][c]; }
            // a brick registered again may hold new voxels: forget its device copy and its value range
            const size_t bi = (size_t)b[0] + (size_t)v->nhb[0] * ((size_t)b[1] + (size_t)v->nhb[1] * b[2]);
            if (v->brick_slot[bi] >= 0) { v->slot_brick[(size_t)v->brick_slot[bi]] = -1; v->brick_slot[bi] = -1; }
            v->brick_mm_state[bi] = 0;
        }
        bool all = true;
        for (const HostBrick& hb : v->bricks) all = all && hb.ptr != nullptr;
        v->uploaded = all;
        return VR_OK;
    }
    for (int q = 0; q < n; ++q) {
        const bool whole = origin[q][0] == 0 && origin[q][1] == 0 && origin[q][2] == 0 &&
                           dims[q][0] == N[0] && dims[q][1] == N[1] && dims[q][2] == N[2];
        const cudaMemcpyKind kind = ptrs_are_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
        if (v->tex) {
            // every chunk takes the layers of the box it holds (a shared layer goes to both neighbours)
            for (int c = 0; c < (int)v->chunk_arr.size(); ++c) {
                const int c0 = c * v->chunk_step, c1 = std::min(c0 + v->chunk_step, N[2] - 1);   // layers [c0, c1]
                const int z0 = std::max(origin[q][2], c0), z1 = std::min(origin[q][2] + dims[q][2] - 1, c1);
                if (z0 > z1) continue;
                const int pos[3] = {origin[q][0], origin[q][1], z0 - c0};
                const int ext[3] = {dims[q][0], dims[q][1], z1 - z0 + 1};
                const float* src = ptrs[q] + (size_t)(z0 - origin[q][2]) * (size_t)dims[q][0] * (size_t)dims[q][1];
                VR_CUDA(copy_box_to_array(v->chunk_arr[(size_t)c], pos, ext, src, kind, s));
            }
        } else if (whole) {
            if ((const void*)ptrs[q] != v->desc.d_storage)
                VR_CUDA(cudaMemcpyAsync(v->desc.d_storage, ptrs[q],
                                        (size_t)N[0] * N[1] * N[2] * sizeof(float), kind, s));
        } else {
            cudaMemcpy3DParms p{};
            p.srcPtr = make_cudaPitchedPtr((void*)ptrs[q], (size_t)dims[q][0] * sizeof(float),
                                           (size_t)dims[q][0], (size_t)dims[q][1]);
            p.dstPtr = make_cudaPitchedPtr(v->desc.d_storage, (size_t)N[0] * sizeof(float),
                                           (size_t)N[0], (size_t)N[1]);
            p.dstPos = make_cudaPos((size_t)origin[q][0] * sizeof(float), (size_t)origin[q][1],
                                    (size_t)origin[q][2]);
            p.extent = make_cudaExtent((size_t)dims[q][0] * sizeof(float), (size_t)dims[q][1],
                                       (size_t)dims[q][2]);
            p.kind = kind;
            VR_CUDA(cudaMemcpy3DAsync(&p, s));
        }
        if (v->blank && !v->tex) {
            float* first = (float*)v->desc.d_storage + ((size_t)origin[q][2] * N[1] + (size_t)origin[q][1]) * N[0] + origin[q][0];
            VR_CUDA(vr::launch_blank(first, dims[q], (long long)N[0], (long long)N[0] * N[1], v->blank_value, s));
        }
    }
    v->uploaded = true;
    v->minmax_valid = false;
    v->skip_valid = false;
    return VR_OK;
}

vr_status vr_set_transfer_function(vr_volume* v, const float* lut, int n, float vmin, float vmax)
{
    if (!v || !lut) return fail(VR_ERR_INVALID_ARG, "vr_set_transfer_function: null argument");
    if (n < 2 || n > vr::kMaxLut)
        return fail(VR_ERR_INVALID_ARG, "vr_set_transfer_function: n_entries must be in [2, %d]", vr::kMaxLut);
    if (!std::isfinite(vmin) || !std::isfinite(vmax) || !(vmax > vmin))
        return fail(VR_ERR_INVALID_ARG, "vr_set_transfer_function: need finite vmin < vmax");
    for (int i = 0; i < 4 * n; ++i)
        if (!std::isfinite(lut[i])) return fail(VR_ERR_INVALID_ARG, "vr_set_transfer_function: non-finite entry");
    v->lut.assign(lut, lut + (size_t)4 * n);
    v->n_lut = n;
    v->vmin = vmin;
    v->vmax = vmax;
    v->scale = (float)((double)(n - 1) / ((double)vmax - (double)vmin));
    v->lut_valid = false;
    v->skip_valid = false;
    return VR_OK;
}

vr_status vr_set_option(vr_volume* v, int key, double value)
{
    if (!v) return fail(VR_ERR_INVALID_ARG, "vr_set_option: null handle");
    switch (key) {
    case VR_OPT_ERT_TAU:
        if (!(value > 0.0)) return fail(VR_ERR_INVALID_ARG, "vr_set_option: tau must be > 0");
        v->tau = (float)value;
        return VR_OK;
    case VR_OPT_SKIP:
        if (v->streamed && value != 0.0)
            return fail(VR_ERR_UNSUPPORTED, "vr_set_option: min/max skipping is for resident volumes");
        v->opt_skip = value != 0.0;
        return VR_OK;
    case VR_OPT_KERNEL:
        if (value != 0.0 && value != 1.0 && value != 2.0) return fail(VR_ERR_INVALID_ARG, "vr_set_option: kernel must be 0, 1 or 2");
        v->opt_kernel = (int)value;
        return VR_OK;
    case VR_OPT_COUNT: v->opt_count = value != 0.0; return VR_OK;
    case VR_OPT_COMPOSITOR:
        if (!v->streamed && value != 0.0)
            return fail(VR_ERR_UNSUPPORTED, "vr_set_option: compositor mode is for streamed volumes");
        v->opt_compositor = value != 0.0;
        return VR_OK;
    case VR_OPT_BEAM_STAGE:
        if (value != 0.0 && (!(value >= 4096.0 && value <= 196608.0) || ((long long)value & 15) != 0))
            return fail(VR_ERR_INVALID_ARG, "vr_set_option: the beam stage must be 0 (automatic) or a multiple of 16 in "
                        "[4096, 196608] bytes");
        v->beam_params.stage_bytes = (int)value;
        return VR_OK;
    case VR_OPT_BEAM_PAD:
        if (value != 0.0 && value != 1.0) return fail(VR_ERR_INVALID_ARG, "vr_set_option: beam padding must be 0 or 1");
        v->beam_params.pad_mode = (int)value;
        return VR_OK;
    case VR_OPT_BEAM_BULK:
        if (value != 0.0 && value != 1.0) return fail(VR_ERR_INVALID_ARG, "vr_set_option: beam bulk copies must be 0 or 1");
        v->beam_params.bulk = (int)value;
        return VR_OK;
    case VR_OPT_BEAM_STAGES:
        if (value != 1.0 && value != 2.0) return fail(VR_ERR_INVALID_ARG, "vr_set_option: beam stages must be 1 or 2");
        v->beam_params.n_stages = (int)value;
        return VR_OK;
    case VR_OPT_MM_BRICK: {
        const int B = (int)value;
        if (v->streamed) return fail(VR_ERR_UNSUPPORTED, "vr_set_option: the min/max table is for resident volumes");
        if ((double)B != value || B < 2 || B > 4096 || (B & (B - 1)) != 0)
            return fail(VR_ERR_INVALID_ARG, "vr_set_option: the min/max brick edge must be a power of two in [2, 4096]");
        if (B == v->mm_B) return VR_OK;
        VR_CUDA(cudaSetDevice(v->desc.device));
        VR_CUDA(cudaDeviceSynchronize());      // frames in flight still read the old tables
        const cudaError_t e = alloc_mm_tables(v, B);
        if (e != cudaSuccess) {
            cudaGetLastError();
            return fail(e == cudaErrorMemoryAllocation ? VR_ERR_OOM_DEVICE : VR_ERR_CUDA, "vr_set_option: %s", cudaGetErrorString(e));
        }
        return VR_OK;
    }
    case VR_OPT_BLANK_VALUE:
        // NaN switches blanking off; a finite value switches it on for the voxels uploaded / streamed from now on
        if (std::isinf(value)) return fail(VR_ERR_INVALID_ARG, "vr_set_option: the blank value must be finite (NaN = off)");
        if (!std::isnan(value) && v->tex)
            return fail(VR_ERR_UNSUPPORTED, "vr_set_option: blanking of non-finite voxels needs VR_LAYOUT_LINEAR");
        v->blank = !std::isnan(value);
        v->blank_value = v->blank ? (float)value : 0.f;
        if (v->streamed) {       // cached bricks and measured ranges were made under the old setting
            for (size_t q = 0; q < v->brick_slot.size(); ++q) {
                if (v->brick_slot[q] >= 0) { v->slot_brick[(size_t)v->brick_slot[q]] = -1; v->brick_slot[q] = -1; }
                v->brick_mm_state[q] = 0;
            }
        }
        return VR_OK;
    case VR_OPT_REUSE:
        if (value != 0.0 && value != 1.0 && value != 2.0)
            return fail(VR_ERR_INVALID_ARG, "vr_set_option: cell reuse must be 0 (automatic), 1 (off) or 2 (on)");
        v->opt_reuse = (int)value;
        return VR_OK;
    case VR_OPT_SPACING_X:
    case VR_OPT_SPACING_Y:
    case VR_OPT_SPACING_Z:
        if (!(value > 0.0) || !std::isfinite(value) || !((float)value > 0.0f) || !std::isfinite((float)value))
            return fail(VR_ERR_INVALID_ARG, "vr_set_option: the voxel spacing must be finite and > 0");
        v->spacing[key - VR_OPT_SPACING_X] = (float)value;
        return VR_OK;
    case VR_OPT_PIPELINE:
        if (value != 0.0 && value != 1.0 && value != 2.0 && value != 4.0)
            return fail(VR_ERR_INVALID_ARG, "vr_set_option: pipeline depth must be 0 (automatic), 1, 2 or 4");
        v->opt_pipeline = (int)value;
        return VR_OK;
    case VR_OPT_TILE_ORDER:
        if (value != 0.0 && value != 1.0) return fail(VR_ERR_INVALID_ARG, "vr_set_option: tile order must be 0 or 1");
        v->opt_tile_order = (int)value;
        return VR_OK;
    case VR_OPT_STREAM_CULL:
        if (!v->streamed && value != 0.0)
            return fail(VR_ERR_UNSUPPORTED, "vr_set_option: brick culling is for streamed volumes");
        v->opt_cull = value != 0.0;
        return VR_OK;
    case VR_OPT_STREAM_CACHE:
        if (!v->streamed && value != 0.0)
            return fail(VR_ERR_UNSUPPORTED, "vr_set_option: the brick cache is for streamed volumes");
        v->opt_cache = value != 0.0;
        return VR_OK;
    default: return fail(VR_ERR_INVALID_ARG, "vr_set_option: unknown key %d", key);
    }
}

vr_status vr_set_aux_output(vr_volume* v, float* d_aux)
{
    if (!v) return fail(VR_ERR_INVALID_ARG, "vr_set_aux_output: null handle");
    v->d_aux = d_aux;
    return VR_OK;
}

vr_status vr_render(vr_volume* v, const vr_camera* cam, int W, int H, float step, int mode,
                    float* out, void* stream)
{
    vr_status st = check_render_args(v, cam, W, H, step, mode, out);
    if (st != VR_OK) return st;
    VR_CUDA(cudaSetDevice(v->desc.device));
    cudaStream_t s = (cudaStream_t)stream;
    if (v->part) return render_part(v, cam, W, H, step, mode, out, s);
    return v->streamed ? render_streamed(v, cam, W, H, step, mode, out, s)
                       : render_resident(v, cam, W, H, step, mode, out, s);
}

vr_status vr_render_wall(vr_volume* v, const vr_camera* cam, int W, int H, int K, int L, float step, int mode,
                         float* const* outs, void* stream)
{
    if (!outs) return fail(VR_ERR_INVALID_ARG, "vr_render_wall: null tile list");
    if (K < 1 || L < 1 || K * L > vr::kMaxWallTiles)
        return fail(VR_ERR_INVALID_ARG, "vr_render_wall: a wall has 1 .. %d tiles (%d x %d asked)", vr::kMaxWallTiles, K, L);
    for (int q = 0; q < K * L; ++q)
        if (!outs[q]) return fail(VR_ERR_INVALID_ARG, "vr_render_wall: tile %d has a null buffer", q);
    vr_status st = check_render_args(v, cam, W, H, step, mode, outs[0]);
    if (st != VR_OK) return st;
    if (W % K != 0 || H % L != 0)
        return fail(VR_ERR_INVALID_ARG, "vr_render_wall: %d x %d pixels do not divide into %d x %d tiles", W, H, K, L);
    if (v->streamed || v->part) return fail(VR_ERR_UNSUPPORTED, "vr_render_wall: resident whole cubes only");
    if (v->d_aux) return fail(VR_ERR_UNSUPPORTED, "vr_render_wall: no aux output (vr_set_aux_output(vol, NULL) first)");
    VR_CUDA(cudaSetDevice(v->desc.device));
    const Wall wall{K, L, outs};
    return render_resident(v, cam, W, H, step, mode, nullptr, (cudaStream_t)stream, &wall);
}

vr_status vr_autotune(vr_volume* v, const vr_camera* cam, int W, int H, float step, int mode, float* out,
                      void* stream, int* pipeline_out, int* tile_order_out, int* reuse_out)
{
    vr_status st = check_render_args(v, cam, W, H, step, mode, out);
    if (st != VR_OK) return st;
    if (v->streamed || v->part) return fail(VR_ERR_UNSUPPORTED, "vr_autotune: resident whole cubes only");
    VR_CUDA(cudaSetDevice(v->desc.device));
    cudaStream_t s = (cudaStream_t)stream;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    VR_CUDA(cudaEventCreateWithFlags(&e0, cudaEventDefault));
    if (cudaEventCreateWithFlags(&e1, cudaEventDefault) != cudaSuccess) {
        cudaEventDestroy(e0);
        return fail(VR_ERR_CUDA, "vr_autotune: cannot create events");
    }
    const int save_p = v->opt_pipeline, save_t = v->opt_tile_order, save_k = v->opt_kernel, save_s = v->opt_skip,
              save_r = v->opt_reuse;
    v->opt_kernel = 1;                          // the direct kernel family
    v->opt_skip = 0;
    float best = INFINITY;
    int best_p = 1, best_t = 0, best_r = 1;
    st = VR_OK;
    // (pipeline depth, cell reuse): plain, 2 and 4 samples in flight, cell reuse -- each under both tile orders
    const int cand[4][2] = {{1, 1}, {2, 1}, {4, 1}, {1, 2}};
    for (int t = 0; t < 2 && st == VR_OK; ++t)
        for (int d = 0; d < 4 && st == VR_OK; ++d) {
            v->opt_pipeline = cand[d][0];
            v->opt_reuse = cand[d][1];
            v->opt_tile_order = t;
            float ms_best = INFINITY;
            for (int rep = 0; rep < 3 && st == VR_OK; ++rep) {       // first repetition = warm-up
                cudaError_t ce = cudaEventRecord(e0, s);
                if (ce == cudaSuccess) st = render_resident(v, cam, W, H, step, mode, out, s);
                if (st != VR_OK) break;
                if (ce == cudaSuccess) ce = cudaEventRecord(e1, s);
                if (ce == cudaSuccess) ce = cudaEventSynchronize(e1);
                float ms = 0.f;
                if (ce == cudaSuccess) ce = cudaEventElapsedTime(&ms, e0, e1);
                if (ce != cudaSuccess) { st = fail(VR_ERR_CUDA, "vr_autotune: %s", cudaGetErrorString(ce)); break; }
                if (rep > 0) ms_best = std::fmin(ms_best, ms);
            }
            if (st == VR_OK && ms_best < best) { best = ms_best; best_p = cand[d][0]; best_r = cand[d][1]; best_t = t; }
        }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    v->opt_kernel = save_k;
    v->opt_skip = save_s;
    if (st != VR_OK) { v->opt_pipeline = save_p; v->opt_tile_order = save_t; v->opt_reuse = save_r; return st; }
    v->opt_pipeline = best_p;
    v->opt_tile_order = best_t;
    v->opt_reuse = best_r;
    if (pipeline_out) *pipeline_out = best_p;
    if (tile_order_out) *tile_order_out = best_t;
    if (reuse_out) *reuse_out = best_r;
    return VR_OK;
}

vr_status vr_render_host(vr_volume* v, const vr_camera* cam, int W, int H, float step, int mode,
                         float* d_staging, float* h_out, void* stream)
{
    if (!h_out) return fail(VR_ERR_INVALID_ARG, "vr_render_host: null host buffer");
    vr_status st = vr_render(v, cam, W, H, step, mode, d_staging, stream);
    if (st != VR_OK) return st;
    VR_CUDA(cudaMemcpyAsync(h_out, d_staging, (size_t)W * H * 4 * sizeof(float), cudaMemcpyDeviceToHost,
                            (cudaStream_t)stream));
    return VR_OK;
}

vr_status vr_get_minmax(vr_volume* v, float* h_min, float* h_max, void* stream)
{
    if (!v || !h_min || !h_max) return fail(VR_ERR_INVALID_ARG, "vr_get_minmax: null argument");
    if (v->streamed || v->part) return fail(VR_ERR_UNSUPPORTED, "vr_get_minmax: resident whole cubes only");
    if (!v->uploaded) return fail(VR_ERR_STATE, "vr_get_minmax: no voxels uploaded yet");
    VR_CUDA(cudaSetDevice(v->desc.device));
    cudaStream_t s = (cudaStream_t)stream;
    vr_status st = ensure_minmax(v, s);
    if (st != VR_OK) return st;
    std::vector<float2> tmp((size_t)v->n_mm);
    VR_CUDA(cudaMemcpyAsync(tmp.data(), v->d_minmax, tmp.size() * sizeof(float2), cudaMemcpyDeviceToHost, s));
    VR_CUDA(cudaStreamSynchronize(s));
    for (int q = 0; q < v->n_mm; ++q) { h_min[q] = tmp[q].x; h_max[q] = tmp[q].y; }
    return VR_OK;
}

vr_status vr_get_stats(vr_volume* v, vr_stats* out)
{
    if (!v || !out) return fail(VR_ERR_INVALID_ARG, "vr_get_stats: null argument");
    VR_CUDA(cudaSetDevice(v->desc.device));
    if (v->opt_count) {
        unsigned long long c[4] = {0, 0, 0, 0};
        VR_CUDA(cudaDeviceSynchronize());
        VR_CUDA(cudaMemcpy(c, v->d_counters, sizeof(c), cudaMemcpyDeviceToHost));
        v->stats.rays_hit = c[0];
        v->stats.samples = c[1];
        v->stats.fetches = v->stats.kernel == 4 ? c[2] : c[1];      // only the cell-reuse kernel fetches less often than it samples
    }
    if (v->streamed && v->frame_no > 0 && !v->stats.timing_valid) {
        VR_CUDA(cudaEventSynchronize(v->ev_f1));
        VR_CUDA(cudaStreamSynchronize(v->copy_stream));
        float ms = 0.f;
        VR_CUDA(cudaEventElapsedTime(&ms, v->ev_f0, v->ev_f1));
        v->stats.frame_ms = ms;
        double copy_ms = 0.0;
        for (int q = 0; q + 1 < v->n_tev; q += 2) {
            VR_CUDA(cudaEventElapsedTime(&ms, v->tev[(size_t)q], v->tev[(size_t)q + 1]));
            copy_ms += ms;
        }
        v->stats.h2d_ms = copy_ms;
        v->stats.h2d_gbs = copy_ms > 0.0 ? (double)v->stats.h2d_bytes / (copy_ms * 1e-3) / 1e9 : 0.0;
        v->stats.overlap_ratio = v->stats.frame_ms > 0.0 ? copy_ms / v->stats.frame_ms : 0.0;
        v->stats.timing_valid = 1;
    }
    if (v->skip_valid) {
        unsigned int ns = 0;
        VR_CUDA(cudaDeviceSynchronize());
        VR_CUDA(cudaMemcpy(&ns, v->d_nskip, sizeof(ns), cudaMemcpyDeviceToHost));
        v->stats.bricks_skippable = ns;
    }
    *out = v->stats;
    return VR_OK;
}

vr_status vr_get_brick_flags(vr_volume* v, int* flags_out)
{
    if (!v || !flags_out) return fail(VR_ERR_INVALID_ARG, "vr_get_brick_flags: null argument");
    if (!v->streamed) return fail(VR_ERR_UNSUPPORTED, "vr_get_brick_flags: streamed volumes only");
    for (size_t q = 0; q < v->brick_flags.size(); ++q) flags_out[q] = v->brick_flags[q];
    return VR_OK;
}

vr_status vr_host_alloc(size_t bytes, void** out)
{
    if (out) *out = nullptr;
    if (!out || bytes == 0) return fail(VR_ERR_INVALID_ARG, "vr_host_alloc: null argument or zero size");
    cudaError_t e = cudaHostAlloc(out, bytes, cudaHostAllocDefault);
    if (e != cudaSuccess) {
        *out = nullptr;
        cudaGetLastError();
        return fail(e == cudaErrorMemoryAllocation ? VR_ERR_OOM_HOST : VR_ERR_CUDA, "vr_host_alloc(%zu): %s", bytes,
                    cudaGetErrorString(e));
    }
    return VR_OK;
}

void vr_host_free(void* p)
{
    if (p) cudaFreeHost(p);
}

vr_status vr_beam_plan(const vr_volume_desc* d, const vr_camera* cam, int W, int H, int tile_i, int tile_j,
                       int stage_bytes, int pad_mode, int max_slabs, int* slabs_out, int* info_out)
{
    if (!valid_dims(d) || !cam || !slabs_out || !info_out || W < 1 || H < 1 || max_slabs < 1 || tile_i < 0 || tile_j < 0 ||
        tile_i * vr::kTileW >= W || tile_j * vr::kTileH >= H || d->nx % 4 != 0)
        return fail(VR_ERR_INVALID_ARG, "vr_beam_plan: bad argument");
    vr::FrameParams P;
    std::memset(&P, 0, sizeof(P));
    for (int c = 0; c < 3; ++c) {
        P.eye[c] = cam->eye[c]; P.right[c] = cam->right[c];
        P.up[c] = cam->up[c];   P.fwd[c] = cam->forward[c];
    }
    P.projection = cam->projection;
    P.th = cam->tan_half_fovy;
    P.hh = cam->ortho_half_height;
    P.W = W; P.H = H;
    P.n[0] = d->nx; P.n[1] = d->ny; P.n[2] = d->nz;
    P.x1 = W; P.y1 = H;
    vr::BeamParams B{};
    vr::beam::default_params(B);
    if (stage_bytes > 0) B.stage_bytes = stage_bytes;
    if (pad_mode >= 0) B.pad_mode = pad_mode ? 1 : 0;
    P.tiles_x = ceil_div(W, vr::kTileW);
    P.tiles_y = ceil_div(H, vr::kTileH);
    if (stage_bytes <= 0) B.stage_bytes = vr::beam::auto_stage_bytes(P, B);
    // the same steps as raycast_beam_kernel (vr_beam.cu), in the same order
    const int tile_x = tile_i * vr::kTileW, tile_y = tile_j * vr::kTileH;
    vr::beam::TileGeom G;
    std::memset(&G, 0, sizeof(G));
    const int alive = vr::beam::tile_geometry(P, tile_x, tile_y, G);
    const bool pos = G.pos != 0;
    int n_slabs = 0;
    int cursor = pos ? G.cmin : G.cmax;
    while (alive > 0 && !vr::beam::march_over(G, cursor)) {
        vr::beam::Slab sl;
        vr::beam::plan_slab_any(P.n, B, G, cursor, sl);
        if (n_slabs < max_slabs) {
            int* o = slabs_out + (size_t)16 * n_slabs;
            o[0] = sl.kind; o[1] = sl.clo; o[2] = sl.depth;
            for (int c = 0; c < 3; ++c) { o[3 + c] = sl.org[c]; o[6 + c] = sl.dim[c]; o[9 + c] = sl.str[c]; }
            o[12] = sl.floats; o[13] = sl.lim; o[14] = sl.cx; o[15] = sl.set;
        }
        ++n_slabs;
    }
    info_out[0] = G.AX; info_out[1] = pos ? 1 : 0; info_out[2] = G.cmin; info_out[3] = G.cmax;
    info_out[4] = n_slabs; info_out[5] = G.flags ? 1 : 0; info_out[6] = alive; info_out[7] = B.stage_bytes;
    info_out[8] = G.FAST; info_out[9] = B.pad_mode;
    return VR_OK;
}

vr_status vr_brick_order(const vr_volume_desc* d, int brick_edge, const vr_camera* cam,
                         int* order_out, int* keys_out)
{
    if (!valid_dims(d) || !cam || !order_out || brick_edge < 1)
        return fail(VR_ERR_INVALID_ARG, "vr_brick_order: bad argument");
    const int nhb[3] = {ceil_div(d->nx - 1, brick_edge), ceil_div(d->ny - 1, brick_edge),
                        ceil_div(d->nz - 1, brick_edge)};
    std::vector<Keyed> ks;
    order_bricks(nhb, brick_edge, cam, ks);
    for (size_t q = 0; q < ks.size(); ++q) {
        order_out[q] = ks[q].idx;
        if (keys_out) keys_out[q] = ks[q].key;
    }
    return VR_OK;
}

}  // extern "C"
