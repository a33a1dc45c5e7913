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
// The per-thread phases (vr_beam_core.cuh) and the CTA body that orders them (vr_beam_cta.cuh) are
// host + device code; tests/beam_harness.cu runs them on the host against the oracle, the CTA body
// with 128 OS threads under ThreadSanitizer.  This file only binds the CTA body to the hardware's
// barriers, warp votes, shared-memory atomics and cp.async.
#include "vr_beam_cta.cuh"

namespace vr {

namespace {

// The context of beam_cta (vr_beam_cta.cuh) on the device: the hardware's barriers, votes and atomics.
// (__host__ __device__ only so that the host + device CTA body may name them; the bodies are device code.)
// Set by bulk_wait when an mbarrier phase did not complete within kBulkSpinLimit polls (a box whose announced bytes
// differ from the bytes its row copies deliver would otherwise hang every CTA); launch_raycast_beam's caller reads it
// back through beam_fault_flag() and reports VR_ERR_CUDA.
__device__ unsigned int g_beam_fault = 0;
constexpr unsigned int kBulkSpinLimit = 1u << 22;

struct DeviceCtx {
#if defined(__CUDA_ARCH__) && !defined(VR_HOSTEMU)
    __host__ __device__ __forceinline__ int tid() const { return (int)threadIdx.x; }
    __host__ __device__ __forceinline__ int block() const { return (int)blockIdx.x; }
    __host__ __device__ __forceinline__ void sync() const { __syncthreads(); }
    __host__ __device__ __forceinline__ bool any(bool p) const { return __any_sync(0xffffffffu, p) != 0; }
    __host__ __device__ __forceinline__ int warp_min(int v) const { return __reduce_min_sync(0xffffffffu, v); }
    __host__ __device__ __forceinline__ int warp_max(int v) const { return __reduce_max_sync(0xffffffffu, v); }
    __host__ __device__ __forceinline__ unsigned int warp_sum(unsigned int v) const { return __reduce_add_sync(0xffffffffu, v); }
    __host__ __device__ __forceinline__ void smem_min(int* p, int v) const { atomicMin(p, v); }
    __host__ __device__ __forceinline__ void smem_max(int* p, int v) const { atomicMax(p, v); }
    __host__ __device__ __forceinline__ void smem_add(int* p, int v) const { atomicAdd(p, v); }
    __host__ __device__ __forceinline__ void smem_or(int* p, int v) const { atomicOr(p, v); }
    __host__ __device__ __forceinline__ int smem_peek(const int* p) const { return *(const volatile int*)p; }
    __host__ __device__ __forceinline__ void copies_done() const
    {
        asm volatile("cp.async.commit_group;\n\tcp.async.wait_group 0;" ::: "memory");
    }
    __host__ __device__ __forceinline__ void count(unsigned long long* p, unsigned long long v) const { atomicAdd(p, v); }
    // mbarrier of the bulk copies: one arrival per phase (thread 0's, which also announces the bytes to come)
    __host__ __device__ __forceinline__ void bulk_init(unsigned long long* bar) const
    {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n\tfence.mbarrier_init.release.cluster;"
                     ::"r"((uint32_t)__cvta_generic_to_shared(bar)) : "memory");
    }
    __host__ __device__ __forceinline__ void bulk_expect(unsigned long long* bar, unsigned int bytes) const
    {
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;"
                     ::"r"((uint32_t)__cvta_generic_to_shared(bar)), "r"(bytes) : "memory");
    }
    __host__ __device__ __forceinline__ void bulk_row(unsigned long long* bar, float* dst, const float* src,
                                                       unsigned int bytes) const
    {
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                     ::"r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src), "r"(bytes),
                       "r"((uint32_t)__cvta_generic_to_shared(bar)) : "memory");
    }
    // bounded: after kBulkSpinLimit polls the thread gives up, flags the fault and goes on (the frame is then wrong
    // and reported as such, but no CTA spins for ever)
    __host__ __device__ __forceinline__ void bulk_wait(unsigned long long* bar, unsigned int parity) const
    {
        const uint32_t a = (uint32_t)__cvta_generic_to_shared(bar);
        uint32_t ok = 0;
        for (unsigned int spin = 0; spin < kBulkSpinLimit; ++spin) {
            asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                         "selp.u32 %0, 1, 0, p;\n\t}"
                         : "=r"(ok) : "r"(a), "r"(parity) : "memory");
            if (ok) return;
        }
        atomicOr(&g_beam_fault, 1u);
    }
#elif defined(VR_HOSTEMU)
    // tests/hostemu: barriers, votes and atomics are the emulation's; a 16-byte cp.async lands at once (VR_CP16); the
    // mbarrier is modelled in its 8 bytes as {pending arrivals : 16 | phase : 16 | transaction bytes still owed : 32}
    int tid() const { return (int)threadIdx.x; }
    int block() const { return (int)blockIdx.x; }
    void sync() const { __syncthreads(); }
    bool any(bool p) const { return __any_sync(0xffffffffu, p) != 0; }
    int warp_min(int v) const { return __reduce_min_sync(0xffffffffu, v); }
    int warp_max(int v) const { return __reduce_max_sync(0xffffffffu, v); }
    unsigned int warp_sum(unsigned int v) const { return __reduce_add_sync(0xffffffffu, v); }
    void smem_min(int* p, int v) const { atomicMin(p, v); }
    void smem_max(int* p, int v) const { atomicMax(p, v); }
    void smem_add(int* p, int v) const { atomicAdd(p, v); }
    void smem_or(int* p, int v) const { atomicOr(p, v); }
    int smem_peek(const int* p) const { return *(const volatile int*)p; }
    void copies_done() const {}
    void count(unsigned long long* p, unsigned long long v) const { atomicAdd(p, v); }
    struct Mbar { short pending; unsigned short phase; int tx; };
    static void mbar_settle(Mbar* m) { if (m->pending == 0 && m->tx == 0) { m->phase ^= 1; m->pending = 1; } }
    void bulk_init(unsigned long long* bar) const { Mbar* m = (Mbar*)bar; m->pending = 1; m->phase = 0; m->tx = 0; }
    void bulk_expect(unsigned long long* bar, unsigned int bytes) const
    {
        Mbar* m = (Mbar*)bar; m->tx += (int)bytes; --m->pending; mbar_settle(m);
    }
    void bulk_row(unsigned long long* bar, float* dst, const float* src, unsigned int bytes) const
    {
        std::memcpy(dst, src, bytes);
        Mbar* m = (Mbar*)bar; m->tx -= (int)bytes; mbar_settle(m);
    }
    void bulk_wait(unsigned long long* bar, unsigned int parity) const
    {
        const Mbar* m = (const Mbar*)bar;
        for (unsigned int spin = 0; spin < kBulkSpinLimit; ++spin) {
            if ((unsigned int)(*(const volatile unsigned short*)&m->phase) != parity) return;
            emu::yield();                                // lets the other fibers of the CTA run
        }
        atomicOr(&g_beam_fault, 1u);
    }
#else
    int tid() const { return 0; }
    int block() const { return 0; }
    void sync() const {}
    bool any(bool p) const { return p; }
    int warp_min(int v) const { return v; }
    int warp_max(int v) const { return v; }
    unsigned int warp_sum(unsigned int v) const { return v; }
    void smem_min(int*, int) const {}
    void smem_max(int*, int) const {}
    void smem_add(int*, int) const {}
    void smem_or(int*, int) const {}
    int smem_peek(const int* p) const { return *p; }
    void copies_done() const {}
    void count(unsigned long long*, unsigned long long) const {}
    void bulk_init(unsigned long long*) const {}
    void bulk_expect(unsigned long long*, unsigned int) const {}
    void bulk_row(unsigned long long*, float*, const float*, unsigned int) const {}
    void bulk_wait(unsigned long long*, unsigned int) const {}
#endif
};

template <int MODE, bool COUNT, bool GREY, int NSTAGE>
__global__ void __launch_bounds__(kThreads, 8)
raycast_beam_kernel(const __grid_constant__ FrameParams P, const __grid_constant__ BeamParams B)
{
    VR_DYN_SHARED(unsigned char, s_dyn);
    __shared__ beam::BeamShared sh;
    DeviceCtx cx;
    beam::beam_cta<MODE, COUNT, GREY, NSTAGE>(P, B, sh, s_dyn, cx);
}

template <int MODE, bool COUNT, bool GREY, int NSTAGE>
cudaError_t launch_stages(const FrameParams& P, const BeamParams& B, cudaStream_t stream)
{
    const size_t lut_bytes = MODE == VR_MODE_EA ? (size_t)(GREY ? 1 : 2) * P.n_lut * sizeof(float4) : 0;
    const size_t smem = lut_bytes + (size_t)NSTAGE * (size_t)B.stage_bytes;
    auto kern = raycast_beam_kernel<MODE, COUNT, GREY, NSTAGE>;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    const int tiles = P.tiles_x * P.tiles_y;
    if (tiles <= 0) return cudaSuccess;
    VR_LAUNCH(kern, tiles, kThreads, smem, stream, P, B);
    return cudaGetLastError();
}

template <int MODE, bool COUNT, bool GREY>
cudaError_t launch_beam(const FrameParams& P, const BeamParams& B, cudaStream_t stream)
{
    return B.n_stages == 2 ? launch_stages<MODE, COUNT, GREY, 2>(P, B, stream) : launch_stages<MODE, COUNT, GREY, 1>(P, B, stream);
}

}  // namespace

// reads and clears the fault flag of the bulk-copy wait (synchronises the device)
cudaError_t beam_fault_flag(unsigned int* flag)
{
#ifdef VR_HOSTEMU
    cudaError_t e = cudaDeviceSynchronize();
    *flag = g_beam_fault;
    g_beam_fault = 0;
    return e;
#else
    cudaError_t e = cudaMemcpyFromSymbol(flag, g_beam_fault, sizeof(unsigned int));
    if (e != cudaSuccess) return e;
    const unsigned int zero = 0;
    return cudaMemcpyToSymbol(g_beam_fault, &zero, sizeof(unsigned int));
#endif
}

cudaError_t launch_raycast_beam(const FrameParams& P, const BeamParams& B, int mode, bool count, cudaStream_t stream)
{
    if (mode == VR_MODE_EA) {
        if (B.lut_grey)
            return count ? launch_beam<VR_MODE_EA, true, true>(P, B, stream) : launch_beam<VR_MODE_EA, false, true>(P, B, stream);
        return count ? launch_beam<VR_MODE_EA, true, false>(P, B, stream) : launch_beam<VR_MODE_EA, false, false>(P, B, stream);
    }
    return count ? launch_beam<VR_MODE_MIP, true, false>(P, B, stream) : launch_beam<VR_MODE_MIP, false, false>(P, B, stream);
}

}  // namespace vr
