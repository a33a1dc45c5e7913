// cuda_runtime.h -- TEST INFRASTRUCTURE: a host emulation of the CUDA subset libvr.so uses.
//
// tests/hostemu/build.py compiles the product's own sources (paper_1001_2049_b200/csrc/*.cu, unchanged) with g++
// against this header instead of the CUDA toolkit's, giving tests/hostemu/libvr_hostemu.so: the same C ABI
// (include/vr.h), "device memory" = host memory, every kernel run thread by thread on the host cores.  It exists so that
// the host logic of the library (validation, layouts, the out-of-core scheduler, stream / event ordering) and the
// kernels' C++ (everything except inline PTX) can be held against the CPU oracle in `-m "not gpu"` tests on a box with
// no GPU.  It is NOT a CPU fallback: the package never loads it, nothing outside tests/ names it, and it is far too slow
// to render anything but test images.
//
// What is modelled, and how faithfully:
//   * every intrinsic by its IEEE-754 / PTX definition (fma by fmaf, __fadd_rd by an add under FE_DOWNWARD, float -> int
//     conversions with the PTX saturation rules, min / max with PTX's signed-zero and NaN rules) -- never by "what the
//     caller expects it to do";
//   * a CTA = a set of fibers (ucontext) on one OS thread, CTAs spread over the host cores; __syncthreads() and the
//     warp collectives (__shfl_xor_sync, votes, __reduce_*_sync) are real rendezvous points between the fibers, exited
//     threads do not take part; static __shared__ variables are per OS thread, the dynamic shared memory is a buffer
//     refilled with NaNs before every CTA;
//   * streams are queues executed LATER (emu_runtime.cpp): a kernel or an asynchronous copy runs when something waits
//     for it, in an order chosen by the policy VR_EMU_SCHED (lazy: as late as allowed; eager: private non-blocking
//     streams as early as allowed; sync: at once), so that a missing event wait between the copy stream and the compute
//     stream shows up as wrong pixels; copies from / to pageable host memory are taken at call time like the real
//     runtime does, copies from / to pinned memory (cudaHostAlloc) when the stream reaches them;
//   * 2D-layered CUDA arrays with point-sampled, unnormalised, clamped texture objects read by the tld4 gather.
// What is not: inline PTX (cp.async, mbarrier -- the sources give a plain C++ path under VR_HOSTEMU), timing, caches.
#pragma once

#define VR_HOSTEMU 1

#include <cfenv>
#include <cmath>
#include <cstddef>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <functional>
#include <tuple>
#include <type_traits>
#include <utility>

#define __host__
#define __device__
#define __global__
#define __forceinline__ inline __attribute__((always_inline))
#define __grid_constant__
#define __launch_bounds__(...)
#define __shared__ static thread_local
#define __align__(n) alignas(n)

// ---- vector types ---------------------------------------------------------------------------------
struct alignas(8) float2 { float x, y; };
struct alignas(16) float4 { float x, y, z, w; };
struct uint3 { unsigned int x, y, z; };
struct dim3 {
    unsigned int x, y, z;
    dim3(unsigned int a = 1, unsigned int b = 1, unsigned int c = 1) : x(a), y(b), z(c) {}
};
static inline float2 make_float2(float x, float y) { float2 r; r.x = x; r.y = y; return r; }
static inline float4 make_float4(float x, float y, float z, float w) { float4 r; r.x = x; r.y = y; r.z = z; r.w = w; return r; }

// ---- runtime API (emu_runtime.cpp) -------------------------------------------------------------------
enum cudaError_t {
    cudaSuccess = 0, cudaErrorInvalidValue = 1, cudaErrorMemoryAllocation = 2, cudaErrorInvalidDevice = 101,
    cudaErrorNotReady = 600, cudaErrorLaunchFailure = 719
};
enum cudaMemcpyKind { cudaMemcpyHostToHost = 0, cudaMemcpyHostToDevice = 1, cudaMemcpyDeviceToHost = 2,
                      cudaMemcpyDeviceToDevice = 3, cudaMemcpyDefault = 4 };
struct emu_stream;
struct emu_event;
typedef emu_stream* cudaStream_t;
typedef emu_event* cudaEvent_t;
enum { cudaStreamDefault = 0, cudaStreamNonBlocking = 1 };
enum { cudaEventDefault = 0, cudaEventBlockingSync = 1, cudaEventDisableTiming = 2 };
enum { cudaHostAllocDefault = 0 };
enum cudaFuncAttribute { cudaFuncAttributeMaxDynamicSharedMemorySize = 8 };

const char* cudaGetErrorString(cudaError_t e);
cudaError_t cudaGetLastError();
cudaError_t cudaGetDeviceCount(int* n);
cudaError_t cudaSetDevice(int d);
cudaError_t cudaMalloc(void** p, size_t bytes);
template <class T> static inline cudaError_t cudaMalloc(T** p, size_t bytes) { return cudaMalloc((void**)p, bytes); }
cudaError_t cudaFree(void* p);
cudaError_t cudaHostAlloc(void** p, size_t bytes, unsigned int flags);
cudaError_t cudaFreeHost(void* p);
cudaError_t cudaMemcpy(void* dst, const void* src, size_t bytes, cudaMemcpyKind kind);
cudaError_t cudaMemcpyAsync(void* dst, const void* src, size_t bytes, cudaMemcpyKind kind, cudaStream_t s = nullptr);
cudaError_t cudaMemset(void* p, int value, size_t bytes);
cudaError_t cudaMemsetAsync(void* p, int value, size_t bytes, cudaStream_t s = nullptr);
cudaError_t cudaStreamCreateWithFlags(cudaStream_t* s, unsigned int flags);
cudaError_t cudaStreamDestroy(cudaStream_t s);
cudaError_t cudaStreamSynchronize(cudaStream_t s);
cudaError_t cudaStreamWaitEvent(cudaStream_t s, cudaEvent_t e, unsigned int flags = 0);
cudaError_t cudaDeviceSynchronize();
cudaError_t cudaEventCreateWithFlags(cudaEvent_t* e, unsigned int flags);
cudaError_t cudaEventDestroy(cudaEvent_t e);
cudaError_t cudaEventRecord(cudaEvent_t e, cudaStream_t s = nullptr);
cudaError_t cudaEventSynchronize(cudaEvent_t e);
cudaError_t cudaEventQuery(cudaEvent_t e);
cudaError_t cudaEventElapsedTime(float* ms, cudaEvent_t a, cudaEvent_t b);
cudaError_t cudaMemGetInfo(size_t* free_b, size_t* total_b);

// ---- CUDA arrays and texture objects (2D layered, float32, point sampled) ------------------------------
struct cudaArray { int w, h, layers; float* data; };
typedef cudaArray* cudaArray_t;
typedef unsigned long long cudaTextureObject_t;
struct cudaChannelFormatDesc { int x, y, z, w, f; };
template <class T> static inline cudaChannelFormatDesc cudaCreateChannelDesc()
{
    static_assert(std::is_same<T, float>::value, "the emulation holds float32 arrays only");
    return cudaChannelFormatDesc{32, 0, 0, 0, 2};
}
struct cudaExtent { size_t width, height, depth; };
struct cudaPos { size_t x, y, z; };
struct cudaPitchedPtr { void* ptr; size_t pitch, xsize, ysize; };
static inline cudaExtent make_cudaExtent(size_t w, size_t h, size_t d) { return cudaExtent{w, h, d}; }
static inline cudaPos make_cudaPos(size_t x, size_t y, size_t z) { return cudaPos{x, y, z}; }
static inline cudaPitchedPtr make_cudaPitchedPtr(void* p, size_t pitch, size_t xs, size_t ys) { return cudaPitchedPtr{p, pitch, xs, ys}; }
struct cudaMemcpy3DParms {
    cudaArray_t srcArray; cudaPos srcPos; cudaPitchedPtr srcPtr;
    cudaArray_t dstArray; cudaPos dstPos; cudaPitchedPtr dstPtr;
    cudaExtent extent; cudaMemcpyKind kind;
};
enum { cudaArrayDefault = 0, cudaArrayLayered = 1 };
enum cudaResourceType { cudaResourceTypeArray = 0 };
struct cudaResourceDesc { cudaResourceType resType; struct { struct { cudaArray_t array; } array; } res; };
enum cudaTextureAddressMode { cudaAddressModeWrap = 0, cudaAddressModeClamp = 1 };
enum cudaTextureFilterMode { cudaFilterModePoint = 0, cudaFilterModeLinear = 1 };
enum cudaTextureReadMode { cudaReadModeElementType = 0 };
struct cudaTextureDesc {
    cudaTextureAddressMode addressMode[3]; cudaTextureFilterMode filterMode; cudaTextureReadMode readMode;
    int normalizedCoords;
};
cudaError_t cudaMalloc3DArray(cudaArray_t* arr, const cudaChannelFormatDesc* cd, cudaExtent ext, unsigned int flags);
cudaError_t cudaFreeArray(cudaArray_t arr);
cudaError_t cudaMemcpy3DAsync(const cudaMemcpy3DParms* p, cudaStream_t s = nullptr);
cudaError_t cudaCreateTextureObject(cudaTextureObject_t* tex, const cudaResourceDesc* rd, const cudaTextureDesc* td, const void*);
cudaError_t cudaDestroyTextureObject(cudaTextureObject_t tex);

// ---- kernel launches: fibers ------------------------------------------------------------------------
namespace emu {

struct ThreadInfo { uint3 tid; };
struct BlockInfo { dim3 grid, block; uint3 bid; };
extern thread_local ThreadInfo* g_thr;
extern thread_local BlockInfo* g_blk;

void* dyn_smem();                                           // the dynamic shared memory of the running CTA
void syncthreads();
void yield();                                               // lets the other threads of the CTA run (spin loops)
// every live lane of the warp contributes `v`; all[l] = lane l's value, *present = mask of live lanes; returns own lane
int warp_exchange(unsigned int v, unsigned int all[32], unsigned int* present);
cudaError_t enqueue_kernel(cudaStream_t s, dim3 grid, dim3 block, size_t smem, std::function<void()> body);
cudaError_t set_max_dyn_smem(int bytes);

template <class... P, class... A>
cudaError_t launch(void (*kern)(P...), dim3 grid, dim3 block, size_t smem, cudaStream_t s, A&&... a)
{
    // parameters are copied at launch time, like a real launch
    auto args = std::make_tuple(typename std::decay<P>::type(std::forward<A>(a))...);
    return enqueue_kernel(s, grid, block, smem, [kern, args]() { std::apply(kern, args); });
}

// tld4.r.a2d: the four texels bilinear filtering would use at (x, y) of `layer`, clamped addressing
float4 tld4_a2d(cudaTextureObject_t tex, int layer, float x, float y);

template <class T> static inline unsigned int bits_of(T v)
{
    static_assert(sizeof(T) == 4, "32-bit values only");
    unsigned int u; std::memcpy(&u, &v, 4); return u;
}
template <class T> static inline T from_bits(unsigned int u) { T v; std::memcpy(&v, &u, 4); return v; }

static inline float add_rounded(float a, float b, int mode)
{
    volatile float x = a, y = b;
    const int old = fegetround();
    fesetround(mode);
    volatile float r = x + y;
    fesetround(old);
    return r;
}

static inline int sat_int(float r)                         // cvt.rXi.s32.f32: NaN -> 0, saturating
{
    if (r != r) return 0;
    if (r >= 2147483648.0f) return 2147483647;
    if (r <= -2147483648.0f) return (-2147483647 - 1);
    return (int)r;
}

}  // namespace emu

template <class F> static inline cudaError_t cudaFuncSetAttribute(F, cudaFuncAttribute, int value)
{
    return emu::set_max_dyn_smem(value);
}

#define threadIdx (emu::g_thr->tid)
#define blockIdx (emu::g_blk->bid)
#define blockDim (emu::g_blk->block)
#define gridDim (emu::g_blk->grid)

static inline void __syncthreads() { emu::syncthreads(); }
static inline void __syncwarp(unsigned int = 0xffffffffu) { unsigned int a[32], p; emu::warp_exchange(0u, a, &p); }

template <class T> static inline T __shfl_xor_sync(unsigned int, T v, int lane_mask)
{
    unsigned int all[32], present;
    const int lane = emu::warp_exchange(emu::bits_of(v), all, &present);
    const int src = lane ^ lane_mask;
    return ((present >> src) & 1u) ? emu::from_bits<T>(all[src]) : v;
}
static inline int __any_sync(unsigned int, int p)
{
    unsigned int all[32], present; emu::warp_exchange(p ? 1u : 0u, all, &present);
    for (int l = 0; l < 32; ++l) if (((present >> l) & 1u) && all[l]) return 1;
    return 0;
}
static inline int __all_sync(unsigned int, int p)
{
    unsigned int all[32], present; emu::warp_exchange(p ? 1u : 0u, all, &present);
    for (int l = 0; l < 32; ++l) if (((present >> l) & 1u) && !all[l]) return 0;
    return 1;
}
static inline unsigned int __ballot_sync(unsigned int, int p)
{
    unsigned int all[32], present, r = 0; emu::warp_exchange(p ? 1u : 0u, all, &present);
    for (int l = 0; l < 32; ++l) if (((present >> l) & 1u) && all[l]) r |= 1u << l;
    return r;
}
static inline int __reduce_min_sync(unsigned int, int v)
{
    unsigned int all[32], present; emu::warp_exchange((unsigned int)v, all, &present);
    int r = v;
    for (int l = 0; l < 32; ++l) if ((present >> l) & 1u) r = (int)all[l] < r ? (int)all[l] : r;
    return r;
}
static inline int __reduce_max_sync(unsigned int, int v)
{
    unsigned int all[32], present; emu::warp_exchange((unsigned int)v, all, &present);
    int r = v;
    for (int l = 0; l < 32; ++l) if ((present >> l) & 1u) r = (int)all[l] > r ? (int)all[l] : r;
    return r;
}
static inline unsigned int __reduce_add_sync(unsigned int, unsigned int v)
{
    unsigned int all[32], present, r = 0; emu::warp_exchange(v, all, &present);
    for (int l = 0; l < 32; ++l) if ((present >> l) & 1u) r += all[l];
    return r;
}

// ---- intrinsics, by their definitions ---------------------------------------------------------------------
static inline float __fmaf_rn(float a, float b, float c) { return fmaf(a, b, c); }
static inline float __fsqrt_rn(float x) { return sqrtf(x); }
static inline float __fdiv_rn(float a, float b) { volatile float x = a, y = b; return x / y; }
static inline float __fadd_rn(float a, float b) { volatile float x = a, y = b; return x + y; }
static inline float __fadd_rd(float a, float b) { return emu::add_rounded(a, b, FE_DOWNWARD); }
static inline float __fadd_ru(float a, float b) { return emu::add_rounded(a, b, FE_UPWARD); }
static inline float __fadd_rz(float a, float b) { return emu::add_rounded(a, b, FE_TOWARDZERO); }
static inline float2 __ffma2_rn(float2 a, float2 b, float2 c) { return make_float2(fmaf(a.x, b.x, c.x), fmaf(a.y, b.y, c.y)); }
static inline float2 __fadd2_rn(float2 a, float2 b) { return make_float2(__fadd_rn(a.x, b.x), __fadd_rn(a.y, b.y)); }
static inline float2 __fadd2_rd(float2 a, float2 b) { return make_float2(__fadd_rd(a.x, b.x), __fadd_rd(a.y, b.y)); }
static inline int __float2int_rd(float x) { return emu::sat_int(floorf(x)); }
static inline int __float2int_ru(float x) { return emu::sat_int(ceilf(x)); }
static inline int __float2int_rz(float x) { return emu::sat_int(truncf(x)); }
static inline int __float2int_rn(float x) { return emu::sat_int(nearbyintf(x)); }     // ties to even (FE_TONEAREST)
static inline unsigned int __umulhi(unsigned int a, unsigned int b) { return (unsigned int)(((unsigned long long)a * b) >> 32); }
template <class T> static inline T __ldg(const T* p) { return *p; }

// min.f32 / max.f32 (PTX): a NaN operand gives the other one; -0 < +0
static inline float emu_fminf(float a, float b)
{
    if (a != a) return b;
    if (b != b) return a;
    if (a == 0.0f && b == 0.0f) return std::signbit(a) ? a : b;
    return a < b ? a : b;
}
static inline float emu_fmaxf(float a, float b)
{
    if (a != a) return b;
    if (b != b) return a;
    if (a == 0.0f && b == 0.0f) return std::signbit(a) ? b : a;
    return a > b ? a : b;
}
#define fminf emu_fminf
#define fmaxf emu_fmaxf

static inline int min(int a, int b) { return a < b ? a : b; }
static inline int max(int a, int b) { return a > b ? a : b; }
static inline unsigned int min(unsigned int a, unsigned int b) { return a < b ? a : b; }
static inline unsigned int max(unsigned int a, unsigned int b) { return a > b ? a : b; }
static inline long long min(long long a, long long b) { return a < b ? a : b; }
static inline long long max(long long a, long long b) { return a > b ? a : b; }

// ---- atomics (CTAs run on several OS threads) -----------------------------------------------------------
static inline int atomicAdd(int* p, int v) { return __atomic_fetch_add(p, v, __ATOMIC_RELAXED); }
static inline unsigned int atomicAdd(unsigned int* p, unsigned int v) { return __atomic_fetch_add(p, v, __ATOMIC_RELAXED); }
static inline unsigned long long atomicAdd(unsigned long long* p, unsigned long long v) { return __atomic_fetch_add(p, v, __ATOMIC_RELAXED); }
static inline int atomicOr(int* p, int v) { return __atomic_fetch_or(p, v, __ATOMIC_RELAXED); }
static inline unsigned int atomicOr(unsigned int* p, unsigned int v) { return __atomic_fetch_or(p, v, __ATOMIC_RELAXED); }
static inline int atomicMin(int* p, int v)
{
    int old = __atomic_load_n(p, __ATOMIC_RELAXED);
    while (v < old && !__atomic_compare_exchange_n(p, &old, v, true, __ATOMIC_RELAXED, __ATOMIC_RELAXED)) {}
    return old;
}
static inline int atomicMax(int* p, int v)
{
    int old = __atomic_load_n(p, __ATOMIC_RELAXED);
    while (v > old && !__atomic_compare_exchange_n(p, &old, v, true, __ATOMIC_RELAXED, __ATOMIC_RELAXED)) {}
    return old;
}
static inline unsigned int atomicMin(unsigned int* p, unsigned int v)
{
    unsigned int old = __atomic_load_n(p, __ATOMIC_RELAXED);
    while (v < old && !__atomic_compare_exchange_n(p, &old, v, true, __ATOMIC_RELAXED, __ATOMIC_RELAXED)) {}
    return old;
}
static inline int __float_as_int(float v) { return (int)emu::bits_of(v); }
static inline unsigned int __float_as_uint(float v) { return emu::bits_of(v); }
static inline float __int_as_float(int v) { return emu::from_bits<float>((unsigned int)v); }
static inline unsigned int atomicMax(unsigned int* p, unsigned int v)
{
    unsigned int old = __atomic_load_n(p, __ATOMIC_RELAXED);
    while (v > old && !__atomic_compare_exchange_n(p, &old, v, true, __ATOMIC_RELAXED, __ATOMIC_RELAXED)) {}
    return old;
}
