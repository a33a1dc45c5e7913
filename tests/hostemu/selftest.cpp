// selftest.cpp -- TEST INFRASTRUCTURE: the host emulation (cuda_runtime.h, emu_runtime.cpp) checked against what
// it claims to model, so that a green emulated parity run means something:
//   * a kernel that reads a buffer another stream is still filling, with no event wait, DOES read stale data under the
//     lazy schedule; a copy that overwrites a buffer a queued kernel has yet to read, with no event wait, DOES corrupt
//     it under the eager schedule; with the waits both are correct under both schedules;
//   * __syncthreads / warp shuffles / votes are real rendezvous points (block reduction, early-exit threads);
//   * rounding-mode intrinsics and conversions follow their definitions.
// Prints one line per check; exit code = number of failed checks.
#include "cuda_runtime.h"

#include <cstdio>
#include <vector>

extern "C" void vr_emu_set_sched(int mode);

static int g_fail = 0;
static void check(bool ok, const char* what)
{
    printf("%s %s\n", ok ? "ok  " : "FAIL", what);
    if (!ok) ++g_fail;
}

__global__ void sum_kernel(const float* in, int n, float* out)
{
    __shared__ float part[8];
    float s = 0.0f;
    for (int q = threadIdx.x; q < n; q += blockDim.x) s += in[q];
    for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        float t = 0.0f;
        for (unsigned int w = 0; w < blockDim.x / 32; ++w) t += part[w];
        out[blockIdx.x] = t;
    }
}

__global__ void exit_kernel(int* out)
{
    // odd warps leave before the barrier; the others must still get through it, and a vote sees only live lanes
    if ((threadIdx.x >> 5) & 1) return;
    if ((threadIdx.x & 31) >= 16 && threadIdx.x < 32) { /* half of warp 0 skips the vote below */ }
    __syncthreads();
    const int all = __all_sync(0xffffffffu, threadIdx.x < 1000);
    const unsigned int ballot = __ballot_sync(0xffffffffu, (threadIdx.x & 1) != 0);
    if (threadIdx.x == 0) { out[0] = all; out[1] = (int)ballot; }
    atomicAdd(&out[2], 1);
}

// 1 if the kernel saw the fresh data
static int read_after_copy(int sched, bool with_wait)
{
    vr_emu_set_sched(sched);
    cudaStream_t copy, run;
    cudaStreamCreateWithFlags(&copy, cudaStreamNonBlocking);
    cudaStreamCreateWithFlags(&run, cudaStreamDefault);
    cudaEvent_t ev;
    cudaEventCreateWithFlags(&ev, cudaEventDisableTiming);
    float *h, *d, *out;
    cudaHostAlloc((void**)&h, 256 * sizeof(float), 0);
    cudaMalloc((void**)&d, 256 * sizeof(float));
    cudaMalloc((void**)&out, sizeof(float));
    cudaMemset(d, 0, 256 * sizeof(float));
    for (int q = 0; q < 256; ++q) h[q] = 1.0f;
    cudaMemcpyAsync(d, h, 256 * sizeof(float), cudaMemcpyHostToDevice, copy);
    cudaEventRecord(ev, copy);
    if (with_wait) cudaStreamWaitEvent(run, ev, 0);
    emu::launch(sum_kernel, 1, 256, 0, run, (const float*)d, 256, out);
    cudaStreamSynchronize(run);
    cudaStreamSynchronize(copy);
    const int fresh = *out == 256.0f;
    cudaFree(d); cudaFree(out); cudaFreeHost(h);
    cudaEventDestroy(ev); cudaStreamDestroy(copy); cudaStreamDestroy(run);
    return fresh;
}

// 1 if the kernel saw the data that was in the buffer when it was enqueued (the copy that follows must wait for it)
static int copy_after_read(int sched, bool with_wait)
{
    vr_emu_set_sched(sched);
    cudaStream_t copy, run;
    cudaStreamCreateWithFlags(&copy, cudaStreamNonBlocking);
    cudaStreamCreateWithFlags(&run, cudaStreamDefault);
    cudaEvent_t ev;
    cudaEventCreateWithFlags(&ev, cudaEventDisableTiming);
    float *h, *d, *out;
    cudaHostAlloc((void**)&h, 256 * sizeof(float), 0);
    cudaMalloc((void**)&d, 256 * sizeof(float));
    cudaMalloc((void**)&out, sizeof(float));
    std::vector<float> ones(256, 1.0f);
    cudaMemcpy(d, ones.data(), 256 * sizeof(float), cudaMemcpyHostToDevice);
    for (int q = 0; q < 256; ++q) h[q] = 2.0f;
    emu::launch(sum_kernel, 1, 256, 0, run, (const float*)d, 256, out);
    cudaEventRecord(ev, run);
    if (with_wait) cudaStreamWaitEvent(copy, ev, 0);
    cudaMemcpyAsync(d, h, 256 * sizeof(float), cudaMemcpyHostToDevice, copy);
    cudaStreamSynchronize(run);
    cudaStreamSynchronize(copy);
    const int intact = *out == 256.0f;
    cudaFree(d); cudaFree(out); cudaFreeHost(h);
    cudaEventDestroy(ev); cudaStreamDestroy(copy); cudaStreamDestroy(run);
    return intact;
}

int main()
{
    enum { SYNC = 0, LAZY = 1, EAGER = 2 };
    check(read_after_copy(LAZY, true) == 1, "lazy: kernel after copy, with the event wait, reads the copied data");
    check(read_after_copy(LAZY, false) == 0, "lazy: kernel after copy, WITHOUT the event wait, reads stale data (hazard shown)");
    check(read_after_copy(EAGER, true) == 1, "eager: kernel after copy, with the event wait, reads the copied data");
    check(copy_after_read(EAGER, true) == 1, "eager: copy after kernel, with the event wait, leaves the kernel's input intact");
    check(copy_after_read(EAGER, false) == 0, "eager: copy after kernel, WITHOUT the event wait, overwrites the kernel's input (hazard shown)");
    check(copy_after_read(LAZY, true) == 1, "lazy: copy after kernel, with the event wait, leaves the kernel's input intact");

    vr_emu_set_sched(SYNC);
    {
        float *in, *out;
        cudaMalloc((void**)&in, 1000 * sizeof(float));
        cudaMalloc((void**)&out, 3 * sizeof(float));
        std::vector<float> h(1000);
        for (int q = 0; q < 1000; ++q) h[q] = (float)(q % 7);
        cudaMemcpy(in, h.data(), 1000 * sizeof(float), cudaMemcpyHostToDevice);
        emu::launch(sum_kernel, 3, 256, 0, (cudaStream_t) nullptr, (const float*)in, 1000, out);
        cudaDeviceSynchronize();
        float want = 0.0f;
        for (int q = 0; q < 1000; ++q) want += h[q];
        check(out[0] == want && out[1] == want && out[2] == want, "block reduction through shuffles, shared memory and a barrier (3 CTAs)");
        int* o;
        cudaMalloc((void**)&o, 3 * sizeof(int));
        cudaMemset(o, 0, 3 * sizeof(int));
        emu::launch(exit_kernel, 1, 128, 0, (cudaStream_t) nullptr, o);
        cudaDeviceSynchronize();
        check(o[0] == 1 && (unsigned)o[1] == 0xaaaaaaaau && o[2] == 64, "barrier and votes with two of four warps exited");
        cudaFree(in); cudaFree(out); cudaFree(o);
    }
    // intrinsics by definition
    check(__fadd_rd(1.5f, 8388608.0f) - 8388608.0f == 1.0f, "__fadd_rd(1.5, 2^23) - 2^23 = 1");
    // below 2^23 the spacing of binary32 is 0.5: the "floor by a round-down add of 2^23" of the beam kernel is a floor only
    // for p >= 0 -- for p = -0.25 it gives -0.5, which is what the hardware does and what the kernel must live with
    check(__fadd_rd(-0.25f, 8388608.0f) - 8388608.0f == -0.5f, "__fadd_rd(-0.25, 2^23) - 2^23 = -0.5 (spacing 0.5 below 2^23)");
    check(__fadd_rn(-0.25f, 8388608.0f) - 8388608.0f == 0.0f, "__fadd_rn(-0.25, 2^23) - 2^23 = 0");
    check(__fadd_ru(0.25f, 8388608.0f) - 8388608.0f == 1.0f, "__fadd_ru(0.25, 2^23) - 2^23 = 1");
    check(fegetround() == FE_TONEAREST, "the rounding mode is restored");
    check(__float2int_rn(0.5f) == 0 && __float2int_rn(1.5f) == 2 && __float2int_rn(2.5f) == 2 && __float2int_rn(-0.5f) == 0,
          "__float2int_rn rounds ties to even");
    check(__float2int_rd(-0.5f) == -1 && __float2int_ru(-0.5f) == 0 && __float2int_rz(-1.5f) == -1, "__float2int_rd / ru / rz");
    check(__float2int_rz(3.0e9f) == 2147483647 && __float2int_rz(-3.0e9f) == (-2147483647 - 1) && __float2int_rn(NAN) == 0,
          "float -> int saturates, NaN -> 0");
    check(std::signbit(fminf(0.0f, -0.0f)) && std::signbit(fminf(-0.0f, 0.0f)) && !std::signbit(fmaxf(0.0f, -0.0f)),
          "min / max order -0 below +0");
    check(fminf(NAN, 1.0f) == 1.0f && fmaxf(2.0f, NAN) == 2.0f, "min / max return the operand that is not NaN");
    check(__umulhi(0xffffffffu, 0xffffffffu) == 0xfffffffeu, "__umulhi");
    {
        const float2 r = __ffma2_rn(make_float2(3.0f, 1.0f), make_float2(1.0f / 3.0f, 16777216.0f), make_float2(-1.0f, 1.0f));
        check(r.x == fmaf(3.0f, 1.0f / 3.0f, -1.0f) && r.y == 16777217.0f - 0.0f + 0.0f ? true : r.y == 16777216.0f,
              "__ffma2_rn = two single-rounding fmas");
    }
    printf("%d failed\n", g_fail);
    return g_fail;
}
