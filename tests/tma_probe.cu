// tma_probe.cu -- standalone check of the TMA mechanics the beam kernel relies on (test infrastructure).
//   tma_probe <mode> [bx by bz [ox oy oz [nx ny nz]]]
// mode 0: tensor map passed as a __grid_constant__ kernel parameter; 1: in global memory, no fence;
// 2: in global memory, acquired with fence.proxy.tensormap::generic.acquire.sys before use (what
// csrc/vr_beam.cu does).  Loads one 3-D box of a float32 cube into shared memory, copies it out and
// compares with the host (out-of-range voxels must read 0).  Exit code 0 = match.
#include <cuda.h>
#include <cuda_runtime.h>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>
#include <stdint.h>
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__global__ void probe(const __grid_constant__ CUtensorMap pm, const void* gm, int use_global, int x, int y, int z,
                      int nfloats, float* out)
{
    extern __shared__ __align__(128) unsigned char s_dyn[];
    __shared__ uint64_t bar;
    float* buf = (float*)s_dyn;
    if (threadIdx.x == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(&bar)), "r"(1) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        const void* map = use_global ? gm : (const void*)&pm;
        if (use_global == 2) asm volatile("fence.proxy.tensormap::generic.acquire.sys [%0], 128;" ::"l"(map) : "memory");
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(&bar)), "r"(nfloats * 4) : "memory");
        asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                     ::"r"(smem_u32(buf)), "l"(map), "r"(x), "r"(y), "r"(z), "r"(smem_u32(&bar)) : "memory");
    }
    uint32_t ok;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(smem_u32(&bar)), "r"(0) : "memory");
    } while (!ok);
    for (int q = threadIdx.x; q < nfloats; q += blockDim.x) out[q] = buf[q];
}
int main(int argc, char** argv)
{
    int n[3] = {64, 64, 64};
    int box[3] = {12, 5, 9};
    int org[3] = {3, 4, 5};
    int use_global = 0;
    if (argc > 1) use_global = atoi(argv[1]);
    if (argc > 4) { box[0] = atoi(argv[2]); box[1] = atoi(argv[3]); box[2] = atoi(argv[4]); }
    if (argc > 7) { org[0] = atoi(argv[5]); org[1] = atoi(argv[6]); org[2] = atoi(argv[7]); }
    if (argc > 10) { n[0] = atoi(argv[8]); n[1] = atoi(argv[9]); n[2] = atoi(argv[10]); }
    size_t nv = (size_t)n[0] * n[1] * n[2];
    std::vector<float> h(nv);
    for (size_t q = 0; q < nv; ++q) h[q] = (float)q + 1.0f;
    float* d; cudaMalloc(&d, nv * 4); cudaMemcpy(d, h.data(), nv * 4, cudaMemcpyHostToDevice);
    void* fn = nullptr; cudaDriverEntryPointQueryResult qr;
    cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr);
    EncodeTiledFn encode = (EncodeTiledFn)fn;
    CUtensorMap m; memset(&m, 0, sizeof(m));
    cuuint64_t gdim[3] = {(cuuint64_t)n[0], (cuuint64_t)n[1], (cuuint64_t)n[2]};
    cuuint64_t gstr[2] = {(cuuint64_t)n[0] * 4, (cuuint64_t)n[0] * n[1] * 4};
    cuuint32_t bx[3] = {(cuuint32_t)box[0], (cuuint32_t)box[1], (cuuint32_t)box[2]};
    cuuint32_t es[3] = {1, 1, 1};
    CUresult r = encode(&m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, d, gdim, gstr, bx, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                        CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    printf("encode rc=%d global=%d box=%d,%d,%d org=%d,%d,%d n=%d,%d,%d\n", (int)r, use_global, box[0], box[1], box[2], org[0], org[1], org[2], n[0], n[1], n[2]);
    if (r != CUDA_SUCCESS) return 1;
    void* gm; cudaMalloc(&gm, 128); cudaMemcpy(gm, &m, 128, cudaMemcpyHostToDevice);
    int nf = box[0] * box[1] * box[2];
    float* out; cudaMalloc(&out, nf * 4);
    probe<<<1, 128, nf * 4 + 128>>>(m, gm, use_global, org[0], org[1], org[2], nf, out);
    cudaError_t e = cudaDeviceSynchronize();
    printf("kernel: %s\n", cudaGetErrorString(e));
    if (e != cudaSuccess) return 2;
    std::vector<float> o(nf); cudaMemcpy(o.data(), out, nf * 4, cudaMemcpyDeviceToHost);
    int bad = 0;
    for (int z = 0; z < box[2]; ++z) for (int y = 0; y < box[1]; ++y) for (int x = 0; x < box[0]; ++x) {
        int gx = org[0] + x, gy = org[1] + y, gz = org[2] + z;
        float want = (gx < 0 || gy < 0 || gz < 0 || gx >= n[0] || gy >= n[1] || gz >= n[2]) ? 0.0f : h[((size_t)gz * n[1] + gy) * n[0] + gx];
        if (o[(z * box[1] + y) * box[0] + x] != want) ++bad;
    }
    printf("mismatches: %d of %d\n", bad, nf);
    return bad != 0;
}
