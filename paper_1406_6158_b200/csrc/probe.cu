// probe.cu -- measures the FP32 CUDA-core rate the force kernels are bounded by (the roofline denominator
// bench.py reports beside the derived one): independent chains of packed fma.rn.f32x2 (the form the pair
// kernels of pairs.cuh use) and of scalar fma.rn.f32, nothing else in the loop.  Not on the hot path.
#include "common.cuh"

namespace hyb {

template <bool PACKED>
__global__ void __launch_bounds__(512) fp32_probe_kernel(float *out, int iters, float a, float b)
{
    if (PACKED) {
        unsigned long long x[8];
        const unsigned long long aa = ((unsigned long long)__float_as_uint(a) << 32) | __float_as_uint(a);
        const unsigned long long bb = ((unsigned long long)__float_as_uint(b) << 32) | __float_as_uint(b);
#pragma unroll
        for (int i = 0; i < 8; i++) x[i] = ((unsigned long long)__float_as_uint((float)(threadIdx.x + i)) << 32) | (unsigned)i;
        for (int it = 0; it < iters; it++) {
#pragma unroll
            for (int i = 0; i < 8; i++) asm volatile("fma.rn.f32x2 %0, %1, %0, %2;" : "+l"(x[i]) : "l"(aa), "l"(bb));
        }
        unsigned long long s = 0;
#pragma unroll
        for (int i = 0; i < 8; i++) s ^= x[i];
        out[blockIdx.x * blockDim.x + threadIdx.x] = __uint_as_float((unsigned)s ^ (unsigned)(s >> 32));
    } else {
        float x[8];
#pragma unroll
        for (int i = 0; i < 8; i++) x[i] = (float)(threadIdx.x + i);
        for (int it = 0; it < iters; it++) {
#pragma unroll
            for (int i = 0; i < 8; i++) asm volatile("fma.rn.f32 %0, %1, %0, %2;" : "+f"(x[i]) : "f"(a), "f"(b));
        }
        float s = 0.0f;
#pragma unroll
        for (int i = 0; i < 8; i++) s += x[i];
        out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    }
}

}  // namespace hyb

using namespace hyb;

extern "C" int hyb_probe_fp32(int device, void *cuda_stream, float *d_scratch, size_t scratch_floats, double *h_tflops)
{
    if (!d_scratch || !h_tflops) return HYB_ERR_INVALID_ARG;
    if (cudaSetDevice(device) != cudaSuccess) return HYB_ERR_CUDA;
    int sms = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess) return HYB_ERR_CUDA;
    const int block = 512, grid = sms * 2, iters = 20000;
    if (scratch_floats < (size_t)block * grid) return HYB_ERR_WORKSPACE_TOO_SMALL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return HYB_ERR_CUDA;
    for (int mode = 0; mode < 2; mode++) {
        float best = 1e30f;
        for (int rep = 0; rep < 4; rep++) {         // the first launch warms up
            cudaEventRecord(e0, st);
            if (mode == 0) fp32_probe_kernel<true><<<grid, block, 0, st>>>(d_scratch, iters, 1.0001f, 0.5f);
            else fp32_probe_kernel<false><<<grid, block, 0, st>>>(d_scratch, iters, 1.0001f, 0.5f);
            cudaEventRecord(e1, st);
            if (cudaEventSynchronize(e1) != cudaSuccess) { cudaEventDestroy(e0); cudaEventDestroy(e1); return HYB_ERR_CUDA; }
            float ms = 0.0f;
            cudaEventElapsedTime(&ms, e0, e1);
            if (rep > 0 && ms < best) best = ms;
        }
        h_tflops[mode] = (double)grid * block * iters * 8.0 * 2.0 * (mode == 0 ? 2.0 : 1.0) / ((double)best * 1e9);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    return HYB_OK;
}
