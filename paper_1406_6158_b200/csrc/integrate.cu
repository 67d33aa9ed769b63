// integrate.cu -- step a10: fused leapfrog kick / drift (Eq. 3-4; R21).
#include "common.cuh"

namespace hyb {

// v += c_soft a_soft + c_hard a_hard;  x += dt_drift v   (dt_drift == 0: kick only)
__global__ void __launch_bounds__(256) kick_drift_kernel(float4 *__restrict__ pos, float4 *__restrict__ vel,
                                                         const float4 *__restrict__ a_soft,
                                                         const float4 *__restrict__ a_hard, u32 n, float c_soft,
                                                         float c_hard, float dt_drift)
{
    for (u32 i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        float4 v = vel[i];
        if (c_soft != 0.0f) {
            const float4 s = __ldg(a_soft + i);
            v.x = fmaf(c_soft, s.x, v.x); v.y = fmaf(c_soft, s.y, v.y); v.z = fmaf(c_soft, s.z, v.z);
        }
        if (c_hard != 0.0f) {
            const float4 h = __ldg(a_hard + i);
            v.x = fmaf(c_hard, h.x, v.x); v.y = fmaf(c_hard, h.y, v.y); v.z = fmaf(c_hard, h.z, v.z);
        }
        vel[i] = v;
        if (dt_drift != 0.0f) {
            float4 p = pos[i];
            p.x = fmaf(dt_drift, v.x, p.x); p.y = fmaf(dt_drift, v.y, p.y); p.z = fmaf(dt_drift, v.z, p.z);
            pos[i] = p;
        }
    }
}

cudaError_t launch_kick_drift(Ctx *c, float c_soft, float c_hard, float dt_drift)
{
    const int grid = (int)imin64((c->n + 255) / 256, (int64_t)c->num_sms * 8);
    kick_drift_kernel<<<grid, 256, 0, c->stream>>>(reinterpret_cast<float4 *>(c->pos), reinterpret_cast<float4 *>(c->vel),
                                                   reinterpret_cast<const float4 *>(c->a_soft),
                                                   reinterpret_cast<const float4 *>(c->a_hard), (u32)c->n, c_soft,
                                                   c_hard, dt_drift);
    return cudaGetLastError();
}

}  // namespace hyb
