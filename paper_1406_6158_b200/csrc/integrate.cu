// integrate.cu -- step a10: fused leapfrog kick / drift (Eq. 3-4; R21).
#include "common.cuh"

namespace hyb {

// v += c_soft a_soft + c_hard a_hard;  x += dt_drift v   (dt_drift == 0: kick only)
// BBOX: the kernel also reduces the bounding box (and checks the validity) of the positions it writes and
// derives the root cube, so that the tree build that follows starts at the keys (a1 folded into a10).
template <bool BBOX>
__global__ void __launch_bounds__(256) kick_drift_kernel(float4 *__restrict__ pos, float4 *__restrict__ vel,
                                                         const float4 *__restrict__ a_soft,
                                                         const float4 *__restrict__ a_hard, u32 n, float c_soft,
                                                         float c_hard, float dt_drift, DevCtl *ctl)
{
    float lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
    bool bad = false;
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
            if (BBOX) {
                bad |= !(isfinite(p.x) && isfinite(p.y) && isfinite(p.z) && isfinite(p.w)) || p.w < 0.0f;
                lo[0] = fminf(lo[0], p.x); hi[0] = fmaxf(hi[0], p.x);
                lo[1] = fminf(lo[1], p.y); hi[1] = fmaxf(hi[1], p.y);
                lo[2] = fminf(lo[2], p.z); hi[2] = fmaxf(hi[2], p.z);
            }
        }
    }
    if (BBOX) bbox_block_reduce(lo, hi, bad, ctl);
}

cudaError_t launch_kick_drift(Ctx *c, float c_soft, float c_hard, float dt_drift, bool with_bbox)
{
    const int grid = (int)imin64((c->n + 255) / 256, (int64_t)c->num_sms * 8);
    float4 *pos = reinterpret_cast<float4 *>(c->pos), *vel = reinterpret_cast<float4 *>(c->vel);
    const float4 *as = reinterpret_cast<const float4 *>(c->a_soft), *ah = reinterpret_cast<const float4 *>(c->a_hard);
    if (with_bbox && dt_drift != 0.0f) {
        kick_drift_kernel<true><<<grid, 256, 0, c->stream>>>(pos, vel, as, ah, (u32)c->n, c_soft, c_hard, dt_drift, c->ctl);
        c->bbox_ready = true;
    } else {
        kick_drift_kernel<false><<<grid, 256, 0, c->stream>>>(pos, vel, as, ah, (u32)c->n, c_soft, c_hard, dt_drift, c->ctl);
    }
    return cudaGetLastError();
}

}  // namespace hyb
