// energy.cu -- total-energy diagnostic on the device ("error in total
// energy of the system that is the sum of kinetic and potential energy"; R23).
//
//   T = sum_i 1/2 m_i |v_i|^2,     W = - G sum_{i<j} m_i m_j / sqrt(r_ij^2 + eps^2)
//
// W is the potential of the UNSPLIT softened force (Eq. 1-2): hard + soft add up to it for any K.  It is
// summed directly over all pairs -- a diagnostic beside the hot path, exact up to fp32 rounding of each
// pair term; 2^20 bodies take a fraction of a second.  Pair terms are fp32, every 256 of them are
// added to an fp64 accumulator; the per-block partial sums are combined in a fixed order, so the result
// does not depend on the scheduling of the blocks.
#include "common.cuh"

namespace hyb {

constexpr int EN_THREADS = 256;
constexpr int EN_SINKS = 2 * EN_THREADS;      // two sinks per thread share every shared-memory read

__device__ __forceinline__ double block_sum(double v, double *sh)
{
#pragma unroll
    for (int off = 16; off; off >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, off);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0) sh[warp] = v;
    __syncthreads();
    double s = 0.0;
    if (threadIdx.x == 0)
        for (int w = 0; w < EN_THREADS / 32; w++) s += sh[w];
    return s;                                  // valid in thread 0
}

// block (x, y): sinks [512 x, 512 x + 512), sources [y jchunk, (y + 1) jchunk); part[y gridDim.x + x] =
// sum over those sinks i and sources j != i of m_i m_j / sqrt(r_ij^2 + eps^2)
__global__ void __launch_bounds__(EN_THREADS) energy_pot_kernel(const float4 *__restrict__ pos, u32 n, float eps2,
                                                                u32 jchunk, double *__restrict__ part)
{
    __shared__ float4 tile[EN_THREADS];
    __shared__ double sh[EN_THREADS / 32];
    const u32 ib = blockIdx.x * EN_SINKS;
    const u32 i0 = ib + threadIdx.x, i1 = i0 + EN_THREADS;
    const float4 p0 = i0 < n ? pos[i0] : make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    const float4 p1 = i1 < n ? pos[i1] : make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    const u32 jbeg = blockIdx.y * jchunk, jend = min(n, jbeg + jchunk);
    double acc0 = 0.0, acc1 = 0.0;
    for (u32 jt = jbeg; jt < jend; jt += EN_THREADS) {
        const u32 j = jt + threadIdx.x;
        tile[threadIdx.x] = j < jend ? pos[j] : make_float4(0.0f, 0.0f, 0.0f, 0.0f);     // padding: mass 0
        __syncthreads();
        float s0 = 0.0f, s1 = 0.0f;
        const bool diag = jt < ib + EN_SINKS && jt + EN_THREADS > ib;      // the tile may hold a sink itself
        if (!diag) {
#pragma unroll 8
            for (int k = 0; k < EN_THREADS; k++) {
                const float4 q = tile[k];
                const float ax = q.x - p0.x, ay = q.y - p0.y, az = q.z - p0.z;
                const float bx = q.x - p1.x, by = q.y - p1.y, bz = q.z - p1.z;
                s0 = fmaf(q.w, rsqrtf(fmaf(ax, ax, fmaf(ay, ay, fmaf(az, az, eps2)))), s0);
                s1 = fmaf(q.w, rsqrtf(fmaf(bx, bx, fmaf(by, by, fmaf(bz, bz, eps2)))), s1);
            }
        } else {
#pragma unroll 4
            for (int k = 0; k < EN_THREADS; k++) {
                const float4 q = tile[k];
                const float ax = q.x - p0.x, ay = q.y - p0.y, az = q.z - p0.z;
                const float bx = q.x - p1.x, by = q.y - p1.y, bz = q.z - p1.z;
                const float t0 = q.w * rsqrtf(fmaf(ax, ax, fmaf(ay, ay, fmaf(az, az, eps2))));
                const float t1 = q.w * rsqrtf(fmaf(bx, bx, fmaf(by, by, fmaf(bz, bz, eps2))));
                s0 += (jt + (u32)k != i0) ? t0 : 0.0f;
                s1 += (jt + (u32)k != i1) ? t1 : 0.0f;
            }
        }
        acc0 += (double)s0; acc1 += (double)s1;
        __syncthreads();
    }
    const double w = (double)p0.w * acc0 + (double)p1.w * acc1;      // sinks beyond n have mass 0
    const double s = block_sum(w, sh);
    if (threadIdx.x == 0) part[(size_t)blockIdx.y * gridDim.x + blockIdx.x] = s;
}

// part[b] = sum over the particles of block b (grid-stride in a fixed pattern) of 1/2 m v^2
__global__ void __launch_bounds__(EN_THREADS) energy_kin_kernel(const float4 *__restrict__ pos, const float4 *__restrict__ vel,
                                                                u32 n, double *__restrict__ part)
{
    __shared__ double sh[EN_THREADS / 32];
    double k = 0.0;
    for (u32 i = blockIdx.x * EN_THREADS + threadIdx.x; i < n; i += gridDim.x * EN_THREADS) {
        const float4 v = vel[i];
        const double vx = v.x, vy = v.y, vz = v.z;
        k += 0.5 * (double)pos[i].w * (vx * vx + vy * vy + vz * vz);
    }
    const double s = block_sum(k, sh);
    if (threadIdx.x == 0) part[blockIdx.x] = s;
}

// out[0] = sum kin[0 .. nk), out[1] = -G/2 sum pot[0 .. np)   (every pair was counted from both ends)
__global__ void __launch_bounds__(EN_THREADS) energy_final_kernel(const double *__restrict__ kin, u32 nk,
                                                                  const double *__restrict__ pot, u32 np, float G,
                                                                  double *__restrict__ out)
{
    __shared__ double sh[EN_THREADS / 32];
    double a = 0.0, b = 0.0;
    for (u32 i = threadIdx.x; i < nk; i += EN_THREADS) a += kin[i];
    for (u32 i = threadIdx.x; i < np; i += EN_THREADS) b += pot[i];
    const double sa = block_sum(a, sh);
    __syncthreads();
    const double sb = block_sum(b, sh);
    if (threadIdx.x == 0) { out[0] = sa; out[1] = -0.5 * (double)G * sb; }
}

size_t energy_scratch_doubles(const Ctx *c, u32 *ni, u32 *nj, u32 *nk)
{
    const u32 n = (u32)c->n;
    *ni = (n + EN_SINKS - 1) / EN_SINKS;
    // enough source chunks to fill the machine a few times over when there are few sink tiles
    const u32 want = (u32)c->num_sms * 8u;
    u32 y = *ni >= want ? 1u : (want + *ni - 1) / *ni;
    const u32 jtiles = (n + EN_THREADS - 1) / EN_THREADS;
    if (y > jtiles) y = jtiles;
    *nj = y;
    *nk = (u32)imin64((n + EN_THREADS - 1) / EN_THREADS, (int64_t)c->num_sms * 4);
    return (size_t)*ni * *nj + *nk + 2;
}

cudaError_t launch_energy(Ctx *c, double *d_scratch, u32 ni, u32 nj, u32 nk)
{
    const u32 n = (u32)c->n;
    const float4 *pos = reinterpret_cast<const float4 *>(c->pos), *vel = reinterpret_cast<const float4 *>(c->vel);
    double *out = d_scratch, *kin = d_scratch + 2, *pot = kin + nk;
    const u32 jtiles = (n + EN_THREADS - 1) / EN_THREADS;
    const u32 jchunk = ((jtiles + nj - 1) / nj) * EN_THREADS;
    energy_kin_kernel<<<nk, EN_THREADS, 0, c->stream>>>(pos, vel, n, kin);
    energy_pot_kernel<<<dim3(ni, nj), EN_THREADS, 0, c->stream>>>(pos, n, c->p.eps * c->p.eps, jchunk, pot);
    energy_final_kernel<<<1, EN_THREADS, 0, c->stream>>>(kin, nk, pot, ni * nj, c->p.G, out);
    return cudaGetLastError();
}

// ------------------------------------------------------------------ hyb_energy_noalloc (include/hyb.h)
// The same three kernels with their partial sums in a file-scope device array instead of a context's workspace, for
// callers that can neither allocate device memory nor hold a context.  Every GPU that loads the library holds the
// array (128 KiB) until the process ends.  In host code the name of the array is a host-side stand-in, not a device
// address: the address comes from cudaGetSymbolAddress, once per device, with that device current.
constexpr size_t EN_STATIC_DOUBLES = 16384;
static __device__ __align__(256) double g_energy_scratch[EN_STATIC_DOUBLES];

// *too_large: the partial sums of n particles do not fit (the caller reports it; nothing was launched).
// Nothing in the array has to start from zero: each kernel writes every element the next one reads.
cudaError_t launch_energy_noalloc(const hyb_float4 *d_pos_m, const hyb_float4 *d_vel, int64_t n, float G, float eps, int device,
                                  cudaStream_t st, double *d_energy, bool *too_large)
{
    static unsigned long long ready = 0ull;
    static double *scratch_of[64];
    static int sms_of[64];
    *too_large = false;
    double *scratch = nullptr;
    int sms = 0;
    if (device >= 0 && device < 64 && device_ready(&ready, device)) { scratch = scratch_of[device]; sms = sms_of[device]; }
    else {
        cudaError_t e = cudaGetSymbolAddress((void **)&scratch, g_energy_scratch);      // of the current device (set by the caller)
        if (e != cudaSuccess) return e;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
        if (e != cudaSuccess) return e;
        if (device >= 0 && device < 64) { scratch_of[device] = scratch; sms_of[device] = sms; device_set_ready(&ready, device); }
    }
    Ctx c{};                      // the launch geometry and the launches are those of hyb_energy (same bits)
    c.n = n; c.num_sms = sms; c.stream = st; c.device = device;
    c.pos = const_cast<hyb_float4 *>(d_pos_m); c.vel = const_cast<hyb_float4 *>(d_vel);
    c.p.G = G; c.p.eps = eps;
    u32 ni, nj, nk;
    if (energy_scratch_doubles(&c, &ni, &nj, &nk) > EN_STATIC_DOUBLES) { *too_large = true; return cudaSuccess; }
    cudaError_t e = launch_energy(&c, scratch, ni, nj, nk);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_energy, scratch, 2 * sizeof(double), cudaMemcpyDeviceToDevice, st);
    return e;
}

}  // namespace hyb
