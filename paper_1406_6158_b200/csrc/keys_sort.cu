// keys_sort.cu -- steps a1-a4: bounding box, 63-bit Morton keys, stable onesweep radix sort,
// re-order of the particle store.  (T2-T6.)
#include "common.cuh"
#include "sort.cuh"

namespace hyb {

// ------------------------------------------------------------------ a1: bounding box (T1, T2)
__global__ void __launch_bounds__(256) bbox_kernel(const float4 *__restrict__ pos, u32 n, DevCtl *ctl)
{
    float lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
    bool bad = false;
    for (u32 i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        float4 p = __ldg(pos + i);
        bad |= !(isfinite(p.x) && isfinite(p.y) && isfinite(p.z) && isfinite(p.w)) || p.w < 0.0f;
        lo[0] = fminf(lo[0], p.x); hi[0] = fmaxf(hi[0], p.x);
        lo[1] = fminf(lo[1], p.y); hi[1] = fmaxf(hi[1], p.y);
        lo[2] = fminf(lo[2], p.z); hi[2] = fmaxf(hi[2], p.z);
    }
    bbox_block_reduce(lo, hi, bad, ctl);
}

// ------------------------------------------------------------------ a2: keys (T4, T5)
__device__ __forceinline__ u64 spread21(u32 q)
{
    u64 x = q & 0x1FFFFFu;
    x = (x | (x << 32)) & 0x001F00000000FFFFull;
    x = (x | (x << 16)) & 0x001F0000FF0000FFull;
    x = (x | (x << 8)) & 0x100F00F00F00F00Full;
    x = (x | (x << 4)) & 0x10C30C30C30C30C3ull;
    x = (x | (x << 2)) & 0x1249249249249249ull;
    return x;
}

__device__ __forceinline__ u32 quantise(float x, double o, double inv)
{
    double s = __dmul_rn(__dsub_rn((double)x, o), inv);
    double f = floor(s);
    return f >= 2097151.0 ? 2097151u : (f > 0.0 ? (u32)f : 0u);
}

constexpr int KEYS_THREADS = 1024;      // few CTAs (each ends with up to 2048 global atomics), many warps (the loop is a chain of latencies)
// also accumulates the eight 8-bit digit histograms the onesweep sort needs; its last CTA turns them into bases
__global__ void __launch_bounds__(KEYS_THREADS) keys_kernel(const float4 *__restrict__ pos, u32 n, DevCtl *ctl,
                                                   u64 *__restrict__ key)
{
    __shared__ u32 hist[RS_PASSES * 256];
    for (int i = threadIdx.x; i < RS_PASSES * 256; i += blockDim.x) hist[i] = 0;
    // the box reduction has been consumed (root cube derived): clear it for the next bbox_kernel / drift
    if (blockIdx.x == 0 && threadIdx.x < 7) (&ctl->bbox_enc[0])[threadIdx.x] = 0u;      // bbox_enc[6], bbox_done
    __syncthreads();
    const double ox = ctl->origin[0], oy = ctl->origin[1], oz = ctl->origin[2], inv = ctl->inv;
    for (u32 i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        float4 p = __ldg(pos + i);
        u64 k = (spread21(quantise(p.x, ox, inv)) << 2) | (spread21(quantise(p.y, oy, inv)) << 1) |
                spread21(quantise(p.z, oz, inv));
        key[i] = k;
#pragma unroll
        for (int d = 0; d < RS_PASSES; d++) atomicAdd(&hist[d * 256 + (u32)((k >> (8 * d)) & 0xFF)], 1u);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < RS_PASSES * 256; i += blockDim.x)
        if (hist[i]) atomicAdd(&ctl->digit_hist[i], hist[i]);
    // the last CTA to get here sees the complete histograms: exclusive scan of each 256-bin histogram -> digit_base
    __shared__ bool last;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) last = atomicAdd(&ctl->tile_counter[13], 1u) == gridDim.x - 1;
    __syncthreads();
    if (!last || threadIdx.x >= 256) return;
    __threadfence();
    {   // warp w scans the histogram of pass w: lane l takes bins 8 l .. 8 l + 7
        static_assert(RS_PASSES == 8 && KEYS_THREADS >= 256, "one warp of the CTA's first eight per pass");
        const int pass = threadIdx.x >> 5, lane = threadIdx.x & 31;
        u32 v[8], sum = 0;
#pragma unroll
        for (int i = 0; i < 8; i++) { v[i] = ld_volatile_u32(&ctl->digit_hist[pass * 256 + 8 * lane + i]); sum += v[i]; }
        u32 incl = sum;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const u32 t = __shfl_up_sync(0xFFFFFFFFu, incl, off);
            if (lane >= off) incl += t;
        }
        u32 run = incl - sum;
#pragma unroll
        for (int i = 0; i < 8; i++) { ctl->digit_base[pass * 256 + 8 * lane + i] = run; run += v[i]; }
    }
}

// ------------------------------------------------------------------ a4: re-order (T6)
__global__ void __launch_bounds__(256) permute_kernel(const u32 *__restrict__ perm, u32 n,
                                                      const float4 *__restrict__ pos, const float4 *__restrict__ vel,
                                                      const u32 *__restrict__ id, float4 *__restrict__ pos_o,
                                                      float4 *__restrict__ vel_o, u32 *__restrict__ id_o)
{
    for (u32 j = blockIdx.x * blockDim.x + threadIdx.x; j < n; j += gridDim.x * blockDim.x) {
        u32 s = perm[j];
        pos_o[j] = __ldg(pos + s);
        vel_o[j] = __ldg(vel + s);
        id_o[j] = __ldg(id + s);
    }
}

cudaError_t launch_keys_sort_permute(Ctx *c)
{
    const Layout &L = c->L;
    const u32 n = (u32)c->n;
    cudaStream_t st = c->stream;
    DevCtl *ctl = c->ctl;
    const int grid = (int)imin64((c->n + 255) / 256, (int64_t)c->num_sms * 8);

    // the drift of hyb_step has already reduced the box of the positions it wrote (integrate.cu)
    if (!c->bbox_ready) bbox_kernel<<<grid, 256, 0, st>>>(reinterpret_cast<const float4 *>(c->pos), n, ctl);
    c->bbox_ready = false;
    u64 *key_orig = wsptr<u64>(c, L.key_orig), *key_a = wsptr<u64>(c, L.key_a), *key_b = wsptr<u64>(c, L.key_b);
    u32 *val_a = wsptr<u32>(c, L.val_a), *val_b = wsptr<u32>(c, L.val_b);
    // few CTAs: every CTA ends with up to 2048 global atomics for its share of the digit histograms
    const int kgrid = (int)imin64((c->n + KEYS_THREADS - 1) / KEYS_THREADS, (int64_t)c->num_sms * 2);
    keys_kernel<<<kgrid, KEYS_THREADS, 0, st>>>(reinterpret_cast<const float4 *>(c->pos), n, ctl, key_orig);

    u32 *status = wsptr<u32>(c, L.rs_status);
    const int sgrid = (int)imin64(L.rs_tiles, (int64_t)c->num_sms * 3);
    const u64 *kin = key_orig; const u32 *vin = nullptr;
    for (int pass = 0; pass < RS_PASSES; pass++) {
        u64 *kout = (pass & 1) ? key_b : key_a;
        u32 *vout = (pass & 1) ? val_b : val_a;
        cudaError_t e = launch_radix_pass<u64>(kin, vin, kout, vout, nullptr, n, nullptr, 8 * pass,
                                               ctl->digit_base + pass * 256,
                                               status + (size_t)pass * (L.rs_tiles + L.rs_blocks) * 256, (u32)L.rs_tiles,
                                               &ctl->tile_counter[pass], &ctl->status, sgrid, st, c->device, L.rs_kpt);
        if (e != cudaSuccess) return e;
        kin = kout; vin = vout;
    }
    // RS_PASSES is even: sorted keys in key_b, permutation in val_b.
    // The re-order of the store runs on the auxiliary stream, next to the octree build (which needs
    // only the sorted keys); later stages read the permuted positions from pos_tmp.
    cudaStream_t ax = c->aux;
    cudaEventRecord(c->ev_sorted, st);
    cudaStreamWaitEvent(ax, c->ev_sorted, 0);
    float4 *pos_w = wsptr<float4>(c, L.pos_tmp), *vel_w = wsptr<float4>(c, L.vel_tmp);
    u32 *id_w = wsptr<u32>(c, L.id_tmp);
    // destination: the copy the store is not in
    float4 *pos_t = c->store_away ? reinterpret_cast<float4 *>(c->pos_home) : pos_w;
    float4 *vel_t = c->store_away ? reinterpret_cast<float4 *>(c->vel_home) : vel_w;
    u32 *id_t = c->store_away ? c->id_home : id_w;
    permute_kernel<<<grid, 256, 0, ax>>>(val_b, n, reinterpret_cast<const float4 *>(c->pos),
                                         reinterpret_cast<const float4 *>(c->vel), c->id, pos_t, vel_t, id_t);
    cudaEventRecord(c->ev_perm, ax);
    c->pos_sorted = pos_t;
    if (c->store_away) {                    // re-ordered straight into the caller's arrays
        c->pos = c->pos_home; c->vel = c->vel_home; c->id = c->id_home; c->store_away = false;
    } else if (c->defer_copy) {             // hyb_step: stay in the workspace copy until the next build
        c->pos = reinterpret_cast<hyb_float4 *>(pos_w); c->vel = reinterpret_cast<hyb_float4 *>(vel_w); c->id = id_w;
        c->store_away = true;
    } else {
        cudaMemcpyAsync(c->pos, pos_t, sizeof(float4) * (size_t)n, cudaMemcpyDeviceToDevice, ax);
        cudaMemcpyAsync(c->vel, vel_t, sizeof(float4) * (size_t)n, cudaMemcpyDeviceToDevice, ax);
        cudaMemcpyAsync(c->id, id_t, sizeof(u32) * (size_t)n, cudaMemcpyDeviceToDevice, ax);
    }
    return cudaGetLastError();
}

cudaError_t store_come_home(Ctx *c)
{
    if (!c->store_away) return cudaSuccess;
    const size_t n = (size_t)c->n;
    cudaMemcpyAsync(c->pos_home, c->pos, sizeof(float4) * n, cudaMemcpyDeviceToDevice, c->stream);
    cudaMemcpyAsync(c->vel_home, c->vel, sizeof(float4) * n, cudaMemcpyDeviceToDevice, c->stream);
    cudaMemcpyAsync(c->id_home, c->id, sizeof(u32) * n, cudaMemcpyDeviceToDevice, c->stream);
    c->pos = c->pos_home; c->vel = c->vel_home; c->id = c->id_home; c->store_away = false;
    return cudaGetLastError();
}

}  // namespace hyb
