// sort.cuh -- one pass of a stable least-significant-digit radix sort, "onesweep" style:
// every tile ranks its keys locally and obtains the global offset of each of its 256 digit
// buckets by decoupled look-back over the tiles before it, so keys are read once and written
// once per pass.  Stability (ties keep input order, T6) holds because the local rank
// is taken in input order and tile prefixes follow tile order.
#pragma once
#include "common.cuh"

namespace hyb {

constexpr u32 RS_FLAG_AGG = 1u << 30, RS_FLAG_PREFIX = 2u << 30, RS_VALUE_MASK = (1u << 30) - 1;

template <int KPT>
struct RadixSmem {
    u64 keys[RS_THREADS * KPT];
    u32 vals[RS_THREADS * KPT];
    u32 warp_cnt[RS_THREADS / 32][256];
    u32 digit_start[256];
    u32 global_off[256];
    u32 scan_tmp[8];
    u32 tile;
};

// n_dev (optional) overrides n with a device-side count (tree nodes).
// vin == nullptr: values are the global input indices (first pass).
// inv_out (optional): inv_out[value] = output position (the inverse permutation).
template <typename KeyT, int KPT>
__global__ void __launch_bounds__(RS_THREADS) radix_pass_kernel(
    const KeyT *__restrict__ kin, const u32 *__restrict__ vin, KeyT *__restrict__ kout, u32 *__restrict__ vout,
    u32 *__restrict__ inv_out, u32 n_host, const u32 *__restrict__ n_dev, int shift,
    const u32 *__restrict__ digit_base, u32 *status, u32 tiles_alloc, u32 *tile_counter, u32 *dev_status, int static_first)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int RS_KPT = KPT, RS_TILE = RS_THREADS * KPT;      // (shadow the names of the large-run tile)
    RadixSmem<KPT> &sm = *reinterpret_cast<RadixSmem<KPT> *>(smem_raw);
    pdl_begin();
    const u32 n = n_dev ? *n_dev : n_host;
    const u32 ntiles = (n + RS_TILE - 1) / RS_TILE;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const u32 lt_mask = (1u << lane) - 1u;
    // Tile ids are normally drawn from a counter, so that a tile never waits (look-back) for a tile that has not
    // started.  When every CTA of the grid is resident at once (static_first, set by the launcher: the grid is not
    // larger than two CTAs per SM, which registers and shared memory allow) no tile can be left out, and the
    // first tile of a CTA is simply its block index: the pass starts loading without the counter's round trip.
    bool first = static_first != 0;

    for (;;) {
        __syncthreads();   // previous iteration's smem is dead
        if (tid == 0) sm.tile = first ? blockIdx.x : (static_first ? gridDim.x : 0u) + atomicAdd(tile_counter, 1u);
        first = false;
        for (int i = tid; i < (RS_THREADS / 32) * 256; i += RS_THREADS) (&sm.warp_cnt[0][0])[i] = 0;
        __syncthreads();
        const u32 tile = sm.tile;
        if (tile >= ntiles) break;
        const u32 base = tile * RS_TILE + warp * (32 * RS_KPT);
        const u32 tile_n = min((u32)RS_TILE, n - tile * RS_TILE);

        KeyT key[RS_KPT];
        u32 val[RS_KPT];
        u32 rank[RS_KPT];
#pragma unroll
        for (int k = 0; k < RS_KPT; k++) {
            u32 idx = base + k * 32 + lane;
            bool ok = idx < n;
            key[k] = ok ? kin[idx] : (KeyT)0;
            val[k] = ok ? (vin ? vin[idx] : idx) : 0xFFFFFFFFu;
        }
        // stable rank of every key among the keys of this warp with the same digit.  The peer masks come
        // from eight ballots per key (one per digit bit; match.any is far slower when the 32 digits of a
        // warp are mostly distinct, as they are in the low passes) and are independent across the keys;
        // only the counter update below is a serial chain.
        u32 peers[RS_KPT];
#pragma unroll
        for (int k = 0; k < RS_KPT; k++) {
            const bool ok = base + k * 32 + lane < n;
            const u32 d = (u32)((key[k] >> shift) & 0xFF);
            u32 m = __ballot_sync(0xFFFFFFFFu, ok);
#pragma unroll
            for (int b = 0; b < 8; b++) {
                const u32 bal = __ballot_sync(0xFFFFFFFFu, (d >> b) & 1u);
                m &= ((d >> b) & 1u) ? bal : ~bal;
            }
            peers[k] = ok ? m : 0u;
        }
#pragma unroll
        for (int k = 0; k < RS_KPT; k++) {
            const bool ok = peers[k] != 0u;
            const u32 d = (u32)((key[k] >> shift) & 0xFF);
            const u32 c = ok ? sm.warp_cnt[warp][d] : 0u;
            __syncwarp();
            rank[k] = c + __popc(peers[k] & lt_mask);
            if (ok && (peers[k] & lt_mask) == 0) sm.warp_cnt[warp][d] = c + __popc(peers[k]);
            __syncwarp();
        }
        __syncthreads();
        // thread d: exclusive scan of digit d over the warps, tile total
        u32 total = 0;
#pragma unroll
        for (int w = 0; w < RS_THREADS / 32; w++) {
            u32 t = sm.warp_cnt[w][tid];
            sm.warp_cnt[w][tid] = total;
            total += t;
        }
        // publish + look back (thread d for digit d).  All tiles of a pass are usually resident at once
        // and publish at about the same time, so a plain decoupled look-back would walk back to tile 0
        // (O(tiles^2) status reads).  Two levels instead: LB_WIN consecutive tiles form a block; a tile
        // sums the aggregates of the earlier tiles of its block (one round trip); the last tile of a block
        // publishes the block aggregate and looks back over BLOCK statuses, LB_WIN at a time, then
        // publishes the block's inclusive prefix, which the tiles of the next block wait for.
        u32 excl = 0;
        {
            volatile u32 *st = status;
            volatile u32 *bs = status + (size_t)tiles_alloc * 256;
            const u32 blk = tile / LB_WIN, r = tile % LB_WIN;
            st[(size_t)tile * 256 + tid] = RS_FLAG_AGG | total;
            u32 inblk = 0;
            int spins = 0;
            if (r > 0) {
                u32 s[LB_WIN - 1];
                bool ready;
                do {
                    ready = true;
#pragma unroll
                    for (int i = 0; i < LB_WIN - 1; i++)
                        s[i] = ((u32)i < r) ? st[((size_t)blk * LB_WIN + i) * 256 + tid] : (1u << 30);
#pragma unroll
                    for (int i = 0; i < LB_WIN - 1; i++) ready = ready && (s[i] >> 30) != 0u;
                } while (!ready && ++spins < LB_SPIN_LIMIT);
#pragma unroll
                for (int i = 0; i < LB_WIN - 1; i++) inblk += ((u32)i < r) ? (s[i] & RS_VALUE_MASK) : 0u;
            }
            u32 bexcl = 0;
            const bool leader = r == LB_WIN - 1 || tile == ntiles - 1;
            if (leader) {
                const size_t me = (size_t)blk * 256 + tid;
                if (blk == 0) bs[me] = RS_FLAG_PREFIX | (inblk + total);
                else {
                    bs[me] = RS_FLAG_AGG | (inblk + total);
                    long long t = (long long)blk - 1;
                    bool done = false;
                    while (!done) {
                        u32 s[LB_WIN];
#pragma unroll
                        for (int i = 0; i < LB_WIN; i++)
                            s[i] = (t - i >= 0) ? bs[(size_t)(t - i) * 256 + tid] : (2u << 30);
#pragma unroll
                        for (int i = 0; i < LB_WIN; i++) {
                            if (done) break;
                            const u32 f = s[i] >> 30;
                            if (f == 0) break;                   // not published yet: poll again from here
                            bexcl += s[i] & RS_VALUE_MASK;
                            t--;
                            if (f == 2) done = true;
                        }
                        if (!done && ++spins >= LB_SPIN_LIMIT) break;
                    }
                    bs[me] = RS_FLAG_PREFIX | (bexcl + inblk + total);
                }
            } else if (blk > 0) {
                u32 sv;
                do { sv = bs[(size_t)(blk - 1) * 256 + tid]; } while ((sv >> 30) != 2u && ++spins < LB_SPIN_LIMIT);
                bexcl = sv & RS_VALUE_MASK;
            }
            if (spins >= LB_SPIN_LIMIT) atomicOr(dev_status, ST_WAIT_EXPIRED);
            excl = bexcl + inblk;
        }
        // block exclusive scan of the digit totals -> digit_start
        u32 incl = total;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            u32 t = __shfl_up_sync(0xFFFFFFFFu, incl, off);
            if (lane >= off) incl += t;
        }
        if (lane == 31) sm.scan_tmp[warp] = incl;
        __syncthreads();
        u32 wbase = 0;
#pragma unroll
        for (int w = 0; w < RS_THREADS / 32; w++) wbase += (w < warp) ? sm.scan_tmp[w] : 0u;
        const u32 dstart = wbase + incl - total;
        sm.digit_start[tid] = dstart;
        sm.global_off[tid] = digit_base[tid] + excl - dstart;
        __syncthreads();
        // scatter into shared memory in sorted-by-digit order
#pragma unroll
        for (int k = 0; k < RS_KPT; k++) {
            u32 idx = base + k * 32 + lane;
            if (idx < n) {
                u32 d = (u32)((key[k] >> shift) & 0xFF);
                u32 lp = sm.digit_start[d] + sm.warp_cnt[warp][d] + rank[k];
                reinterpret_cast<KeyT *>(sm.keys)[lp] = key[k];
                sm.vals[lp] = val[k];
            }
        }
        __syncthreads();
        for (u32 i = tid; i < tile_n; i += RS_THREADS) {
            KeyT k = reinterpret_cast<KeyT *>(sm.keys)[i];
            u32 d = (u32)((k >> shift) & 0xFF);
            u32 g = sm.global_off[d] + i;
            kout[g] = k;
            u32 v = sm.vals[i];
            vout[g] = v;
            if (inv_out) inv_out[v] = g;
        }
    }
}

template <typename KeyT, int KPT>
static cudaError_t launch_radix_pass_kpt(const KeyT *kin, const u32 *vin, KeyT *kout, u32 *vout, u32 *inv_out, u32 n_host,
                                         const u32 *n_dev, int shift, const u32 *digit_base, u32 *status, u32 tiles_alloc,
                                         u32 *tile_counter, u32 *dev_status, int grid, cudaStream_t st, int device)
{
    static unsigned long long ready = 0ull;
    if (!device_ready(&ready, device)) {
        cudaError_t e = cudaFuncSetAttribute(radix_pass_kernel<KeyT, KPT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)sizeof(RadixSmem<KPT>));
        if (e != cudaSuccess) return e;
        device_set_ready(&ready, device);
    }
    int sms = 0;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
    const int static_first = grid <= 2 * sms ? 1 : 0;
    return launch_pdl(radix_pass_kernel<KeyT, KPT>, dim3((unsigned)grid), dim3(RS_THREADS), sizeof(RadixSmem<KPT>), st, kin, vin, kout,
                      vout, inv_out, n_host, n_dev, shift, digit_base, status, tiles_alloc, tile_counter, dev_status, static_first);
}

// kpt: Layout::rs_kpt (the status arrays were planned for tiles of RS_THREADS x kpt keys)
template <typename KeyT>
static cudaError_t launch_radix_pass(const KeyT *kin, const u32 *vin, KeyT *kout, u32 *vout, u32 *inv_out, u32 n_host,
                                     const u32 *n_dev, int shift, const u32 *digit_base, u32 *status, u32 tiles_alloc,
                                     u32 *tile_counter, u32 *dev_status, int grid, cudaStream_t st, int device, int kpt)
{
    if (kpt == RS_KPT_SMALL)
        return launch_radix_pass_kpt<KeyT, RS_KPT_SMALL>(kin, vin, kout, vout, inv_out, n_host, n_dev, shift, digit_base, status,
                                                        tiles_alloc, tile_counter, dev_status, grid, st, device);
    return launch_radix_pass_kpt<KeyT, RS_KPT>(kin, vin, kout, vout, inv_out, n_host, n_dev, shift, digit_base, status, tiles_alloc,
                                               tile_counter, dev_status, grid, st, device);
}

}  // namespace hyb
