// common.cuh -- shared declarations of the hyb CUDA library (sm_100a).
// Product code: shares nothing with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>

#include "../../include/hyb.h"

namespace hyb {

typedef unsigned int u32;
typedef unsigned long long u64;

constexpr u32 NOCHILD = 0xFFFFFFFFu;
constexpr int MAXLEVEL = 21;

// status bits (device control block)
constexpr u32 ST_NONFINITE = 1u;
constexpr u32 ST_NODE_OVERFLOW = 2u;
constexpr u32 ST_STACK_OVERFLOW = 4u;
constexpr u32 ST_WAIT_EXPIRED = 8u;

// radix sort tiling (onesweep): 256 threads x 14 keys = 3584 keys per tile (2^20 keys = 293 tiles, two per SM on
// 148 SMs; with 4096-key tiles 40 SMs had one tile and 108 had two)
constexpr int RS_THREADS = 256;
constexpr int RS_KPT = 14;        // keys per thread of a radix tile: 3584 keys per tile ...
constexpr int RS_KPT_SMALL = 4;   // ... 1024 for small runs, where a pass is one tile's chain of latencies and most SMs have none
#ifndef RS_SMALL_N
#define RS_SMALL_N 300000         // (4 against 14 keys per thread: build -20 % at n = 2^12, -15 % at 2^17, -6 % at 2^18, +17 % at 2^19)
#endif
inline int rs_kpt_for(int64_t n) { return n < RS_SMALL_N ? RS_KPT_SMALL : RS_KPT; }
constexpr int RS_PASSES = 8;      // 8 x 8 bits >= 63 bits
constexpr int LB_WIN = 16;        // radix look-back: tiles per block = status words requested together

// single-value scan tiles (octree preorder, group compaction)
constexpr int SC_THREADS = 256;
constexpr int SC_IPT = 16;
constexpr int SC_TILE = SC_THREADS * SC_IPT;
constexpr int PO_IPT = 4;                // octree preorder: heavy per-item work, small tiles
constexpr int PO_TILE = SC_THREADS * PO_IPT;

// walk kernel geometry
constexpr int WK_WARPS = 8;              // warps per CTA
#ifndef SMALL_RUN_PER_WARP
#define SMALL_RUN_PER_WARP 160         // particles per resident warp below which a run counts as small (Ctx::soft_split, hard_small)
#endif
constexpr int WK_U = 4;                  // sources per iteration of the pair loops (pairs.cuh)
constexpr int WK_CELL_CAP = 320;         // monopole buffer entries per warp
constexpr int WK_PART_CAP = 192;         // K-weighted (near) particle buffer entries per warp

enum WalkMode { WALK_HYBRID = 0, WALK_HARD = 1, WALK_NORMAL = 2 };

// Device control block.  It sits in the workspace right in front of the look-back statuses, and its last
// block of fields is what a build starts from zero: ONE memset per build clears from build_zero_begin to the end of
// the status arrays (Layout::zero_end).
struct DevCtl {
    u32 status;
    u32 nn, ng;
    u32 level_offset[MAXLEVEL + 2];
    // ---- derived ----
    float bbox[6];
    double L, inv, origin[3];
    float Lf;
    u32 digit_base[RS_PASSES * 256];
    u32 node_base[256];
    // ---- walk ----
    // work distribution: launch k uses slot k & 1 and clears the other slot for launch k + 1 (no memset)
    u32 group_counter[2];
    u32 nheavy[2];              // sink ranges of split groups (split_group)
    u32 walk_ng;                // number of groups of the last walk (is its nhard[] comparable?)
    u32 split_t[3];             // hard walk scheduling thresholds (pairs): queue first / cut in 2 / cut in 4 (set by hyb_init)
    u32 split_cap;              // entries the queue of sink ranges can hold
    // fused (soft) walk scheduling: thresholds in 1/64 of the ideal makespan soft_work / soft_slots (hyb_init)
    u32 soft_a[3];              // queue first / cut in 2 / cut in 4
    u32 soft_slots;             // warps the fused walk keeps resident (hyb_init)
    u32 soft_ng;                // number of groups of the last fused walk (is its scost[] comparable?)
    u64 soft_work[2];           // sum over the groups of the last fused walk of members x cost (slot: WalkArgs::spar)
    u64 inter_soft, inter_hard, inter_hard_fused;   // pair counts: soft lists, hard lists (all walks), hard lists of fused walks
    u64 inter_hard_leaf;        // hard-only walks: members x particles of the leaves within r_out (the hard list without the particle cut)
    // ---- bounding box reduction: filled by bbox_kernel or by the drift, cleared again by keys_kernel ----
    alignas(32) u32 bbox_enc[6]; // (one 32-byte sector with bbox_done) order-preserving encodings: ~min xyz, max xyz (atomicMax from 0 for both)
    u32 bbox_done;              // CTAs that have contributed (the last one derives the root cube)
    // ---- zero at the start of every build (keep last) ----
    u32 build_zero_begin;       // (marks the start of the memset range)
    u32 digit_hist[RS_PASSES * 256];
    u32 node_hist[256];
    u32 tile_counter[16];       // dynamic tile ids, one slot per lookback kernel instance
    u32 nn_total;               // un-clamped node count
};

// Programmatic dependent launch, used between the passes of the radix sort (sort.cuh).  A kernel
// launched with launch_pdl may become resident while the previous kernel of the stream is still running; it
// starts with pdl_begin(), which waits until that kernel has completed and its writes are visible, and only
// then lets the next launch_pdl kernel of the stream start early.  This hides the launch and
// CTA-scheduling latency between short dependent kernels.  Rules: nothing is read from global memory before
// pdl_begin(); and what the kernel reads through the non-coherent path (const __restrict__, __ldg) must not
// have been read by the previous kernel at addresses that kernel also wrote (a stale L1 line could survive:
// the previous kernel ran on the same SMs after this one's launch).  A radix pass only writes what the next
// pass reads, so it qualifies; the other kernels of the build read and write shared control words and are
// launched the ordinary way (pdl_begin() then returns at once).
__device__ __forceinline__ void pdl_begin()
{
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}

template <typename... Exp, typename... Act>
static inline cudaError_t launch_pdl(void (*kern)(Exp...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Act &&...args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, static_cast<Exp>(args)...);
}

// One tree node as the walk reads it: 64 bytes, children of a cell are contiguous (T7).
struct __align__(16) NodeRec {
    float4 A;        // centre of mass, mass (T9)
    float4 B;        // tight box minimum, squared opening radius (T8, T10)
    float4 C;        // tight box maximum, 0
    uint2 meta;      // cell: (first child, nchild);  leaf: (first particle, count | 0x80000000)
    uint2 pad;       // (first particle, count) of the node, cell or leaf
};

struct Layout {   // byte offsets into the workspace; computed by plan_workspace
    size_t ctl;
    size_t key_orig, key_a, key_b, val_a, val_b;
    size_t pos_tmp, vel_tmp, id_tmp;
    size_t rs_status;           // [RS_PASSES][rs_tiles + rs_blocks][256] u32 (tile and block look-back statuses)
    size_t sc_status;           // u64 [po_tiles] (preorder scan) then [sc_tiles] (group scan)
    size_t gnode_at;            // u32[n]: node a group hangs from, by first particle (scratch of the group kernels)
    size_t gflag;               // u8[n]
    size_t pre_level, pre_first, pre_of_bfs, bfs_of_pre;   // u8, u32, u32, u32 [node_cap]
    size_t node_status;         // [ntiles(node_cap)][256] u32
    size_t level, first, count, child, nchild, parent, arrived;
    size_t nodes;                              // NodeRec[node_cap]
    size_t MS64, C64, B2, bmax2;               // double[4nc] (M, Sx, Sy, Sz), [3nc], [nc], u64[nc]
    size_t leaf_of;             // u32[n]
    size_t gfirst, gcount, glo, ghi, ncell, npart, nhard;   // [group_cap]
    size_t gnode, ganc;         // u32[group_cap]: tree node a group hangs from; start node of its hard walk
    size_t splitq;              // u32[4 group_cap]: sink ranges of split groups, processed first (walk.cu)
    size_t scost;               // u32[group_cap]: list length of the group at the last fused walk (ncell + npart + nhard)
    size_t scratch, scratch_bytes; // hyb_energy / hyb_let_count
    size_t zero_begin, zero_end; // look-back statuses and group flags: cleared by one memset per build
    size_t total;
    int64_t n, node_cap, group_cap;
    int64_t rs_tiles, node_tiles, sc_tiles, po_tiles;
    int64_t rs_blocks, node_blocks;      // look-back blocks of LB_WIN tiles
    int rs_kpt;                          // keys per thread of the radix tiles this workspace is planned for (rs_kpt_for(n))
};

inline int64_t node_capacity(int64_t n) { return 2 * n + 4096; }
inline int64_t imin64(int64_t a, int64_t b) { return a < b ? a : b; }
Layout plan_workspace(int64_t n);

struct Ctx {
    bool split_ready = false;   // ginfo_kernel has already queued the heavy groups for the walk that uses slot split_par
    u32 split_par = 0;
    int split_kind = 0;         // ... and that walk is a hard-only walk (1) or a fused walk (2)
    int next_kind = 2;          // the walk the build being enqueued is for
    u32 soft_par = 0;           // slot of DevCtl::soft_work the next fused walk adds to
    bool soft_split = false;    // the fused walk follows a prepared work order (few groups per resident warp; hyb_init)
    // The store (positions, velocities, ids) lives in the caller's arrays.  A build re-orders it into the workspace copy
    // and copies it back -- unless hyb_step has set defer_copy: then pos / vel / id simply point to the workspace copy
    // afterwards (store_away) and the next build re-orders straight back into the caller's arrays; hyb_step returns with
    // the store at home (one copy if the number of builds of the call was odd).
    const float4 *pos_sorted = nullptr;          // where the build being enqueued puts the re-ordered positions
    hyb_float4 *pos_home = nullptr, *vel_home = nullptr;
    u32 *id_home = nullptr;
    bool defer_copy = false, store_away = false;
    bool hard_small = false;    // the hard walk runs its small-N variant (SmemLayout<WALK_HARD, true>; hyb_init)
    // hyb_run_host: called by hyb_step right after it has enqueued the LAST tree build of the call -- from ev_groups on
    // the store (positions, ids) has its final order and values, and can travel while the last walk runs
    void (*store_final)(Ctx *, void *) = nullptr;
    void *store_final_arg = nullptr;
    bool bbox_ready = false;    // the last drift has already reduced the bounding box of the current positions
    u32 walk_par = 0;           // slot of the walk work counters the next launch uses (DevCtl::group_counter)
    hyb_params p;
    u32 sink_lo, sink_hi;       // hyb_set_sink_range: the sinks this context evaluates (store slots), default all
    int64_t n;
    int device;
    cudaStream_t stream;
    cudaStream_t aux;              // library-owned: runs the parts of a build that are off the critical path
    cudaEvent_t ev_sorted, ev_perm, ev_linked, ev_groups;
    int num_sms;
    hyb_float4 *pos, *vel, *a_soft, *a_hard;
    u32 *id;
    char *ws;
    Layout L;
    bool tree_valid, acc_valid;
    bool tree_refit;               // the tree's boxes were refitted after a drift: valid for the direct hard walk only
    int group_max_now;
    int grouping_now;              // HYB_GROUP_NODE / SIBLINGS of the build being enqueued
    bool boxes_only;               // the build being enqueued is read by a hard walk only: no moments
    cudaEvent_t ev[5];
    cudaEvent_t *evpool;           // stage timers of hyb_step, kept between calls
    size_t evpool_n;
    float t_acc[8];
    bool timing;
    unsigned long long launches;   // kernels launched since hyb_init
    char err[256];
    // typed views of the workspace
    DevCtl *ctl;
};

// Per-device one-time set-up (function attributes, constant tables): bit d of *mask says device d is done.
// Two threads may both do the set-up; that is harmless.
static inline bool device_ready(const unsigned long long *mask, int device)
{
    return (__atomic_load_n(mask, __ATOMIC_ACQUIRE) >> (device & 63)) & 1ull;
}
static inline void device_set_ready(unsigned long long *mask, int device)
{
    __atomic_fetch_or(mask, 1ull << (device & 63), __ATOMIC_RELEASE);
}

template <typename T>
static inline T *wsptr(const Ctx *c, size_t off) { return reinterpret_cast<T *>(c->ws + off); }

// stage launchers (each enqueues on c->stream and returns the last CUDA error)
cudaError_t launch_build_tree(Ctx *c);
cudaError_t store_come_home(Ctx *c);        // no-op unless store_away: the workspace copy goes to the caller's arrays
cudaError_t launch_regroup(Ctx *c);        // sink groups again (group_max_now / grouping_now) on the existing topology
cudaError_t launch_refit_tree(Ctx *c);     // tight boxes of nodes and groups for the current positions, same topology
cudaError_t launch_walk(Ctx *c, int mode);
cudaError_t launch_kick_drift(Ctx *c, float c_soft, float c_hard, float dt_drift, bool with_bbox = false);
cudaError_t launch_zero_acc(Ctx *c, hyb_float4 *a);
cudaError_t launch_let_count(Ctx *c, int ndom, const float *d_boxes, unsigned long long *d_out);
size_t energy_scratch_doubles(const Ctx *c, u32 *ni, u32 *nj, u32 *nk);
cudaError_t launch_energy(Ctx *c, double *d_scratch, u32 ni, u32 nj, u32 nk);
cudaError_t launch_energy_noalloc(const hyb_float4 *d_pos_m, const hyb_float4 *d_vel, int64_t n, float G, float eps, int device,
                                  cudaStream_t st, double *d_energy, bool *too_large);

// ---- device helpers ------------------------------------------------------------------
__device__ __forceinline__ u32 enc_float(float f)
{
    u32 u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float dec_float(u32 e)
{
    return __uint_as_float((e & 0x80000000u) ? (e ^ 0x80000000u) : ~e);
}
__device__ __forceinline__ u32 ld_volatile_u32(const u32 *p)
{
    return *reinterpret_cast<const volatile u32 *>(p);
}
__device__ __forceinline__ u64 ld_volatile_u64(const u64 *p)
{
    return *reinterpret_cast<const volatile u64 *>(p);
}

// a1 (T1-T3): bounding box of the particles and the root cube.  Every thread brings the minima / maxima and
// the validity of the particles it has seen; the block combines them, adds them to the control block, and the
// last block to arrive derives the root cube.  Used by bbox_kernel and by the drift (integrate.cu), which
// sees every new position anyway.  All threads of the block must call it (256 threads).
__device__ __forceinline__ void root_cube(DevCtl *ctl)
{
    double L = 0.0;
    for (int a = 0; a < 3; a++) {
        float lo = dec_float(~ld_volatile_u32(&ctl->bbox_enc[a])), hi = dec_float(ld_volatile_u32(&ctl->bbox_enc[3 + a]));
        ctl->bbox[a] = lo; ctl->bbox[3 + a] = hi;
        double e = __dsub_rn((double)hi, (double)lo);
        if (e > L) L = e;
        ctl->origin[a] = (double)lo;
    }
    if (!(L > 0.0) || !isfinite(L)) L = 1.0;
    ctl->L = L;
    ctl->inv = __ddiv_rn(2097152.0, L);
    ctl->Lf = __double2float_rn(L);
}

__device__ __forceinline__ void bbox_block_reduce(const float lo[3], const float hi[3], bool bad, DevCtl *ctl)
{
    __shared__ u32 s_enc[6];
    if (threadIdx.x < 3) s_enc[threadIdx.x] = 0xFFFFFFFFu;
    else if (threadIdx.x < 6) s_enc[threadIdx.x] = 0u;
    __syncthreads();
#pragma unroll
    for (int a = 0; a < 3; a++) {
        u32 mn = __reduce_min_sync(0xFFFFFFFFu, enc_float(lo[a]));
        u32 mx = __reduce_max_sync(0xFFFFFFFFu, enc_float(hi[a]));
        if ((threadIdx.x & 31) == 0) { atomicMin(&s_enc[a], mn); atomicMax(&s_enc[3 + a], mx); }
    }
    if (__any_sync(0xFFFFFFFFu, bad) && (threadIdx.x & 31) == 0) atomicOr(&ctl->status, ST_NONFINITE);
    __syncthreads();
    // the minima are kept complemented, so that both halves grow by atomicMax from zero
    if (threadIdx.x < 3) atomicMax(&ctl->bbox_enc[threadIdx.x], ~s_enc[threadIdx.x]);
    else if (threadIdx.x < 6) atomicMax(&ctl->bbox_enc[threadIdx.x], s_enc[threadIdx.x]);
    // the last CTA to get here sees every CTA's contribution and derives the root cube
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0 && atomicAdd(&ctl->bbox_done, 1u) == gridDim.x - 1) {
        __threadfence();
        root_cube(ctl);
    }
}

// Walk scheduling: a group whose list was long at the previous walk of the same kind (members x list length of the
// group with the same index -- an estimate that steers the order of work: the lists are the group's either way, only
// the last bits of a sum can differ, because a range of fewer sinks combines its partial sums differently) is queued
// in front of everything else, the heaviest ones cut into 2 or 4 sink ranges; the walk skips it in the ordinary
// sequence.  kind 1: the hard-only walk, estimate from nhard[], fixed thresholds (DevCtl::split_t).  kind 2: the
// fused walk, estimate from scost[], thresholds relative to the ideal makespan of the previous fused walk (all its
// pairs / the warps that run side by side): with few groups per warp the longest group sets the duration of the
// kernel, so it has to start first, and be shared by several warps when it alone is longer than the rest.
// Called once per group by ginfo_kernel (during the build, off the critical path) or by split_kernel.
struct SplitArgs {
    DevCtl *ctl; const u32 *nhard_prev, *scost_prev; u32 *heavy; unsigned char *is_split;
    u32 par, kind, soft_slot;
};

__device__ __forceinline__ void split_group(const SplitArgs &x, u32 g, u32 ng, u32 n)
{
    DevCtl *ctl = x.ctl;
    unsigned long long est, t0, t1, t2;
    if (x.kind == 0u) { x.is_split[g] = 0; return; }
    if (x.kind == 1u) {
        const u32 prev = ctl->walk_ng;
        const bool comparable = (prev > ng ? prev - ng : ng - prev) <= ng / 16u;
        est = (unsigned long long)n * (unsigned long long)(comparable ? x.nhard_prev[g] : 0u);
        t0 = ctl->split_t[0]; t1 = ctl->split_t[1]; t2 = ctl->split_t[2];
    } else {
        const u32 prev = ctl->soft_ng;
        const bool comparable = (prev > ng ? prev - ng : ng - prev) <= ng / 16u;
        est = (unsigned long long)n * (unsigned long long)(comparable ? x.scost_prev[g] : 0u);
        const unsigned long long u = ctl->soft_work[x.soft_slot] / (64ull * (unsigned long long)ctl->soft_slots) + 1ull;
        t0 = u * ctl->soft_a[0]; t1 = u * ctl->soft_a[1]; t2 = u * ctl->soft_a[2];
    }
    u32 nsub = 0;                                   // 0: stays in the ordinary sequence
    if (est >= t2 && n >= 32u) nsub = 4;
    else if (est >= t1 && n >= 16u) nsub = 2;
    else if (est >= t0) nsub = 1;                   // whole, but queued in front
    if (est == 0ull) nsub = 0;
    if (nsub) {
        const u32 at = atomicAdd(&ctl->nheavy[x.par], nsub);
        if (at + nsub <= ctl->split_cap) {
            for (u32 i = 0; i < nsub; i++) x.heavy[at + i] = g | (i << 28) | ((nsub - 1u) << 30);
        } else {
            atomicSub(&ctl->nheavy[x.par], nsub);   // the queue is full (it cannot be: 4 entries per group): leave the group where it is
            nsub = 0;
        }
    }
    x.is_split[g] = nsub > 0;
}

// Decoupled look-back over one value per tile (status word: bits 63..62 flag, low 62 bits value).
constexpr u64 LB_AGG = 1ull << 62, LB_PREFIX = 2ull << 62, LB_MASK = (1ull << 62) - 1;
constexpr int LB_SPIN_LIMIT = 1 << 22;
// The 32 lanes of one warp each inspect a different predecessor.  Called by all lanes of ONE warp of the
// CTA that owns `tile`; every lane returns the exclusive prefix of the earlier tiles.
__device__ __forceinline__ u64 lookback_warp(u64 *status, u32 tile, u64 aggregate, u32 *dev_status, int lane)
{
    volatile u64 *st = status;
    if (tile == 0) {
        if (lane == 0) st[0] = LB_PREFIX | aggregate;
        return 0;
    }
    if (lane == 0) st[tile] = LB_AGG | aggregate;
    u64 excl = 0;
    long long t = (long long)tile - 1;
    int spins = 0;
    for (;;) {
        const long long idx = t - lane;
        const u64 s = idx >= 0 ? st[idx] : (2ull << 62);
        const u32 f = (u32)(s >> 62);
        const u32 notready = __ballot_sync(0xFFFFFFFFu, f == 0u), prefix = __ballot_sync(0xFFFFFFFFu, f == 2u);
        const int lim_nr = notready ? __ffs(notready) - 1 : 32, lim_p = prefix ? __ffs(prefix) - 1 : 32;
        const bool done = lim_p < lim_nr;
        const int use = done ? lim_p + 1 : lim_nr;          // lanes 0 .. use-1 contribute
        u64 v = lane < use ? (s & LB_MASK) : 0ull;
#pragma unroll
        for (int off = 16; off; off >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, off);
        excl += v;
        if (done) break;
        t -= use;
        if (use == 0 && ++spins >= LB_SPIN_LIMIT) {
            if (lane == 0) atomicOr(dev_status, ST_WAIT_EXPIRED);
            break;
        }
    }
    if (lane == 0) st[tile] = LB_PREFIX | (excl + aggregate);
    return excl;
}

}  // namespace hyb
