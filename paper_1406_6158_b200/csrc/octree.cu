// octree.cu -- steps a5-a7: linear octree in breadth-first numbering, moment upsweep with the
// opening radius, sink groups.  (T7-T11.)
//
// Construction is depth-independent (a handful of launches):
//   preorder : per particle i, the levels at which a node starts at i form the contiguous range
//              (d(i), top(i)], d(i) = common leading 3-bit digits of key[i-1], key[i] and top(i)
//              derived from a sliding window of leaf_max+1 keys.  A scan gives each node its
//              preorder index.
//   bfs      : one stable counting-sort pass by level turns preorder into breadth-first order.
//   link     : every node finds its range end, children and parent from the two orders (a leaf ends
//              where the next preorder node starts; sibling runs are consecutive in breadth-first
//              order); only a cell's range end needs a binary search in the keys.
//   upsweep  : leaves first, the last child to arrive computes the parent (fixed summation order).
#include "common.cuh"
#include "sort.cuh"

namespace hyb {

__device__ __forceinline__ int lcp_levels(u64 a, u64 b)
{
    u64 x = a ^ b;
    return x ? (__clzll((long long)x) - 1) / 3 : MAXLEVEL;
}

// ------------------------------------------------------------------ a5: preorder emission
// level_offset and the counting-sort bases (clamped to the node pool).  One thread of the last CTA of
// preorder_kernel to finish (every CTA has added its share of node_hist by then).
__device__ void level_offsets(DevCtl *ctl)
{
    {
        // node pool overflow: the counting-sort bases would point past the pool, so drop the tree
        // (nn = 0 makes every later stage a no-op); the status bit reports the failure.
        if (ld_volatile_u32(&ctl->status) & ST_NODE_OVERFLOW) ctl->nn = 0;
        const u32 nn = ld_volatile_u32(&ctl->nn);
        u32 run = 0;
        for (int l = 0; l <= MAXLEVEL; l++) {
            ctl->level_offset[l] = min(run, nn);
            ctl->node_base[l] = run;
            run += ld_volatile_u32(&ctl->node_hist[l]);
        }
        ctl->level_offset[MAXLEVEL + 1] = min(run, nn);
        for (int l = MAXLEVEL + 1; l < 256; l++) ctl->node_base[l] = run;
    }
}


constexpr int PO_HALO = 64;

__global__ void __launch_bounds__(SC_THREADS) preorder_kernel(
    const u64 *__restrict__ key, u32 n, int leaf_max, u32 node_cap, DevCtl *ctl, u64 *sc_status,
    unsigned char *__restrict__ pre_level, u32 *__restrict__ pre_first)
{
    __shared__ u64 s_key[PO_TILE + 2 * PO_HALO];
    __shared__ signed char s_w[PO_TILE + PO_HALO];
    __shared__ u32 s_hist[MAXLEVEL + 1];
    __shared__ u32 s_warp[SC_THREADS / 32];
    __shared__ u32 s_tile;
    __shared__ u64 s_prefix;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const u32 ntiles = (n + PO_TILE - 1) / PO_TILE;
    for (;;) {
        __syncthreads();
        if (tid == 0) s_tile = atomicAdd(&ctl->tile_counter[8], 1u);
        if (tid <= MAXLEVEL) s_hist[tid] = 0;
        __syncthreads();
        const u32 tile = s_tile;
        if (tile >= ntiles) break;
        const long long t0 = (long long)tile * PO_TILE;
        for (int q = tid; q < PO_TILE + 2 * PO_HALO; q += SC_THREADS) {
            long long g = t0 - PO_HALO + q;
            s_key[q] = (g >= 0 && g < (long long)n) ? key[g] : 0ull;
        }
        __syncthreads();
        for (int q = tid; q < PO_TILE + PO_HALO; q += SC_THREADS) {       // w(s), s = t0 - HALO + q
            long long s = t0 - PO_HALO + q;
            int w = -1;
            if (s >= 0 && s + leaf_max < (long long)n) w = lcp_levels(s_key[q], s_key[q + leaf_max]);
            s_w[q] = (signed char)w;
        }
        __syncthreads();
        int d[PO_IPT], cnt[PO_IPT];
        u32 mysum = 0;
#pragma unroll
        for (int k = 0; k < PO_IPT; k++) {
            const int li = tid * PO_IPT + k;                 // local index in tile
            const long long i = t0 + li;
            d[k] = 0; cnt[k] = 0;
            if (i < (long long)n) {
                d[k] = (i == 0) ? -1 : lcp_levels(s_key[PO_HALO + li - 1], s_key[PO_HALO + li]);
                int lfull = -1;
                for (int s = 0; s <= leaf_max; s++) lfull = max(lfull, (int)s_w[PO_HALO + li - s]);
                int top = min(lfull + 1, MAXLEVEL);
                cnt[k] = max(0, top - d[k]);
            }
            mysum += cnt[k];
        }
        // block exclusive scan of mysum
        u32 incl = mysum;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            u32 t = __shfl_up_sync(0xFFFFFFFFu, incl, off);
            if (lane >= off) incl += t;
        }
        if (lane == 31) s_warp[warp] = incl;
        __syncthreads();
        u32 wbase = 0, tile_total = 0;
#pragma unroll
        for (int w = 0; w < SC_THREADS / 32; w++) { if (w < warp) wbase += s_warp[w]; tile_total += s_warp[w]; }
        if (warp == 0) {
            const u64 pre = lookback_warp(sc_status, tile, tile_total, &ctl->status, lane);
            if (lane == 0) s_prefix = pre;
            if (lane == 0 && tile == ntiles - 1) {
                u64 tot = pre + tile_total;
                ctl->nn_total = (u32)min(tot, (u64)0xFFFFFFFFu);
                ctl->nn = (u32)min(tot, (u64)node_cap);
                if (tot > node_cap) atomicOr(&ctl->status, ST_NODE_OVERFLOW);
            }
        }
        __syncthreads();
        u64 p = s_prefix + wbase + incl - mysum;
#pragma unroll
        for (int k = 0; k < PO_IPT; k++) {
            const long long i = t0 + tid * PO_IPT + k;
            if (i < (long long)n) {
                for (int j = 0; j < cnt[k]; j++) {
                    if (p + j < node_cap) {
                        pre_level[p + j] = (unsigned char)(d[k] + 1 + j);
                        pre_first[p + j] = (u32)i;
                    }
                    atomicAdd(&s_hist[d[k] + 1 + j], 1u);
                }
                p += cnt[k];
            }
        }
        __syncthreads();
        if (tid <= MAXLEVEL && s_hist[tid]) atomicAdd(&ctl->node_hist[tid], s_hist[tid]);
    }
    // the last CTA to leave sees the complete level histogram and the node count
    __threadfence();
    __syncthreads();
    if (tid == 0 && atomicAdd(&ctl->tile_counter[12], 1u) == gridDim.x - 1) {
        __threadfence();
        level_offsets(ctl);
    }
}

// ------------------------------------------------------------------ a5: link
__device__ __forceinline__ u32 lower_bound_key(const u64 *__restrict__ key, u32 lo, u32 hi, u64 target)
{
    while (lo < hi) {           // first index in [lo,hi) with key >= target
        u32 mid = lo + ((hi - lo) >> 1);
        if (__ldg(key + mid) < target) lo = mid + 1; else hi = mid;
    }
    return lo;
}
// Topology from the two orders.  In preorder a node is followed by its first child (one level deeper) if
// it has children, else by the next node that starts where it ends; a node is a FIRST child exactly when
// its preorder predecessor is one level up (its parent).  In breadth-first order the children of a cell
// are consecutive, so the first child of a sibling run is at most seven steps back and the run ends at
// most seven steps ahead: a handful of grouped loads instead of binary searches in the keys.
__global__ void __launch_bounds__(256) link_kernel(
    const u64 *__restrict__ key, u32 n, int leaf_max, const DevCtl *__restrict__ ctl,
    const unsigned char *__restrict__ level, const u32 *__restrict__ pre_of_bfs, const u32 *__restrict__ bfs_of_pre,
    const unsigned char *__restrict__ pre_level, const u32 *__restrict__ pre_first,
    u32 *__restrict__ first, u32 *__restrict__ count, u32 *__restrict__ child, unsigned char *__restrict__ nchild,
    u32 *__restrict__ parent, u32 *__restrict__ arrived, NodeRec *__restrict__ rec, u64 *__restrict__ bmax2)
{
    const u32 nn = ctl->nn;
    for (u32 b = blockIdx.x * blockDim.x + threadIdx.x; b < nn; b += gridDim.x * blockDim.x) {
        const u32 p = pre_of_bfs[b];
        const int lev = level[b];
        const u32 f = pre_first[p];
        const bool has_kids = p + 1 < nn && (int)pre_level[p + 1] == lev + 1;
        u32 end;
        if (lev == 0) end = n;
        else if (!has_kids) end = p + 1 < nn ? pre_first[p + 1] : n;     // the next node starts where this one ends
        else {
            const u64 k0 = __ldg(key + f);
            const int sh = 63 - 3 * lev;
            end = lower_bound_key(key, f, n, ((k0 >> sh) + 1ull) << sh);
        }
        const u32 c = end - f;
        const bool internal = has_kids && (c > (u32)leaf_max) && lev < MAXLEVEL;
        u32 ch = NOCHILD, nc = 0;
        if (internal) {
            ch = bfs_of_pre[p + 1];
            const u32 lim = ctl->level_offset[lev + 2];                   // end of the children's level
            u32 pq[7];
#pragma unroll
            for (int i = 0; i < 7; i++) pq[i] = ch + 1 + i < lim ? pre_of_bfs[ch + 1 + i] : 0u;
            bool fst[7];
#pragma unroll
            for (int i = 0; i < 7; i++) fst[i] = ch + 1 + i >= lim || (int)pre_level[pq[i] - 1] == lev;
            nc = 8;
#pragma unroll
            for (int i = 6; i >= 0; i--) if (fst[i]) nc = 1 + i;          // the run ends before the next first child
        }
        u32 par = NOCHILD;
        if (lev > 0) {
            const u32 lo = ctl->level_offset[lev];
            u32 pb[8];
            pb[0] = p;
#pragma unroll
            for (int i = 1; i < 8; i++) pb[i] = (b >= lo + i) ? pre_of_bfs[b - i] : 1u;
            bool fst[8];
#pragma unroll
            for (int i = 0; i < 8; i++) fst[i] = (b >= lo + i) && (int)pre_level[pb[i] - 1] == lev - 1;
            u32 pp = pb[0] - 1;
#pragma unroll
            for (int i = 7; i >= 0; i--) if (fst[i]) pp = pb[i] - 1;      // nearest first child at or before b
            par = bfs_of_pre[pp];
        }
        first[b] = f; count[b] = c; child[b] = ch; nchild[b] = (unsigned char)nc; parent[b] = par;
        arrived[b] = 0; bmax2[b] = 0ull;
        rec[b].meta = internal ? make_uint2(ch, nc) : make_uint2(f, c | 0x80000000u);
        rec[b].pad = make_uint2(f, c);
    }
}

// ------------------------------------------------------------------ a6: upsweep (T8-T10)
struct NodeArrays {
    const u32 *first, *count, *child, *parent;
    const unsigned char *nchild, *level;
    u32 *arrived;
    NodeRec *rec;               // A = com_m, B = lo | ropen2, C = hi | 0
    double4 *MS64;              // (M, Sx, Sy, Sz) before the division
    double *C64, *B2;
    u32 *leaf_of;
};

__device__ __forceinline__ double4 ldcg_d4(const double4 *p)
{
    const double2 *q = reinterpret_cast<const double2 *>(p);
    const double2 a = __ldcg(q), b = __ldcg(q + 1);
    return make_double4(a.x, a.y, b.x, b.y);
}

__device__ __forceinline__ double dist2_rn(double ax, double ay, double az, double bx, double by, double bz)
{
    double dx = __dsub_rn(ax, bx), dy = __dsub_rn(ay, by), dz = __dsub_rn(az, bz);
    return __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
}

__device__ __forceinline__ void finish_node(const NodeArrays &na, u32 b, int lev, double M, double Sx, double Sy,
                                            double Sz, float3 lo, float3 hi, int mac, float Lf, float theta,
                                            double &Cx, double &Cy, double &Cz)
{
    if (M == 0.0) { Cx = (double)lo.x; Cy = (double)lo.y; Cz = (double)lo.z; }
    else { Cx = __ddiv_rn(Sx, M); Cy = __ddiv_rn(Sy, M); Cz = __ddiv_rn(Sz, M); }
    float ropen2 = 0.0f;
    if (mac == HYB_MAC_THETA) {
        float l = __fmul_rn(Lf, __uint_as_float((u32)(127 - lev) << 23));     // Lf * 2^-lev, exact
        float r = __fdiv_rn(l, theta);
        ropen2 = __fmul_rn(r, r);
    }
    na.rec[b].A = make_float4(__double2float_rn(Cx), __double2float_rn(Cy), __double2float_rn(Cz), __double2float_rn(M));
    na.rec[b].B = make_float4(lo.x, lo.y, lo.z, ropen2);
    // C.w: the largest squared opening radius among the children (walk.cu: a cell farther away than this has only
    // accepted children).  theta-mode: a child's cell side is half of this one's, so its r_open^2 is exactly a quarter;
    // absolute MAC: filled in by ropen_abs_kernel once every node has its own radius
    na.rec[b].C = make_float4(hi.x, hi.y, hi.z, mac == HYB_MAC_THETA ? __fmul_rn(ropen2, 0.25f) : INFINITY);
    na.MS64[b] = make_double4(M, Sx, Sy, Sz);
    na.C64[3 * (size_t)b] = Cx; na.C64[3 * (size_t)b + 1] = Cy; na.C64[3 * (size_t)b + 2] = Cz;
}

// MOMENTS = false: tight boxes only.  hyb_step uses it for the trees that only a hard walk reads (rule
// (b) and the hard list need the boxes and the topology, not the centres of mass).
template <bool MOMENTS>
__global__ void __launch_bounds__(128) upsweep_kernel(NodeArrays na, const float4 *__restrict__ pos,
                                                      const DevCtl *__restrict__ ctl, int mac, float theta)
{
    const u32 nn = ctl->nn;
    const float Lf = ctl->Lf;
    // deepest leaves first (breadth-first numbering: the highest indices): their climbs are the longest chains
    for (u32 idx = blockIdx.x * blockDim.x + threadIdx.x; idx < nn; idx += gridDim.x * blockDim.x) {
    const u32 b = nn - 1u - idx;
    if (na.child[b] != NOCHILD) continue;
    u32 par = na.parent[b];            // requested now, needed after the leaf sums
    // ---- leaf: sequential sums over its particles, ascending (T9)
    {
        const u32 f = na.first[b], c = na.count[b];
        double M = 0.0, Sx = 0.0, Sy = 0.0, Sz = 0.0;
        float4 p0 = __ldg(pos + f);
        float3 lo = make_float3(p0.x, p0.y, p0.z), hi = lo;
        for (u32 j = f; j < f + c; j++) {
            float4 p = __ldg(pos + j);
            if (MOMENTS) {
                double m = (double)p.w;
                M = __dadd_rn(M, m);
                Sx = __dadd_rn(Sx, __dmul_rn(m, (double)p.x));
                Sy = __dadd_rn(Sy, __dmul_rn(m, (double)p.y));
                Sz = __dadd_rn(Sz, __dmul_rn(m, (double)p.z));
            }
            lo.x = fminf(lo.x, p.x); lo.y = fminf(lo.y, p.y); lo.z = fminf(lo.z, p.z);
            hi.x = fmaxf(hi.x, p.x); hi.y = fmaxf(hi.y, p.y); hi.z = fmaxf(hi.z, p.z);
            if (MOMENTS && mac == HYB_MAC_ABS) na.leaf_of[j] = b;
        }
        if (!MOMENTS) {
            na.rec[b].B = make_float4(lo.x, lo.y, lo.z, 0.0f);
            na.rec[b].C = make_float4(hi.x, hi.y, hi.z, 0.0f);
        } else {
            double Cx, Cy, Cz;
            finish_node(na, b, na.level[b], M, Sx, Sy, Sz, lo, hi, mac, Lf, theta, Cx, Cy, Cz);
            if (mac == HYB_MAC_ABS) {
                double B2 = 0.0;
                for (u32 j = f; j < f + c; j++) {
                    float4 p = __ldg(pos + j);
                    double d2 = dist2_rn((double)p.x, (double)p.y, (double)p.z, Cx, Cy, Cz);
                    B2 = __dadd_rn(B2, __dmul_rn((double)p.w, d2));
                }
                na.B2[b] = B2;
            }
        }
    }
    // ---- climb: the last child to arrive computes the parent, children in ascending order
    // (the topology of the parent and the index of ITS parent come back in one round trip)
    while (par != NOCHILD) {
        const u32 nc = na.nchild[par], c0 = na.child[par];      // topology: requested before the fence
        const int plev = na.level[par];
        const u32 gpar = na.parent[par];
        // arrival counter with release (this node's record is written) / acquire (the siblings' records
        // are read next) ordering at device scope
        u32 old;
        asm volatile("atom.acq_rel.gpu.global.add.u32 %0, [%1], %2;" : "=r"(old) : "l"(na.arrived + par), "r"(1u) : "memory");
        if (old + 1 != nc) break;
        double M = 0.0, Sx = 0.0, Sy = 0.0, Sz = 0.0;
        float3 lo, hi;
        for (u32 q = c0; q < c0 + nc; q++) {
            if (MOMENTS) {
                const double4 cm = ldcg_d4(na.MS64 + q);
                M = __dadd_rn(M, cm.x); Sx = __dadd_rn(Sx, cm.y); Sy = __dadd_rn(Sy, cm.z); Sz = __dadd_rn(Sz, cm.w);
            }
            const float4 bl = __ldcg(&na.rec[q].B), bh = __ldcg(&na.rec[q].C);
            if (q == c0) { lo = make_float3(bl.x, bl.y, bl.z); hi = make_float3(bh.x, bh.y, bh.z); }
            else {
                lo.x = fminf(lo.x, bl.x); lo.y = fminf(lo.y, bl.y); lo.z = fminf(lo.z, bl.z);
                hi.x = fmaxf(hi.x, bh.x); hi.y = fmaxf(hi.y, bh.y); hi.z = fmaxf(hi.z, bh.z);
            }
        }
        if (!MOMENTS) {
            na.rec[par].B = make_float4(lo.x, lo.y, lo.z, 0.0f);
            na.rec[par].C = make_float4(hi.x, hi.y, hi.z, 0.0f);
        } else {
            double Cx, Cy, Cz;
            finish_node(na, par, plev, M, Sx, Sy, Sz, lo, hi, mac, Lf, theta, Cx, Cy, Cz);
            if (mac == HYB_MAC_ABS) {            // parallel-axis sum of the children's B_2 (T10)
                double B2 = 0.0;
                for (u32 q = c0; q < c0 + nc; q++) {
                    double d2 = dist2_rn(__ldcg(na.C64 + 3 * (size_t)q), __ldcg(na.C64 + 3 * (size_t)q + 1),
                                         __ldcg(na.C64 + 3 * (size_t)q + 2), Cx, Cy, Cz);
                    B2 = __dadd_rn(B2, __dadd_rn(__ldcg(na.B2 + q), __dmul_rn(__ldcg(&na.MS64[q].x), d2)));
                }
                na.B2[par] = B2;
            }
        }
        par = gpar;
    }
    }
}

// exact b_max^2 (Eq. 5; R9): every particle visits its ancestors, one level per iteration so that
// the lanes of a warp meet at the same node; bit patterns of non-negative doubles order as u64.
__global__ void __launch_bounds__(256) bmax_kernel(const float4 *__restrict__ pos, u32 n,
                                                   const u32 *__restrict__ leaf_of, const u32 *__restrict__ parent,
                                                   const unsigned char *__restrict__ level,
                                                   const double *__restrict__ C64, u64 *bmax2)
{
    const u32 j = blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = j < n;
    float4 p = live ? __ldg(pos + j) : make_float4(0, 0, 0, 0);
    u32 node = live ? leaf_of[j] : NOCHILD;
    int nl = live ? (int)level[node] : -1;
    for (int l = MAXLEVEL; l >= 0; --l) {
        const bool act = (nl == l);
        u64 bits = 0;
        if (act) {
            double d2 = dist2_rn((double)p.x, (double)p.y, (double)p.z, C64[3 * (size_t)node],
                                 C64[3 * (size_t)node + 1], C64[3 * (size_t)node + 2]);
            bits = (u64)__double_as_longlong(d2);
        }
        int same;
        __match_all_sync(0xFFFFFFFFu, act ? node : NOCHILD, &same);
        if (same) {
            if (act) {                       // whole warp at one node
#pragma unroll
                for (int off = 16; off; off >>= 1) {
                    u64 o = __shfl_xor_sync(0xFFFFFFFFu, bits, off);
                    bits = o > bits ? o : bits;
                }
                if ((threadIdx.x & 31) == 0) atomicMax(bmax2 + node, bits);
            }
        } else if (act) atomicMax(bmax2 + node, bits);
        if (act) { node = parent[node]; nl = l - 1; }
    }
}

__global__ void __launch_bounds__(256) ropen_abs_kernel(const DevCtl *__restrict__ ctl, const u64 *__restrict__ bmax2,
                                                        const double *__restrict__ B2, float a_err, NodeRec *rec)
{
    const u32 nn = ctl->nn;
    const u32 b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= nn) return;
    double bm = __dsqrt_rn(__longlong_as_double((long long)bmax2[b]));
    double t3 = __dsqrt_rn(__ddiv_rn(__dmul_rn(3.0, B2[b]), (double)a_err));
    double t5 = __ddiv_rn(__dmul_rn(bm, bm), 4.0);
    double rb = __dadd_rn(__ddiv_rn(bm, 2.0), __dsqrt_rn(__dadd_rn(t5, t3)));
    float r = __double2float_rn(rb);
    rec[b].B.w = __fmul_rn(r, r);
}

// absolute MAC: NodeRec::C.w = largest squared opening radius among the children (see finish_node)
__global__ void __launch_bounds__(256) cmax_kernel(const DevCtl *__restrict__ ctl, const u32 *__restrict__ child,
                                                   const unsigned char *__restrict__ nchild, NodeRec *rec)
{
    const u32 nn = ctl->nn;
    for (u32 b = blockIdx.x * blockDim.x + threadIdx.x; b < nn; b += gridDim.x * blockDim.x) {
        const u32 c0 = child[b];
        float m = 0.0f;
        if (c0 != NOCHILD)
            for (u32 q = c0; q < c0 + nchild[b]; q++) m = fmaxf(m, rec[q].B.w);
        rec[b].C.w = m;
    }
}

// ------------------------------------------------------------------ a7: groups (T11)
__global__ void __launch_bounds__(256) gmark_kernel(const DevCtl *__restrict__ ctl, const u32 *__restrict__ first,
                                                    const u32 *__restrict__ count, const u32 *__restrict__ child,
                                                    const unsigned char *__restrict__ nchild,
                                                    const u32 *__restrict__ parent, int group_max, int grouping,
                                                    unsigned char *gflag, u32 *__restrict__ gnode_at)
{
    const u32 nn = ctl->nn;
    for (u32 b = blockIdx.x * blockDim.x + threadIdx.x; b < nn; b += gridDim.x * blockDim.x) {
    const u32 c = count[b], f = first[b], gm = (u32)group_max;
    if (c > gm && child[b] == NOCHILD) {
        for (u32 s = f; s < f + c; s += gm) { gflag[s] = 1; gnode_at[s] = b; }     // level-21 leaf cut into chunks
    } else if (grouping == HYB_GROUP_NODE) {
        if (c <= gm && (b == 0 || count[parent[b]] > gm)) { gflag[f] = 1; gnode_at[f] = b; }
    } else if (c <= gm) {
        if (b == 0) { gflag[f] = 1; gnode_at[f] = b; }          // the whole system is one group
    } else {
        // the children in order: consecutive small ones are packed greedily into runs of <= gm sinks
        u32 run = 0;
        bool open = false;
        const u32 c0 = child[b], nc = nchild[b];
        for (u32 q = c0; q < c0 + nc; q++) {
            const u32 cq = count[q];
            if (cq > gm) { open = false; run = 0; continue; }
            if (!open || run + cq > gm) { gflag[first[q]] = 1; gnode_at[first[q]] = b; run = 0; open = true; }
            run += cq;
        }
    }
    }
}

__global__ void __launch_bounds__(SC_THREADS) gscan_kernel(const unsigned char *__restrict__ gflag, u32 n, DevCtl *ctl,
                                                           u64 *sc_status, u32 *__restrict__ gfirst,
                                                           const u32 *__restrict__ gnode_at, u32 *__restrict__ gnode)
{
    __shared__ u32 s_warp[SC_THREADS / 32];
    __shared__ u32 s_tile;
    __shared__ u64 s_prefix;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const u32 ntiles = (n + SC_TILE - 1) / SC_TILE;
    for (;;) {
        __syncthreads();
        if (tid == 0) s_tile = atomicAdd(&ctl->tile_counter[9], 1u);
        __syncthreads();
        const u32 tile = s_tile;
        if (tile >= ntiles) break;
        const u32 i0 = tile * SC_TILE + tid * SC_IPT;
        u32 fl[SC_IPT], mysum = 0;
#pragma unroll
        for (int k = 0; k < SC_IPT; k++) fl[k] = 0u;
        if (i0 + SC_IPT <= n) {                      // 16 flags in one 16-byte load
            static_assert(SC_IPT == 16, "vector load of the flags assumes 16 items per thread");
            const uint4 v = *reinterpret_cast<const uint4 *>(gflag + i0);
            const u32 w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int k = 0; k < SC_IPT; k++) fl[k] = (w[k >> 2] >> (8 * (k & 3))) & 0xFFu;
        } else {
#pragma unroll
            for (int k = 0; k < SC_IPT; k++) fl[k] = (i0 + k < n) ? gflag[i0 + k] : 0u;
        }
#pragma unroll
        for (int k = 0; k < SC_IPT; k++) mysum += fl[k];
        u32 incl = mysum;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            u32 t = __shfl_up_sync(0xFFFFFFFFu, incl, off);
            if (lane >= off) incl += t;
        }
        if (lane == 31) s_warp[warp] = incl;
        __syncthreads();
        u32 wbase = 0, tile_total = 0;
#pragma unroll
        for (int w = 0; w < SC_THREADS / 32; w++) { if (w < warp) wbase += s_warp[w]; tile_total += s_warp[w]; }
        if (warp == 0) {
            const u64 pre = lookback_warp(sc_status, tile, tile_total, &ctl->status, lane);
            if (lane == 0) s_prefix = pre;
            if (lane == 0 && tile == ntiles - 1) ctl->ng = (u32)(pre + tile_total);
        }
        __syncthreads();
        u32 g = (u32)s_prefix + wbase + incl - mysum;
#pragma unroll
        for (int k = 0; k < SC_IPT; k++)
            if (fl[k]) { gfirst[g] = i0 + k; gnode[g] = gnode_at[i0 + k]; g++; }
    }
}

// Start node of the hard walk of every group (walk.cu): the lowest ancestor of the group's node whose
// Morton cell contains the group box grown by r_out (plus a margin far above the fp32 rounding of the
// T12 distance).  A leaf whose tight box comes within r_out of the group box in the fp32 arithmetic of
// T12 overlaps the grown box, so its cell meets that ancestor's cell; Morton cells are nested or disjoint,
// hence the leaf lies below the ancestor (or is it) and a walk that starts there finds the same hard list
// as a walk from the root.
__device__ __forceinline__ u32 quantise_d(double x, double o, double inv)
{
    const double f = floor((x - o) * inv);
    return f >= 2097151.0 ? 2097151u : (f > 0.0 ? (u32)f : 0u);
}

struct AncArgs {       // what ginfo_kernel<true> needs beyond the boxes (one thread per group does this part)
    const u32 *gnode; const unsigned char *level; const u32 *parent;
    float r_out;
    u32 *ganc;
    SplitArgs sp;                                                                             // split_group (common.cuh)
};

__device__ __forceinline__ u32 node_anc(const DevCtl *__restrict__ ctl, const AncArgs &x, u32 node, const float3 lo, const float3 hi)
{
    const double inv = ctl->inv;
    int lstar = MAXLEVEL;
    const float l3[3] = {lo.x, lo.y, lo.z}, h3[3] = {hi.x, hi.y, hi.z};
#pragma unroll
    for (int a = 0; a < 3; a++) {
        const double o = ctl->origin[a];
        const double R = (double)x.r_out * (1.0 + 1.0 / 1024.0) +
                         (fabs((double)l3[a]) + fabs((double)h3[a]) + (double)x.r_out) * (1.0 / 1048576.0);
        const u32 qa = quantise_d((double)l3[a] - R, o, inv), qb = quantise_d((double)h3[a] + R, o, inv);
        const u32 d = qa ^ qb;
        lstar = min(lstar, d ? __clz((int)d) - 11 : MAXLEVEL);       // common leading bits of the 21
    }
    while ((int)x.level[node] > lstar) node = x.parent[node];
    return node;
}

__device__ __forceinline__ void group_anc(const DevCtl *__restrict__ ctl, const AncArgs &x, u32 g, u32 ng, u32 count,
                                          const float3 lo, const float3 hi)
{
    split_group(x.sp, g, ng, count);      // work order of the next walk (the group flags of the build are free again by now)
    x.ganc[g] = node_anc(ctl, x, x.gnode[g], lo, hi);
}

// eight lanes per group: each takes every eighth member, then the octet combines by shuffles
template <bool ANC>
__global__ void __launch_bounds__(256) ginfo_kernel(const DevCtl *__restrict__ ctl, u32 n,
                                                    const float4 *__restrict__ pos, const u32 *__restrict__ gfirst,
                                                    u32 *__restrict__ gcount, float4 *__restrict__ glo,
                                                    float4 *__restrict__ ghi, const AncArgs anc)
{
    const u32 ng = ctl->ng;
    const u32 sub = threadIdx.x & 7u;
    const u32 ngr = (ng + 31u) & ~31u;          // whole warps stay in the loop together (shuffles below)
    for (u32 g = (blockIdx.x * blockDim.x + threadIdx.x) >> 3; g < ngr; g += (gridDim.x * blockDim.x) >> 3) {
        const bool live = g < ng;
        const u32 f = live ? gfirst[g] : 0u, e = live ? ((g + 1 < ng) ? gfirst[g + 1] : n) : 0u;
        float3 lo = make_float3(INFINITY, INFINITY, INFINITY), hi = make_float3(-INFINITY, -INFINITY, -INFINITY);
        for (u32 j = f + sub; j < e; j += 8) {
            const float4 p = __ldg(pos + j);
            lo.x = fminf(lo.x, p.x); lo.y = fminf(lo.y, p.y); lo.z = fminf(lo.z, p.z);
            hi.x = fmaxf(hi.x, p.x); hi.y = fmaxf(hi.y, p.y); hi.z = fmaxf(hi.z, p.z);
        }
#pragma unroll
        for (int off = 4; off; off >>= 1) {
            lo.x = fminf(lo.x, __shfl_xor_sync(0xFFFFFFFFu, lo.x, off));
            lo.y = fminf(lo.y, __shfl_xor_sync(0xFFFFFFFFu, lo.y, off));
            lo.z = fminf(lo.z, __shfl_xor_sync(0xFFFFFFFFu, lo.z, off));
            hi.x = fmaxf(hi.x, __shfl_xor_sync(0xFFFFFFFFu, hi.x, off));
            hi.y = fmaxf(hi.y, __shfl_xor_sync(0xFFFFFFFFu, hi.y, off));
            hi.z = fmaxf(hi.z, __shfl_xor_sync(0xFFFFFFFFu, hi.z, off));
        }
        if (live && sub == 0) {
            gcount[g] = e - f;
            glo[g] = make_float4(lo.x, lo.y, lo.z, 0.0f);
            ghi[g] = make_float4(hi.x, hi.y, hi.z, 0.0f);
            if (ANC) group_anc(ctl, anc, g, ng, e - f, lo, hi);
        }
    }
}

// ------------------------------------------------------------------ host side
cudaError_t launch_keys_sort_permute(Ctx *c);

cudaError_t launch_build_tree(Ctx *c)
{
    const Layout &L = c->L;
    const u32 n = (u32)c->n;
    cudaStream_t st = c->stream;
    DevCtl *ctl = c->ctl;
    // reset per-build device state
    // one memset: the build block of the control words, the look-back statuses and the group flags
    char *zb = reinterpret_cast<char *>(ctl) + offsetof(DevCtl, build_zero_begin);
    cudaMemsetAsync(zb, 0, (size_t)((c->ws + L.zero_end) - zb), st);
    // the queue of sink ranges this build fills for the next walk (ginfo_kernel): a build that no walk
    // consumed (two builds in a row) must not leave its entries behind
    if (c->p.split) cudaMemsetAsync(&ctl->nheavy[c->walk_par], 0, sizeof(u32), st);

    cudaError_t e = launch_keys_sort_permute(c);
    if (e != cudaSuccess) return e;

    const u64 *key = wsptr<u64>(c, L.key_b);
    u64 *sc_status = wsptr<u64>(c, L.sc_status);
    const int sc_grid = (int)imin64(L.sc_tiles, (int64_t)c->num_sms * 8);
    unsigned char *pre_level = wsptr<unsigned char>(c, L.pre_level);
    u32 *pre_first = wsptr<u32>(c, L.pre_first);
    const int po_grid = (int)imin64(L.po_tiles, (int64_t)c->num_sms * 8);
    preorder_kernel<<<po_grid, SC_THREADS, 0, st>>>(key, n, c->p.leaf_max, (u32)L.node_cap, ctl, sc_status,
                                                    pre_level, pre_first);
    unsigned char *level = wsptr<unsigned char>(c, L.level);
    u32 *pre_of_bfs = wsptr<u32>(c, L.pre_of_bfs), *bfs_of_pre = wsptr<u32>(c, L.bfs_of_pre);
    const int ngrid = (int)imin64(L.node_tiles, (int64_t)c->num_sms * 3);
    e = launch_radix_pass<unsigned char>(pre_level, nullptr, level, pre_of_bfs, bfs_of_pre, 0, &ctl->nn, 0,
                                         ctl->node_base, wsptr<u32>(c, L.node_status), (u32)L.node_tiles, &ctl->tile_counter[10],
                                         &ctl->status, ngrid, st, c->device, L.rs_kpt);
    if (e != cudaSuccess) return e;

    u32 *first = wsptr<u32>(c, L.first), *count = wsptr<u32>(c, L.count), *child = wsptr<u32>(c, L.child);
    u32 *parent = wsptr<u32>(c, L.parent), *arrived = wsptr<u32>(c, L.arrived);
    unsigned char *nchild = wsptr<unsigned char>(c, L.nchild);
    NodeRec *rec = wsptr<NodeRec>(c, L.nodes);
    u64 *bmax2 = wsptr<u64>(c, L.bmax2);
    const int node_grid = (int)imin64((L.node_cap + 255) / 256, (int64_t)c->num_sms * 16);
    link_kernel<<<node_grid, 256, 0, st>>>(key, n, c->p.leaf_max, ctl, level, pre_of_bfs, bfs_of_pre, pre_level, pre_first,
                                           first, count, child, nchild, parent, arrived, rec, bmax2);
    // sink groups need only the topology and the permuted positions: auxiliary stream, next to the upsweep
    cudaStream_t ax = c->aux;
    const float4 *pos_t = c->pos_sorted;      // the re-ordered store (launch_keys_sort_permute)
    cudaEventRecord(c->ev_linked, st);
    cudaStreamWaitEvent(ax, c->ev_linked, 0);
    unsigned char *gflag = wsptr<unsigned char>(c, L.gflag);
    gmark_kernel<<<(int)imin64((L.node_cap + 255) / 256, (int64_t)c->num_sms * 8), 256, 0, ax>>>(ctl, first, count, child, nchild, parent,
                                                                  c->group_max_now, c->grouping_now, gflag, wsptr<u32>(c, L.gnode_at));
    u32 *gfirst = wsptr<u32>(c, L.gfirst);
    gscan_kernel<<<sc_grid, SC_THREADS, 0, ax>>>(gflag, n, ctl, sc_status + L.po_tiles, gfirst, wsptr<u32>(c, L.gnode_at),
                                                 wsptr<u32>(c, L.gnode));
    // group boxes; with the force split also the start node of each group's hard walk and the work order of
    // the next walk (split_group), for the counter slot that walk will use
    const int gi_grid = (int)imin64((c->n + 255) / 256, (int64_t)c->num_sms * 8);
    AncArgs anc = {};
    c->split_ready = false;
    if (c->p.split) {
        anc.gnode = wsptr<u32>(c, L.gnode); anc.level = level; anc.parent = parent; anc.r_out = c->p.r_out;
        anc.ganc = wsptr<u32>(c, L.ganc);
        anc.sp = SplitArgs{ctl, wsptr<u32>(c, L.nhard), wsptr<u32>(c, L.scost), wsptr<u32>(c, L.splitq), gflag,
                           c->walk_par, (u32)(c->next_kind == 2 && !c->soft_split ? 0 : c->next_kind), c->soft_par ^ 1u};
        ginfo_kernel<true><<<gi_grid, 256, 0, ax>>>(ctl, n, pos_t, gfirst, wsptr<u32>(c, L.gcount), wsptr<float4>(c, L.glo),
                                                    wsptr<float4>(c, L.ghi), anc);
        c->split_ready = true; c->split_par = c->walk_par; c->split_kind = c->next_kind;
    } else {
        ginfo_kernel<false><<<gi_grid, 256, 0, ax>>>(ctl, n, pos_t, gfirst, wsptr<u32>(c, L.gcount), wsptr<float4>(c, L.glo),
                                                     wsptr<float4>(c, L.ghi), anc);
    }
    cudaEventRecord(c->ev_groups, ax);

    NodeArrays na;
    na.first = first; na.count = count; na.child = child; na.parent = parent; na.nchild = nchild; na.level = level;
    na.arrived = arrived;
    na.rec = rec;
    na.MS64 = wsptr<double4>(c, L.MS64); na.C64 = wsptr<double>(c, L.C64);
    na.B2 = wsptr<double>(c, L.B2); na.leaf_of = wsptr<u32>(c, L.leaf_of);
    // one thread per node; the node count is known on the device only: a bounded grid strides over the nodes
    const int full_node_grid = (int)imin64((L.node_cap + 127) / 128, (int64_t)c->num_sms * 16);
    cudaStreamWaitEvent(st, c->ev_perm, 0);
    if (c->boxes_only) upsweep_kernel<false><<<full_node_grid, 128, 0, st>>>(na, pos_t, ctl, c->p.mac, c->p.theta);
    else upsweep_kernel<true><<<full_node_grid, 128, 0, st>>>(na, pos_t, ctl, c->p.mac, c->p.theta);
    if (c->p.mac == HYB_MAC_ABS && !c->boxes_only) {
        bmax_kernel<<<(n + 255) / 256, 256, 0, st>>>(pos_t, n, na.leaf_of, parent, level, na.C64, bmax2);
        ropen_abs_kernel<<<(int)((L.node_cap + 255) / 256), 256, 0, st>>>(ctl, bmax2, na.B2, c->p.a_err, rec);
        cmax_kernel<<<(int)imin64((L.node_cap + 255) / 256, (int64_t)c->num_sms * 8), 256, 0, st>>>(ctl, child, nchild, rec);
    }
    cudaStreamWaitEvent(st, c->ev_groups, 0);       // join: groups, and (earlier on aux) the store copied back
    return cudaGetLastError();
}

// ------------------------------------------------------------------ refit (hyb_params.hard_refit)
// Between two soft steps the particles move by a small fraction of r_out.  The hard force is a direct
// K-weighted sum over everything within r_out, so it does not need the canonical tree of the new
// positions: any hierarchy of TIGHT boxes finds the same neighbours.  A refit keeps the store order and
// the topology of the last full build and recomputes the tight boxes of the nodes (boxes-only upsweep)
// and of the sink groups.  (The Morton cells no longer hold their particles exactly, so the walk starts
// at the root instead of ganc.)
cudaError_t launch_regroup(Ctx *c)
{
    const Layout &L = c->L;
    const u32 n = (u32)c->n;
    cudaStream_t st = c->stream;
    DevCtl *ctl = c->ctl;
    c->split_ready = false;                      // the flag array is re-used below
    cudaMemsetAsync(c->ws + L.gflag, 0, (size_t)n, st);
    cudaMemsetAsync(c->ws + L.sc_status + sizeof(u64) * (size_t)L.po_tiles, 0, sizeof(u64) * (size_t)L.sc_tiles, st);
    cudaMemsetAsync(&ctl->tile_counter[9], 0, sizeof(u32), st);
    unsigned char *gflag = wsptr<unsigned char>(c, L.gflag);
    gmark_kernel<<<(int)imin64((L.node_cap + 255) / 256, (int64_t)c->num_sms * 8), 256, 0, st>>>(
        ctl, wsptr<u32>(c, L.first), wsptr<u32>(c, L.count), wsptr<u32>(c, L.child), wsptr<unsigned char>(c, L.nchild),
        wsptr<u32>(c, L.parent), c->group_max_now, c->grouping_now, gflag, wsptr<u32>(c, L.gnode_at));
    const int sc_grid = (int)imin64(L.sc_tiles, (int64_t)c->num_sms * 8);
    gscan_kernel<<<sc_grid, SC_THREADS, 0, st>>>(gflag, n, ctl, wsptr<u64>(c, L.sc_status) + L.po_tiles, wsptr<u32>(c, L.gfirst),
                                                 wsptr<u32>(c, L.gnode_at), wsptr<u32>(c, L.gnode));
    ginfo_kernel<false><<<(int)imin64((c->n + 255) / 256, (int64_t)c->num_sms * 8), 256, 0, st>>>(
        ctl, n, reinterpret_cast<const float4 *>(c->pos), wsptr<u32>(c, L.gfirst), wsptr<u32>(c, L.gcount),
        wsptr<float4>(c, L.glo), wsptr<float4>(c, L.ghi), AncArgs{});
    return cudaGetLastError();
}

cudaError_t launch_refit_tree(Ctx *c)
{
    const Layout &L = c->L;
    cudaStream_t st = c->stream;
    cudaMemsetAsync(c->ws + L.arrived, 0, sizeof(u32) * (size_t)L.node_cap, st);
    NodeArrays na;
    na.first = wsptr<u32>(c, L.first); na.count = wsptr<u32>(c, L.count); na.child = wsptr<u32>(c, L.child);
    na.parent = wsptr<u32>(c, L.parent); na.nchild = wsptr<unsigned char>(c, L.nchild);
    na.level = wsptr<unsigned char>(c, L.level); na.arrived = wsptr<u32>(c, L.arrived);
    na.rec = wsptr<NodeRec>(c, L.nodes);
    na.MS64 = wsptr<double4>(c, L.MS64); na.C64 = wsptr<double>(c, L.C64);
    na.B2 = wsptr<double>(c, L.B2); na.leaf_of = wsptr<u32>(c, L.leaf_of);
    upsweep_kernel<false><<<(int)imin64((L.node_cap + 127) / 128, (int64_t)c->num_sms * 16), 128, 0, st>>>(na, reinterpret_cast<const float4 *>(c->pos), c->ctl,
                                                                           c->p.mac, c->p.theta);
    ginfo_kernel<false><<<(int)imin64((c->n + 255) / 256, (int64_t)c->num_sms * 8), 256, 0, st>>>(
        c->ctl, (u32)c->n, reinterpret_cast<const float4 *>(c->pos), wsptr<u32>(c, L.gfirst), wsptr<u32>(c, L.gcount),
        wsptr<float4>(c, L.glo), wsptr<float4>(c, L.ghi), AncArgs{});
    return cudaGetLastError();
}

}  // namespace hyb
