// walk.cu -- steps a8, a9, a11: group tree walk with interaction lists staged in shared memory
// and evaluated on the FP32 pipes.  (T12-T15.)
//
// One warp owns one sink group at a time (groups are handed out by an atomic counter; the next
// group id is requested while the current group is processed).
//   traversal : the per-warp stack (shared memory) holds one descriptor per OPENED cell
//               (first child | (nchild-1) << 29).  An iteration pops up to four descriptors; the
//               eight lanes of an octet test the up-to-eight children of one of them (children are
//               contiguous in breadth-first numbering, T7).  Accepted cells are compacted by
//               ballot into the monopole buffer, opened cells push their descriptor, opened
//               leaves queue (first, count) and are expanded 32 leaves at a time into the
//               monopole buffer (farther than r_out: K == 0 for every pair) or the near buffer.
//               The node records of the next batch are requested before the current batch is
//               appended / evaluated, so their latency overlaps that work.
//   evaluation: whenever a buffer fills, all lanes stream it from shared memory.  Lane l holds
//               S sinks (l mod A) + k A, k < S, and works on every P-th buffer entry starting at
//               l / A, A = ceil(members / S), P = floor(32 / A); S in {2, 3, 4} is chosen per group
//               to maximise the fraction of busy lanes.  The P partial sums per sink are combined
//               through shared memory at the end.
// The whole per-group control flow is one loop with a single call site for each evaluation
// routine (flags request a flush and the loop comes back to it), which keeps the code small.
#include "common.cuh"

namespace hyb {

struct WalkArgs {
    const float4 *pos;            // Morton-ordered particles (x,y,z,m)
    const float4 *nodeA, *nodeB, *nodeC;
    const uint2 *meta;
    const u32 *gfirst, *gcount;
    const float4 *glo, *ghi;
    u32 *ncell, *npart, *nhard;
    float4 *a_soft, *a_hard;
    DevCtl *ctl;
    float G, eps2, rout, kc0, kc1;   // Y = sat(kc0 + kc1 r)
};

constexpr int WK_SMAX = 4;          // most sinks per lane
constexpr u32 FULL = 0xFFFFFFFFu;
constexpr u32 DESC_MASK = 0x1FFFFFFFu;      // node index bits of a stack descriptor

template <int MODE>
struct SmemLayout {                 // per warp
    static constexpr int cell_cap = MODE == WALK_HARD ? 0 : WK_CELL_CAP;
    static constexpr int part_cap = MODE == WALK_NORMAL ? 0 : WK_PART_CAP;
    static constexpr int stack_cap = MODE == WALK_HARD ? 512 : 768;
    static constexpr int lq_cap = 64;
    static constexpr size_t bytes = 16 * (size_t)(cell_cap + part_cap) + 4 * (size_t)stack_cap + 8 * 2 * (size_t)lq_cap;
    static constexpr int ctas_per_sm = MODE == WALK_HARD ? 3 : 2;
};

// ---- pair kernels ---------------------------------------------------------------------------
__device__ __forceinline__ float rsqrt_approx(float x)
{
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float sqrt_approx(float x)
{
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// monopole (Eq. 2): 3 sub + 3 fma + rsqrt + 3 mul + 3 fma = 12 FP32-pipe instructions + 1 MUFU
__device__ __forceinline__ void mono(const float4 s, const float3 x, float eps2, float3 &a)
{
    float dx = s.x - x.x, dy = s.y - x.y, dz = s.z - x.z;
    float r2 = fmaf(dx, dx, eps2);
    r2 = fmaf(dy, dy, r2);
    r2 = fmaf(dz, dz, r2);
    float ri = rsqrt_approx(r2);
    float ri2 = ri * ri;
    float mr = s.w * ri;
    float mr3 = mr * ri2;
    a.x = fmaf(mr3, dx, a.x);
    a.y = fmaf(mr3, dy, a.y);
    a.z = fmaf(mr3, dz, a.z);
}

// Eq. 10 with Y clamped to [0,1]: K = t^3 (10 - 15 t + 6 t^2), t = Y^2 (T15)
__device__ __forceinline__ float kfun(float r, float kc0, float kc1)
{
    float Y = __saturatef(fmaf(r, kc1, kc0));
    float t = Y * Y;
    float poly = fmaf(fmaf(6.0f, t, -15.0f), t, 10.0f);
    return (t * t) * (t * poly);
}

// K-weighted pair (Eq. 8, 9): hard part K F, and (SOFT) the soft part (1 - K) F
template <bool SOFT>
__device__ __forceinline__ void kpair(const float4 s, const float3 x, float eps2, float kc0, float kc1, float3 &as,
                                      float3 &ah)
{
    float dx = s.x - x.x, dy = s.y - x.y, dz = s.z - x.z;
    float r2u = dx * dx;
    r2u = fmaf(dy, dy, r2u);
    r2u = fmaf(dz, dz, r2u);
    float ri = rsqrt_approx(r2u + eps2);
    float r = sqrt_approx(r2u);
    float ri2 = ri * ri;
    float mr = s.w * ri;
    float mr3 = mr * ri2;
    float wh = kfun(r, kc0, kc1) * mr3;
    ah.x = fmaf(wh, dx, ah.x);
    ah.y = fmaf(wh, dy, ah.y);
    ah.z = fmaf(wh, dz, ah.z);
    if (SOFT) {
        float ws = mr3 - wh;
        as.x = fmaf(ws, dx, as.x);
        as.y = fmaf(ws, dy, as.y);
        as.z = fmaf(ws, dz, as.z);
    }
}

template <int S>
__device__ __forceinline__ void eval_mono(const float4 *buf, int cnt, int part, int P, const float3 (&x)[WK_SMAX],
                                          float eps2, float3 (&acc)[WK_SMAX])
{
#pragma unroll 2
    for (int j = part; j < cnt; j += P) {
        const float4 s = buf[j];
#pragma unroll
        for (int k = 0; k < S; k++) mono(s, x[k], eps2, acc[k]);
    }
}

template <int S, bool SOFT>
__device__ __forceinline__ void eval_near(const float4 *buf, int cnt, int part, int P, const float3 (&x)[WK_SMAX],
                                          float eps2, float kc0, float kc1, float3 (&as)[WK_SMAX],
                                          float3 (&ah)[WK_SMAX])
{
#pragma unroll 1
    for (int j = part; j < cnt; j += P) {
        const float4 s = buf[j];
#pragma unroll
        for (int k = 0; k < S; k++) kpair<SOFT>(s, x[k], eps2, kc0, kc1, as[k], ah[k]);
    }
}

__device__ __forceinline__ u32 warp_excl_scan(u32 v, int lane, u32 &total)
{
    u32 incl = v;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        u32 t = __shfl_up_sync(FULL, incl, off);
        if (lane >= off) incl += t;
    }
    total = __shfl_sync(FULL, incl, 31);
    return incl - v;
}

template <int MODE>
__global__ void __launch_bounds__(WK_WARPS * 32, SmemLayout<MODE>::ctas_per_sm) walk_kernel(const WalkArgs a)
{
    using SL = SmemLayout<MODE>;
    constexpr bool HAS_MONO = MODE != WALK_HARD;      // monopole buffer (cells, far particles)
    constexpr bool HAS_NEAR = MODE != WALK_NORMAL;    // K-weighted buffer
    constexpr int C = MODE == WALK_HYBRID ? 6 : 3;    // accumulated components per sink
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int oct = lane >> 3, sub = lane & 7;
    unsigned char *wbase = smem_raw + (size_t)warp * SL::bytes;
    float4 *cellbuf = reinterpret_cast<float4 *>(wbase);
    float4 *partbuf = cellbuf + SL::cell_cap;
    u32 *stack = reinterpret_cast<u32 *>(partbuf + SL::part_cap);
    uint2 *lq0 = reinterpret_cast<uint2 *>(stack + SL::stack_cap);     // far leaves
    uint2 *lq1 = lq0 + SL::lq_cap;                                     // near leaves
    float *red = reinterpret_cast<float *>(wbase);                     // reduction scratch (buffers are empty then)

    const u32 lt_mask = (1u << lane) - 1u;
    const u32 ng = a.ctl->ng;
    const float rout2 = __fmul_rn(a.rout, a.rout);
    const float eps2 = a.eps2, kc0 = a.kc0, kc1 = a.kc1;
    unsigned long long isoft = 0, ihard = 0;

    u32 g = 0;
    if (lane == 0) g = atomicAdd(&a.ctl->group_counter, 1u);
    g = __shfl_sync(FULL, g, 0);

    while (g < ng) {
        u32 g_next = 0;
        if (lane == 0) g_next = atomicAdd(&a.ctl->group_counter, 1u);      // consumed at the end of this group
        const u32 gf = a.gfirst[g];
        const int n = (int)a.gcount[g];
        const float4 glo = a.glo[g], ghi = a.ghi[g];
        // sinks per lane: maximise n P / (32 S) over S in {2,3,4}; ties go to the larger S
        int S = 2, A = (n + 1) >> 1, P = 32 / A;
        {
            const int A3 = (n + 2) / 3, P3 = 32 / A3, A4 = (n + 3) >> 2, P4 = 32 / A4;
            int best = 6 * P;
            if (4 * P3 >= best) { best = 4 * P3; S = 3; A = A3; P = P3; }
            if (3 * P4 >= best) { S = 4; A = A4; P = P4; }
        }
        const int aidx = lane % A;
        const int part = (lane / A < P) ? lane / A : 0x40000000;     // idle lanes never enter the loops
        float3 x[WK_SMAX], as[WK_SMAX], ah[WK_SMAX];
#pragma unroll
        for (int k = 0; k < WK_SMAX; k++) {
            const int si = aidx + k * A;
            const float4 p = __ldg(a.pos + gf + ((k < S && si < n) ? si : 0));
            x[k] = make_float3(p.x, p.y, p.z);
            as[k] = make_float3(0.0f, 0.0f, 0.0f);
            ah[k] = make_float3(0.0f, 0.0f, 0.0f);
        }

        u32 ncell = 0, npart = 0, nhard = 0;
        int ncb = 0, npb = 0;             // buffer fills
        int nlq0 = 0, nlq1 = 0;           // leaf queue fills
        int sp = 0;
        bool trav_done = false, flush_mono = false, flush_near = false, overflow = false;
        int ex_near = 0;                  // pending expansion: target buffer, this lane's leaf, progress
        u32 ex_first = 0, ex_cnt = 0, ex_off = 0, ex_T = 0, ex_done = 0;

        // current batch of nodes (one per lane); starts with the root alone
        bool have = lane == 0;
        u32 node = 0;
        float4 nA = make_float4(0, 0, 0, 0), nB = nA, nC = nA;
        uint2 mt = make_uint2(0, 0);
        if (have) {
            nB = __ldg(a.nodeB); nC = __ldg(a.nodeC); mt = __ldg(a.meta);
            if (MODE != WALK_HARD) nA = __ldg(a.nodeA);
        }

        for (;;) {
            // ---- evaluation: the only call sites
            if (HAS_MONO && flush_mono) {
                __syncwarp();
                if (S == 2) eval_mono<2>(cellbuf, ncb, part, P, x, eps2, as);
                else if (S == 3) eval_mono<3>(cellbuf, ncb, part, P, x, eps2, as);
                else eval_mono<4>(cellbuf, ncb, part, P, x, eps2, as);
                ncb = 0; flush_mono = false;
                __syncwarp();
            }
            if (HAS_NEAR && flush_near) {
                __syncwarp();
                if (S == 2) eval_near<2, MODE == WALK_HYBRID>(partbuf, npb, part, P, x, eps2, kc0, kc1, as, ah);
                else if (S == 3) eval_near<3, MODE == WALK_HYBRID>(partbuf, npb, part, P, x, eps2, kc0, kc1, as, ah);
                else eval_near<4, MODE == WALK_HYBRID>(partbuf, npb, part, P, x, eps2, kc0, kc1, as, ah);
                npb = 0; flush_near = false;
                __syncwarp();
            }
            // ---- pending leaf expansion: every lane copies the part of its leaf that fits
            if (ex_done < ex_T) {
                const bool tonear = HAS_NEAR && (!HAS_MONO || ex_near);
                float4 *buf = tonear ? partbuf : cellbuf;
                const int cap = tonear ? SL::part_cap : SL::cell_cap;
                int fill = tonear ? npb : ncb;
                const u32 take = min((u32)(cap - fill), ex_T - ex_done);
                const u32 lo = max(ex_off, ex_done), hi = min(ex_off + ex_cnt, ex_done + take);
                for (u32 e = lo; e < hi; e++) buf[fill + (e - ex_done)] = __ldg(a.pos + ex_first + (e - ex_off));
                fill += (int)take; ex_done += take;
                if (tonear) npb = fill; else ncb = fill;
                if (ex_done < ex_T) { if (tonear) flush_near = true; else flush_mono = true; }    // buffer is full
                continue;
            }
            // ---- start an expansion when a leaf queue holds a full batch (or at the end)
            {
                int cls = -1;
                if (HAS_MONO && (nlq0 >= 32 || (trav_done && nlq0 > 0))) cls = 0;
                else if (HAS_NEAR && (nlq1 >= 32 || (trav_done && nlq1 > 0))) cls = 1;
                if (cls >= 0) {
                    __syncwarp();
                    int &nlq = cls ? nlq1 : nlq0;
                    const uint2 *q = cls ? lq1 : lq0;
                    const int m = min(32, nlq);
                    uint2 lf = make_uint2(0, 0);
                    if (lane < m) lf = q[nlq - m + lane];
                    nlq -= m;
                    ex_first = lf.x; ex_cnt = lf.y;
                    ex_off = warp_excl_scan(ex_cnt, lane, ex_T);
                    ex_done = 0; ex_near = cls;
                    __syncwarp();
                    continue;
                }
            }
            if (trav_done) {
                if (HAS_MONO && ncb > 0) { flush_mono = true; continue; }
                if (HAS_NEAR && npb > 0) { flush_near = true; continue; }
                break;
            }
            // ---- traversal iteration on the current batch
            if (HAS_MONO && ncb > SL::cell_cap - 32) { flush_mono = true; continue; }
            bool accept = false, open_int = false, leaf_far = false, leaf_near = false;
            if (have) {
                // T12: box-box distance (rule (b)), fp32, one rounding per operation
                float fx = fmaxf(0.0f, fmaxf(__fsub_rn(nB.x, ghi.x), __fsub_rn(glo.x, nC.x)));
                float fy = fmaxf(0.0f, fmaxf(__fsub_rn(nB.y, ghi.y), __fsub_rn(glo.y, nC.y)));
                float fz = fmaxf(0.0f, fmaxf(__fsub_rn(nB.z, ghi.z), __fsub_rn(glo.z, nC.z)));
                float d2b = __fadd_rn(__fadd_rn(__fmul_rn(fx, fx), __fmul_rn(fy, fy)), __fmul_rn(fz, fz));
                const bool near = d2b < rout2;
                bool open;
                if (MODE == WALK_HARD) open = near;
                else {
                    float ex = fmaxf(0.0f, fmaxf(__fsub_rn(glo.x, nA.x), __fsub_rn(nA.x, ghi.x)));
                    float ey = fmaxf(0.0f, fmaxf(__fsub_rn(glo.y, nA.y), __fsub_rn(nA.y, ghi.y)));
                    float ez = fmaxf(0.0f, fmaxf(__fsub_rn(glo.z, nA.z), __fsub_rn(nA.z, ghi.z)));
                    float d2a = __fadd_rn(__fadd_rn(__fmul_rn(ex, ex), __fmul_rn(ey, ey)), __fmul_rn(ez, ez));
                    const bool mac_open = d2a < nB.w;
                    open = (MODE == WALK_NORMAL) ? mac_open : (mac_open || near);
                }
                const bool is_leaf = (mt.y & 0x80000000u) != 0;
                accept = !open && MODE != WALK_HARD;
                open_int = open && !is_leaf;
                leaf_near = open && is_leaf && near && MODE != WALK_NORMAL;
                leaf_far = open && is_leaf && !leaf_near;
            }
            // opened cells: push one descriptor each
            {
                const u32 bal = __ballot_sync(FULL, open_int);
                const int npush = __popc(bal);
                if (sp + npush > SL::stack_cap) { overflow = true; break; }
                if (open_int) stack[sp + __popc(bal & lt_mask)] = mt.x | ((mt.y - 1u) << 29);
                sp += npush;
            }
            __syncwarp();
            // pop the next batch and request its node records
            const int npop = min(4, sp);
            bool have_n = false;
            u32 node_n = 0;
            if (oct < npop) {
                const u32 d = stack[sp - 1 - oct];
                node_n = (d & DESC_MASK) + (u32)sub;
                have_n = (u32)sub <= (d >> 29);
            }
            sp -= npop;
            float4 nA_n = make_float4(0, 0, 0, 0), nB_n = nA_n, nC_n = nA_n;
            uint2 mt_n = make_uint2(0, 0);
            if (have_n) {
                nB_n = __ldg(a.nodeB + node_n); nC_n = __ldg(a.nodeC + node_n); mt_n = __ldg(a.meta + node_n);
                if (MODE != WALK_HARD) nA_n = __ldg(a.nodeA + node_n);
            }
            // accepted cells -> monopole buffer
            if (HAS_MONO) {
                const u32 bal = __ballot_sync(FULL, accept);
                if (accept) cellbuf[ncb + __popc(bal & lt_mask)] = nA;
                ncb += __popc(bal);
                ncell += __popc(bal);
            }
            // opened leaves -> queues
            if (HAS_MONO) {
                const u32 bal = __ballot_sync(FULL, leaf_far);
                if (bal) {
                    const u32 cnt = leaf_far ? (mt.y & 0x7FFFFFFFu) : 0u;
                    if (leaf_far) lq0[nlq0 + __popc(bal & lt_mask)] = make_uint2(mt.x, cnt);
                    nlq0 += __popc(bal);
                    npart += __reduce_add_sync(FULL, cnt);
                }
            }
            if (HAS_NEAR) {
                const u32 bal = __ballot_sync(FULL, leaf_near);
                if (bal) {
                    const u32 cnt = leaf_near ? (mt.y & 0x7FFFFFFFu) : 0u;
                    if (leaf_near) lq1[nlq1 + __popc(bal & lt_mask)] = make_uint2(mt.x, cnt);
                    nlq1 += __popc(bal);
                    const u32 tot = __reduce_add_sync(FULL, cnt);
                    npart += tot; nhard += tot;
                }
            }
            // rotate
            have = have_n; node = node_n; nA = nA_n; nB = nB_n; nC = nC_n; mt = mt_n;
            if (npop == 0) trav_done = true;
        }
        (void)node;
        __syncwarp();
        if (overflow && lane == 0) atomicOr(&a.ctl->status, ST_STACK_OVERFLOW);

        // ---- combine the P partial sums per sink through shared memory: row r = k C + c holds
        //      component c of sink slot k for all 32 lanes; lane (aidx, part) sums rows part, part+P, ...
        float v[WK_SMAX * C];
#pragma unroll
        for (int k = 0; k < WK_SMAX; k++) {
            if (MODE != WALK_HARD) { v[k * C + 0] = as[k].x; v[k * C + 1] = as[k].y; v[k * C + 2] = as[k].z; }
            if (MODE == WALK_HYBRID) { v[k * C + 3] = ah[k].x; v[k * C + 4] = ah[k].y; v[k * C + 5] = ah[k].z; }
            if (MODE == WALK_HARD) { v[k * C + 0] = ah[k].x; v[k * C + 1] = ah[k].y; v[k * C + 2] = ah[k].z; }
        }
        if (P > 1) {
            const int rows = S * C;
#pragma unroll
            for (int r = 0; r < WK_SMAX * C; r++)
                if (r < rows) red[r * 32 + lane] = v[r];
            __syncwarp();
            for (int r = part; r < rows; r += P) {
                float sum = red[r * 32 + aidx];
                for (int q = 1; q < P; q++) sum += red[r * 32 + aidx + q * A];
                red[r * 32 + aidx] = sum;
            }
            __syncwarp();
            if (lane < A) {
#pragma unroll
                for (int r = 0; r < WK_SMAX * C; r++)
                    if (r < rows) v[r] = red[r * 32 + lane];
            }
            __syncwarp();
        }
        if (lane < A) {
#pragma unroll
            for (int k = 0; k < WK_SMAX; k++) {
                const int si = lane + k * A;
                if (k < S && si < n) {
                    if (MODE == WALK_HYBRID) {
                        a.a_soft[gf + si] = make_float4(a.G * v[k * C], a.G * v[k * C + 1], a.G * v[k * C + 2], 0.0f);
                        a.a_hard[gf + si] = make_float4(a.G * v[k * C + 3], a.G * v[k * C + 4], a.G * v[k * C + 5], 0.0f);
                    } else if (MODE == WALK_NORMAL) {
                        a.a_soft[gf + si] = make_float4(a.G * v[k * C], a.G * v[k * C + 1], a.G * v[k * C + 2], 0.0f);
                        a.a_hard[gf + si] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
                    } else {
                        a.a_hard[gf + si] = make_float4(a.G * v[k * C], a.G * v[k * C + 1], a.G * v[k * C + 2], 0.0f);
                    }
                }
            }
        }
        if (lane == 0) {
            a.ncell[g] = ncell; a.npart[g] = npart; a.nhard[g] = nhard;
            if (MODE != WALK_HARD) isoft += (unsigned long long)n * (unsigned long long)(ncell + npart);
            if (MODE != WALK_NORMAL) ihard += (unsigned long long)n * (unsigned long long)nhard;
        }
        g = __shfl_sync(FULL, g_next, 0);
    }
    if (lane == 0) {
        if (isoft) atomicAdd(&a.ctl->inter_soft, isoft);
        if (ihard) atomicAdd(&a.ctl->inter_hard, ihard);
    }
}

__global__ void zero_acc_kernel(float4 *a, u32 n)
{
    for (u32 i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x)
        a[i] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
}

cudaError_t launch_zero_acc(Ctx *c, hyb_float4 *a)
{
    zero_acc_kernel<<<(int)imin64((c->n + 255) / 256, (int64_t)c->num_sms * 8), 256, 0, c->stream>>>(
        reinterpret_cast<float4 *>(a), (u32)c->n);
    return cudaGetLastError();
}

template <int MODE>
static cudaError_t launch_walk_mode(Ctx *c, const WalkArgs &a)
{
    using SL = SmemLayout<MODE>;
    const size_t smem = SL::bytes * WK_WARPS;
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(walk_kernel<MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    walk_kernel<MODE><<<c->num_sms * SL::ctas_per_sm, WK_WARPS * 32, smem, c->stream>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_walk(Ctx *c, int mode)
{
    const Layout &L = c->L;
    WalkArgs a;
    a.pos = reinterpret_cast<const float4 *>(c->pos);
    a.nodeA = wsptr<float4>(c, L.nodeA); a.nodeB = wsptr<float4>(c, L.nodeB); a.nodeC = wsptr<float4>(c, L.nodeC);
    a.meta = wsptr<uint2>(c, L.meta);
    a.gfirst = wsptr<u32>(c, L.gfirst); a.gcount = wsptr<u32>(c, L.gcount);
    a.glo = wsptr<float4>(c, L.glo); a.ghi = wsptr<float4>(c, L.ghi);
    a.ncell = wsptr<u32>(c, L.ncell); a.npart = wsptr<u32>(c, L.npart); a.nhard = wsptr<u32>(c, L.nhard);
    a.a_soft = reinterpret_cast<float4 *>(c->a_soft); a.a_hard = reinterpret_cast<float4 *>(c->a_hard);
    a.ctl = c->ctl;
    a.G = c->p.G; a.eps2 = c->p.eps * c->p.eps; a.rout = c->p.r_out;
    const float w = c->p.r_out - c->p.r_in;
    a.kc0 = c->p.r_out / w; a.kc1 = -1.0f / w;
    cudaMemsetAsync(&c->ctl->group_counter, 0, sizeof(u32), c->stream);
    if (mode == WALK_HYBRID) return launch_walk_mode<WALK_HYBRID>(c, a);
    if (mode == WALK_HARD) return launch_walk_mode<WALK_HARD>(c, a);
    return launch_walk_mode<WALK_NORMAL>(c, a);
}

}  // namespace hyb
