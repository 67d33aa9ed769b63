// walk.cu -- steps a8, a9, a11: group tree walk with interaction lists staged in shared memory
// and evaluated on the FP32 pipes.  (T12-T15.)
//
// One warp owns one sink group at a time (groups are handed out by an atomic counter).
//   traversal : each lane tests one node of the frontier (a per-warp stack in global memory);
//               ballots/prefix sums compact accepted cells into a monopole buffer, children of
//               opened cells back onto the stack, particles of opened leaves into the monopole
//               buffer (leaf farther than r_out: K == 0 for every pair) or the near buffer.
//   evaluation: whenever a buffer fills, all lanes stream it from shared memory.  Lane l holds
//               S sinks (l mod A) + k A and works on every P-th buffer entry starting at l / A,
//               A = ceil(members / S), P = floor(32 / A); partial sums over the P parts are
//               combined with shuffles at the end.  Small groups therefore still fill the warp.
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
    u32 *stacks;
    float G, eps2, rout, kc0, kc1;   // Y = sat(kc0 + kc1 r)
};

constexpr int WK_S = 2;     // sinks per lane

struct WarpSmem {
    float4 cell[WK_CELL_CAP];
    float4 part[WK_PART_CAP];
    u32 lf_first[32];
    u32 lf_off[33];
};

// ---- pair kernels ---------------------------------------------------------------------------
// monopole: 3 sub + 3 fma + rsqrt + 3 mul + 3 fma
__device__ __forceinline__ void mono(const float4 s, const float3 x, float eps2, float3 &a)
{
    float dx = s.x - x.x, dy = s.y - x.y, dz = s.z - x.z;
    float r2 = fmaf(dx, dx, eps2);
    r2 = fmaf(dy, dy, r2);
    r2 = fmaf(dz, dz, r2);
    float ri = rsqrtf(r2);
    float ri2 = ri * ri;
    float mr = s.w * ri;
    float mr3 = mr * ri2;
    a.x = fmaf(mr3, dx, a.x);
    a.y = fmaf(mr3, dy, a.y);
    a.z = fmaf(mr3, dz, a.z);
}

__device__ __forceinline__ float sqrt_approx(float x)
{
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// Eq. 10 with Y clamped to [0,1]: K = t^3 (10 - 15 t + 6 t^2), t = Y^2 (T15)
__device__ __forceinline__ float kfun(float r, float kc0, float kc1)
{
    float Y = __saturatef(fmaf(r, kc1, kc0));
    float t = Y * Y;
    float poly = fmaf(fmaf(6.0f, t, -15.0f), t, 10.0f);
    return (t * t) * (t * poly);
}

template <bool SOFT>
__device__ __forceinline__ void kpair(const float4 s, const float3 x, float eps2, float kc0, float kc1, float3 &as,
                                      float3 &ah)
{
    float dx = s.x - x.x, dy = s.y - x.y, dz = s.z - x.z;
    float r2u = dx * dx;
    r2u = fmaf(dy, dy, r2u);
    r2u = fmaf(dz, dz, r2u);
    float ri = rsqrtf(r2u + eps2);
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

__device__ __forceinline__ void eval_mono(const float4 *buf, int cnt, int part, int P, const float3 (&x)[WK_S],
                                          float eps2, float3 (&acc)[WK_S])
{
#pragma unroll 4
    for (int j = part; j < cnt; j += P) {
        const float4 s = buf[j];
#pragma unroll
        for (int k = 0; k < WK_S; k++) mono(s, x[k], eps2, acc[k]);
    }
}

template <bool SOFT>
__device__ __forceinline__ void eval_near(const float4 *buf, int cnt, int part, int P, const float3 (&x)[WK_S],
                                          float eps2, float kc0, float kc1, float3 (&as)[WK_S], float3 (&ah)[WK_S])
{
#pragma unroll 2
    for (int j = part; j < cnt; j += P) {
        const float4 s = buf[j];
#pragma unroll
        for (int k = 0; k < WK_S; k++) kpair<SOFT>(s, x[k], eps2, kc0, kc1, as[k], ah[k]);
    }
}

__device__ __forceinline__ u32 warp_excl_scan(u32 v, int lane, u32 &total)
{
    u32 incl = v;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        u32 t = __shfl_up_sync(0xFFFFFFFFu, incl, off);
        if (lane >= off) incl += t;
    }
    total = __shfl_sync(0xFFFFFFFFu, incl, 31);
    return incl - v;
}

template <int MODE>
__global__ void __launch_bounds__(WK_WARPS * 32, 2) walk_kernel(const WalkArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    WarpSmem &sm = reinterpret_cast<WarpSmem *>(smem_raw)[warp];
    u32 *stack = a.stacks + (size_t)(blockIdx.x * WK_WARPS + warp) * WK_STACK_CAP;
    const u32 lt_mask = (1u << lane) - 1u;
    const u32 ng = a.ctl->ng;
    const float rout2 = __fmul_rn(a.rout, a.rout);
    const float eps2 = a.eps2, kc0 = a.kc0, kc1 = a.kc1;

    for (;;) {
        u32 g = 0;
        if (lane == 0) g = atomicAdd(&a.ctl->group_counter, 1u);
        g = __shfl_sync(0xFFFFFFFFu, g, 0);
        if (g >= ng) break;
        const u32 gf = a.gfirst[g];
        const int n = (int)a.gcount[g];
        const float4 glo = a.glo[g], ghi = a.ghi[g];
        const int A = (n + WK_S - 1) / WK_S;
        const int P = 32 / A;
        const int aidx = lane % A;
        const int part = (lane / A < P) ? lane / A : 0x40000000;     // idle lanes never enter the loops
        float3 x[WK_S];
#pragma unroll
        for (int k = 0; k < WK_S; k++) {
            int si = aidx + k * A;
            float4 p = __ldg(a.pos + gf + (si < n ? si : 0));
            x[k] = make_float3(p.x, p.y, p.z);
        }
        float3 as[WK_S], ah[WK_S];
#pragma unroll
        for (int k = 0; k < WK_S; k++) { as[k] = make_float3(0, 0, 0); ah[k] = make_float3(0, 0, 0); }

        u32 ncell = 0, npart = 0, nhard = 0;
        int ncb = 0, npb = 0;       // buffer fills
        int sp = 1;
        if (lane == 0) stack[0] = 0;
        __syncwarp();
        bool overflow = false;

        while (sp > 0) {
            const int npop = min(32, sp);
            sp -= npop;
            const bool have = lane < npop;
            u32 node = 0;
            bool accept = false, open_int = false, leaf_far = false, leaf_near = false;
            uint2 mt = make_uint2(0, 0);
            float4 nA = make_float4(0, 0, 0, 0);
            if (have) {
                node = stack[sp + lane];
                const float4 nB = __ldg(a.nodeB + node), nC = __ldg(a.nodeC + node);
                mt = __ldg(a.meta + node);
                // T12: box-box distance (rule (b)), fp32, one rounding per operation
                float fx = fmaxf(0.0f, fmaxf(__fsub_rn(nB.x, ghi.x), __fsub_rn(glo.x, nC.x)));
                float fy = fmaxf(0.0f, fmaxf(__fsub_rn(nB.y, ghi.y), __fsub_rn(glo.y, nC.y)));
                float fz = fmaxf(0.0f, fmaxf(__fsub_rn(nB.z, ghi.z), __fsub_rn(glo.z, nC.z)));
                float d2b = __fadd_rn(__fadd_rn(__fmul_rn(fx, fx), __fmul_rn(fy, fy)), __fmul_rn(fz, fz));
                const bool near = d2b < rout2;
                bool open;
                if (MODE == WALK_HARD) open = near;
                else {
                    nA = __ldg(a.nodeA + node);
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
            // ---- children of opened cells back onto the stack
            {
                u32 tot;
                const u32 nch = open_int ? mt.y : 0u;
                const u32 off = warp_excl_scan(nch, lane, tot);
                if (sp + (int)tot > WK_STACK_CAP) { overflow = true; break; }
                for (u32 q = 0; q < nch; q++) stack[sp + off + q] = mt.x + q;
                sp += (int)tot;
            }
            // ---- accepted cells -> monopole buffer
            if (MODE != WALK_HARD) {
                if (ncb > WK_CELL_CAP - 32) {
                    __syncwarp();
                    eval_mono(sm.cell, ncb, part, P, x, eps2, as);
                    ncb = 0;
                    __syncwarp();
                }
                const u32 bal = __ballot_sync(0xFFFFFFFFu, accept);
                if (accept) sm.cell[ncb + __popc(bal & lt_mask)] = nA;
                ncb += __popc(bal);
                ncell += __popc(bal);
            }
            // ---- particles of opened leaves: far -> monopole buffer, near -> K buffer
#pragma unroll
            for (int cls = 0; cls < 2; cls++) {
                if (cls == 0 && MODE == WALK_HARD) continue;
                if (cls == 1 && MODE == WALK_NORMAL) continue;
                const bool mine = cls == 0 ? leaf_far : leaf_near;
                const u32 bal = __ballot_sync(0xFFFFFFFFu, mine);
                if (bal == 0) continue;
                u32 tot;
                const u32 cnt = mine ? (mt.y & 0x7FFFFFFFu) : 0u;
                const u32 off = warp_excl_scan(cnt, lane, tot);
                const int nleaf = __popc(bal);
                __syncwarp();
                if (mine) { int r = __popc(bal & lt_mask); sm.lf_first[r] = mt.x; sm.lf_off[r] = off; }
                __syncwarp();
                npart += tot;
                if (cls == 1) nhard += tot;
                float4 *buf = cls == 0 ? sm.cell : sm.part;
                const int cap = cls == 0 ? WK_CELL_CAP : WK_PART_CAP;
                int fill = cls == 0 ? ncb : npb;
                u32 done = 0;
                while (done < tot) {
                    if (fill == cap) {
                        __syncwarp();
                        if (cls == 0) eval_mono(buf, fill, part, P, x, eps2, as);
                        else eval_near<MODE == WALK_HYBRID>(buf, fill, part, P, x, eps2, kc0, kc1, as, ah);
                        fill = 0;
                        __syncwarp();
                    }
                    const u32 take = min((u32)(cap - fill), tot - done);
                    for (u32 e = lane; e < take; e += 32) {
                        const u32 idx = done + e;
                        int lo = 0, hi = nleaf - 1;           // largest l with lf_off[l] <= idx
                        while (lo < hi) {
                            int mid = (lo + hi + 1) >> 1;
                            if (sm.lf_off[mid] <= idx) lo = mid; else hi = mid - 1;
                        }
                        buf[fill + e] = __ldg(a.pos + sm.lf_first[lo] + (idx - sm.lf_off[lo]));
                    }
                    fill += (int)take;
                    done += take;
                }
                if (cls == 0) ncb = fill; else npb = fill;
            }
            __syncwarp();
        }
        // ---- flush what is left in the buffers
        __syncwarp();
        if (MODE != WALK_HARD && ncb > 0) eval_mono(sm.cell, ncb, part, P, x, eps2, as);
        if (MODE != WALK_NORMAL && npb > 0)
            eval_near<MODE == WALK_HYBRID>(sm.part, npb, part, P, x, eps2, kc0, kc1, as, ah);
        __syncwarp();
        if (overflow && lane == 0) atomicOr(&a.ctl->status, ST_STACK_OVERFLOW);
        // ---- combine the P partial sums (lanes aidx + q A) and store
        float v[WK_S][6];
#pragma unroll
        for (int k = 0; k < WK_S; k++) {
            v[k][0] = as[k].x; v[k][1] = as[k].y; v[k][2] = as[k].z;
            v[k][3] = ah[k].x; v[k][4] = ah[k].y; v[k][5] = ah[k].z;
        }
        for (int q = 1; q < P; q++) {
            const int src = (lane + q * A) & 31;
#pragma unroll
            for (int k = 0; k < WK_S; k++)
#pragma unroll
                for (int c = 0; c < 6; c++) {
                    if (MODE == WALK_HARD && c < 3) continue;
                    if (MODE == WALK_NORMAL && c >= 3) continue;
                    float o = __shfl_sync(0xFFFFFFFFu, v[k][c], src);
                    if (lane < A) v[k][c] += o;
                }
        }
        if (lane < A) {
#pragma unroll
            for (int k = 0; k < WK_S; k++) {
                const int si = aidx + k * A;
                if (si < n) {
                    if (MODE != WALK_HARD)
                        a.a_soft[gf + si] = make_float4(a.G * v[k][0], a.G * v[k][1], a.G * v[k][2], 0.0f);
                    if (MODE != WALK_NORMAL)
                        a.a_hard[gf + si] = make_float4(a.G * v[k][3], a.G * v[k][4], a.G * v[k][5], 0.0f);
                    else
                        a.a_hard[gf + si] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
                }
            }
        }
        if (lane == 0) {
            a.ncell[g] = ncell; a.npart[g] = npart; a.nhard[g] = nhard;
            if (MODE != WALK_HARD) atomicAdd(&a.ctl->inter_soft, (u64)n * (u64)(ncell + npart));
            if (MODE != WALK_NORMAL) atomicAdd(&a.ctl->inter_hard, (u64)n * (u64)nhard);
        }
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
    a.stacks = wsptr<u32>(c, L.stacks);
    a.G = c->p.G; a.eps2 = c->p.eps * c->p.eps; a.rout = c->p.r_out;
    const float w = c->p.r_out - c->p.r_in;
    a.kc0 = c->p.r_out / w; a.kc1 = -1.0f / w;
    const size_t smem = sizeof(WarpSmem) * WK_WARPS;
    static bool attr_set = false;
    if (!attr_set) {
        cudaFuncSetAttribute(walk_kernel<WALK_HYBRID>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        cudaFuncSetAttribute(walk_kernel<WALK_HARD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        cudaFuncSetAttribute(walk_kernel<WALK_NORMAL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        attr_set = true;
    }
    const int grid = min(c->num_sms * 2, L.n_walk_warps / WK_WARPS);
    cudaMemsetAsync(&c->ctl->group_counter, 0, sizeof(u32), c->stream);
    if (mode == WALK_HYBRID) walk_kernel<WALK_HYBRID><<<grid, WK_WARPS * 32, smem, c->stream>>>(a);
    else if (mode == WALK_HARD) walk_kernel<WALK_HARD><<<grid, WK_WARPS * 32, smem, c->stream>>>(a);
    else walk_kernel<WALK_NORMAL><<<grid, WK_WARPS * 32, smem, c->stream>>>(a);
    return cudaGetLastError();
}

}  // namespace hyb
