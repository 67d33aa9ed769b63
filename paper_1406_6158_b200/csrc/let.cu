// let.cu -- virtual-domain LET counts (Eq. 14-15, Fig. 4).
//
// The paper's processes exchange locally essential trees: for the soft force every cell that passes
// the MAC against the receiver's domain (Eq. 14) is sent as one entry, opened leaves send particles; for
// the hard force the walk additionally drops what is farther than R_2 + b_max from the domain (Eq. 15).
// On one GPU there is nothing to exchange, but the sizes of those trees -- the paper's N_soft and N_hard
// -- can be COUNTED from the global tree for any set of virtual domains.  One warp walks the tree for one
// domain; a lane tests one node per iteration.  Decisions in fp32 with one rounding per operation (the
// sequence include/hyb.h states for hyb_let_count).
#include "common.cuh"

namespace hyb {

constexpr int LET_STACK = 6144;             // entries per warp (node | hard-walk flag << 31)
constexpr u32 LET_FULL = 0xFFFFFFFFu;

__device__ __forceinline__ float let_gap(float lo, float hi, float c)
{
    const float u = __fsub_rn(lo, c), w = __fsub_rn(c, hi);
    const float m = u > w ? u : w;
    return m > 0.0f ? m : 0.0f;
}

__global__ void __launch_bounds__(32) let_count_kernel(const NodeRec *__restrict__ nodes, const u32 *__restrict__ count,
                                                       const u64 *__restrict__ bmax2,
                                                       const float4 *__restrict__ pos, const float *__restrict__ boxes,
                                                       int ndom, float r_out, DevCtl *ctl,
                                                       unsigned long long *__restrict__ out)
{
    __shared__ u32 stack[LET_STACK];
    const int lane = threadIdx.x;
    const int j = blockIdx.x;
    if (j >= ndom) return;
    const float lox = boxes[6 * j], loy = boxes[6 * j + 1], loz = boxes[6 * j + 2];
    const float hix = boxes[6 * j + 3], hiy = boxes[6 * j + 4], hiz = boxes[6 * j + 5];
    const float R22 = __fmul_rn(r_out, r_out);
    unsigned long long nloc = 0, nsoft = 0, nhard = 0;      // per-lane partial counts
    int sp = 1;
    bool overflow = false;
    if (lane == 0) stack[0] = 0x80000000u;                   // the root, still on the hard walk
    __syncwarp();
    while (sp > 0) {
        const int m = min(32, sp);
        const bool have = lane < m;
        const u32 ent = have ? stack[sp - 1 - lane] : 0u;
        sp -= m;
        __syncwarp();
        const u32 k = ent & 0x7FFFFFFFu;
        const bool alive = (ent >> 31) != 0u;
        u32 nc = 0, ch = 0;
        bool hard_kids = false;
        if (have) {
            const float4 A = __ldg(&nodes[k].A), B = __ldg(&nodes[k].B), C = __ldg(&nodes[k].C);
            const uint2 mt = __ldg(&nodes[k].meta);
            const bool is_leaf = (mt.y & 0x80000000u) != 0u;
            const u32 cnt = is_leaf ? (mt.y & 0x7FFFFFFFu) : 0u;
            const bool inside = B.x >= lox && C.x < hix && B.y >= loy && C.y < hiy && B.z >= loz && C.z < hiz;
            const bool touches = C.x >= lox && B.x < hix && C.y >= loy && B.y < hiy && C.z >= loz && B.z < hiz;
            if (inside) nloc += __ldg(count + k);            // local: nothing to exchange
            else {
                const float ex = let_gap(lox, hix, A.x), ey = let_gap(loy, hiy, A.y), ez = let_gap(loz, hiz, A.z);
                const float r2 = __fadd_rn(__fadd_rn(__fmul_rn(ex, ex), __fmul_rn(ey, ey)), __fmul_rn(ez, ez));
                const float bm = __double2float_rn(__dsqrt_rn(__longlong_as_double((long long)__ldg(bmax2 + k))));
                const float cut = __fadd_rn(r_out, bm);
                const bool hard = alive && r2 < __fmul_rn(cut, cut);             // Eq. 15
                const bool open = r2 < B.w || touches;                           // Eq. 14
                if (!open) { nsoft += 1; nhard += hard ? 1u : 0u; }
                else if (is_leaf) {
                    for (u32 q = mt.x; q < mt.x + cnt; q++) {
                        const float4 p = __ldg(pos + q);
                        const bool in = p.x >= lox && p.x < hix && p.y >= loy && p.y < hiy && p.z >= loz && p.z < hiz;
                        if (in) { nloc += 1; continue; }
                        const float dx = let_gap(lox, hix, p.x), dy = let_gap(loy, hiy, p.y), dz = let_gap(loz, hiz, p.z);
                        const float d2 = __fadd_rn(__fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy)), __fmul_rn(dz, dz));
                        nsoft += 1;
                        if (hard && d2 < R22) nhard += 1;
                    }
                } else { nc = mt.y; ch = mt.x; hard_kids = hard; }
            }
        }
        // push the children of the opened cells
        u32 incl = nc;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const u32 t = __shfl_up_sync(LET_FULL, incl, off);
            if (lane >= off) incl += t;
        }
        const u32 total = __shfl_sync(LET_FULL, incl, 31);
        if (sp + (int)total > LET_STACK) { overflow = true; break; }
        const u32 at = (u32)sp + incl - nc;
        for (u32 i = 0; i < nc; i++) stack[at + i] = (ch + i) | (hard_kids ? 0x80000000u : 0u);
        sp += (int)total;
        __syncwarp();
    }
#pragma unroll
    for (int off = 16; off; off >>= 1) {
        nloc += __shfl_xor_sync(LET_FULL, nloc, off);
        nsoft += __shfl_xor_sync(LET_FULL, nsoft, off);
        nhard += __shfl_xor_sync(LET_FULL, nhard, off);
    }
    if (lane == 0) {
        out[3 * j] = nloc; out[3 * j + 1] = nsoft; out[3 * j + 2] = nhard;
        if (overflow) atomicOr(&ctl->status, ST_STACK_OVERFLOW);
    }
}

cudaError_t launch_let_count(Ctx *c, int ndom, const float *d_boxes, unsigned long long *d_out)
{
    const Layout &L = c->L;
    let_count_kernel<<<ndom, 32, 0, c->stream>>>(wsptr<NodeRec>(c, L.nodes), wsptr<u32>(c, L.count), wsptr<u64>(c, L.bmax2),
                                                 reinterpret_cast<const float4 *>(c->pos), d_boxes, ndom, c->p.r_out,
                                                 c->ctl, d_out);
    return cudaGetLastError();
}

}  // namespace hyb
