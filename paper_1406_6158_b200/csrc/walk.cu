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
#include "pairs.cuh"

namespace hyb {

struct WalkArgs {
    const float4 *pos;            // Morton-ordered particles (x,y,z,m)
    const NodeRec *nodes;
    const u32 *gfirst, *gcount;
    const float4 *glo, *ghi;
    u32 *ncell, *npart, *nhard;
    u32 *scost;                   // fused walk: list length per group, the estimate of the next fused walk's work order
    const u32 *heavy;             // sink ranges of split groups (split_group, common.cuh)
    u32 par;                      // which slot of DevCtl::group_counter / nheavy this launch uses
    u32 spar;                     // fused walk: which slot of DevCtl::soft_work it adds to
    const u32 *ganc;              // hard walk: start node of every group (octree.cu, group_anc)
    const unsigned char *is_split; // group is handled as ranges
    float4 *a_soft, *a_hard;
    DevCtl *ctl;
    u32 sink_lo, sink_hi;            // only groups whose first sink lies in [sink_lo, sink_hi) are evaluated
    float G, eps2, rout, kc0, kc1;   // Y = sat(kc0 + kc1 r)
    unsigned long long zero64;       // 0, passed as an argument so that it is opaque to the compiler
};

// hard walk: estimated pair count (members x hard-list length) above which a group is cut in 2 / 4 ranges
constexpr u32 DESC_MASK = 0x1FFFFFFFu;      // node index bits of a stack descriptor

// SMALL (hard walk only): the variant for runs with about one work item per resident warp (Ctx::hard_small), where
// the walk is a chain of round trips and nothing else: 128 particles per expansion step instead of 64, and 2 CTAs per SM
// with 128 registers (no spills) instead of 3 with 80.
template <int MODE, bool SMALL = false>
struct SmemLayout {                 // per warp
    static constexpr int cell_cap = MODE == WALK_HARD ? 0 : WK_CELL_CAP;
    // the hard walk has no monopole buffer, so its K-weighted buffer can be larger (fewer flushes) at 3 CTAs per SM
    static constexpr int part_cap = MODE == WALK_NORMAL ? 0 : (MODE == WALK_HARD ? (SMALL ? 384 : 256) : WK_PART_CAP);
    static constexpr int NE = SMALL ? 4 : 2;          // x 32 particles per expansion step
    static constexpr int stack_cap = MODE == WALK_HYBRID ? 320 : 512;
    static constexpr int lq_cap = 96;
    static constexpr int nqueues = MODE == WALK_HYBRID ? 3 : 2;      // far leaves, near leaves, runs of accepted children
    static constexpr int cell_alloc = cell_cap ? cell_cap + WK_PAD_SLACK : 0;
    static constexpr int part_alloc = part_cap ? part_cap + WK_PAD_SLACK : 0;
    static constexpr size_t bytes = 16 * (size_t)(cell_alloc + part_alloc) + 4 * (size_t)stack_cap + 8 * (size_t)nqueues * (size_t)lq_cap;
    // measured in round 2 (profiles/r02_profile.md): 2 x 8, 2 x 10, 3 x 7, 4 x 6 warps per SM make no difference to the hard
    // walk; the fused walk needs its 128 registers (anything that caps them lower spills and loses 20 %)
    static constexpr int ctas_per_sm = (MODE == WALK_HARD && !SMALL) ? 3 : 2;
    static constexpr int warps = WK_WARPS;      // per CTA
};

// TREE (hyb_params.hard_tree): the paper-literal hard force.  The MAC is applied in the hard walk too and a
// cell accepted within r_out of the group box is evaluated like a particle at its centre of mass with
// the K weights (hard K, soft 1 - K); the soft walk drops rule (b).  TREE = false: every node within
// r_out is opened, i.e. the hard force is the direct K-weighted sum (R20).
// CUT (hyb_params.hard_cut, R30): the hard list holds only the particles that are themselves within
// r_out of the group box; the other particles of a near leaf are plain Eq. 2 pairs (monopole buffer).
// SPLIT: the work order prepared by split_group is followed (always in the hard-only walk; in the fused walk when
// the particle number is small, Ctx::soft_split).
template <int MODE, int KF, bool TREE, bool CUT, bool SPLIT, bool SMALL>
__global__ void __launch_bounds__(SmemLayout<MODE, SMALL>::warps * 32, SmemLayout<MODE, SMALL>::ctas_per_sm) walk_kernel(const WalkArgs a)
{
    using SL = SmemLayout<MODE, SMALL>;
    constexpr bool HAS_MONO = MODE != WALK_HARD;      // monopole buffer (cells, far particles)
    constexpr bool HAS_NEAR = MODE != WALK_NORMAL;    // K-weighted buffer
    constexpr int C = MODE == WALK_HYBRID ? 6 : 3;    // accumulated components per sink
    // An opened cell that is not within r_out and is at least as far from the group box as the largest opening
    // radius of its children (NodeRec::C.w) has only accepted children: every child's centre of mass lies in the
    // cell's tight box, so its T12 distances are not smaller than the cell's box distance.  Such a cell is not
    // pushed; its children go to the monopole buffer as one run, without being tested (same lists, T13).
    constexpr bool HAS_RUNS = MODE == WALK_HYBRID;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int oct = lane >> 3, sub = lane & 7;
    unsigned char *wbase = smem_raw + (size_t)warp * SL::bytes;
    float4 *cellbuf = reinterpret_cast<float4 *>(wbase);
    float4 *partbuf = cellbuf + SL::cell_alloc;
    u32 *stack = reinterpret_cast<u32 *>(partbuf + SL::part_alloc);
    uint2 *lq0 = reinterpret_cast<uint2 *>(stack + SL::stack_cap);     // far leaves
    uint2 *lq1 = lq0 + SL::lq_cap;                                     // near leaves
    uint2 *lq2 = lq1 + SL::lq_cap;                                     // cells whose children are all accepted (HAS_RUNS)
    float *red = reinterpret_cast<float *>(wbase);                     // reduction scratch (buffers are empty then)

    const u32 lt_mask = (1u << lane) - 1u;
    const u32 ng = a.ctl->ng;
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        if (MODE == WALK_HARD) a.ctl->walk_ng = ng;                     // read by the next split_group
        else { a.ctl->soft_ng = ng; a.ctl->soft_work[a.spar ^ 1u] = 0ull; }
        a.ctl->group_counter[a.par ^ 1u] = 0u; a.ctl->nheavy[a.par ^ 1u] = 0u;      // the next launch's slots
    }
    const float rout2 = __fmul_rn(a.rout, a.rout);
    const float eps2 = a.eps2, kc0 = a.kc0, kc1 = a.kc1;
    unsigned long long isoft = 0, ihard = 0, ileaf = 0;

    // Work items come from one atomic counter.  The heaviest sink groups (by the estimate of split_group)
    // have been queued, some cut into 2 or 4 sink ranges, and are handed out first, so
    // that the longest items start early and run side by side; then the other groups in Morton order.
    // Every range walks with the box of the WHOLE group, so its lists are the group's lists (T12-T13);
    // only the sinks differ.
    const u32 nheavy = SPLIT ? a.ctl->nheavy[a.par] : 0u;
    const u32 nitems = ng + nheavy;
    u32 item = 0;
    if (lane == 0) item = atomicAdd(&a.ctl->group_counter[a.par], 1u);
    item = __shfl_sync(FULL, item, 0);

    while (item < nitems) {
        u32 item_next = 0;
        if (lane == 0) item_next = atomicAdd(&a.ctl->group_counter[a.par], 1u);      // consumed at the end of this item
        u32 g, rsub = 0, nsub = 1;
        if (SPLIT && item < nheavy) {
            const u32 it = __ldg(a.heavy + item);
            g = it & 0x0FFFFFFFu; rsub = (it >> 28) & 3u; nsub = (it >> 30) + 1u;
        } else {
            g = item - nheavy;
            if (SPLIT && a.is_split[g]) {                      // handled as ranges
                item = __shfl_sync(FULL, item_next, 0);
                continue;
            }
        }
        const u32 gf0 = a.gfirst[g];
        if (gf0 < a.sink_lo || gf0 >= a.sink_hi) {             // another replica's sinks (hyb_set_sink_range)
            item = __shfl_sync(FULL, item_next, 0);
            continue;
        }
        const u32 n_all = a.gcount[g];
        const u32 n_rng = (n_all + nsub - 1u) / nsub;                  // sinks per range
        const u32 gf = gf0 + rsub * n_rng;
        const int n = (int)(min(n_all, (rsub + 1u) * n_rng) - rsub * n_rng);
        const float4 glo = a.glo[g], ghi = a.ghi[g];
        // sinks per lane S in {2,3,4}, lanes per copy A = ceil(n / S), copies P: from the table of
        // sink_layout() (maximises the busy fraction n P / (32 S)); lane / A by a 15-bit reciprocal
        const ushort4 lay = c_layout[n];
        const int S = lay.x, A = lay.y, P = lay.z;
        const int US = WK_U;                                             // sources per evaluation iteration (monopoles)
        const int copy = (lane * (int)lay.w) >> 15;                   // = lane / A  (lane < 32, A <= 32)
        const int aidx = lane - copy * A;
        const int part = copy < P ? copy : 0x40000000;               // idle lanes never enter the loops
        const float4 dummy = make_float4(glo.x, glo.y, glo.z, 0.0f); // zero-mass padding entry
        Sinks sk;
#pragma unroll
        for (int q = 0; q < 2; q++) {
            const int s0 = aidx + 2 * q * A, s1 = s0 + A;
            const float4 p0 = __ldg(a.pos + gf + ((2 * q < S && s0 < n) ? s0 : 0));
            const float4 p1 = __ldg(a.pos + gf + ((2 * q + 1 < S && s1 < n) ? s1 : 0));
            // the 64-bit integer add of an (opaque) zero makes each pair the result of a real instruction,
            // so it lives in an aligned register pair instead of being re-packed from p0 / p1 at every use
            sk.nx[q] = pk(-p0.x, -p1.x) + a.zero64; sk.ny[q] = pk(-p0.y, -p1.y) + a.zero64;
            sk.nz[q] = pk(-p0.z, -p1.z) + a.zero64;
            sk.sx[q] = sk.sy[q] = sk.sz[q] = 0ull;
            sk.hx[q] = sk.hy[q] = sk.hz[q] = 0ull;
        }

        u32 ncell = 0, npart = 0, nhard = 0;
        int ncb = 0, npb = 0;             // buffer fills
        int nlq0 = 0, nlq1 = 0, nlq2 = 0; // leaf queue fills, cell-run queue fill
        int sp = 1;
        bool trav_done = false, flush_mono = false, flush_near = false, overflow = false;
        bool slow = false;                // something other than a plain traversal iteration is pending
        int ex_near = 0;                  // pending expansion: target buffer, this lane's leaf, progress
        u32 ex_first = 0, ex_cnt = 0, ex_off = 0, ex_T = 0, ex_done = 0;
        // the start node alone ("first child" = the node, nchild - 1 = 0): the root, or for a hard walk
        // the lowest ancestor that holds every leaf within r_out of the group box
        // (TREE: from the root -- a cell above that ancestor may be accepted by the MAC)
        if (lane == 0) stack[0] = (MODE == WALK_HARD && !TREE && a.ganc) ? __ldg(a.ganc + g) : 0u;
        __syncwarp();

        for (;;) {
            if (slow) {
                // ---- evaluation: the only call sites
                if (HAS_MONO && flush_mono) {
                    const int cnt = pad_buffer(cellbuf, ncb, P * US, dummy, lane);
                    __syncwarp();
                    if (S == 2) eval_mono<2, WK_U>(cellbuf, cnt, part, P, sk, eps2);
                    else if (S == 3) eval_mono<3, WK_U>(cellbuf, cnt, part, P, sk, eps2);
                    else eval_mono<4, WK_U>(cellbuf, cnt, part, P, sk, eps2);
                    ncb = 0; flush_mono = false;
                    __syncwarp();
                }
                if (HAS_NEAR && flush_near) {
                    const int cnt = pad_buffer(partbuf, npb, P * WK_U, dummy, lane);
                    __syncwarp();
                    if (S == 2) eval_near<2, WK_U, MODE == WALK_HYBRID, KF>(partbuf, cnt, part, P, sk, eps2, kc0, kc1);
                    else if (S == 3) eval_near<3, WK_U, MODE == WALK_HYBRID, KF>(partbuf, cnt, part, P, sk, eps2, kc0, kc1);
                    else eval_near<4, WK_U, MODE == WALK_HYBRID, KF>(partbuf, cnt, part, P, sk, eps2, kc0, kc1);
                    npb = 0; flush_near = false;
                    __syncwarp();
                }
                // ---- pending leaf expansion, 64 particles per step: the particles of the (up to 32) leaves of the batch
                //      are numbered by the prefix sum ex_off of their counts; lane l takes particles ex_done + l and
                //      ex_done + 32 + l (binary search of the leaf in the prefix sums the lanes hold), so the loads are
                //      dense whatever the leaf sizes.  CUT: a particle of a near leaf goes to the K-weighted buffer only
                //      if it is itself within r_out of the group box, else to the monopole buffer.
                if (ex_done < ex_T) {
                    const bool tonear = HAS_NEAR && (!HAS_MONO || ex_near == 1);
                    const bool cutting = CUT && tonear;
                    constexpr int NE = SL::NE;
                    if (tonear && npb + 32 * NE > SL::part_cap) { flush_near = true; continue; }
                    if (HAS_MONO && (!tonear || cutting) && ncb + 32 * NE > SL::cell_cap) { flush_mono = true; continue; }
                    float4 p[NE];
                    bool ok[NE];
#pragma unroll
                    for (int u = 0; u < NE; u++) {
                        if (NE > 2 && ex_done + 32u * u >= ex_T) { ok[u] = false; continue; }      // (uniform) nothing left for this quarter
                        const u32 slot = ex_done + 32u * u + (u32)lane;
                        ok[u] = slot < ex_T;
                        int j = 0;                      // the last leaf that starts at or before this particle
#pragma unroll
                        for (int st = 16; st; st >>= 1) {
                            const u32 t = __shfl_sync(FULL, ex_off, j + st);
                            if (t <= slot) j += st;
                        }
                        const u32 fj = __shfl_sync(FULL, ex_first, j), oj = __shfl_sync(FULL, ex_off, j);
                        if (ok[u]) p[u] = __ldg(a.pos + fj + (slot - oj));
                    }
#pragma unroll
                    for (int u = 0; u < NE; u++) {
                        if (NE > 2 && ex_done + 32u * u >= ex_T) continue;
                        if (cutting) {
                            bool nr = false;
                            if (ok[u]) {
                                const float ex = fmaxf(0.0f, fmaxf(__fsub_rn(glo.x, p[u].x), __fsub_rn(p[u].x, ghi.x)));
                                const float ey = fmaxf(0.0f, fmaxf(__fsub_rn(glo.y, p[u].y), __fsub_rn(p[u].y, ghi.y)));
                                const float ez = fmaxf(0.0f, fmaxf(__fsub_rn(glo.z, p[u].z), __fsub_rn(p[u].z, ghi.z)));
                                const float d2 = __fadd_rn(__fadd_rn(__fmul_rn(ex, ex), __fmul_rn(ey, ey)), __fmul_rn(ez, ez));
                                nr = d2 < rout2;
                            }
                            u32 bal = __ballot_sync(FULL, nr);
                            if (nr) partbuf[npb + __popc(bal & lt_mask)] = p[u];
                            npb += __popc(bal); nhard += __popc(bal);
                            if (HAS_MONO) {
                                bal = __ballot_sync(FULL, ok[u] && !nr);
                                if (ok[u] && !nr) cellbuf[ncb + __popc(bal & lt_mask)] = p[u];
                                ncb += __popc(bal);
                            }
                        } else {
                            const int cnt = (int)min(32u, ex_T - min(ex_T, ex_done + 32u * u));
                            if (tonear) { if (ok[u]) partbuf[npb + lane] = p[u]; npb += cnt; }
                            else { if (ok[u]) cellbuf[ncb + lane] = p[u]; ncb += cnt; }
                        }
                    }
                    ex_done += 32u * NE;
                    continue;
                }
                // ---- runs of accepted children: eight runs per step, lane (oct, sub) copies child sub of runs oct and
                //      oct + 4 (the centre-of-mass record only; nothing is tested)
                if (HAS_RUNS && (nlq2 >= 32 || (trav_done && nlq2 > 0))) {
                    __syncwarp();
                    while (nlq2 > 0) {
                        if (ncb + 64 > SL::cell_cap) { flush_mono = true; break; }
                        const int m = min(8, nlq2);
                        float4 p[2];
                        bool hv[2];
#pragma unroll
                        for (int h = 0; h < 2; h++) {
                            hv[h] = false;
                            const int slot = oct + 4 * h;
                            if (slot < m) {
                                const uint2 r = lq2[nlq2 - 1 - slot];
                                hv[h] = (u32)sub < r.y;
                                if (hv[h]) p[h] = __ldg(&a.nodes[r.x + (u32)sub].A);
                            }
                        }
                        nlq2 -= m;
#pragma unroll
                        for (int h = 0; h < 2; h++) {
                            const u32 bal = __ballot_sync(FULL, hv[h]);
                            if (hv[h]) cellbuf[ncb + __popc(bal & lt_mask)] = p[h];
                            ncb += __popc(bal);
                        }
                    }
                    __syncwarp();
                    if (flush_mono) continue;
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
                if (HAS_MONO && ncb > SL::cell_cap - 64) { flush_mono = true; continue; }
                if (TREE && HAS_NEAR && npb > SL::part_cap - 64) { flush_near = true; continue; }
                if (trav_done) {
                    if (HAS_MONO && ncb > 0) { flush_mono = true; continue; }
                    if (HAS_NEAR && npb > 0) { flush_near = true; continue; }
                    break;
                }
                slow = false;
            }
            // ---- traversal iteration: pop up to eight descriptors, lane (oct, sub) tests child sub of
            //      descriptors oct and oct + 4
            const int npop = min(8, sp);
            // hard walk: its first iterations below the start node pop four descriptors or fewer, and then no lane has a
            // second node to test (uniform branch; the other walks are wide almost always and keep the straight code)
            const bool wide = MODE != WALK_HARD || npop > 4;
            bool have[2];
            float4 nA[2], nB[2], nC[2];
            uint2 mt[2];
#pragma unroll
            for (int h = 0; h < 2; h++) if (h == 0 || wide) {
                have[h] = false;
                const int slot = oct + 4 * h;
                if (slot < npop) {
                    const u32 d = stack[sp - 1 - slot];
                    have[h] = (u32)sub <= (d >> 29);
                    if (have[h]) {
                        const NodeRec *r = a.nodes + ((d & DESC_MASK) + (u32)sub);
                        nB[h] = __ldg(&r->B); nC[h] = __ldg(&r->C); mt[h] = __ldg(&r->meta);
                        if (MODE != WALK_HARD || TREE) nA[h] = __ldg(&r->A);
                    }
                }
            }
            sp -= npop;
            __syncwarp();
            bool accept[2], accept_near[2], open_int[2], leaf_far[2], leaf_near[2], cell_run[2];
#pragma unroll
            for (int h = 0; h < 2; h++) if (h == 0 || wide) {
                accept[h] = accept_near[h] = open_int[h] = leaf_far[h] = leaf_near[h] = cell_run[h] = false;
                if (have[h]) {
                    // T12: box-box distance (rule (b)), fp32, one rounding per operation
                    float fx = fmaxf(0.0f, fmaxf(__fsub_rn(nB[h].x, ghi.x), __fsub_rn(glo.x, nC[h].x)));
                    float fy = fmaxf(0.0f, fmaxf(__fsub_rn(nB[h].y, ghi.y), __fsub_rn(glo.y, nC[h].y)));
                    float fz = fmaxf(0.0f, fmaxf(__fsub_rn(nB[h].z, ghi.z), __fsub_rn(glo.z, nC[h].z)));
                    float d2b = __fadd_rn(__fadd_rn(__fmul_rn(fx, fx), __fmul_rn(fy, fy)), __fmul_rn(fz, fz));
                    const bool near = d2b < rout2;
                    bool open, mac_open = true;
                    if (MODE != WALK_HARD || TREE) {
                        float ex = fmaxf(0.0f, fmaxf(__fsub_rn(glo.x, nA[h].x), __fsub_rn(nA[h].x, ghi.x)));
                        float ey = fmaxf(0.0f, fmaxf(__fsub_rn(glo.y, nA[h].y), __fsub_rn(nA[h].y, ghi.y)));
                        float ez = fmaxf(0.0f, fmaxf(__fsub_rn(glo.z, nA[h].z), __fsub_rn(nA[h].z, ghi.z)));
                        float d2a = __fadd_rn(__fadd_rn(__fmul_rn(ex, ex), __fmul_rn(ey, ey)), __fmul_rn(ez, ez));
                        mac_open = d2a < nB[h].w;
                    }
                    if (MODE == WALK_HARD) open = near && mac_open;            // (!near: discarded)
                    else open = (MODE == WALK_NORMAL || TREE) ? mac_open : (mac_open || near);
                    const bool is_leaf = (mt[h].y & 0x80000000u) != 0;
                    const bool acc = !open && (MODE != WALK_HARD || (TREE && near));
                    accept_near[h] = TREE && acc && near && MODE != WALK_NORMAL;
                    accept[h] = acc && !accept_near[h];
                    open_int[h] = open && !is_leaf;
                    if (HAS_RUNS) {        // every child will be accepted: list them as one run instead of testing them
                        cell_run[h] = open_int[h] && !near && d2b >= nC[h].w;
                        open_int[h] = open_int[h] && !cell_run[h];
                    }
                    leaf_near[h] = open && is_leaf && near && MODE != WALK_NORMAL;
                    leaf_far[h] = open && is_leaf && !leaf_near[h];
                }
            }
            // opened cells: push one descriptor each
#pragma unroll
            for (int h = 0; h < 2; h++) if (h == 0 || wide) {
                const u32 bal = __ballot_sync(FULL, open_int[h]);
                const int npush = __popc(bal);
                if (sp + npush > SL::stack_cap) { overflow = true; break; }
                if (open_int[h]) stack[sp + __popc(bal & lt_mask)] = mt[h].x | ((mt[h].y - 1u) << 29);
                sp += npush;
            }
            if (overflow) break;
            // cells with accepted children only -> queue of runs of node records (counted as cells now)
            if (HAS_RUNS) {
#pragma unroll
                for (int h = 0; h < 2; h++) if (h == 0 || wide) {
                    const u32 bal = __ballot_sync(FULL, cell_run[h]);
                    if (bal) {
                        const u32 cnt = cell_run[h] ? mt[h].y : 0u;
                        if (cell_run[h]) lq2[nlq2 + __popc(bal & lt_mask)] = make_uint2(mt[h].x, cnt);
                        nlq2 += __popc(bal);
                        ncell += __reduce_add_sync(FULL, cnt);
                    }
                }
            }
            // accepted cells -> monopole buffer
            if (HAS_MONO) {
#pragma unroll
                for (int h = 0; h < 2; h++) if (h == 0 || wide) {
                    const u32 bal = __ballot_sync(FULL, accept[h]);
                    if (accept[h]) cellbuf[ncb + __popc(bal & lt_mask)] = nA[h];
                    ncb += __popc(bal);
                    ncell += __popc(bal);
                }
            }
            // TREE: cells accepted within r_out -> K-weighted buffer (counted as cells and as hard-list entries)
            if (TREE && HAS_NEAR) {
#pragma unroll
                for (int h = 0; h < 2; h++) if (h == 0 || wide) {
                    const u32 bal = __ballot_sync(FULL, accept_near[h]);
                    if (accept_near[h]) partbuf[npb + __popc(bal & lt_mask)] = nA[h];
                    npb += __popc(bal);
                    ncell += __popc(bal); nhard += __popc(bal);
                }
            }
            // opened leaves -> queues
            if (HAS_MONO) {
#pragma unroll
                for (int h = 0; h < 2; h++) if (h == 0 || wide) {
                    const u32 bal = __ballot_sync(FULL, leaf_far[h]);
                    if (bal) {
                        const u32 cnt = leaf_far[h] ? (mt[h].y & 0x7FFFFFFFu) : 0u;
                        if (leaf_far[h]) lq0[nlq0 + __popc(bal & lt_mask)] = make_uint2(mt[h].x, cnt);
                        nlq0 += __popc(bal);
                        npart += __reduce_add_sync(FULL, cnt);
                    }
                }
            }
            if (HAS_NEAR) {
#pragma unroll
                for (int h = 0; h < 2; h++) if (h == 0 || wide) {
                    const u32 bal = __ballot_sync(FULL, leaf_near[h]);
                    if (bal) {
                        const u32 cnt = leaf_near[h] ? (mt[h].y & 0x7FFFFFFFu) : 0u;
                        if (leaf_near[h]) lq1[nlq1 + __popc(bal & lt_mask)] = make_uint2(mt[h].x, cnt);
                        nlq1 += __popc(bal);
                        const u32 tot = __reduce_add_sync(FULL, cnt);
                        npart += tot;
                        if (!CUT) nhard += tot;         // CUT: counted particle by particle at the expansion
                    }
                }
            }
            __syncwarp();
            trav_done = sp == 0;
            slow = trav_done || nlq0 >= 32 || nlq1 >= 32 || (HAS_RUNS && nlq2 >= 32) || (HAS_MONO && ncb > SL::cell_cap - 64) ||
                   (TREE && HAS_NEAR && npb > SL::part_cap - 64);
        }
        __syncwarp();
        if (overflow && lane == 0) atomicOr(&a.ctl->status, ST_STACK_OVERFLOW);

        // ---- combine the P partial sums per sink through shared memory: row r = k C + c holds
        //      component c of sink slot k for all 32 lanes; lane (aidx, part) sums rows part, part+P, ...
        float v[WK_SMAX * C];
#pragma unroll
        for (int q = 0; q < 2; q++) {
            const int k0 = 2 * q, k1 = 2 * q + 1;
            if (MODE != WALK_HARD) {
                upk(sk.sx[q], v[k0 * C + 0], v[k1 * C + 0]); upk(sk.sy[q], v[k0 * C + 1], v[k1 * C + 1]);
                upk(sk.sz[q], v[k0 * C + 2], v[k1 * C + 2]);
            }
            if (MODE == WALK_HYBRID) {
                upk(sk.hx[q], v[k0 * C + 3], v[k1 * C + 3]); upk(sk.hy[q], v[k0 * C + 4], v[k1 * C + 4]);
                upk(sk.hz[q], v[k0 * C + 5], v[k1 * C + 5]);
            }
            if (MODE == WALK_HARD) {
                upk(sk.hx[q], v[k0 * C + 0], v[k1 * C + 0]); upk(sk.hy[q], v[k0 * C + 1], v[k1 * C + 1]);
                upk(sk.hz[q], v[k0 * C + 2], v[k1 * C + 2]);
            }
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
            if (rsub == 0) {
                a.ncell[g] = ncell; a.npart[g] = npart; a.nhard[g] = nhard;
                if (MODE != WALK_HARD) a.scost[g] = ncell + npart + nhard;
            }
            if (MODE != WALK_HARD) isoft += (unsigned long long)n * (unsigned long long)(ncell + npart);
            if (MODE != WALK_NORMAL) ihard += (unsigned long long)n * (unsigned long long)nhard;
            if (MODE == WALK_HARD) ileaf += (unsigned long long)n * (unsigned long long)npart;
        }
        item = __shfl_sync(FULL, item_next, 0);
    }
    if (lane == 0) {
        if (isoft) atomicAdd(&a.ctl->inter_soft, isoft);
        if (ihard) atomicAdd(&a.ctl->inter_hard, ihard);
        if (ihard && MODE == WALK_HYBRID) atomicAdd(&a.ctl->inter_hard_fused, ihard);
        if (ileaf) atomicAdd(&a.ctl->inter_hard_leaf, ileaf);
        if (MODE != WALK_HARD && isoft + ihard) atomicAdd(&a.ctl->soft_work[a.spar], isoft + ihard);
    }
}

// Walk scheduling (split_group, common.cuh) for a walk whose tree build has not done it: a second
// force call on the same tree, a refitted tree, or a build that expected the other kind of walk.
__global__ void __launch_bounds__(256) split_kernel(const SplitArgs x, const u32 *__restrict__ gcount)
{
    const u32 ng = x.ctl->ng;
    for (u32 g = blockIdx.x * blockDim.x + threadIdx.x; g < ng; g += gridDim.x * blockDim.x)
        split_group(x, g, ng, gcount[g]);
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

template <int MODE, int KF, bool TREE, bool CUT, bool SPLIT, bool SMALL>
static cudaError_t launch_walk_mode(Ctx *c, const WalkArgs &a)
{
    using SL = SmemLayout<MODE, SMALL>;
    const size_t smem = SL::bytes * SL::warps;
    static unsigned long long ready = 0ull;
    if (!device_ready(&ready, c->device)) {
        ushort4 t[65];
        sink_layout(t);
        cudaError_t e = cudaMemcpyToSymbol(c_layout, t, sizeof t);
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(walk_kernel<MODE, KF, TREE, CUT, SPLIT, SMALL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        device_set_ready(&ready, c->device);
    }
    walk_kernel<MODE, KF, TREE, CUT, SPLIT, SMALL><<<c->num_sms * SL::ctas_per_sm, SL::warps * 32, smem, c->stream>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_walk(Ctx *c, int mode)
{
    const Layout &L = c->L;
    WalkArgs a;
    a.pos = reinterpret_cast<const float4 *>(c->pos);
    a.nodes = wsptr<NodeRec>(c, L.nodes);
    a.gfirst = wsptr<u32>(c, L.gfirst); a.gcount = wsptr<u32>(c, L.gcount);
    a.glo = wsptr<float4>(c, L.glo); a.ghi = wsptr<float4>(c, L.ghi);
    a.ncell = wsptr<u32>(c, L.ncell); a.npart = wsptr<u32>(c, L.npart); a.nhard = wsptr<u32>(c, L.nhard);
    a.a_soft = reinterpret_cast<float4 *>(c->a_soft); a.a_hard = reinterpret_cast<float4 *>(c->a_hard);
    a.ctl = c->ctl;
    a.G = c->p.G; a.eps2 = c->p.eps * c->p.eps; a.rout = c->p.r_out;
    const float w = c->p.r_out - c->p.r_in;
    a.kc0 = c->p.r_out / w; a.kc1 = -1.0f / w;
    a.zero64 = 0ull;
    a.sink_lo = c->sink_lo; a.sink_hi = c->sink_hi;
    if (c->sink_lo > 0u || (int64_t)c->sink_hi < c->n) {      // a sink range: everything outside it reads zero
        if (mode != WALK_HARD) cudaMemsetAsync(c->a_soft, 0, sizeof(hyb_float4) * (size_t)c->n, c->stream);
        cudaMemsetAsync(c->a_hard, 0, sizeof(hyb_float4) * (size_t)c->n, c->stream);
    }
    a.heavy = wsptr<u32>(c, L.splitq);
    a.ganc = c->tree_refit ? nullptr : wsptr<u32>(c, L.ganc);      // refitted boxes: the Morton cells are stale
    a.is_split = wsptr<unsigned char>(c, L.gflag);      // the build's flag array is free between builds
    a.par = c->walk_par; c->walk_par ^= 1u;      // both slots start at zero (hyb_init); each walk clears the other one
    a.scost = wsptr<u32>(c, L.scost);
    a.spar = c->soft_par;
    const int kind = mode == WALK_HARD ? 1 : 2;
    const bool sched = mode == WALK_HARD || (mode == WALK_HYBRID && c->soft_split);
    if (sched && !(c->split_ready && c->split_par == a.par && c->split_kind == kind)) {
        if (c->split_ready && c->split_par == a.par)       // the build queued the groups for the other kind of walk
            cudaMemsetAsync(&c->ctl->nheavy[a.par], 0, sizeof(u32), c->stream);
        split_kernel<<<(int)imin64((c->n + 255) / 256, (int64_t)c->num_sms * 4), 256, 0, c->stream>>>(
            SplitArgs{c->ctl, a.nhard, a.scost, wsptr<u32>(c, L.splitq), wsptr<unsigned char>(c, L.gflag), a.par, (u32)kind,
                      c->soft_par ^ 1u}, a.gcount);
        c->launches += 1;
    }
    if (mode != WALK_HARD) c->soft_par ^= 1u;
    c->split_ready = false;
    const bool poly7 = c->p.kfunc == HYB_K_POLY7, tree = c->p.hard_tree != 0, cut = c->p.hard_cut != 0;
    if (mode == WALK_NORMAL) return launch_walk_mode<WALK_NORMAL, HYB_K_PAPER, false, false, false, false>(c, a);
#define HYB_WALK_CASE(M, K, T, C, S) if (poly7 == (K == HYB_K_POLY7) && tree == T && cut == C && sched == S && small == SM) return launch_walk_mode<M, K, T, C, S, SM>(c, a)
#define HYB_WALK_CASES(M, S) \
    HYB_WALK_CASE(M, HYB_K_PAPER, false, false, S); HYB_WALK_CASE(M, HYB_K_PAPER, false, true, S); \
    HYB_WALK_CASE(M, HYB_K_PAPER, true, false, S); HYB_WALK_CASE(M, HYB_K_PAPER, true, true, S); \
    HYB_WALK_CASE(M, HYB_K_POLY7, false, false, S); HYB_WALK_CASE(M, HYB_K_POLY7, false, true, S); \
    HYB_WALK_CASE(M, HYB_K_POLY7, true, false, S); HYB_WALK_CASE(M, HYB_K_POLY7, true, true, S)
    const bool small = mode == WALK_HARD && c->hard_small;
#define SM false
    if (mode == WALK_HYBRID) { HYB_WALK_CASES(WALK_HYBRID, false); HYB_WALK_CASES(WALK_HYBRID, true); }
    HYB_WALK_CASES(WALK_HARD, true);
#undef SM
#define SM true
    HYB_WALK_CASES(WALK_HARD, true);
#undef SM
#undef HYB_WALK_CASES
#undef HYB_WALK_CASE
    return cudaErrorInvalidValue;
}

}  // namespace hyb
