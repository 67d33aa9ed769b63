// api.cu -- the C-ABI of include/hyb.h: argument checks, workspace carving, step driver, export.
#include <math.h>
#include <stdio.h>
#include <stddef.h>
#include <string.h>
#include <stdlib.h>

#include <mutex>
#include <new>
#include <vector>

#include "common.cuh"

namespace hyb {

static thread_local char g_err[256] = "";

static size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

Layout plan_workspace(int64_t n)
{
    Layout L;
    memset(&L, 0, sizeof L);
    L.n = n;
    L.node_cap = node_capacity(n);
    L.group_cap = n;
    L.rs_kpt = rs_kpt_for(n);
    const int64_t rs_tile = (int64_t)RS_THREADS * L.rs_kpt;
    L.rs_tiles = (n + rs_tile - 1) / rs_tile;
    L.node_tiles = (L.node_cap + rs_tile - 1) / rs_tile;
    L.sc_tiles = (n + SC_TILE - 1) / SC_TILE;
    L.po_tiles = (n + PO_TILE - 1) / PO_TILE;
    L.rs_blocks = (L.rs_tiles + LB_WIN - 1) / LB_WIN;
    L.node_blocks = (L.node_tiles + LB_WIN - 1) / LB_WIN;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes); return o; };
    const size_t N = (size_t)n, NC = (size_t)L.node_cap, GC = (size_t)L.group_cap;
    L.key_orig = take(8 * N); L.key_a = take(8 * N); L.key_b = take(8 * N);
    L.val_a = take(4 * N); L.val_b = take(4 * N);
    L.pos_tmp = take(16 * N); L.vel_tmp = take(16 * N); L.id_tmp = take(4 * N);
    // cleared at the start of every build by ONE memset: the tail of the control block and [zero_begin, zero_end)
    L.ctl = take(sizeof(DevCtl));
    L.rs_status = take(4 * 256 * (size_t)(L.rs_tiles + L.rs_blocks) * RS_PASSES);
    L.zero_begin = L.rs_status;
    L.sc_status = take(8 * (size_t)(L.sc_tiles + L.po_tiles));
    L.node_status = take(4 * 256 * (size_t)(L.node_tiles + L.node_blocks));
    L.gflag = take(N);
    L.zero_end = off;
    L.gnode_at = take(4 * N);
    L.pre_level = take(NC); L.pre_first = take(4 * NC); L.pre_of_bfs = take(4 * NC); L.bfs_of_pre = take(4 * NC);
    L.level = take(NC); L.first = take(4 * NC); L.count = take(4 * NC); L.child = take(4 * NC);
    L.nchild = take(NC); L.parent = take(4 * NC); L.arrived = take(4 * NC);
    L.nodes = take(sizeof(NodeRec) * NC);
    L.MS64 = take(32 * NC); L.C64 = take(24 * NC); L.B2 = take(8 * NC); L.bmax2 = take(8 * NC);
    L.leaf_of = take(4 * N);
    L.gfirst = take(4 * GC); L.gcount = take(4 * GC); L.glo = take(16 * GC); L.ghi = take(16 * GC);
    L.ncell = take(4 * GC); L.npart = take(4 * GC); L.nhard = take(4 * GC);
    L.splitq = take(4 * 4 * GC);
    L.scost = take(4 * GC);
    L.gnode = take(4 * GC); L.ganc = take(4 * GC);
    // scratch of hyb_energy and hyb_let_count (partial sums; domain boxes and counts)
    L.scratch_bytes = 8 * (N / 16 + 32768);
    L.scratch = take(L.scratch_bytes);
    L.total = off;
    return L;
}

static bool params_ok(const hyb_params *p, int64_t n, char *msg)
{
    auto bad = [&](const char *m) { snprintf(msg, 256, "%s", m); return false; };
    if (!p) return bad("params is NULL");
    if (n < 1 || node_capacity(n) > (1ll << 29)) return bad("n must be in [1, 2^28 - 2048]");
    if (!(p->eps > 0.0f) || !isfinite(p->eps)) return bad("eps must be finite and > 0");
    if (!isfinite(p->G)) return bad("G must be finite");
    if (p->n_sub < 1) return bad("n_sub must be >= 1");
    if (!isfinite(p->dt_soft)) return bad("dt_soft must be finite");
    if (p->leaf_max < 1 || p->group_max < p->leaf_max || p->group_max > 64) return bad("need 1 <= leaf_max <= group_max <= 64");
    if (p->mac != HYB_MAC_THETA && p->mac != HYB_MAC_ABS) return bad("unknown mac");
    if (p->mac == HYB_MAC_THETA && !(p->theta >= 0.0f && isfinite(p->theta))) return bad("theta must be finite and >= 0");
    if (p->mac == HYB_MAC_ABS && !(p->a_err > 0.0f && isfinite(p->a_err))) return bad("a_err must be finite and > 0");
    if (p->kfunc != HYB_K_PAPER && p->kfunc != HYB_K_POLY7) return bad("unknown kfunc");
    if (p->split != 0 && p->split != 1) return bad("split must be 0 or 1");
    if (p->hard_tree != 0 && p->hard_tree != 1) return bad("hard_tree must be 0 or 1");
    if (p->hard_refit != 0 && p->hard_refit != 1) return bad("hard_refit must be 0 or 1");
    if (p->hard_cut != 0 && p->hard_cut != 1) return bad("hard_cut must be 0 or 1");
    if (p->hard_refit == 1 && (p->split != 1 || p->hard_tree != 0)) return bad("hard_refit needs split = 1 and hard_tree = 0");
    if (p->grouping != HYB_GROUP_NODE && p->grouping != HYB_GROUP_SIBLINGS && p->grouping != HYB_GROUP_AUTO) return bad("unknown grouping");
    if (p->split == 1 && !(p->r_in >= 0.0f && p->r_out > p->r_in && isfinite(p->r_out))) return bad("need 0 <= r_in < r_out");
    return true;
}

static int fail(Ctx *c, int code, const char *msg)
{
    snprintf(g_err, sizeof g_err, "%s", msg);
    if (c) snprintf(c->err, sizeof c->err, "%s", msg);
    return code;
}
static int cuda_fail(Ctx *c, cudaError_t e, const char *where)
{
    char m[256];
    snprintf(m, sizeof m, "%s: %s", where, cudaGetErrorString(e));
    return fail(c, HYB_ERR_CUDA, m);
}

static int status_to_error(Ctx *c, u32 st)
{
    if (st & ST_NONFINITE) return fail(c, HYB_ERR_NONFINITE_INPUT, "non-finite position/mass or negative mass");
    if (st & ST_NODE_OVERFLOW) return fail(c, HYB_ERR_CAPACITY_OVERFLOW, "tree node pool overflow");
    if (st & ST_STACK_OVERFLOW) return fail(c, HYB_ERR_CAPACITY_OVERFLOW, "traversal stack overflow");
    if (st & ST_WAIT_EXPIRED) return fail(c, HYB_ERR_INTERNAL, "device-side look-back wait expired");
    return HYB_OK;
}

// a box reduced by a drift that no build consumed (a step that failed in between): drop it, the positions
// are the caller's and may have changed
static void discard_pending_bbox(Ctx *c)
{
    if (!c->bbox_ready) return;
    cudaMemsetAsync(&c->ctl->bbox_enc[0], 0, 7 * sizeof(u32), c->stream);      // bbox_enc[6], bbox_done
    c->bbox_ready = false;
}

static int do_build(Ctx *c, bool hard_only = false)
{
    const bool had_bbox = c->bbox_ready;
    // HYB_GROUP_AUTO: runs of sibling cells, of up to group_max sinks for the soft walk and up to
    // group_max / 2 when only a hard walk follows
    c->grouping_now = c->p.grouping == HYB_GROUP_AUTO ? HYB_GROUP_SIBLINGS : c->p.grouping;
    c->group_max_now = c->p.group_max;
    if (hard_only && c->p.grouping == HYB_GROUP_AUTO)                 // smaller runs: fewer listed particles beyond r_out
        c->group_max_now = c->p.group_max / 2 > c->p.leaf_max ? c->p.group_max / 2 : c->p.leaf_max;      // (cfg2: 16 / 24 / 40 / 48 / 64 are 4-25 % slower than 32)
    c->boxes_only = hard_only && !c->p.hard_tree;      // the tree-approximated hard walk needs the moments
    c->next_kind = hard_only ? 1 : 2;                  // whose work order ginfo_kernel prepares
    cudaError_t e = launch_build_tree(c);
    if (e != cudaSuccess) return cuda_fail(c, e, "build_tree");
    c->tree_valid = true;
    c->tree_refit = false;
    c->acc_valid = false;
    // bbox (+ root cube), keys (+ digit bases), 8 sort passes, permute | preorder (+ level offsets), level sort,
    // link, upsweep, group mark / scan / info (+ b_max, r_b in absolute-MAC mode)
    c->launches += 11 + 7 + (c->p.mac == HYB_MAC_ABS && !hard_only ? 3 : 0) - (had_bbox ? 1 : 0);
    return HYB_OK;
}

// hard-only substep with hard_refit: boxes of the existing topology for the drifted positions; the first
// one of a cycle also forms the (smaller) sink groups of the hard walks
static int do_refit(Ctx *c, bool regroup)
{
    cudaError_t e = cudaSuccess;
    if (regroup) {
        c->grouping_now = c->p.grouping == HYB_GROUP_AUTO ? HYB_GROUP_SIBLINGS : c->p.grouping;
        c->group_max_now = c->p.group_max;
        if (c->p.grouping == HYB_GROUP_AUTO)
            c->group_max_now = c->p.group_max / 2 > c->p.leaf_max ? c->p.group_max / 2 : c->p.leaf_max;
        e = launch_regroup(c);
        c->launches += 3;
    }
    if (e == cudaSuccess) e = launch_refit_tree(c);
    if (e != cudaSuccess) return cuda_fail(c, e, "refit_tree");
    c->launches += 2;
    c->tree_refit = true;
    c->acc_valid = false;
    return HYB_OK;
}

static int do_soft(Ctx *c)
{
    cudaError_t e = launch_walk(c, c->p.split ? WALK_HYBRID : WALK_NORMAL);
    if (e != cudaSuccess) return cuda_fail(c, e, "soft walk");
    c->launches += 1;
    return HYB_OK;
}

static int do_hard(Ctx *c)
{
    cudaError_t e = c->p.split ? launch_walk(c, WALK_HARD) : launch_zero_acc(c, c->a_hard);
    if (e != cudaSuccess) return cuda_fail(c, e, "hard walk");
    c->launches += 1;                           // the walk (launch_walk counts a split_kernel), or the zero fill
    return HYB_OK;
}

}  // namespace hyb

using namespace hyb;

// device buffer, stream and context kept between hyb_run_host calls
static struct { char *ptr; size_t bytes; int device; cudaStream_t st, st2; hyb_ctx *ctx; hyb_params p; int64_t n; } g_host =
    {nullptr, 0, -1, nullptr, nullptr, nullptr, {}, 0};
struct EarlyCopy { hyb_float4 *h_pos; uint32_t *h_id; size_t n; cudaStream_t st2; bool done; };
// the store is final once the last build's re-order has been copied back (ev_groups follows it on the auxiliary stream)
static void early_copy(Ctx *c, void *arg)
{
    EarlyCopy *x = static_cast<EarlyCopy *>(arg);
    cudaStreamWaitEvent(x->st2, c->ev_groups, 0);
    cudaMemcpyAsync(x->h_pos, c->pos, 16 * x->n, cudaMemcpyDeviceToHost, x->st2);      // (wherever the store is right now)
    cudaMemcpyAsync(x->h_id, c->id, 4 * x->n, cudaMemcpyDeviceToHost, x->st2);
    x->done = true;
}
static std::mutex g_host_mutex;
static void release_host_cache()
{
    if (g_host.ptr) {
        cudaSetDevice(g_host.device);
        if (g_host.st) cudaStreamSynchronize(g_host.st);
        if (g_host.st2) cudaStreamSynchronize(g_host.st2);
        if (g_host.ctx) hyb_free(g_host.ctx);
        if (g_host.st) cudaStreamDestroy(g_host.st);
        if (g_host.st2) cudaStreamDestroy(g_host.st2);
        cudaFree(g_host.ptr);
    }
    g_host.ptr = nullptr; g_host.bytes = 0; g_host.device = -1; g_host.st = nullptr; g_host.st2 = nullptr; g_host.ctx = nullptr; g_host.n = 0;
}

extern "C" {

size_t hyb_workspace_bytes(int64_t n, const hyb_params *params)
{
    char msg[256];
    if (!params_ok(params, n, msg)) return 0;
    return plan_workspace(n).total;
}

int hyb_init(hyb_ctx **out, const hyb_params *params, int64_t n, hyb_float4 *d_pos_m, hyb_float4 *d_vel,
             hyb_float4 *d_a_soft, hyb_float4 *d_a_hard, uint32_t *d_id, void *d_workspace, size_t workspace_bytes,
             int device, void *cuda_stream)
{
    char msg[256];
    if (!out) return fail(nullptr, HYB_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (!params_ok(params, n, msg)) return fail(nullptr, HYB_ERR_INVALID_ARG, msg);
    if (!d_pos_m || !d_vel || !d_a_soft || !d_a_hard || !d_id || !d_workspace)
        return fail(nullptr, HYB_ERR_INVALID_ARG, "a device pointer is NULL");
    if (((uintptr_t)d_workspace & 255) || ((uintptr_t)d_pos_m & 15) || ((uintptr_t)d_vel & 15) ||
        ((uintptr_t)d_a_soft & 15) || ((uintptr_t)d_a_hard & 15))
        return fail(nullptr, HYB_ERR_INVALID_ARG, "misaligned device pointer");
    Layout L = plan_workspace(n);
    if (workspace_bytes < L.total) return fail(nullptr, HYB_ERR_WORKSPACE_TOO_SMALL, "workspace too small");
    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaSetDevice");
    Ctx *c = new (std::nothrow) Ctx;
    if (!c) return fail(nullptr, HYB_ERR_INTERNAL, "out of host memory");
    memset(c, 0, sizeof *c);
    c->sink_lo = 0u; c->sink_hi = (u32)n;
    c->p = *params; c->n = n; c->device = device; c->stream = (cudaStream_t)cuda_stream;
    c->pos = d_pos_m; c->vel = d_vel; c->a_soft = d_a_soft; c->a_hard = d_a_hard; c->id = d_id;
    c->pos_home = d_pos_m; c->vel_home = d_vel; c->id_home = d_id;
    c->ws = (char *)d_workspace; c->L = L; c->ctl = (DevCtl *)(c->ws + L.ctl);
    e = cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, device);
    if (e != cudaSuccess) { const int rc = cuda_fail(nullptr, e, "cudaDeviceGetAttribute"); hyb_free(reinterpret_cast<hyb_ctx *>(c)); return rc; }
    for (int i = 0; i < 5; i++) {
        e = cudaEventCreate(&c->ev[i]);
        if (e != cudaSuccess) { const int rc = cuda_fail(nullptr, e, "cudaEventCreate"); hyb_free(reinterpret_cast<hyb_ctx *>(c)); return rc; }
    }
    e = cudaStreamCreateWithFlags(&c->aux, cudaStreamNonBlocking);
    if (e != cudaSuccess) { const int rc = cuda_fail(nullptr, e, "cudaStreamCreate"); hyb_free(reinterpret_cast<hyb_ctx *>(c)); return rc; }
    cudaEvent_t *evs[4] = {&c->ev_sorted, &c->ev_perm, &c->ev_linked, &c->ev_groups};
    for (int i = 0; i < 4; i++) {
        e = cudaEventCreateWithFlags(evs[i], cudaEventDisableTiming);
        if (e != cudaSuccess) { const int rc = cuda_fail(nullptr, e, "cudaEventCreate"); hyb_free(reinterpret_cast<hyb_ctx *>(c)); return rc; }
    }
    c->timing = true;
    // with fewer than a few sink groups per resident warp the longest groups set the duration of the fused walk: it
    // then follows the work order of split_group (measured: cfg1 soft walk 0.60 -> 0.45 ms; from 2^20 particles up the
    // Morton order is 1-2 % faster, its neighbours share cache lines)
    c->soft_split = params->split && n < (int64_t)SMALL_RUN_PER_WARP * c->num_sms * 2 * WK_WARPS;
    // (cfg1: 7 hard walks 0.29 -> 0.24 ms, cfg0 0.094 -> 0.077; at N = 2^20 the same variant is 6 % slower for the direct
    // hard sum, but 3-6 % faster for the tree-approximated hard walk, whose 80-register instantiation spills)
    c->hard_small = c->soft_split || params->hard_tree != 0;
    e = cudaMemsetAsync(c->ctl, 0, sizeof(DevCtl), c->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(c->ws + L.nhard, 0, 4 * (size_t)L.group_cap, c->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(c->ws + L.scost, 0, 4 * (size_t)L.group_cap, c->stream);
    {
        // walk scheduling (split_group).  Hard walk: estimated pairs above which a group is queued in front / cut in 2 /
        // cut in 4.  Fused walk: the same three in 1/64 of the ideal makespan (all pairs / resident warps).
        // (cfg1, soft walk: 0.60 ms in Morton order; 0.44-0.46 ms with 0-24 / 48 / 96; 0.50-0.52 with x / 64 / 128 or x / 32 / 64)
        const u32 t[8] = {8192u, 24576u, 65536u, (u32)imin64(4 * L.group_cap, 0xFFFFFFFFll), 16u, 48u, 96u, (u32)c->num_sms * 2u * (u32)WK_WARPS};
        static_assert(offsetof(DevCtl, soft_slots) - offsetof(DevCtl, split_t) == 7 * sizeof(u32), "split_t .. soft_slots are contiguous");
        if (e == cudaSuccess) e = cudaMemcpyAsync(&c->ctl->split_t[0], t, sizeof t, cudaMemcpyHostToDevice, c->stream);
    }
    if (e != cudaSuccess) { const int rc = cuda_fail(nullptr, e, "cudaMemsetAsync"); hyb_free(reinterpret_cast<hyb_ctx *>(c)); return rc; }
    *out = reinterpret_cast<hyb_ctx *>(c);
    return HYB_OK;
}

int hyb_set_params(hyb_ctx *ctx, const hyb_params *params)
{
    Ctx *c = reinterpret_cast<Ctx *>(ctx);
    char msg[256];
    if (!c) return fail(nullptr, HYB_ERR_INVALID_ARG, "ctx is NULL");
    if (!params_ok(params, c->n, msg)) return fail(c, HYB_ERR_INVALID_ARG, msg);
    if (params->leaf_max != c->p.leaf_max || params->group_max != c->p.group_max || params->grouping != c->p.grouping)
        return fail(c, HYB_ERR_INVALID_ARG, "leaf_max / group_max / grouping cannot change after hyb_init");
    c->p = *params;
    c->soft_split = params->split && c->n < (int64_t)SMALL_RUN_PER_WARP * c->num_sms * 2 * WK_WARPS;
    c->hard_small = c->soft_split || params->hard_tree != 0;
    c->split_ready = false;
    c->tree_valid = false; c->acc_valid = false;
    return HYB_OK;
}

int hyb_build_tree(hyb_ctx *ctx)
{
    Ctx *c = reinterpret_cast<Ctx *>(ctx);
    if (!c) return fail(nullptr, HYB_ERR_INVALID_ARG, "ctx is NULL");
    cudaSetDevice(c->device);
    discard_pending_bbox(c);
    return do_build(c);
}

int hyb_build_tree_hard(hyb_ctx *ctx)
{
    Ctx *c = reinterpret_cast<Ctx *>(ctx);
    if (!c) return fail(nullptr, HYB_ERR_INVALID_ARG, "ctx is NULL");
    if (c->p.split != 1) return fail(c, HYB_ERR_INVALID_ARG, "a hard-step tree needs split = 1");
    cudaSetDevice(c->device);
    discard_pending_bbox(c);
    return do_build(c, true);
}

int hyb_refit_tree(hyb_ctx *ctx)
{
    Ctx *c = reinterpret_cast<Ctx *>(ctx);
    if (!c) return fail(nullptr, HYB_ERR_INVALID_ARG, "ctx is NULL");
    if (!c->tree_valid) return fail(c, HYB_ERR_NO_TREE, "nothing to refit: call hyb_build_tree first");
    if (c->p.split != 1 || c->p.hard_tree != 0) return fail(c, HYB_ERR_INVALID_ARG, "a refitted tree serves the direct hard force only (split = 1, hard_tree = 0)");
    cudaSetDevice(c->device);
    return do_refit(c, false);
}

int hyb_soft_force(hyb_ctx *ctx)
{
    Ctx *c = reinterpret_cast<Ctx *>(ctx);
    if (!c) return fail(nullptr, HYB_ERR_INVALID_ARG, "ctx is NULL");
    if (!c->tree_valid || c->tree_refit || c->boxes_only)
        return fail(c, HYB_ERR_NO_TREE, "no tree with moments for the current positions");
    cudaSetDevice(c->device);
    int rc = do_soft(c);
    if (rc == HYB_OK) c->acc_valid = true;
    return rc;
}

int hyb_hard_force(hyb_ctx *ctx)
{
    Ctx *c = reinterpret_cast<Ctx *>(ctx);
    if (!c) return fail(nullptr, HYB_ERR_INVALID_ARG, "ctx is NULL");
    if (!c->tree_valid) return fail(c, HYB_ERR_NO_TREE, "no tree for the current positions");
    cudaSetDevice(c->device);
    return do_hard(c);
}

int hyb_set_sink_range(hyb_ctx *ctx, int64_t first, int64_t last)
{
    Ctx *c = reinterpret_cast<Ctx *>(ctx);
    if (!c) return fail(nullptr, HYB_ERR_INVALID_ARG, "ctx is NULL");
    if (first < 0 || last < first || last > c->n) return fail(c, HYB_ERR_INVALID_ARG, "need 0 <= first <= last <= n");
    c->sink_lo = (u32)first; c->sink_hi = (u32)last;
    c->acc_valid = false;
    return HYB_OK;
}

int hyb_kick_drift(hyb_ctx *ctx, float c_soft, float c_hard, float dt)
{
    Ctx *c = reinterpret_cast<Ctx *>(ctx);
    if (!c) return fail(nullptr, HYB_ERR_INVALID_ARG, "ctx is NULL");
    if (!isfinite(c_soft) || !isfinite(c_hard) || !isfinite(dt)) return fail(c, HYB_ERR_INVALID_ARG, "non-finite coefficient");
    cudaSetDevice(c->device);
    discard_pending_bbox(c);
    cudaError_t e = launch_kick_drift(c, c_soft, c_hard, dt, false);
    if (e != cudaSuccess) return cuda_fail(c, e, "kick_drift");
    c->launches += 1;
    if (dt != 0.0f) { c->tree_valid = false; c->acc_valid = false; }
    return HYB_OK;
}

int hyb_sync(hyb_ctx *ctx)
{
    Ctx *c = reinterpret_cast<Ctx *>(ctx);
    if (!c) return fail(nullptr, HYB_ERR_INVALID_ARG, "ctx is NULL");
    cudaSetDevice(c->device);
    u32 st = 0;
    cudaError_t e = cudaMemcpyAsync(&st, &c->ctl->status, sizeof st, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e, "hyb_sync");
    if (st) {       // reported once: the word is cleared, what was computed from the bad state is dropped
        cudaMemsetAsync(&c->ctl->status, 0, sizeof(u32), c->stream);
        c->tree_valid = false; c->acc_valid = false; c->bbox_ready = false;
        cudaMemsetAsync(&c->ctl->bbox_enc[0], 0, 7 * sizeof(u32), c->stream);
    }
    return status_to_error(c, st);
}

int hyb_step(hyb_ctx *ctx, int32_t n_soft_steps)
{
    Ctx *c = reinterpret_cast<Ctx *>(ctx);
    if (!c) return fail(nullptr, HYB_ERR_INVALID_ARG, "ctx is NULL");
    if (n_soft_steps < 0) return fail(c, HYB_ERR_INVALID_ARG, "n_soft_steps < 0");
    if (c->sink_lo != 0u || (int64_t)c->sink_hi != c->n)
        return fail(c, HYB_ERR_INVALID_ARG, "hyb_step needs the full sink range: with hyb_set_sink_range the caller exchanges the accelerations between the force calls and the kicks");
    cudaSetDevice(c->device);
    const bool split = c->p.split != 0;
    const int nsub = c->p.n_sub;
    const float dts = c->p.dt_soft, dth = dts / (float)nsub;
    int rc;
    discard_pending_bbox(c);
    if (!c->acc_valid || (c->p.hard_refit && (!c->tree_valid || c->tree_refit))) {
        if ((rc = do_build(c)) != HYB_OK) return rc;
        if ((rc = do_soft(c)) != HYB_OK) return rc;
        c->acc_valid = true;
    }
    struct Seg { int kind; cudaEvent_t a, b; };     // kind: 0 build, 1 soft, 2 hard, 3 integrate
    std::vector<Seg> segs;
    // stage timers: events come from a pool the context keeps (it grows to the longest call and is destroyed by hyb_free)
    if (c->timing) {
        const size_t need = 5 * (size_t)nsub * (size_t)n_soft_steps;
        if (need > c->evpool_n) {
            cudaEvent_t *np = (cudaEvent_t *)realloc(c->evpool, need * sizeof(cudaEvent_t));
            if (!np) return fail(c, HYB_ERR_INTERNAL, "out of host memory");
            c->evpool = np;
            for (; c->evpool_n < need; c->evpool_n++)
                if (cudaEventCreate(&c->evpool[c->evpool_n]) != cudaSuccess) return cuda_fail(c, cudaGetLastError(), "cudaEventCreate");
        }
    }
    size_t ev_used = 0;
    auto ev = [&]() { cudaEvent_t e = c->evpool[ev_used++]; cudaEventRecord(e, c->stream); return e; };
    auto bail = [&](int code) {
        c->defer_copy = false; store_come_home(c);
        c->tree_valid = false; c->acc_valid = false; return code;
    };
    c->defer_copy = true;      // builds leave the store where they re-ordered it to; it is home again when the call returns
    for (int32_t cyc = 0; cyc < n_soft_steps; cyc++) {
        for (int k = 0; k < nsub; k++) {
            cudaEvent_t e0 = c->timing ? ev() : nullptr;
            cudaError_t e;
            // opening kick(s) + drift.  split = 0: the whole force lives in a_soft and is kicked at dt_h.
            // Inside a cycle the closing half kick of one substep and the opening half kick of the next
            // use the same acceleration, so they are one full kick fused with the drift (k > 0).
            const float open_c = k == 0 ? 0.5f * dth : dth;
            const bool soft_step = !split || k == nsub - 1;
            const bool rebuild = soft_step || !c->p.hard_refit;      // a full build follows: the drift reduces its bounding box
            if (split) e = launch_kick_drift(c, k == 0 ? 0.5f * dts : 0.0f, open_c, dth, rebuild);
            else e = launch_kick_drift(c, open_c, 0.0f, dth, rebuild);
            if (e != cudaSuccess) return bail(cuda_fail(c, e, "kick_drift"));
            cudaEvent_t e1 = c->timing ? ev() : nullptr;
            if (!soft_step && c->p.hard_refit) rc = do_refit(c, k == 0 && c->p.grouping == HYB_GROUP_AUTO);
            else rc = do_build(c, !soft_step);
            if (rc != HYB_OK) return bail(rc);
            if (c->store_final && cyc == n_soft_steps - 1 && k == nsub - 1) c->store_final(c, c->store_final_arg);
            cudaEvent_t e2 = c->timing ? ev() : nullptr;
            if (soft_step) rc = do_soft(c); else rc = do_hard(c);
            if (rc != HYB_OK) return bail(rc);
            cudaEvent_t e3 = c->timing ? ev() : nullptr;
            const bool last = k == nsub - 1;           // the closing half kick of the other substeps is fused above
            if (last) {
                if (split) e = launch_kick_drift(c, 0.5f * dts, 0.5f * dth, 0.0f);
                else e = launch_kick_drift(c, 0.5f * dth, 0.0f, 0.0f);
                if (e != cudaSuccess) return bail(cuda_fail(c, e, "kick"));
            }
            c->launches += last ? 2 : 1;
            if (c->timing) {
                cudaEvent_t e4 = ev();
                segs.push_back({3, e0, e1}); segs.push_back({0, e1, e2});
                segs.push_back({soft_step ? 1 : 2, e2, e3}); segs.push_back({3, e3, e4});
            }
        }
        c->acc_valid = true;
    }
    c->defer_copy = false;
    {
        const cudaError_t e = store_come_home(c);
        if (e != cudaSuccess) return bail(cuda_fail(c, e, "store copy"));
    }
    rc = hyb_sync(ctx);
    if (rc == HYB_OK)
        for (auto &s : segs) { float ms = 0; cudaEventElapsedTime(&ms, s.a, s.b); c->t_acc[s.kind] += ms; }
    c->t_acc[7] += (float)n_soft_steps;
    return rc;
}

int hyb_export(hyb_ctx *ctx, int32_t what, void *host_dst, size_t bytes, size_t *written)
{
    Ctx *c = reinterpret_cast<Ctx *>(ctx);
    if (!c) return fail(nullptr, HYB_ERR_INVALID_ARG, "ctx is NULL");
    if (!host_dst) return fail(c, HYB_ERR_INVALID_ARG, "host_dst is NULL");
    cudaSetDevice(c->device);
    cudaError_t e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e, "hyb_export sync");
    DevCtl h;
    e = cudaMemcpy(&h, c->ctl, sizeof h, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return cuda_fail(c, e, "hyb_export ctl");
    const Layout &L = c->L;
    const size_t n = (size_t)c->n, nn = h.nn, ng = h.ng;
    const void *src = nullptr; size_t sz = 0;
    std::vector<char> tmp;
    switch (what) {
    case HYB_X_COUNTS: {
        int64_t v[8] = {(int64_t)n, (int64_t)nn, (int64_t)ng, L.node_cap, (int64_t)h.status, (int64_t)h.nn_total, (int64_t)c->launches,
                        (int64_t)h.nheavy[c->walk_par ^ 1u]};
        if (bytes < sizeof v) return fail(c, HYB_ERR_INVALID_ARG, "buffer too small");
        memcpy(host_dst, v, sizeof v); if (written) *written = sizeof v; return HYB_OK; }
    case HYB_X_LEVEL_OFFSET:
        if (bytes < sizeof h.level_offset) return fail(c, HYB_ERR_INVALID_ARG, "buffer too small");
        memcpy(host_dst, h.level_offset, sizeof h.level_offset); if (written) *written = sizeof h.level_offset; return HYB_OK;
    case HYB_X_BBOX:
        if (bytes < sizeof h.bbox) return fail(c, HYB_ERR_INVALID_ARG, "buffer too small");
        memcpy(host_dst, h.bbox, sizeof h.bbox); if (written) *written = sizeof h.bbox; return HYB_OK;
    case HYB_X_INTERACTIONS: {
        u64 v[4] = {h.inter_soft, h.inter_hard, h.inter_hard_fused, h.inter_hard_leaf};
        if (bytes < sizeof v) return fail(c, HYB_ERR_INVALID_ARG, "buffer too small");
        memcpy(host_dst, v, sizeof v); if (written) *written = sizeof v;
        cudaMemset(&c->ctl->inter_soft, 0, 4 * sizeof(u64));
        return HYB_OK; }
    case HYB_X_TIMINGS:
        if (bytes < sizeof c->t_acc) return fail(c, HYB_ERR_INVALID_ARG, "buffer too small");
        memcpy(host_dst, c->t_acc, sizeof c->t_acc); if (written) *written = sizeof c->t_acc;
        memset(c->t_acc, 0, sizeof c->t_acc);
        return HYB_OK;
    case HYB_X_KEYS_SORTED: src = c->ws + L.key_b; sz = 8 * n; break;
    case HYB_X_KEYS: src = c->ws + L.key_orig; sz = 8 * n; break;
    case HYB_X_PERM: src = c->ws + L.val_b; sz = 4 * n; break;
    case HYB_X_LEVEL: src = c->ws + L.level; sz = nn; break;
    case HYB_X_FIRST: src = c->ws + L.first; sz = 4 * nn; break;
    case HYB_X_COUNT: src = c->ws + L.count; sz = 4 * nn; break;
    case HYB_X_CHILD: src = c->ws + L.child; sz = 4 * nn; break;
    case HYB_X_NCHILD: src = c->ws + L.nchild; sz = nn; break;
    case HYB_X_PARENT: src = c->ws + L.parent; sz = 4 * nn; break;
    case HYB_X_COM_M: case HYB_X_NLO: case HYB_X_NHI: case HYB_X_ROPEN2: {      // strided fields of NodeRec
        const size_t off = what == HYB_X_COM_M ? offsetof(NodeRec, A) : what == HYB_X_NHI ? offsetof(NodeRec, C)
                           : what == HYB_X_NLO ? offsetof(NodeRec, B) : offsetof(NodeRec, B) + 12;
        const size_t w = what == HYB_X_ROPEN2 ? 4 : 16;
        if (bytes < w * nn) return fail(c, HYB_ERR_INVALID_ARG, "buffer too small");
        if (nn) {
            e = cudaMemcpy2D(host_dst, w, c->ws + L.nodes + off, sizeof(NodeRec), w, nn, cudaMemcpyDeviceToHost);
            if (e != cudaSuccess) return cuda_fail(c, e, "hyb_export copy");
        }
        if (written) *written = w * nn;
        return HYB_OK; }
    case HYB_X_GFIRST: src = c->ws + L.gfirst; sz = 4 * ng; break;
    case HYB_X_GCOUNT: src = c->ws + L.gcount; sz = 4 * ng; break;
    case HYB_X_GLO: src = c->ws + L.glo; sz = 16 * ng; break;
    case HYB_X_GHI: src = c->ws + L.ghi; sz = 16 * ng; break;
    case HYB_X_NCELL: src = c->ws + L.ncell; sz = 4 * ng; break;
    case HYB_X_NPART: src = c->ws + L.npart; sz = 4 * ng; break;
    case HYB_X_NHARD: src = c->ws + L.nhard; sz = 4 * ng; break;
    case HYB_X_M64:                                                            // strided field of (M, Sx, Sy, Sz)
        if (bytes < 8 * nn) return fail(c, HYB_ERR_INVALID_ARG, "buffer too small");
        if (nn) {
            e = cudaMemcpy2D(host_dst, 8, c->ws + L.MS64, 32, 8, nn, cudaMemcpyDeviceToHost);
            if (e != cudaSuccess) return cuda_fail(c, e, "hyb_export copy");
        }
        if (written) *written = 8 * nn;
        return HYB_OK;
    case HYB_X_C64: src = c->ws + L.C64; sz = 24 * nn; break;
    case HYB_X_B2: src = c->ws + L.B2; sz = 8 * nn; break;
    case HYB_X_BMAX: {
        if (bytes < 8 * nn) return fail(c, HYB_ERR_INVALID_ARG, "buffer too small");
        e = cudaMemcpy(host_dst, c->ws + L.bmax2, 8 * nn, cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) return cuda_fail(c, e, "hyb_export copy");
        for (size_t i = 0; i < nn; i++) ((double *)host_dst)[i] = sqrt(((double *)host_dst)[i]);
        if (written) *written = 8 * nn;
        return HYB_OK; }
    default: return fail(c, HYB_ERR_INVALID_ARG, "unknown export selector");
    }
    if (bytes < sz) return fail(c, HYB_ERR_INVALID_ARG, "buffer too small");
    if (sz) {
        e = cudaMemcpy(host_dst, src, sz, cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) return cuda_fail(c, e, "hyb_export copy");
    }
    if (written) *written = sz;
    return HYB_OK;
}

int hyb_run_host(const hyb_params *params, int64_t n, hyb_float4 *h_pos_m, hyb_float4 *h_vel, hyb_float4 *h_a_soft,
                 hyb_float4 *h_a_hard, uint32_t *h_id, int32_t n_soft_steps, int32_t acc_valid, int device,
                 uint64_t *h_interactions)
{
    char msg[256];
    if (!params_ok(params, n, msg)) return fail(nullptr, HYB_ERR_INVALID_ARG, msg);
    if (!h_pos_m || !h_vel || !h_a_soft || !h_a_hard || !h_id) return fail(nullptr, HYB_ERR_INVALID_ARG, "a host pointer is NULL");
    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaSetDevice");
    const size_t ws_bytes = plan_workspace(n).total, N = (size_t)n;
    const size_t o_pos = 0, o_vel = 16 * N, o_as = 32 * N, o_ah = 48 * N, o_id = 64 * N;
    const size_t o_ws = (68 * N + 255) & ~(size_t)255;
    // the device buffer and the stream are kept for the next call (hyb_run_host_release frees them):
    // cudaMalloc / cudaFree of half a gigabyte cost more than the copies of a million particles
    std::lock_guard<std::mutex> lock(g_host_mutex);
    if (g_host.ptr && (g_host.device != device || g_host.bytes < o_ws + ws_bytes)) release_host_cache();
    if (!g_host.ptr) {
        e = cudaMalloc(&g_host.ptr, o_ws + ws_bytes);
        if (e != cudaSuccess) { g_host.ptr = nullptr; return cuda_fail(nullptr, e, "cudaMalloc"); }
        g_host.bytes = o_ws + ws_bytes; g_host.device = device;
        if ((e = cudaStreamCreate(&g_host.st)) != cudaSuccess) { release_host_cache(); return cuda_fail(nullptr, e, "cudaStreamCreate"); }
        if ((e = cudaStreamCreateWithFlags(&g_host.st2, cudaStreamNonBlocking)) != cudaSuccess) { release_host_cache(); return cuda_fail(nullptr, e, "cudaStreamCreate"); }
    }
    char *d = g_host.ptr;
    cudaStream_t st = g_host.st;
    int rc = HYB_OK;
    // the context is kept as well while n and the parameters stay the same: a run that advances call by call then
    // keeps what a device-resident run keeps (the work order of the walks follows the list lengths of the previous
    // ones, split_group), and gives the same bits
    if (g_host.ctx && (g_host.n != n || memcmp(&g_host.p, params, sizeof(hyb_params)) != 0)) {
        cudaStreamSynchronize(st);
        hyb_free(g_host.ctx); g_host.ctx = nullptr;
    }
    do {
        cudaMemcpyAsync(d + o_pos, h_pos_m, 16 * N, cudaMemcpyHostToDevice, st);
        cudaMemcpyAsync(d + o_vel, h_vel, 16 * N, cudaMemcpyHostToDevice, st);
        cudaMemcpyAsync(d + o_id, h_id, 4 * N, cudaMemcpyHostToDevice, st);
        if (acc_valid) {       // the caller continues a run: the accelerations of these positions come with them
            cudaMemcpyAsync(d + o_as, h_a_soft, 16 * N, cudaMemcpyHostToDevice, st);
            cudaMemcpyAsync(d + o_ah, h_a_hard, 16 * N, cudaMemcpyHostToDevice, st);
        }
        if (!g_host.ctx) {
            rc = hyb_init(&g_host.ctx, params, n, (hyb_float4 *)(d + o_pos), (hyb_float4 *)(d + o_vel), (hyb_float4 *)(d + o_as),
                          (hyb_float4 *)(d + o_ah), (uint32_t *)(d + o_id), d + o_ws, ws_bytes, device, st);
            if (rc != HYB_OK) { g_host.ctx = nullptr; break; }
            g_host.p = *params; g_host.n = n;
        }
        Ctx *c = reinterpret_cast<Ctx *>(g_host.ctx);
        c->timing = false;
        discard_pending_bbox(c);                              // new positions: nothing of the last call's tree applies
        c->tree_valid = false; c->tree_refit = false;
        c->acc_valid = acc_valid != 0 && params->hard_refit == 0;
        // positions and ids go back on a second stream as soon as the last build of the call has re-ordered them, next to
        // the last walk (which only reads them); velocities and accelerations follow when the step is done
        EarlyCopy ec = {h_pos_m, h_id, N, g_host.st2, false};
        c->store_final = early_copy; c->store_final_arg = &ec;
        rc = hyb_step(g_host.ctx, n_soft_steps);
        c->store_final = nullptr; c->store_final_arg = nullptr;
        if (rc != HYB_OK) { cudaStreamSynchronize(g_host.st2); break; }
        cudaMemcpyAsync(h_vel, d + o_vel, 16 * N, cudaMemcpyDeviceToHost, st);
        cudaMemcpyAsync(h_a_soft, d + o_as, 16 * N, cudaMemcpyDeviceToHost, st);
        cudaMemcpyAsync(h_a_hard, d + o_ah, 16 * N, cudaMemcpyDeviceToHost, st);
        if (!ec.done) {          // n_soft_steps = 0: no cycle, the store is the one of the initial build
            cudaMemcpyAsync(h_pos_m, d + o_pos, 16 * N, cudaMemcpyDeviceToHost, st);
            cudaMemcpyAsync(h_id, d + o_id, 4 * N, cudaMemcpyDeviceToHost, st);
        }
        e = cudaStreamSynchronize(st);
        const cudaError_t e2 = cudaStreamSynchronize(g_host.st2);
        if (e == cudaSuccess) e = e2;
        if (e != cudaSuccess) { rc = cuda_fail(nullptr, e, "copy back"); break; }
        uint64_t v[4];                                        // (read every time: the counters run since the last read)
        rc = hyb_export(g_host.ctx, HYB_X_INTERACTIONS, v, sizeof v, nullptr);
        if (h_interactions)
            for (int i = 0; i < 4; i++) h_interactions[i] = v[i];
    } while (0);
    if (rc != HYB_OK) release_host_cache();      // (the message stays in the thread's hyb_last_error(NULL))
    return rc;
}

void hyb_run_host_release(void)
{
    std::lock_guard<std::mutex> lock(g_host_mutex);
    release_host_cache();
}

int hyb_let_count(hyb_ctx *ctx, int32_t ndom, const float *h_boxes, uint64_t *h_counts)
{
    Ctx *c = reinterpret_cast<Ctx *>(ctx);
    if (!c) return fail(nullptr, HYB_ERR_INVALID_ARG, "ctx is NULL");
    if (ndom < 1 || !h_boxes || !h_counts) return fail(c, HYB_ERR_INVALID_ARG, "need ndom >= 1 and two host pointers");
    if (!c->tree_valid || c->tree_refit || c->boxes_only)
        return fail(c, HYB_ERR_NO_TREE, "no tree with moments for the current positions");
    if (c->p.mac != HYB_MAC_ABS) return fail(c, HYB_ERR_INVALID_ARG, "hyb_let_count needs HYB_MAC_ABS (r_b and b_max per node)");
    for (int32_t i = 0; i < ndom; i++)
        for (int a = 0; a < 3; a++)
            if (!(h_boxes[6 * i + a] < h_boxes[6 * i + 3 + a])) return fail(c, HYB_ERR_INVALID_ARG, "a domain box is empty or NaN");
    cudaSetDevice(c->device);
    // boxes and counts go through the scratch area of the workspace, as many domains at a time as fit
    char *d = c->ws + c->L.scratch;
    const int32_t chunk = (int32_t)imin64((int64_t)(c->L.scratch_bytes / 64), (int64_t)ndom);
    int rc = HYB_OK;
    for (int32_t d0 = 0; d0 < ndom && rc == HYB_OK; d0 += chunk) {
        const int32_t nd = ndom - d0 < chunk ? ndom - d0 : chunk;
        const size_t bb = sizeof(float) * 6 * (size_t)nd, ob = sizeof(uint64_t) * 3 * (size_t)nd;
        unsigned long long *d_out = reinterpret_cast<unsigned long long *>(d + 32 * (size_t)chunk);
        cudaError_t e = cudaMemcpyAsync(d, h_boxes + 6 * (size_t)d0, bb, cudaMemcpyHostToDevice, c->stream);
        if (e == cudaSuccess) e = launch_let_count(c, nd, reinterpret_cast<const float *>(d), d_out);
        if (e == cudaSuccess) e = cudaMemcpyAsync(h_counts + 3 * (size_t)d0, d_out, ob, cudaMemcpyDeviceToHost, c->stream);
        if (e != cudaSuccess) rc = cuda_fail(c, e, "hyb_let_count");
        else { c->launches += 1; rc = hyb_sync(ctx); }
    }
    return rc;
}

int hyb_energy(hyb_ctx *ctx, double *h_energy)
{
    Ctx *c = reinterpret_cast<Ctx *>(ctx);
    if (!c) return fail(nullptr, HYB_ERR_INVALID_ARG, "ctx is NULL");
    if (!h_energy) return fail(c, HYB_ERR_INVALID_ARG, "h_energy is NULL");
    cudaSetDevice(c->device);
    u32 ni, nj, nk;
    const size_t nd = energy_scratch_doubles(c, &ni, &nj, &nk);
    if (nd * sizeof(double) > c->L.scratch_bytes) return fail(c, HYB_ERR_INTERNAL, "energy scratch does not fit the workspace");
    double *d = reinterpret_cast<double *>(c->ws + c->L.scratch);
    int rc = HYB_OK;
    cudaError_t e = launch_energy(c, d, ni, nj, nk);
    if (e == cudaSuccess) e = cudaMemcpyAsync(h_energy, d, 2 * sizeof(double), cudaMemcpyDeviceToHost, c->stream);
    if (e != cudaSuccess) rc = cuda_fail(c, e, "hyb_energy");
    else { c->launches += 3; rc = hyb_sync(ctx); }
    return rc;
}

int hyb_energy_noalloc(const hyb_float4 *d_pos_m, const hyb_float4 *d_vel, int64_t n, float G, float eps, int device,
                       void *cuda_stream, double *d_energy)
{
    if (!d_pos_m || !d_vel || !d_energy) return fail(nullptr, HYB_ERR_INVALID_ARG, "a device pointer is NULL");
    if (n < 1) return fail(nullptr, HYB_ERR_INVALID_ARG, "n < 1");
    if (n > HYB_ENERGY_NOALLOC_MAX_N)
        return fail(nullptr, HYB_ERR_INVALID_ARG, "hyb_energy_noalloc: n exceeds HYB_ENERGY_NOALLOC_MAX_N (4194304): the partial sums would not fit the static scratch; use hyb_energy");
    if (!isfinite(G) || !isfinite(eps) || eps < 0.0f) return fail(nullptr, HYB_ERR_INVALID_ARG, "G / eps not finite or eps < 0");
    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaSetDevice");
    bool too_large = false;
    e = launch_energy_noalloc(d_pos_m, d_vel, n, G, eps, device, (cudaStream_t)cuda_stream, d_energy, &too_large);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "hyb_energy_noalloc");
    if (too_large) return fail(nullptr, HYB_ERR_INVALID_ARG, "hyb_energy_noalloc: the partial sums of n particles do not fit the static scratch on this device; use hyb_energy");
    return HYB_OK;
}

const char *hyb_last_error(const hyb_ctx *ctx)
{
    const Ctx *c = reinterpret_cast<const Ctx *>(ctx);
    return c ? c->err : g_err;
}

void hyb_free(hyb_ctx *ctx)
{
    Ctx *c = reinterpret_cast<Ctx *>(ctx);
    if (!c) return;
    for (int i = 0; i < 5; i++) if (c->ev[i]) cudaEventDestroy(c->ev[i]);
    for (size_t i = 0; i < c->evpool_n; i++) cudaEventDestroy(c->evpool[i]);
    free(c->evpool);
    if (c->aux) { cudaStreamSynchronize(c->aux); cudaStreamDestroy(c->aux); }
    cudaEvent_t evs[4] = {c->ev_sorted, c->ev_perm, c->ev_linked, c->ev_groups};
    for (int i = 0; i < 4; i++) if (evs[i]) cudaEventDestroy(evs[i]);
    delete c;
}

}  // extern "C"
