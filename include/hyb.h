/* hyb.h -- C-ABI of the B200-native hybrid tree force evaluation
 * (Watanabe & Nakasato, "GPU accelerated Hybrid Tree Algorithm for Collision-less N-body
 * Simulations", arXiv:1406.6158; citations are PAPER.md line numbers).
 *
 * One CUDA device, one stream.  The caller (PyTorch in this repository) owns all particle
 * memory and the scratch workspace; the library only launches kernels on the caller's stream.
 * No torch types, no C++ types, no exceptions cross this boundary; nothing is printed.
 *
 * Every function returns HYB_OK (0) or a negative HYB_ERR_* code; hyb_last_error() gives a
 * short message for the last failure on that context.
 *
 * The canonical computation (what every stage must produce, bit for bit where it is integer)
 * is the "T-spec" restated in DESIGN.md section 3 from SURVEY.md 8(c).
 */
#ifndef HYB_H
#define HYB_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* (x, y, z, w) -- 16-byte aligned.  Positions carry the mass in w (Eq. 2:
 * r_j and m_j); velocities and accelerations leave w unused (written as 0). */
typedef struct hyb_float4 {
    float x, y, z, w;
} hyb_float4;

typedef struct hyb_ctx hyb_ctx; /* opaque; created by hyb_init, destroyed by hyb_free */

enum { HYB_MAC_THETA = 0, HYB_MAC_ABS = 1 };
enum { HYB_K_PAPER = 0, HYB_K_POLY7 = 1 };
enum { HYB_GROUP_NODE = 0, HYB_GROUP_SIBLINGS = 1, HYB_GROUP_AUTO = 2 };

/* The paper's statement of the problem. */
typedef struct hyb_params {
    float G;           /* gravitational constant, Eq. 2                                        */
    float eps;         /* softening length, Eq. 2; must be > 0                                 */
    float theta;       /* opening angle for HYB_MAC_THETA (open if d < l/theta); 0 opens all   */
    float a_err;       /* absolute-MAC accuracy parameter of Eq. 5 (paper: 2^-8); > 0 if used  */
    float r_in;        /* R_1 of Eq. 10                                                        */
    float r_out;       /* R_2 of Eq. 10; 0 <= r_in < r_out                                     */
    float dt_soft;     /* Delta t_s                                              */
    int32_t n_sub;     /* n: Delta t_h = Delta t_s / n, >= 1                                   */
    int32_t leaf_max;  /* n_crit: a cell with more particles is split; 1..64     */
    int32_t group_max; /* sinks that share one traversal (n_vec); leaf_max..64   */
    int32_t mac;       /* HYB_MAC_THETA or HYB_MAC_ABS (Eq. 5-6)                               */
    int32_t kfunc;     /* HYB_K_PAPER (Eq. 10, the default) or HYB_K_POLY7 (north_star's alternative) */
    int32_t split;     /* 1 = hybrid (Eq. 7-9); 0 = normal tree (K == 0)     */
    int32_t grouping;  /* sink groups (consecutive sorted sinks share a traversal):
                          HYB_GROUP_SIBLINGS = runs of consecutive sibling cells of <= group_max particles
                          in all, HYB_GROUP_NODE = one tree node per group (R17);
                          HYB_GROUP_AUTO = SIBLINGS, except that hyb_step builds the trees that only a
                          hard walk uses with runs of at most group_max / 2 sinks (the hard force is a
                          direct sum whatever the groups are; smaller groups list fewer particles beyond
                          r_out)                                                                        */
    int32_t hard_tree; /* 0 = the hard force is the direct K-weighted sum over every particle of the leaves
                          within r_out (R20); 1 = the paper's hard walk: the
                          MAC applies there too, a cell accepted within r_out contributes K(r_COM) F_COM and
                          (1 - K(r_COM)) F_COM to the soft force, and the soft walk drops rule (b)        */
    int32_t hard_refit;/* hyb_step only, needs split = 1 and hard_tree = 0.  0 = the tree is rebuilt before
                          every force evaluation, as the paper does (R21).  1 = it is
                          rebuilt at soft steps only; the hard-only substeps keep the store order and the
                          topology and refit the tight boxes (see hyb_refit_tree): the hard force is the same
                          direct sum, only the order of the fp32 additions differs                          */
    int32_t hard_cut;  /* the hard list of a sink group (K = 0 beyond R_2; R30).
                          0 = every particle of every leaf whose tight box comes within r_out of the group box;
                          1 = only the particles that are themselves within r_out of the group box (what the
                          fused walk drops from the hard list it evaluates as plain Eq. 2 pairs).  The forces are
                          the same (the dropped pairs carry K = 0); HYB_X_NHARD and the hard interaction count
                          report the list that was evaluated                                               */
} hyb_params;

enum {
    HYB_OK = 0,
    HYB_ERR_INVALID_ARG = -1,
    HYB_ERR_WORKSPACE_TOO_SMALL = -2,
    HYB_ERR_NONFINITE_INPUT = -3,   /* a position or mass is NaN/Inf, or a mass is negative     */
    HYB_ERR_CAPACITY_OVERFLOW = -4, /* node pool or a walk stack overflowed; results invalid    */
    HYB_ERR_NO_TREE = -5,           /* force call without a tree built for the current positions*/
    HYB_ERR_CUDA = -6,
    HYB_ERR_INTERNAL = -7           /* a bounded device-side wait expired (should never happen) */
};

/* hyb_export selectors.  "n" = particles, "nn" = tree nodes, "ng" = sink groups (read them
 * with HYB_X_COUNTS first).  All arrays refer to the store order after the last
 * hyb_build_tree (Morton order). */
enum {
    HYB_X_COUNTS = 0,      /* int64[8]: n, nn, ng, node_cap, status bits, nodes before clamping,
                              kernels launched since hyb_init, sink ranges the last walk was handed
                              in front of the ordinary sequence (its work order, see hyb_soft_force) */
    HYB_X_KEYS_SORTED = 1, /* uint64[n]  63-bit Morton keys, ascending                          */
    HYB_X_PERM = 2,        /* uint32[n]  perm[j] = index, in the order the build found the
                              store in, of the particle now in slot j (stable sort)            */
    HYB_X_LEVEL = 3,       /* uint8[nn]                                                         */
    HYB_X_FIRST = 4,       /* uint32[nn]                                                        */
    HYB_X_COUNT = 5,       /* uint32[nn]                                                        */
    HYB_X_CHILD = 6,       /* uint32[nn] index of first child, 0xFFFFFFFF for a leaf            */
    HYB_X_NCHILD = 7,      /* uint8[nn]                                                         */
    HYB_X_PARENT = 8,      /* uint32[nn] 0xFFFFFFFF for the root                                */
    HYB_X_LEVEL_OFFSET = 9,/* uint32[23]                                                        */
    HYB_X_COM_M = 10,      /* float[4 nn] centre of mass and mass                               */
    HYB_X_ROPEN2 = 11,     /* float[nn]  squared opening radius                                 */
    HYB_X_NLO = 12,        /* float[4 nn] tight box minimum (w unused)                          */
    HYB_X_NHI = 13,        /* float[4 nn] tight box maximum (w unused)                          */
    HYB_X_GFIRST = 14,     /* uint32[ng]                                                        */
    HYB_X_GCOUNT = 15,     /* uint32[ng]                                                        */
    HYB_X_GLO = 16,        /* float[4 ng]                                                       */
    HYB_X_GHI = 17,        /* float[4 ng]                                                       */
    HYB_X_NCELL = 18,      /* uint32[ng] cell-list length of the last walk                      */
    HYB_X_NPART = 19,      /* uint32[ng] particle-list length of the last walk                  */
    HYB_X_NHARD = 20,      /* uint32[ng] hard-list length of the last walk                      */
    HYB_X_INTERACTIONS = 21,/* uint64[4] since the last read: sum over groups of members x (ncell+npart),
                              members x nhard (all walks), members x nhard of the fused soft+hard walks (those pairs
                              are on both lists but evaluated once), members x npart of the hard-only walks (their
                              hard lists at leaf granularity, whatever hard_cut is) */
    HYB_X_TIMINGS = 22,    /* float[8] ms accumulated in hyb_step since the last read:
                              build, soft walk, hard walk, integrate, 0, 0, 0, cycles           */
    HYB_X_BBOX = 23,       /* float[6] lo xyz, hi xyz of the last build                         */
    HYB_X_KEYS = 24,       /* uint64[n] keys in the order the build found the store in          */
    HYB_X_M64 = 25,        /* double[nn] node mass before rounding                              */
    HYB_X_C64 = 26,        /* double[3 nn] node centre of mass before rounding                  */
    HYB_X_B2 = 27,         /* double[nn]  B_2 of Eq. 6 (HYB_MAC_ABS only)                       */
    HYB_X_BMAX = 28        /* double[nn]  b_max of Eq. 5 (HYB_MAC_ABS only)                     */
};

/* Bytes of device scratch hyb_init needs for n particles with these parameters.
 * Pure host function (no CUDA call).  Returns 0 if n < 1 or the parameters are invalid. */
size_t hyb_workspace_bytes(int64_t n, const hyb_params *params);

/* Create a context.
 *  params          host pointer; copied.
 *  n               number of particles, 1 <= n <= 2^28 - 2048 (tree node indices are 29-bit).
 *  d_pos_m         DEVICE float4[n], in/out: positions and masses.  Re-ordered
 *                  into Morton order by every tree build, advanced by hyb_step.
 *  d_vel           DEVICE float4[n], in/out: velocities, re-ordered with the positions.
 *  d_a_soft        DEVICE float4[n], out: soft accelerations, Eq. 9 summed over j
 *                  (split = 0: the full normal-tree acceleration).
 *  d_a_hard        DEVICE float4[n], out: hard accelerations, Eq. 8 summed over j.
 *  d_id            DEVICE uint32[n], in/out: caller's particle labels, re-ordered with the
 *                  positions (fill with 0..n-1 to track the permutation).
 *  d_workspace     DEVICE scratch of at least hyb_workspace_bytes(n, params), 256-byte aligned.
 *  device, cuda_stream   CUDA device ordinal and cudaStream_t (as void*) all work is issued on.
 * All device buffers stay owned by the caller and must outlive the context.  A context allocates no
 * device memory: every call, hyb_energy and hyb_let_count included, works inside d_workspace (the only
 * device allocation of the library is the buffer hyb_run_host keeps, see there).  The context owns host
 * memory, one auxiliary CUDA stream and CUDA events.  hyb_init itself only zeroes its control block. */
int hyb_init(hyb_ctx **out, const hyb_params *params, int64_t n,
             hyb_float4 *d_pos_m, hyb_float4 *d_vel, hyb_float4 *d_a_soft, hyb_float4 *d_a_hard,
             uint32_t *d_id, void *d_workspace, size_t workspace_bytes, int device, void *cuda_stream);

/* Change parameters that do not affect workspace size (theta, a_err, r_in, r_out, eps, G,
 * dt_soft, n_sub, mac, split); leaf_max / group_max must be unchanged.  Invalidates the tree. */
int hyb_set_params(hyb_ctx *ctx, const hyb_params *params);

/* Steps a1-a7: bounding box, 63-bit Morton keys, stable radix sort, re-order of pos/vel/id,
 * linear octree, centre-of-mass / opening-radius upsweep
 * and sink groups for the current positions.  Asynchronous. */
int hyb_build_tree(hyb_ctx *ctx);

/* The tree of a hard-step (a hard-step computes only the hard force; the tree is
 * rebuilt for it): steps a1-a5 and a7 as in hyb_build_tree and the tight boxes of a6, but no moments and no
 * opening radius, which only the soft walk reads (with hard_tree = 1 they are computed, the hard walk applies
 * the MAC).  With grouping = HYB_GROUP_AUTO the sink groups are runs of at most group_max / 2 sinks
 * (R17).  This is the build hyb_step uses in front of every hard-only force
 * evaluation.  Afterwards hyb_hard_force works; hyb_soft_force and hyb_let_count return HYB_ERR_NO_TREE.
 * Needs split = 1.  Asynchronous. */
int hyb_build_tree_hard(hyb_ctx *ctx);

/* After the positions have moved a little since the last hyb_build_tree (same store order): recompute the
 * tight boxes of all nodes and sink groups for the current positions, keeping the topology.  The result
 * serves hyb_hard_force with hard_tree = 0 only (a direct K-weighted sum over everything within r_out does
 * not depend on which hierarchy of tight boxes finds the neighbours); hyb_soft_force and hyb_let_count
 * return HYB_ERR_NO_TREE until the next hyb_build_tree.  Asynchronous.
 * Errors: NO_TREE (nothing to refit), INVALID_ARG (split = 0 or hard_tree = 1). */
int hyb_refit_tree(hyb_ctx *ctx);

/* Step a8 (+a9 at a soft-step).  split = 1: one fused group walk that writes d_a_soft
 * (cells accepted by the MAC as monopoles, plus (1-K)-weighted neighbours, Eq. 9)
 * AND d_a_hard (K-weighted neighbours within r_out, Eq. 8).  split = 0: normal-tree walk,
 * d_a_soft = full acceleration, d_a_hard = 0.  Requires a tree.  Asynchronous.
 * Work order: with fewer than about 160 particles per warp the GPU keeps resident (n < 3.8e5 on a B200) the
 * longest sink groups decide how long the walk takes; they are then cut into sink ranges like those of
 * hyb_hard_force, from the list lengths of the previous fused walk (none at the first one).  The same
 * reproducibility statement holds. */
int hyb_soft_force(hyb_ctx *ctx);

/* Step a9 alone (a hard-step): neighbour search cut off at r_out
 * and the K-weighted direct sum; writes d_a_hard only.  split = 0: writes zeros.
 * Requires a tree.  Asynchronous.
 * Reproducibility: the same sequence of calls on the same input gives the same bits.  The heaviest sink
 * groups are cut into sink ranges for load balance, chosen from the list lengths of the previous walk; the
 * neighbour lists never depend on that, but a cut group adds its partial sums in another order, so a walk
 * repeated on one tree can differ from the first in the last bits. */
int hyb_hard_force(hyb_ctx *ctx);

/* n_soft_steps cycles of the two-rate leapfrog (Eq. 3-4), in the
 * kick-drift-kick form of DESIGN.md (reading R21):
 *   v += dt_s/2 a_soft;  n x { v += dt_h/2 a_hard; x += dt_h v; build; a_hard (and a_soft on the
 *   last repeat); v += dt_h/2 a_hard };  v += dt_s/2 a_soft.
 * If the accelerations are not valid for the current positions they are evaluated first.
 * Leaves a_soft / a_hard valid for the final positions.  Synchronises the stream once at the
 * end to read the device status word (capacity overflow, non-finite input). */
int hyb_step(hyb_ctx *ctx, int32_t n_soft_steps);

/* Sink-sharded evaluation (PAPER.md:113-122 without the LET: every replica holds all
 * particles and builds the same tree, the sinks are divided).  After this call hyb_soft_force / hyb_hard_force
 * evaluate only the sink groups whose first particle lies in store slots [first, last) -- groups are never cut,
 * so the ranges of the replicas tile the groups when they tile [0, n) -- and write ZERO accelerations for all
 * other sinks, so that the element-wise sum over the replicas (one all-reduce, or an all-gather of the owned
 * ranges) is the full result: every replica holds the same bits afterwards, and they are the bits of an unsharded
 * evaluation wherever the same groups were cut into sink ranges (see hyb_hard_force; else equal to the last bits).  hyb_step refuses a partial range: the caller runs the cycle with
 * hyb_kick_drift / hyb_build_tree(_hard) / hyb_soft_force / hyb_hard_force and exchanges in between
 * (paper_1406_6158_b200/sharded.py).  Default [0, n).  Errors: INVALID_ARG. */
int hyb_set_sink_range(hyb_ctx *ctx, int64_t first, int64_t last);

/* Step a10 alone (Eq. 3-4): v += c_soft a_soft + c_hard a_hard;  x += dt v  for every
 * particle (dt = 0: kick only), with the accelerations as they are in d_a_soft / d_a_hard now.  The building
 * block of hyb_step's cycle (R21) for callers that run the cycle themselves.  dt != 0 invalidates the tree.
 * Asynchronous.  Errors: INVALID_ARG (non-finite coefficient), CUDA. */
int hyb_kick_drift(hyb_ctx *ctx, float c_soft, float c_hard, float dt);

/* Synchronise the stream and return the device status as an error code.  An error (non-finite input, capacity
 * overflow) is reported once: the status word is cleared, the tree and the accelerations of the context are
 * marked invalid, and the context can be used again after the caller has repaired the input (the next
 * hyb_build_tree / hyb_step starts from the particle arrays as they are). */
int hyb_sync(hyb_ctx *ctx);

/* Debug / test / bench read-back into HOST memory; synchronises the stream.
 * *written (optional) receives the byte count; too small a buffer -> HYB_ERR_INVALID_ARG. */
int hyb_export(hyb_ctx *ctx, int32_t what, void *host_dst, size_t bytes, size_t *written);

/* End-to-end call for HOST buffers: copies the particles to the device, runs hyb_step(n_soft_steps)
 * (n_soft_steps = 0: one build + soft-step evaluation only), copies positions, velocities, ids and both
 * accelerations back.  acc_valid = 0: the accelerations of the incoming positions are evaluated first (one more
 * tree build and soft-step walk); acc_valid = 1: h_a_soft / h_a_hard are INPUTS too -- the accelerations this
 * call returned for exactly these positions the last time -- so a run whose state lives on the host advances
 * one call per cycle with nothing computed twice, and with the bits a device-resident context gives.  The device
 * buffer (particles + workspace, the library's only device allocation), its stream and -- while n and the
 * parameters stay the same -- the context are kept for the next call on the same device (freed by
 * hyb_run_host_release, or replaced when a larger n comes); concurrent calls are serialised.  Positions and ids
 * travel back while the last walk of the call still runs (they are final once its tree is built); when the call
 * returns an error the contents of the host arrays are unspecified.  Every pointer is
 * a HOST pointer to n elements; h_interactions (optional) receives uint64[4] as HYB_X_INTERACTIONS. */
int hyb_run_host(const hyb_params *params, int64_t n, hyb_float4 *h_pos_m, hyb_float4 *h_vel,
                 hyb_float4 *h_a_soft, hyb_float4 *h_a_hard, uint32_t *h_id, int32_t n_soft_steps,
                 int32_t acc_valid, int device, uint64_t *h_interactions);

/* Frees what hyb_run_host keeps between calls (nothing else holds device memory in this library). */
void hyb_run_host_release(void);

/* Virtual-domain LET counts (Eq. 14-15; Fig. 4: N_soft, N_hard).  The paper's processes
 * exchange locally essential trees; on one GPU nothing is exchanged, but for any set of ndom virtual
 * domains (h_boxes: HOST float[6 ndom] = lo xyz, hi xyz, half-open, +-INFINITY allowed) the size of what
 * domain j would have to receive can be counted from the tree: a node wholly inside the domain is local;
 * otherwise it is sent as one cell unless r_ib < r_b (Eq. 14) or part of it is inside, in which case it
 * is opened (an opened leaf sends its particles outside the domain); the hard LET drops nodes with
 * r_ib >= R_2 + b_max (Eq. 15) and particles farther than R_2.  h_counts: HOST uint64[3 ndom] =
 * N_local, N_soft, N_hard per domain.  Needs a valid tree built with HYB_MAC_ABS; synchronises.
 * Errors: INVALID_ARG (theta-MAC tree, empty box), NO_TREE, CAPACITY_OVERFLOW (traversal stack). */
int hyb_let_count(hyb_ctx *ctx, int32_t ndom, const float *h_boxes, uint64_t *h_counts);

/* Total-energy diagnostic ("error in total energy of the system that is the sum of kinetic
 * and potential energy") for the particles as they are in d_pos_m / d_vel now:
 *   h_energy[0] = T = sum_i 1/2 m_i |v_i|^2
 *   h_energy[1] = W = - G sum_{i<j} m_i m_j / sqrt(r_ij^2 + eps^2)   (potential of the unsplit force, Eq. 1-2)
 * h_energy: HOST double[2].  W is a direct sum over all n (n - 1) / 2 pairs on the device (fp32 pair terms,
 * fp64 accumulation, fixed summation order: repeated calls return the same bits); cost grows as n^2 (a
 * fraction of a second at n = 2^20).  Needs no tree, changes nothing, synchronises.  With eps = 0 two
 * coincident particles give W = -inf.  Errors: INVALID_ARG (NULL pointer), CUDA. */
int hyb_energy(hyb_ctx *ctx, double *h_energy);

/* The same diagnostic (T and W as defined for hyb_energy, the same kernels, the same summation order,
 * hence the same bits) for callers that cannot allocate device memory or hold a context: code under CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc.  This entry point allocates nothing, on the
 * device or on the host: the partial sums of the blocks go to ONE static device array of the library (128 KiB,
 * held by every GPU that loads the library until the process ends).
 *  d_pos_m, d_vel  DEVICE float4[n], inputs (positions + masses, velocities); not changed.
 *  n               1 <= n <= HYB_ENERGY_NOALLOC_MAX_N; larger n -> HYB_ERR_INVALID_ARG with a message that says so
 *                  (hyb_energy has no such limit, its scratch is in the caller's workspace).
 *  G, eps          as in hyb_params.
 *  device, cuda_stream   the device the pointers belong to and the stream the work is issued on.
 *  d_energy        DEVICE double[2], output: T, W.  Written by a device-to-device copy on the stream.
 * Asynchronous: nothing is synchronised, no status word is read; the result is there when the stream gets there.
 * The first call on a device looks up the address of the static array (once per device; it may load the module):
 * make one call before a graph capture begins.
 * The array is shared by every call of the process on that device and keeps the last call's contents; nothing in it
 * has to start from zero (each kernel writes what the next one reads).  Calls that overlap on the GPU (two streams,
 * two threads) race on it and give garbage: issue them on one stream or order them with events.
 * Errors: INVALID_ARG (NULL pointer, n out of range, G / eps not finite, eps < 0), CUDA. */
#define HYB_ENERGY_NOALLOC_MAX_N 4194304
int hyb_energy_noalloc(const hyb_float4 *d_pos_m, const hyb_float4 *d_vel, int64_t n, float G, float eps,
                       int device, void *cuda_stream, double *d_energy);

/* Diagnostic, not on the hot path: the FP32 rate of the CUDA cores of `device`, measured with independent chains
 * of packed (h_tflops[0], fma.rn.f32x2 as the pair kernels use) and scalar (h_tflops[1], fma.rn.f32) fused
 * multiply-adds, in TFLOP/s.  bench.py reports it beside the peak derived from the unit counts and the clock.
 * d_scratch: DEVICE float[scratch_floats], caller-owned, at least 1024 x the number of SMs (results of the chains
 * are stored there so that the loops are not optimised away).  h_tflops: HOST double[2].  Synchronises. */
int hyb_probe_fp32(int device, void *cuda_stream, float *d_scratch, size_t scratch_floats, double *h_tflops);

/* Message for the last error on this context ("" if none).  ctx may be NULL (returns the
 * message of the last failed hyb_init / hyb_run_host on this thread). */
const char *hyb_last_error(const hyb_ctx *ctx);

/* Destroys the context (host memory and CUDA events only; device buffers are the caller's). */
void hyb_free(hyb_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* HYB_H */
