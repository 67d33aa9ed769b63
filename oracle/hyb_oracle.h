/* hyb_oracle.h -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct CPU restatement (fp64 forces, step-by-step decision
 * arithmetic) of the hybrid tree force evaluation of Watanabe & Nakasato, arXiv:1406.6158
 * (PAPER.md).  It shares no code, header, table or constant with the CUDA path under
 * paper_1406_6158_b200/ and may be used only by tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py.
 *
 * Every function cites the PAPER.md passage it follows; "T<n>" / "R<n>" refer to the
 * canonical computation and the readings listed in DESIGN.md (taken from SURVEY.md 8(c)).
 *
 * Parity pins (tests/test_oracle_*.py, run with -m "not gpu"):
 *   orc_K            exact rationals of Eq. 10                       pinned
 *   keys / sort      lattice values, stable-sort equivalence          pinned
 *   octree / groups  invariants + independent geometric bisection     pinned
 *   moments / r_b    direct sums, worked value of Eq. 5               pinned
 *   walk lists       completeness, brute-force neighbour superset,
 *                    rule (a) and Eq. 14-15 re-derived as sets, mutated
 *                    oracles fail (test_oracle_mac.py); hard_cut = 1:
 *                    list == brute-force set over all particles      pinned
 *   forces           two-body closed form, theta=0 == brute force,
 *                    momentum of the hard sum, Plummer/Hernquist/ball pinned
 *   step             circular binary, reversibility, 2nd order        pinned
 *   energy-drift bound over 64 soft steps: the paper prints no number: PARITY UNPINNED
 */
#ifndef HYB_ORACLE_H
#define HYB_ORACLE_H
#include <stdint.h>
#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
    float G, eps;          /* Eq. 2 */
    float theta;           /* theta-MAC (R7, R27) */
    float a_err;           /* absolute MAC, Eq. 5 */
    float r_in, r_out;     /* R1, R2 of Eq. 10 */
    float dt_soft;         /* Delta t_s */
    int32_t n_sub;         /* n, Delta t_h = Delta t_s / n */
    int32_t leaf_max;      /* n_crit (R11) */
    int32_t group_max;     /* sink group size (R17) */
    int32_t mac;           /* 0 theta, 1 absolute */
    int32_t kfunc;         /* 0 Eq. 10, 1 north_star's 7th-degree polynomial */
    int32_t split;         /* 1 hybrid, 0 normal tree */
    int32_t grouping;      /* T11: 0 sink group = one tree node, 1 = run of consecutive small siblings (R17) */
    int32_t hard_tree;     /* R20: 0 hard force = direct K-weighted sum, 1 = the paper's MAC-approximated hard walk */
    int32_t hard_cut;      /* R30 (T13): 0 = the hard list holds every particle of a leaf whose box comes within r_out
                              of the group box; 1 = only those particles that are themselves within r_out of the group
                              box ("neighbours within r_out": cut-off beyond R_2) */
} orc_params;

enum { ORC_MODE_HYBRID = 0, ORC_MODE_HARD = 1, ORC_MODE_NORMAL = 2 };

enum {  /* orc_tree_get selectors */
    ORC_GET_KEYS = 1,      /* u64[n]  keys in input order (T5)          */
    ORC_GET_PERM,          /* u32[n]  stable sort permutation (T6)      */
    ORC_GET_KEYS_SORTED,   /* u64[n]                                    */
    ORC_GET_POS_SORTED,    /* f32[4n]                                   */
    ORC_GET_LEVEL,         /* u8[nn]                                    */
    ORC_GET_FIRST,         /* u32[nn]                                   */
    ORC_GET_COUNT,         /* u32[nn]                                   */
    ORC_GET_CHILD,         /* u32[nn] 0xFFFFFFFF for a leaf             */
    ORC_GET_NCHILD,        /* u8[nn]                                    */
    ORC_GET_PARENT,        /* u32[nn] 0xFFFFFFFF for the root           */
    ORC_GET_LEVEL_OFFSET,  /* u32[23]                                   */
    ORC_GET_COM_M,         /* f32[4nn] stored (x,y,z,M) (T9)            */
    ORC_GET_ROPEN2,        /* f32[nn] (T10)                             */
    ORC_GET_NLO,           /* f32[3nn] tight box min (T8)               */
    ORC_GET_NHI,           /* f32[3nn]                                  */
    ORC_GET_M64,           /* f64[nn]                                   */
    ORC_GET_C64,           /* f64[3nn]                                  */
    ORC_GET_B2,            /* f64[nn]                                   */
    ORC_GET_BMAX,          /* f64[nn]                                   */
    ORC_GET_GFIRST,        /* u32[ng]                                   */
    ORC_GET_GCOUNT,        /* u32[ng]                                   */
    ORC_GET_GLO,           /* f32[3ng]                                  */
    ORC_GET_GHI,           /* f32[3ng]                                  */
    ORC_GET_BBOX,          /* f32[6] lo xyz, hi xyz (T2)                */
    ORC_GET_ROOT_L         /* f64[1] (T3)                               */
};

typedef struct orc_tree orc_tree;

/* Eq. 10 (kfunc 0) or north_star's polynomial (kfunc 1); T15 / R4-R6. */
double orc_K(double r, double r_in, double r_out, int kfunc);

/* Eq. 5: r_b from b_max, B_2, a_err (order of operations of T10). */
double orc_rb(double bmax, double B2, double a_err);

/* T2-T11 on pos4 = (x,y,z,m) float[4n] in the caller's order.  NULL on invalid input. */
orc_tree *orc_tree_build(int64_t n, const float *pos4, const orc_params *p);
void orc_tree_free(orc_tree *t);
int64_t orc_tree_nn(const orc_tree *t);
int64_t orc_tree_ng(const orc_tree *t);
/* copies the selected array; returns bytes written or -1 */
int64_t orc_tree_get(const orc_tree *t, int what, void *dst, int64_t bytes);

/* T12-T13: list lengths per group.  npart counts the particles of every opened leaf; nhard the hard list
 * (hard_cut = 0: the particles of the leaves within r_out of the group box; hard_cut = 1: those of them that are
 * themselves within r_out of the group box). */
void orc_walk_counts(const orc_tree *t, int mode, uint32_t *ncell, uint32_t *npart, uint32_t *nhard);
/* T12-T13 for the ngsel groups listed in gsel: output entry k belongs to group gsel[k]. */
void orc_walk_counts_sel(const orc_tree *t, int mode, int64_t ngsel, const int64_t *gsel,
                         uint32_t *ncell, uint32_t *npart, uint32_t *nhard);
/* list contents for one group: cells = node ids, parts = sorted-order particle indices,
 * hard[k] = 1 if parts[k] is on the hard list. Returns 0, or -1 if a capacity is too small. */
int orc_walk_lists(const orc_tree *t, int mode, int64_t g,
                   uint32_t *cells, int64_t cap_cells, int64_t *ncells,
                   uint32_t *parts, uint8_t *hard, int64_t cap_parts, int64_t *nparts);

/* Virtual-domain LET counts (Eq. 14-15): boxes = ndom x
 * (lo xyz, hi xyz) floats, half-open; needs a tree built with mac = 1 (r_b and b_max per node).
 * out[3 j ..] = N_local, N_soft, N_hard of domain j. */
void orc_let_count(const orc_tree *t, int64_t ndom, const float *boxes, uint64_t *out);

/* T14: accelerations in SORTED order, double[3n] each.  If ngsel > 0 only the groups in gsel
 * are evaluated (other entries untouched).  interactions (optional) receives
 * sum over evaluated groups of members x (ncell + npart) resp. members x nhard. */
void orc_forces(const orc_tree *t, int mode, int64_t ngsel, const int64_t *gsel,
                double *a_soft, double *a_hard, double *inter_soft, double *inter_hard);

/* Eq. 1-2 by brute force for the sinks sel[0..nsel) (indices into pos4), split by K (Eq. 7-9):
 * a_tot, a_hard, a_soft double[3 nsel]. */
void orc_direct(int64_t n, const float *pos4, float G, float eps, float r_in, float r_out,
                int kfunc, int64_t nsel, const int64_t *sel,
                double *a_tot, double *a_hard, double *a_soft);

/* T16 / R21: ncycles soft cycles of the KDK two-rate leapfrog on fp64 state (input order kept).
 * acc_valid != 0: a_soft/a_hard hold accelerations for the current x. Returns 0 / -1. */
int orc_step(int64_t n, double *x, double *v, const float *m, const orc_params *p,
             int32_t ncycles, double *a_soft, double *a_hard, int acc_valid);

/* R23: kinetic and (softened, unsplit) potential energy. */
void orc_energy(int64_t n, const double *x, const double *v, const float *m, float G, float eps,
                double *kin, double *pot);

int orc_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
