/* hyb_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE (see hyb_oracle.h).
 *
 * Plain C restatement of the hybrid tree force evaluation of PAPER.md, written from the
 * paper in the paper's order.  Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC.
 * -ffp-contract=off matters: the discrete decisions (T4, T10, T12) are specified as
 * individually rounded IEEE operations.  OpenMP is used only over independent sink groups /
 * sinks; every sum is sequential in the order the definition states.
 */
#include "hyb_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define NOCHILD 0xFFFFFFFFu
#define MAXLEVEL 21

struct orc_tree {
    int64_t n;
    orc_params p;
    float lo[3], hi[3];
    double L, origin[3], inv;
    uint64_t *key, *key_s;
    uint32_t *perm;
    float *pos_s;
    int64_t nn, cap;
    uint8_t *level, *nchild;
    uint32_t *first, *count, *child, *parent;
    uint32_t level_offset[MAXLEVEL + 2];
    double *M, *C, *B2, *bmax;
    float *com_m, *ropen2, *nlo, *nhi;
    int64_t ng;
    uint32_t *gfirst, *gcount;
    float *glo, *ghi;
};

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------ K(r), Eq. 10 (T15) */
/* PAPER.md:82-85.  Y = (R2 - r)/(R2 - R1); K = 1 (Y>=1), 10Y^6 - 15Y^8 + 6Y^10 (0<Y<1),
 * 0 (Y<=0).  r is the unsoftened distance (R4).  kfunc 1 is north_star's alternative
 * K(x) = 1 - x^4 (35 - 84x + 70x^2 - 20x^3), x = (r - R1)/(R2 - R1)  (R6; not the default). */
double orc_K(double r, double r_in, double r_out, int kfunc)
{
    if (kfunc == 1) {
        double x = (r - r_in) / (r_out - r_in);
        if (x <= 0.0) return 1.0;
        if (x >= 1.0) return 0.0;
        return 1.0 - x * x * x * x * (35.0 - 84.0 * x + 70.0 * x * x - 20.0 * x * x * x);
    }
    double Y = (r_out - r) / (r_out - r_in);
    if (Y >= 1.0) return 1.0;
    if (Y <= 0.0) return 0.0;
    double t = Y * Y;
    return t * t * t * (10.0 - 15.0 * t + 6.0 * t * t);
}

/* ------------------------------------------------------------------ r_b, Eq. 5 (T10) */
/* PAPER.md:59.  r_b = b_max/2 + sqrt(b_max^2/4 + sqrt(3 B_2 / a_err)). */
double orc_rb(double bmax, double B2, double a_err)
{
    double t1 = 3.0 * B2;
    double t2 = t1 / a_err;
    double t3 = sqrt(t2);
    double t4 = bmax * bmax;
    double t5 = t4 / 4.0;
    double t6 = t5 + t3;
    double t7 = sqrt(t6);
    return bmax / 2.0 + t7;
}

/* ------------------------------------------------------------------ T2-T5 keys */
/* PAPER.md:103 "we first calculate the region and size of the root cell that include all
 * particles. Then, we calculate keys of the particles ... Morton key". */
static void bbox(int64_t n, const float *pos4, float lo[3], float hi[3])
{
    for (int a = 0; a < 3; a++) { lo[a] = pos4[a]; hi[a] = pos4[a]; }
    for (int64_t i = 1; i < n; i++)
        for (int a = 0; a < 3; a++) {
            float x = pos4[4 * i + a];
            if (x < lo[a]) lo[a] = x;
            if (x > hi[a]) hi[a] = x;
        }
}

static uint64_t morton63(uint32_t qx, uint32_t qy, uint32_t qz)
{
    uint64_t k = 0;
    for (int b = 0; b < 21; b++) {
        k |= (uint64_t)((qx >> b) & 1u) << (3 * b + 2);
        k |= (uint64_t)((qy >> b) & 1u) << (3 * b + 1);
        k |= (uint64_t)((qz >> b) & 1u) << (3 * b);
    }
    return k;
}

static void make_keys(orc_tree *t, const float *pos4)
{
    bbox(t->n, pos4, t->lo, t->hi);                                   /* T2 */
    double L = 0.0;                                                    /* T3 */
    for (int a = 0; a < 3; a++) {
        double e = (double)t->hi[a] - (double)t->lo[a];
        if (e > L) L = e;
        t->origin[a] = (double)t->lo[a];
    }
    if (L == 0.0) L = 1.0;
    t->L = L;
    t->inv = 2097152.0 / L;
    for (int64_t i = 0; i < t->n; i++) {                               /* T4, T5 */
        uint32_t q[3];
        for (int a = 0; a < 3; a++) {
            double d = (double)pos4[4 * i + a] - t->origin[a];
            double s = d * t->inv;
            double f = floor(s);
            uint32_t u = (f >= 2097151.0) ? 2097151u : (uint32_t)f;
            q[a] = u;
        }
        t->key[i] = morton63(q[0], q[1], q[2]);
    }
}

/* ------------------------------------------------------------------ T6 stable sort */
/* PAPER.md:103-105 "we sort the keys ... We also sort the data of the positions".
 * Bottom-up merge sort of indices by key; the left run wins ties, so equal keys keep
 * ascending input index (R15). */
static void stable_sort_perm(int64_t n, const uint64_t *key, uint32_t *perm)
{
    uint32_t *a = perm, *b = (uint32_t *)malloc(sizeof(uint32_t) * (size_t)n);
    for (int64_t i = 0; i < n; i++) a[i] = (uint32_t)i;
    for (int64_t w = 1; w < n; w *= 2) {
        for (int64_t s = 0; s < n; s += 2 * w) {
            int64_t m = s + w < n ? s + w : n, e = s + 2 * w < n ? s + 2 * w : n;
            int64_t i = s, j = m, k = s;
            while (i < m && j < e) {
                if (key[a[j]] < key[a[i]]) b[k++] = a[j++];
                else b[k++] = a[i++];
            }
            while (i < m) b[k++] = a[i++];
            while (j < e) b[k++] = a[j++];
        }
        uint32_t *tmp = a; a = b; b = tmp;
    }
    if (a != perm) { memcpy(perm, a, sizeof(uint32_t) * (size_t)n); free(a); }
    else free(b);
}

/* ------------------------------------------------------------------ T7 octree */
/* PAPER.md:53 "The division is recursively continued while the cell has many particles than
 * a critical number n_crit" (R11: internal <=> count > leaf_max), "we divide the
 * array into eight sub-arrays by the three most significant bits of the keys ... Then we
 * recursively repeat the procedure for every three bits of key".  Breadth-first numbering. */
static int grow(orc_tree *t)
{
    int64_t c = t->cap * 2;
    t->level = (uint8_t *)realloc(t->level, (size_t)c);
    t->nchild = (uint8_t *)realloc(t->nchild, (size_t)c);
    t->first = (uint32_t *)realloc(t->first, 4 * (size_t)c);
    t->count = (uint32_t *)realloc(t->count, 4 * (size_t)c);
    t->child = (uint32_t *)realloc(t->child, 4 * (size_t)c);
    t->parent = (uint32_t *)realloc(t->parent, 4 * (size_t)c);
    t->cap = c;
    return 0;
}

static void build_octree(orc_tree *t)
{
    const uint64_t *ks = t->key_s;
    t->cap = 1024;
    t->level = (uint8_t *)malloc((size_t)t->cap);
    t->nchild = (uint8_t *)malloc((size_t)t->cap);
    t->first = (uint32_t *)malloc(4 * (size_t)t->cap);
    t->count = (uint32_t *)malloc(4 * (size_t)t->cap);
    t->child = (uint32_t *)malloc(4 * (size_t)t->cap);
    t->parent = (uint32_t *)malloc(4 * (size_t)t->cap);
    t->level[0] = 0; t->first[0] = 0; t->count[0] = (uint32_t)t->n;
    t->parent[0] = NOCHILD; t->child[0] = NOCHILD; t->nchild[0] = 0;
    int64_t nn = 1;
    for (int l = 0; l <= MAXLEVEL + 1; l++) t->level_offset[l] = 0;
    int64_t head = 0;
    int curlevel = 0;
    t->level_offset[0] = 0;
    while (head < nn) {
        int l = t->level[head];
        while (curlevel < l) { curlevel++; t->level_offset[curlevel] = (uint32_t)head; }
        uint32_t f = t->first[head], c = t->count[head];
        if ((int64_t)c > t->p.leaf_max && l < MAXLEVEL) {          /* internal */
            int shift = 60 - 3 * l;
            uint32_t pos = f, end = f + c;
            t->child[head] = (uint32_t)nn;
            int nc = 0;
            for (unsigned o = 0; o < 8; o++) {                        /* digits ascending */
                uint32_t s = pos;
                while (pos < end && ((ks[pos] >> shift) & 7u) == o) pos++;
                if (pos > s) {
                    if (nn == t->cap) grow(t);
                    t->level[nn] = (uint8_t)(l + 1);
                    t->first[nn] = s; t->count[nn] = pos - s;
                    t->parent[nn] = (uint32_t)head;
                    t->child[nn] = NOCHILD; t->nchild[nn] = 0;
                    nn++; nc++;
                }
            }
            t->nchild[head] = (uint8_t)nc;
        }
        head++;
    }
    for (int l = curlevel + 1; l <= MAXLEVEL + 1; l++) t->level_offset[l] = (uint32_t)nn;
    t->nn = nn;
}

/* ------------------------------------------------------------------ T8-T10 moments, MAC */
/* PAPER.md:55 centre of mass; Eq. 5-6 (b_max exact, R9; B_2 by the parallel-axis
 * upsweep, R10); theta-mode l/theta with l the geometric cell side (R27). */
static void moments(orc_tree *t)
{
    int64_t nn = t->nn;
    const float *ps = t->pos_s;
    t->M = (double *)calloc((size_t)nn, 8); t->C = (double *)calloc(3 * (size_t)nn, 8);
    t->B2 = (double *)calloc((size_t)nn, 8); t->bmax = (double *)calloc((size_t)nn, 8);
    t->com_m = (float *)calloc(4 * (size_t)nn, 4); t->ropen2 = (float *)calloc((size_t)nn, 4);
    t->nlo = (float *)calloc(3 * (size_t)nn, 4); t->nhi = (float *)calloc(3 * (size_t)nn, 4);
    double *S = (double *)calloc(3 * (size_t)nn, 8);
    for (int64_t k = nn - 1; k >= 0; k--) {        /* children have larger BFS index */
        uint32_t f = t->first[k], c = t->count[k];
        double M = 0.0, Sx = 0.0, Sy = 0.0, Sz = 0.0;
        float lo[3], hi[3];
        if (t->child[k] == NOCHILD) {                                  /* T9 leaf, T8 */
            for (int a = 0; a < 3; a++) { lo[a] = ps[4 * (size_t)f + a]; hi[a] = lo[a]; }
            for (uint32_t j = f; j < f + c; j++) {
                double m = (double)ps[4 * (size_t)j + 3];
                M = M + m;
                Sx = Sx + m * (double)ps[4 * (size_t)j + 0];
                Sy = Sy + m * (double)ps[4 * (size_t)j + 1];
                Sz = Sz + m * (double)ps[4 * (size_t)j + 2];
                for (int a = 0; a < 3; a++) {
                    float x = ps[4 * (size_t)j + a];
                    if (x < lo[a]) lo[a] = x;
                    if (x > hi[a]) hi[a] = x;
                }
            }
        } else {                                                       /* T9 internal */
            uint32_t c0 = t->child[k];
            for (int a = 0; a < 3; a++) { lo[a] = t->nlo[3 * (size_t)c0 + a]; hi[a] = t->nhi[3 * (size_t)c0 + a]; }
            for (uint32_t q = c0; q < c0 + t->nchild[k]; q++) {
                M = M + t->M[q];
                Sx = Sx + S[3 * (size_t)q + 0];
                Sy = Sy + S[3 * (size_t)q + 1];
                Sz = Sz + S[3 * (size_t)q + 2];
                for (int a = 0; a < 3; a++) {
                    if (t->nlo[3 * (size_t)q + a] < lo[a]) lo[a] = t->nlo[3 * (size_t)q + a];
                    if (t->nhi[3 * (size_t)q + a] > hi[a]) hi[a] = t->nhi[3 * (size_t)q + a];
                }
            }
        }
        t->M[k] = M; S[3 * k] = Sx; S[3 * k + 1] = Sy; S[3 * k + 2] = Sz;
        for (int a = 0; a < 3; a++) { t->nlo[3 * k + a] = lo[a]; t->nhi[3 * k + a] = hi[a]; }
        double Cx, Cy, Cz;
        if (M == 0.0) { Cx = (double)lo[0]; Cy = (double)lo[1]; Cz = (double)lo[2]; }
        else { Cx = Sx / M; Cy = Sy / M; Cz = Sz / M; }
        t->C[3 * k] = Cx; t->C[3 * k + 1] = Cy; t->C[3 * k + 2] = Cz;
        t->com_m[4 * k] = (float)Cx; t->com_m[4 * k + 1] = (float)Cy;
        t->com_m[4 * k + 2] = (float)Cz; t->com_m[4 * k + 3] = (float)M;
        float ropen;
        if (t->p.mac == 0) {                                           /* T10 theta-mode */
            float l = ldexpf((float)t->L, -(int)t->level[k]);
            ropen = l / t->p.theta;
        } else {                                                       /* T10 abs-mode */
            double b2max = 0.0;
            for (uint32_t j = f; j < f + c; j++) {
                double dx = (double)ps[4 * (size_t)j + 0] - Cx;
                double dy = (double)ps[4 * (size_t)j + 1] - Cy;
                double dz = (double)ps[4 * (size_t)j + 2] - Cz;
                double d2 = (dx * dx + dy * dy) + dz * dz;
                if (d2 > b2max) b2max = d2;
            }
            double B2 = 0.0;
            if (t->child[k] == NOCHILD) {
                for (uint32_t j = f; j < f + c; j++) {
                    double dx = (double)ps[4 * (size_t)j + 0] - Cx;
                    double dy = (double)ps[4 * (size_t)j + 1] - Cy;
                    double dz = (double)ps[4 * (size_t)j + 2] - Cz;
                    double d2 = (dx * dx + dy * dy) + dz * dz;
                    B2 = B2 + (double)ps[4 * (size_t)j + 3] * d2;
                }
            } else {
                uint32_t c0 = t->child[k];
                for (uint32_t q = c0; q < c0 + t->nchild[k]; q++) {
                    double dx = t->C[3 * (size_t)q + 0] - Cx;
                    double dy = t->C[3 * (size_t)q + 1] - Cy;
                    double dz = t->C[3 * (size_t)q + 2] - Cz;
                    double d2 = (dx * dx + dy * dy) + dz * dz;
                    B2 = B2 + (t->B2[q] + t->M[q] * d2);
                }
            }
            double bm = sqrt(b2max);
            t->B2[k] = B2; t->bmax[k] = bm;
            ropen = (float)orc_rb(bm, B2, (double)t->p.a_err);
        }
        t->ropen2[k] = ropen * ropen;
    }
    free(S);
}

/* ------------------------------------------------------------------ T11 groups */
/* n_vec CONSECUTIVE sorted sinks share one traversal.  R17, two readings:
 *   grouping 0: a sink group is a maximal tree node with count <= group_max;
 *   grouping 1: the children of a cell with more than group_max particles are taken in order and
 *               consecutive children with count <= group_max are packed greedily into runs whose
 *               total stays <= group_max (a child with more than group_max particles closes the run
 *               and is treated recursively); a group is such a run -- consecutive sorted sinks as in
 *               the paper, fuller than single nodes, and still inside one cell.
 * In both, level-21 leaves larger than group_max are cut into chunks of group_max. */
static void groups(orc_tree *t)
{
    int64_t gm = t->p.group_max, ng = 0;
    uint8_t *mark = (uint8_t *)calloc((size_t)t->n, 1);
    if (t->p.grouping == 1) {             /* T11 (siblings): see the comment above */
        for (int64_t k = 0; k < t->nn; k++) {
            uint32_t c = t->count[k], f = t->first[k];
            if ((int64_t)c <= gm) { if (k == 0) mark[f] = 1; continue; }
            if (t->child[k] == NOCHILD) { for (uint32_t s = f; s < f + c; s += (uint32_t)gm) mark[s] = 1; continue; }
            int64_t run = 0; int open = 0;
            for (uint32_t q = t->child[k]; q < t->child[k] + t->nchild[k]; q++) {
                int64_t cq = t->count[q];
                if (cq > gm) { open = 0; run = 0; continue; }
                if (!open || run + cq > gm) { mark[t->first[q]] = 1; run = 0; open = 1; }
                run += cq;
            }
        }
    } else
    for (int64_t k = 0; k < t->nn; k++) {
        uint32_t c = t->count[k], f = t->first[k];
        int is_group = (int64_t)c <= gm && (k == 0 || (int64_t)t->count[t->parent[k]] > gm);
        if (is_group) mark[f] = 1;
        else if (t->child[k] == NOCHILD && (int64_t)c > gm)          /* level-21 leaf */
            for (uint32_t s = f; s < f + c; s += (uint32_t)gm) mark[s] = 1;
    }
    for (int64_t i = 0; i < t->n; i++) ng += mark[i];
    t->ng = ng;
    t->gfirst = (uint32_t *)malloc(4 * (size_t)ng); t->gcount = (uint32_t *)malloc(4 * (size_t)ng);
    t->glo = (float *)malloc(12 * (size_t)ng); t->ghi = (float *)malloc(12 * (size_t)ng);
    int64_t g = -1;
    for (int64_t i = 0; i < t->n; i++) {
        if (mark[i]) { g++; t->gfirst[g] = (uint32_t)i; t->gcount[g] = 0;
            for (int a = 0; a < 3; a++) { t->glo[3 * g + a] = t->pos_s[4 * i + a]; t->ghi[3 * g + a] = t->pos_s[4 * i + a]; } }
        t->gcount[g]++;
        for (int a = 0; a < 3; a++) {
            float x = t->pos_s[4 * i + a];
            if (x < t->glo[3 * g + a]) t->glo[3 * g + a] = x;
            if (x > t->ghi[3 * g + a]) t->ghi[3 * g + a] = x;
        }
    }
    free(mark);
}

orc_tree *orc_tree_build(int64_t n, const float *pos4, const orc_params *p)
{
    if (n < 1 || n > 0x7FFFFFFF || !pos4 || !p) return NULL;
    if (p->leaf_max < 1 || p->group_max < p->leaf_max) return NULL;
    for (int64_t i = 0; i < 4 * n; i++) if (!isfinite(pos4[i])) return NULL;     /* T1 */
    for (int64_t i = 0; i < n; i++) if (pos4[4 * i + 3] < 0.0f) return NULL;
    orc_tree *t = (orc_tree *)calloc(1, sizeof(orc_tree));
    t->n = n; t->p = *p;
    t->key = (uint64_t *)malloc(8 * (size_t)n); t->key_s = (uint64_t *)malloc(8 * (size_t)n);
    t->perm = (uint32_t *)malloc(4 * (size_t)n); t->pos_s = (float *)malloc(16 * (size_t)n);
    make_keys(t, pos4);
    stable_sort_perm(n, t->key, t->perm);
    for (int64_t j = 0; j < n; j++) {
        t->key_s[j] = t->key[t->perm[j]];
        memcpy(t->pos_s + 4 * j, pos4 + 4 * (size_t)t->perm[j], 16);
    }
    build_octree(t);
    moments(t);
    groups(t);
    return t;
}

void orc_tree_free(orc_tree *t)
{
    if (!t) return;
    free(t->key); free(t->key_s); free(t->perm); free(t->pos_s);
    free(t->level); free(t->nchild); free(t->first); free(t->count); free(t->child); free(t->parent);
    free(t->M); free(t->C); free(t->B2); free(t->bmax);
    free(t->com_m); free(t->ropen2); free(t->nlo); free(t->nhi);
    free(t->gfirst); free(t->gcount); free(t->glo); free(t->ghi);
    free(t);
}

int64_t orc_tree_nn(const orc_tree *t) { return t->nn; }
int64_t orc_tree_ng(const orc_tree *t) { return t->ng; }

int64_t orc_tree_get(const orc_tree *t, int what, void *dst, int64_t bytes)
{
    const void *src = NULL; int64_t sz = 0;
    size_t n = (size_t)t->n, nn = (size_t)t->nn, ng = (size_t)t->ng;
    float bb[6]; double L = t->L;
    switch (what) {
    case ORC_GET_KEYS: src = t->key; sz = 8 * n; break;
    case ORC_GET_PERM: src = t->perm; sz = 4 * n; break;
    case ORC_GET_KEYS_SORTED: src = t->key_s; sz = 8 * n; break;
    case ORC_GET_POS_SORTED: src = t->pos_s; sz = 16 * n; break;
    case ORC_GET_LEVEL: src = t->level; sz = nn; break;
    case ORC_GET_FIRST: src = t->first; sz = 4 * nn; break;
    case ORC_GET_COUNT: src = t->count; sz = 4 * nn; break;
    case ORC_GET_CHILD: src = t->child; sz = 4 * nn; break;
    case ORC_GET_NCHILD: src = t->nchild; sz = nn; break;
    case ORC_GET_PARENT: src = t->parent; sz = 4 * nn; break;
    case ORC_GET_LEVEL_OFFSET: src = t->level_offset; sz = 4 * (MAXLEVEL + 2); break;
    case ORC_GET_COM_M: src = t->com_m; sz = 16 * nn; break;
    case ORC_GET_ROPEN2: src = t->ropen2; sz = 4 * nn; break;
    case ORC_GET_NLO: src = t->nlo; sz = 12 * nn; break;
    case ORC_GET_NHI: src = t->nhi; sz = 12 * nn; break;
    case ORC_GET_M64: src = t->M; sz = 8 * nn; break;
    case ORC_GET_C64: src = t->C; sz = 24 * nn; break;
    case ORC_GET_B2: src = t->B2; sz = 8 * nn; break;
    case ORC_GET_BMAX: src = t->bmax; sz = 8 * nn; break;
    case ORC_GET_GFIRST: src = t->gfirst; sz = 4 * ng; break;
    case ORC_GET_GCOUNT: src = t->gcount; sz = 4 * ng; break;
    case ORC_GET_GLO: src = t->glo; sz = 12 * ng; break;
    case ORC_GET_GHI: src = t->ghi; sz = 12 * ng; break;
    case ORC_GET_BBOX: for (int a = 0; a < 3; a++) { bb[a] = t->lo[a]; bb[3 + a] = t->hi[a]; }
        src = bb; sz = 24; break;
    case ORC_GET_ROOT_L: src = &L; sz = 8; break;
    default: return -1;
    }
    if (bytes < sz) return -1;
    memcpy(dst, src, (size_t)sz);
    return sz;
}

/* ------------------------------------------------------------------ T12 walk tests */
/* PAPER.md:66 "If r_b > r_ij ... we further visit ... else we add the force from the cell";
 * PAPER.md:107-109 Eq. 11 (minimum over the sinks sharing the walk; R18: group box to COM);
 * rule (b) of north_star (R19): a cell whose tight box comes within r_out of the group box is
 * opened; "cut-off the tree traversal for distant cells" in the hard walk.
 * All arithmetic here is fp32, one rounding per operation. */
static float fmax0(float a, float b) { float m = a > b ? a : b; return m > 0.0f ? m : 0.0f; }

static float dist2_box_com(const orc_tree *t, int64_t g, int64_t k)
{
    float e[3];
    for (int a = 0; a < 3; a++) {
        float c = t->com_m[4 * k + a];
        float u = t->glo[3 * g + a] - c;
        float w = c - t->ghi[3 * g + a];
        e[a] = fmax0(u, w);
    }
    float xx = e[0] * e[0], yy = e[1] * e[1], zz = e[2] * e[2];
    float s = xx + yy;
    return s + zz;
}

static float dist2_box_box(const orc_tree *t, int64_t g, int64_t k)
{
    float e[3];
    for (int a = 0; a < 3; a++) {
        float u = t->nlo[3 * k + a] - t->ghi[3 * g + a];
        float w = t->glo[3 * g + a] - t->nhi[3 * k + a];
        e[a] = fmax0(u, w);
    }
    float xx = e[0] * e[0], yy = e[1] * e[1], zz = e[2] * e[2];
    float s = xx + yy;
    return s + zz;
}

/* T13 with hard_cut = 1 (R30): is particle j (sorted order) within r_out of the box of group g?
 * the hard force acts only within R_2 ("cut-off").  Every sink of the group lies in
 * the group box, so a particle at least r_out away from the box has K = 0 for all of them.  fp32, one
 * rounding per operation, strict "<" like rule (b). */
static int in_cut(const orc_tree *t, int64_t g, uint32_t j)
{
    float e[3];
    for (int a = 0; a < 3; a++) {
        float x = t->pos_s[4 * (size_t)j + a];
        float u = t->glo[3 * g + a] - x;
        float w = x - t->ghi[3 * g + a];
        e[a] = fmax0(u, w);
    }
    float xx = e[0] * e[0], yy = e[1] * e[1], zz = e[2] * e[2];
    float s = xx + yy;
    float d2 = s + zz;
    float rout = t->p.r_out;
    return d2 < rout * rout;
}

/* T13.  Visits the tree for group g; calls back for accepted cells and opened leaves. */
typedef struct {
    uint32_t *cells; uint8_t *cellhard; int64_t ncells, cap_cells;
    uint32_t *leaves; uint8_t *leafhard; int64_t nleaves, cap_leaves;
    int64_t npart, nhard;
} walk_out;

static void push_cell(walk_out *w, uint32_t k, int hard)
{
    if (w->cells) {
        if (w->ncells == w->cap_cells) { w->cap_cells = w->cap_cells ? 2 * w->cap_cells : 1024;
            w->cells = (uint32_t *)realloc(w->cells, 4 * (size_t)w->cap_cells);
            w->cellhard = (uint8_t *)realloc(w->cellhard, (size_t)w->cap_cells); }
        w->cells[w->ncells] = k; w->cellhard[w->ncells] = (uint8_t)hard;
    }
    w->ncells++;
    if (hard) w->nhard += 1;
}
static void push_leaf(walk_out *w, uint32_t k, int hard, uint32_t count, uint32_t count_hard)
{
    if (w->leaves) {
        if (w->nleaves == w->cap_leaves) { w->cap_leaves = w->cap_leaves ? 2 * w->cap_leaves : 1024;
            w->leaves = (uint32_t *)realloc(w->leaves, 4 * (size_t)w->cap_leaves);
            w->leafhard = (uint8_t *)realloc(w->leafhard, (size_t)w->cap_leaves); }
        w->leaves[w->nleaves] = k; w->leafhard[w->nleaves] = (uint8_t)hard;
    }
    w->nleaves++;
    w->npart += count;
    if (hard) w->nhard += count_hard;
}

static void walk_group(const orc_tree *t, int mode, int64_t g, walk_out *w, int keep)
{
    float rout = t->p.r_out;
    float rout2 = rout * rout;
    int64_t scap = 256, sp = 0;
    uint32_t *stack = (uint32_t *)malloc(4 * (size_t)scap);
    w->ncells = w->nleaves = w->npart = w->nhard = 0;
    if (keep) {
        if (!w->cells) { w->cap_cells = 1024; w->cells = (uint32_t *)malloc(4 * 1024); w->cellhard = (uint8_t *)malloc(1024); }
        if (!w->leaves) { w->cap_leaves = 1024; w->leaves = (uint32_t *)malloc(4 * 1024); w->leafhard = (uint8_t *)malloc(1024); }
    }
    stack[sp++] = 0;
    while (sp > 0) {
        uint32_t k = stack[--sp];
        float d2b = dist2_box_box(t, g, k);
        int near = d2b < rout2;
        int open;
        /* hard_tree ("we use the tree algorithm ... for both of soft and hard
         * forces", "we can cut-off the tree traversal for distant cells"): the hard walk applies the
         * MAC too and an accepted cell within r_out contributes K(r_COM) F_COM; the soft walk is the
         * plain MAC walk (no rule (b)) whose cells within r_out carry 1 - K(r_COM). */
        int tree = t->p.hard_tree && mode != ORC_MODE_NORMAL;
        if (mode == ORC_MODE_HARD) {
            if (!near) continue;                                       /* discarded */
            open = tree ? (dist2_box_com(t, g, k) < t->ropen2[k]) : 1;
        } else {
            float d2a = dist2_box_com(t, g, k);
            int mac_open = d2a < t->ropen2[k];
            open = (mode == ORC_MODE_NORMAL || tree) ? mac_open : (mac_open || near);
        }
        if (!open) { push_cell(w, k, tree && near); continue; }
        if (t->child[k] == NOCHILD) {
            int hard = (mode == ORC_MODE_NORMAL) ? 0 : near;
            uint32_t nh = t->count[k];
            if (hard && t->p.hard_cut) {                               /* R30: particle-level cut */
                nh = 0;
                for (uint32_t j = t->first[k]; j < t->first[k] + t->count[k]; j++) nh += (uint32_t)in_cut(t, g, j);
            }
            push_leaf(w, k, hard, t->count[k], nh);
            continue;
        }
        if (sp + 8 > scap) { scap *= 2; stack = (uint32_t *)realloc(stack, 4 * (size_t)scap); }
        for (int q = (int)t->nchild[k] - 1; q >= 0; q--) stack[sp++] = t->child[k] + (uint32_t)q;
    }
    free(stack);
}

void orc_walk_counts(const orc_tree *t, int mode, uint32_t *ncell, uint32_t *npart, uint32_t *nhard)
{
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t g = 0; g < t->ng; g++) {
        walk_out w; memset(&w, 0, sizeof w);
        walk_group(t, mode, g, &w, 0);
        ncell[g] = (uint32_t)w.ncells; npart[g] = (uint32_t)w.npart; nhard[g] = (uint32_t)w.nhard;
    }
}

/* the same for the groups in gsel only: entry k of each output belongs to group gsel[k] */
void orc_walk_counts_sel(const orc_tree *t, int mode, int64_t ngsel, const int64_t *gsel,
                         uint32_t *ncell, uint32_t *npart, uint32_t *nhard)
{
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t k = 0; k < ngsel; k++) {
        walk_out w; memset(&w, 0, sizeof w);
        walk_group(t, mode, gsel[k], &w, 0);
        ncell[k] = (uint32_t)w.ncells; npart[k] = (uint32_t)w.npart; nhard[k] = (uint32_t)w.nhard;
    }
}

int orc_walk_lists(const orc_tree *t, int mode, int64_t g,
                   uint32_t *cells, int64_t cap_cells, int64_t *ncells,
                   uint32_t *parts, uint8_t *hard, int64_t cap_parts, int64_t *nparts)
{
    walk_out w; memset(&w, 0, sizeof w);
    walk_group(t, mode, g, &w, 1);
    int rc = 0;
    *ncells = w.ncells; *nparts = w.npart;
    if (w.ncells > cap_cells || w.npart > cap_parts) rc = -1;
    else {
        memcpy(cells, w.cells, 4 * (size_t)w.ncells);
        int64_t q = 0;
        for (int64_t l = 0; l < w.nleaves; l++) {
            uint32_t k = w.leaves[l];
            for (uint32_t j = t->first[k]; j < t->first[k] + t->count[k]; j++) {
                parts[q] = j;
                hard[q] = (uint8_t)(w.leafhard[l] && (!t->p.hard_cut || in_cut(t, g, j)));
                q++;
            }
        }
    }
    free(w.cells); free(w.cellhard); free(w.leaves); free(w.leafhard);
    return rc;
}

/* ------------------------------------------------------------------ virtual-domain LET counts */
/* SURVEY.md 8(f) rank 3.  The box is cut into P cuboid domains (the caller's
 * boxes, half-open [lo, hi) per axis).  For domain j the tree is walked as process j's neighbours
 * would walk their local trees to fill j's locally essential tree: a node wholly inside D_j is local;
 * otherwise it is opened when r_ib < r_b (Eq. 14; r_ib = distance from its centre of mass to D_j, r_b
 * the opening radius of T10) or when part of it lies inside D_j, else it is sent as ONE cell; an
 * opened leaf sends its particles that lie outside D_j.  N_soft counts what is sent.  The hard LET
 * (Eq. 15) follows the same walk but drops every node with r_ib >= R_2 + b_max and every particle
 * farther than R_2 from D_j; N_hard counts what is left.  Decisions in fp32, one rounding per
 * operation, like T12.  out[3 j .. 3 j + 2] = N_local, N_soft, N_hard. */
void orc_let_count(const orc_tree *t, int64_t ndom, const float *boxes, uint64_t *out)
{
    float R2 = t->p.r_out, R22 = R2 * R2;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t j = 0; j < ndom; j++) {
        const float *lo = boxes + 6 * j, *hi = lo + 3;
        uint64_t nloc = 0, nsoft = 0, nhard = 0;
        int64_t scap = 1024, sp = 0;
        uint32_t *stack = (uint32_t *)malloc(4 * (size_t)scap);
        stack[sp++] = 0u | 0x80000000u;                            /* bit 31: still on the hard walk */
        while (sp > 0) {
            uint32_t ent = stack[--sp], k = ent & 0x7FFFFFFFu;
            int alive = (ent >> 31) != 0;
            int inside = 1, touches = 1;
            float e[3];
            for (int a = 0; a < 3; a++) {
                float nl = t->nlo[3 * (size_t)k + a], nh = t->nhi[3 * (size_t)k + a], c = t->com_m[4 * (size_t)k + a];
                inside = inside && nl >= lo[a] && nh < hi[a];
                touches = touches && nh >= lo[a] && nl < hi[a];
                float u = lo[a] - c, w = c - hi[a];
                e[a] = fmax0(u, w);
            }
            if (inside) { nloc += t->count[k]; continue; }
            float xx = e[0] * e[0], yy = e[1] * e[1], zz = e[2] * e[2];
            float s2 = xx + yy, r2 = s2 + zz;
            float cut = R2 + (float)t->bmax[k], cut2 = cut * cut;
            int hard = alive && r2 < cut2;                         /* Eq. 15 */
            int open = r2 < t->ropen2[k] || touches;               /* Eq. 14 */
            if (!open) { nsoft++; nhard += (uint64_t)hard; continue; }
            if (t->child[k] == NOCHILD) {
                for (uint32_t q = t->first[k]; q < t->first[k] + t->count[k]; q++) {
                    const float *x = t->pos_s + 4 * (size_t)q;
                    int in = 1; float d[3];
                    for (int a = 0; a < 3; a++) {
                        in = in && x[a] >= lo[a] && x[a] < hi[a];
                        float u = lo[a] - x[a], w = x[a] - hi[a];
                        d[a] = fmax0(u, w);
                    }
                    if (in) { nloc++; continue; }
                    float px = d[0] * d[0], py = d[1] * d[1], pz = d[2] * d[2];
                    float ps = px + py, d2 = ps + pz;
                    nsoft++;
                    if (hard && d2 < R22) nhard++;
                }
                continue;
            }
            if (sp + 8 > scap) { scap *= 2; stack = (uint32_t *)realloc(stack, 4 * (size_t)scap); }
            for (int q = (int)t->nchild[k] - 1; q >= 0; q--)
                stack[sp++] = (t->child[k] + (uint32_t)q) | (hard ? 0x80000000u : 0u);
        }
        free(stack);
        out[3 * j] = nloc; out[3 * j + 1] = nsoft; out[3 * j + 2] = nhard;
    }
}

/* ------------------------------------------------------------------ T14 forces */
/* PAPER.md:35 Eq. 2 (R2: m_j is the source mass); Eq. 7-9 (R3) split by K; "we get
 * the force of a sink particle by summing forces from source cells and particles".  Cells are
 * plain monopoles (R24).  fp64 from the fp32-stored positions, masses and COMs; G once (R26). */
static void pair(const double xi[3], const float *src, double eps2, double *dx, double *s, double *r2)
{
    dx[0] = (double)src[0] - xi[0];
    dx[1] = (double)src[1] - xi[1];
    dx[2] = (double)src[2] - xi[2];
    *r2 = dx[0] * dx[0] + dx[1] * dx[1] + dx[2] * dx[2];
    double d2 = *r2 + eps2;
    *s = 1.0 / (d2 * sqrt(d2));
}

void orc_forces(const orc_tree *t, int mode, int64_t ngsel, const int64_t *gsel,
                double *a_soft, double *a_hard, double *inter_soft, double *inter_hard)
{
    int64_t ngrp = ngsel > 0 ? ngsel : t->ng;
    double eps2 = (double)t->p.eps * (double)t->p.eps;
    double G = (double)t->p.G, rin = (double)t->p.r_in, rout = (double)t->p.r_out;
    double isoft = 0.0, ihard = 0.0;
#pragma omp parallel for schedule(dynamic, 4) reduction(+ : isoft, ihard)
    for (int64_t gi = 0; gi < ngrp; gi++) {
        int64_t g = ngsel > 0 ? gsel[gi] : gi;
        walk_out w; memset(&w, 0, sizeof w);
        walk_group(t, mode, g, &w, 1);
        uint32_t gf = t->gfirst[g], gc = t->gcount[g];
        if (mode != ORC_MODE_HARD) isoft += (double)gc * (double)(w.ncells + w.npart);
        if (mode != ORC_MODE_NORMAL) ihard += (double)gc * (double)w.nhard;
        for (uint32_t i = gf; i < gf + gc; i++) {
            double xi[3] = { (double)t->pos_s[4 * (size_t)i], (double)t->pos_s[4 * (size_t)i + 1], (double)t->pos_s[4 * (size_t)i + 2] };
            double as[3] = { 0, 0, 0 }, ah[3] = { 0, 0, 0 };
            for (int64_t c = 0; c < w.ncells; c++) {                  /* cells */
                const float *src = t->com_m + 4 * (size_t)w.cells[c];
                double dx[3], s, r2;
                pair(xi, src, eps2, dx, &s, &r2);
                double ms = (double)src[3] * s;
                if (w.cellhard[c]) {                                   /* hard_tree: K-weighted cell */
                    double K = orc_K(sqrt(r2), rin, rout, t->p.kfunc);
                    double wh = K * ms, ws = (1.0 - K) * ms;
                    ah[0] += wh * dx[0]; ah[1] += wh * dx[1]; ah[2] += wh * dx[2];
                    if (mode == ORC_MODE_HYBRID) { as[0] += ws * dx[0]; as[1] += ws * dx[1]; as[2] += ws * dx[2]; }
                } else {
                    as[0] += ms * dx[0]; as[1] += ms * dx[1]; as[2] += ms * dx[2];
                }
            }
            for (int64_t l = 0; l < w.nleaves; l++) {                 /* particles */
                uint32_t k = w.leaves[l];
                int hard = w.leafhard[l];
                for (uint32_t j = t->first[k]; j < t->first[k] + t->count[k]; j++) {
                    if (j == i) continue;                              /* R22 */
                    const float *src = t->pos_s + 4 * (size_t)j;
                    double dx[3], s, r2;
                    pair(xi, src, eps2, dx, &s, &r2);
                    double ms = (double)src[3] * s;
                    if (mode == ORC_MODE_NORMAL) {
                        as[0] += ms * dx[0]; as[1] += ms * dx[1]; as[2] += ms * dx[2];
                    } else {
                        double K = orc_K(sqrt(r2), rin, rout, t->p.kfunc);
                        if (mode == ORC_MODE_HYBRID) {
                            double ws = (1.0 - K) * ms;
                            as[0] += ws * dx[0]; as[1] += ws * dx[1]; as[2] += ws * dx[2];
                        }
                        if (hard && (!t->p.hard_cut || in_cut(t, g, j))) {
                            double wh = K * ms;
                            ah[0] += wh * dx[0]; ah[1] += wh * dx[1]; ah[2] += wh * dx[2];
                        }
                    }
                }
            }
            if (mode != ORC_MODE_HARD && a_soft) for (int a = 0; a < 3; a++) a_soft[3 * (size_t)i + a] = G * as[a];
            if (mode != ORC_MODE_NORMAL && a_hard) for (int a = 0; a < 3; a++) a_hard[3 * (size_t)i + a] = G * ah[a];
            if (mode == ORC_MODE_NORMAL && a_hard) for (int a = 0; a < 3; a++) a_hard[3 * (size_t)i + a] = 0.0;
        }
        free(w.cells); free(w.cellhard); free(w.leaves); free(w.leafhard);
    }
    if (inter_soft) *inter_soft = isoft;
    if (inter_hard) *inter_hard = ihard;
}

/* ------------------------------------------------------------------ brute force, Eq. 1-2 */
/* a_i = sum_{j != i} F_ij (R1); split per pair by Eq. 7-9. */
void orc_direct(int64_t n, const float *pos4, float Gf, float epsf, float r_in, float r_out,
                int kfunc, int64_t nsel, const int64_t *sel,
                double *a_tot, double *a_hard, double *a_soft)
{
    double eps2 = (double)epsf * (double)epsf, G = (double)Gf;
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t si = 0; si < nsel; si++) {
        int64_t i = sel ? sel[si] : si;
        double xi[3] = { (double)pos4[4 * i], (double)pos4[4 * i + 1], (double)pos4[4 * i + 2] };
        double at[3] = { 0, 0, 0 }, ah[3] = { 0, 0, 0 }, as[3] = { 0, 0, 0 };
        for (int64_t j = 0; j < n; j++) {
            if (j == i) continue;
            double dx[3], s, r2;
            pair(xi, pos4 + 4 * j, eps2, dx, &s, &r2);
            double ms = (double)pos4[4 * j + 3] * s;
            double K = (r_out > r_in) ? orc_K(sqrt(r2), (double)r_in, (double)r_out, kfunc) : 0.0;
            for (int a = 0; a < 3; a++) {
                double f = ms * dx[a];
                at[a] += f; ah[a] += K * f; as[a] += (1.0 - K) * f;
            }
        }
        for (int a = 0; a < 3; a++) {
            if (a_tot) a_tot[3 * si + a] = G * at[a];
            if (a_hard) a_hard[3 * si + a] = G * ah[a];
            if (a_soft) a_soft[3 * si + a] = G * as[a];
        }
    }
}

/* ------------------------------------------------------------------ T16 step (R21) */
/* PAPER.md:42-45 Eq. 3-4 kick/drift; "Delta t_s = n Delta t_h ... one soft-step and
 * n-1 hard-steps".  KDK form:  v += dt_s/2 a_soft; n x { v += dt_h/2 a_hard; x += dt_h v;
 * rebuild tree; a_hard (and a_soft on the last repeat); v += dt_h/2 a_hard }; v += dt_s/2 a_soft.
 * split = 0 (R29): n x { v += dt_h/2 a; x += dt_h v; a = normal tree; v += dt_h/2 a }, a kept
 * in a_soft, a_hard = 0. */
static int eval_acc(int64_t n, const double *x, const float *m, const orc_params *p, int mode,
                    double *a_soft, double *a_hard)
{
    float *pos4 = (float *)malloc(16 * (size_t)n);
    for (int64_t i = 0; i < n; i++) {
        pos4[4 * i] = (float)x[3 * i]; pos4[4 * i + 1] = (float)x[3 * i + 1];
        pos4[4 * i + 2] = (float)x[3 * i + 2]; pos4[4 * i + 3] = m[i];
    }
    orc_tree *t = orc_tree_build(n, pos4, p);
    free(pos4);
    if (!t) return -1;
    double *s = (double *)calloc(3 * (size_t)n, 8), *h = (double *)calloc(3 * (size_t)n, 8);
    orc_forces(t, mode, 0, NULL, s, h, NULL, NULL);
    for (int64_t j = 0; j < n; j++) {
        size_t i = t->perm[j];
        for (int a = 0; a < 3; a++) {
            if (mode != ORC_MODE_HARD) a_soft[3 * i + a] = s[3 * j + a];
            if (mode != ORC_MODE_NORMAL) a_hard[3 * i + a] = h[3 * j + a];
            else a_hard[3 * i + a] = 0.0;
        }
    }
    free(s); free(h);
    orc_tree_free(t);
    return 0;
}

int orc_step(int64_t n, double *x, double *v, const float *m, const orc_params *p,
             int32_t ncycles, double *a_soft, double *a_hard, int acc_valid)
{
    if (p->n_sub < 1) return -1;
    double dts = (double)p->dt_soft, dth = dts / (double)p->n_sub;
    int split = p->split != 0;
    if (!acc_valid)
        if (eval_acc(n, x, m, p, split ? ORC_MODE_HYBRID : ORC_MODE_NORMAL, a_soft, a_hard)) return -1;
    for (int32_t c = 0; c < ncycles; c++) {
        if (split) for (int64_t i = 0; i < 3 * n; i++) v[i] += 0.5 * dts * a_soft[i];
        for (int32_t k = 0; k < p->n_sub; k++) {
            const double *af = split ? a_hard : a_soft;
            for (int64_t i = 0; i < 3 * n; i++) v[i] += 0.5 * dth * af[i];
            for (int64_t i = 0; i < 3 * n; i++) x[i] += dth * v[i];
            int mode = !split ? ORC_MODE_NORMAL : (k == p->n_sub - 1 ? ORC_MODE_HYBRID : ORC_MODE_HARD);
            if (eval_acc(n, x, m, p, mode, a_soft, a_hard)) return -1;
            for (int64_t i = 0; i < 3 * n; i++) v[i] += 0.5 * dth * af[i];
        }
        if (split) for (int64_t i = 0; i < 3 * n; i++) v[i] += 0.5 * dts * a_soft[i];
    }
    return 0;
}

/* ------------------------------------------------------------------ energy (R23) */
/* PAPER.md:174 "error in total energy of the system that is the sum of kinetic and potential
 * energy".  E = sum 1/2 m v^2 - sum_{i<j} G m_i m_j / sqrt(r_ij^2 + eps^2). */
void orc_energy(int64_t n, const double *x, const double *v, const float *m, float Gf, float epsf,
                double *kin, double *pot)
{
    double eps2 = (double)epsf * (double)epsf, K = 0.0, W = 0.0;
    for (int64_t i = 0; i < n; i++)
        K += 0.5 * (double)m[i] * (v[3 * i] * v[3 * i] + v[3 * i + 1] * v[3 * i + 1] + v[3 * i + 2] * v[3 * i + 2]);
#pragma omp parallel for schedule(dynamic, 64) reduction(+ : W)
    for (int64_t i = 0; i < n; i++) {
        double w = 0.0;
        for (int64_t j = i + 1; j < n; j++) {
            double dx = x[3 * j] - x[3 * i], dy = x[3 * j + 1] - x[3 * i + 1], dz = x[3 * j + 2] - x[3 * i + 2];
            w += (double)m[j] / sqrt(dx * dx + dy * dy + dz * dz + eps2);
        }
        W += (double)m[i] * w;
    }
    *kin = K; *pot = -(double)Gf * W;
}
