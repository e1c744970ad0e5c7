/*
 * treegen.c -- host-side INPUT GENERATOR (harness only, never timed, not on the hot path).
 *
 * Re-creates, for synthetic particle sets, the inputs the gravity hot path consumes:
 * a tree with buckets (binary tree, cells split along the longest axis
 * into equal volumes, leaves of up to b particles, particles and cells "in a
 * hierarchically sorted order"), per-cell centre of mass, b_max, bounding box and raw
 * moments to 4th order about the centre of mass (L69, L71), and per-bucket P-P / P-C
 * interaction lists from an opening-angle acceptance test (L65-69; reading A6).
 *
 * It holds none of the method's evaluation arithmetic (no force, no potential, no
 * expansion): both the fp64 oracle and the CUDA library receive its output arrays.
 *
 * The tree is built over particles already sorted by a 63-bit Morton key of a CUBIC root
 * box (done in numpy by the caller).  Splitting a cube along its longest axis at the
 * midpoint cycles x, y, z, so the paper's binary tree is the bit-by-bit refinement of that
 * key; the octree (BASELINE.json config 1) takes three bits per level.
 *
 * Cells are numbered in depth-first pre-order; subtree_end[c] is the index one past the
 * last descendant of c, so the children of c are c+1, subtree_end[c+1], ... and a list
 * walk needs no stack.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define REC 36 /* floats per canonical cell record (include/pkdg.h) */

typedef struct {
    int64_t n;          /* particles */
    const uint64_t *key; /* sorted keys (borrowed during build only) */
    int mode;           /* 0 = octree (3 bits per level), 1 = binary (1 bit per level) */
    int cap;            /* bucket capacity */
    int64_t ncell, cellcap;
    int32_t *first, *count, *end, *isleaf;
    int64_t nleaf;
} tg_tree;

static void grow(tg_tree *t) {
    if (t->ncell < t->cellcap) return;
    t->cellcap = t->cellcap ? t->cellcap * 2 : 1024;
    t->first = realloc(t->first, sizeof(int32_t) * t->cellcap);
    t->count = realloc(t->count, sizeof(int32_t) * t->cellcap);
    t->end = realloc(t->end, sizeof(int32_t) * t->cellcap);
    t->isleaf = realloc(t->isleaf, sizeof(int32_t) * t->cellcap);
}

/* first index in [lo,hi) whose key, shifted right by sh and masked, is >= v (keys sorted) */
static int64_t lower(const uint64_t *key, int64_t lo, int64_t hi, int sh, uint64_t mask, uint64_t v) {
    while (lo < hi) {
        int64_t mid = (lo + hi) >> 1;
        if (((key[mid] >> sh) & mask) < v) lo = mid + 1; else hi = mid;
    }
    return lo;
}

static void build(tg_tree *t, int64_t lo, int64_t hi, int lvl) {
    grow(t);
    int64_t c = t->ncell++;
    t->first[c] = (int32_t)lo;
    t->count[c] = (int32_t)(hi - lo);
    int step = t->mode == 0 ? 3 : 1;
    int nway = 1 << step;
    if (hi - lo <= t->cap) {
        t->isleaf[c] = 1;
        t->nleaf++;
        t->end[c] = (int32_t)t->ncell;
        return;
    }
    t->isleaf[c] = 0;
    int64_t cut[9];
    for (;;) {
        if (lvl + step > 63) { /* key bits exhausted (coincident points): split by index */
            cut[0] = lo; cut[1] = (lo + hi) / 2; cut[2] = hi;
            nway = 2;
            break;
        }
        int sh = 63 - lvl - step;
        cut[0] = lo;
        for (int o = 1; o < nway; ++o) cut[o] = lower(t->key, lo, hi, sh, (uint64_t)nway - 1, (uint64_t)o);
        cut[nway] = hi;
        int nonempty = 0;
        for (int o = 0; o < nway; ++o) nonempty += cut[o + 1] > cut[o];
        if (nonempty > 1) break;
        lvl += step; /* all particles in one child volume: shrink without making a cell */
    }
    for (int o = 0; o < nway; ++o)
        if (cut[o + 1] > cut[o]) build(t, cut[o], cut[o + 1], lvl + step);
    t->end[c] = (int32_t)t->ncell;
}

tg_tree *tg_tree_build(int64_t n, const uint64_t *sorted_keys, int mode, int cap) {
    tg_tree *t = calloc(1, sizeof(tg_tree));
    t->n = n; t->key = sorted_keys; t->mode = mode; t->cap = cap;
    if (n > 0) build(t, 0, n, 0);
    t->key = NULL;
    return t;
}

int64_t tg_tree_ncells(const tg_tree *t) { return t->ncell; }
int64_t tg_tree_nleaves(const tg_tree *t) { return t->nleaf; }

void tg_tree_free(tg_tree *t) {
    if (!t) return;
    free(t->first); free(t->count); free(t->end); free(t->isleaf); free(t);
}

/* Raw moments of particles [lo,hi) about the fp32-rounded centre of mass, in fp64, stored
 * as fp32 in the canonical record layout; bounding box of the fp32 coordinates. */
static void cell_record(const float *xyzm, int64_t lo, int64_t hi, float *rec, float *bblo,
                        float *bbhi, int par) {
    double m = 0, cx = 0, cy = 0, cz = 0;
    float l0 = INFINITY, l1 = INFINITY, l2 = INFINITY, h0 = -INFINITY, h1 = -INFINITY, h2 = -INFINITY;
#pragma omp parallel for reduction(+ : m, cx, cy, cz) reduction(min : l0, l1, l2) reduction(max : h0, h1, h2) if (par)
    for (int64_t j = lo; j < hi; ++j) {
        const float *p = xyzm + 4 * j;
        double mj = p[3];
        m += mj; cx += mj * p[0]; cy += mj * p[1]; cz += mj * p[2];
        l0 = fminf(l0, p[0]); l1 = fminf(l1, p[1]); l2 = fminf(l2, p[2]);
        h0 = fmaxf(h0, p[0]); h1 = fmaxf(h1, p[1]); h2 = fmaxf(h2, p[2]);
    }
    float com[3];
    if (m > 0) { com[0] = (float)(cx / m); com[1] = (float)(cy / m); com[2] = (float)(cz / m); }
    else { com[0] = 0.5f * (l0 + h0); com[1] = 0.5f * (l1 + h1); com[2] = 0.5f * (l2 + h2); }
    double M[31];
    for (int q = 0; q < 31; ++q) M[q] = 0;
    double b2 = 0;
#pragma omp parallel for reduction(+ : M[:31]) reduction(max : b2) if (par)
    for (int64_t j = lo; j < hi; ++j) {
        const float *p = xyzm + 4 * j;
        double s[3] = {(double)p[0] - com[0], (double)p[1] - com[1], (double)p[2] - com[2]};
        double mj = p[3];
        double d2 = s[0] * s[0] + s[1] * s[1] + s[2] * s[2];
        if (d2 > b2) b2 = d2;
        double pw[3][5];
        for (int d = 0; d < 3; ++d) {
            pw[d][0] = 1;
            for (int e = 1; e < 5; ++e) pw[d][e] = pw[d][e - 1] * s[d];
        }
        int q = 0;
        for (int n = 2; n <= 4; ++n)
            for (int a = n; a >= 0; --a)
                for (int b = n - a; b >= 0; --b) M[q++] += mj * pw[0][a] * pw[1][b] * pw[2][n - a - b];
    }
    rec[0] = com[0]; rec[1] = com[1]; rec[2] = com[2]; rec[3] = (float)m;
    for (int q = 0; q < 31; ++q) rec[4 + q] = (float)M[q];
    rec[35] = (float)sqrt(b2);
    bblo[0] = l0; bblo[1] = l1; bblo[2] = l2; bbhi[0] = h0; bbhi[1] = h1; bbhi[2] = h2;
}

/* Fill caller-allocated arrays: per cell first/count/end/isleaf, 36-float records, bounding
 * boxes; per leaf (in pre-order = particle order) its cell index. */
void tg_tree_export(const tg_tree *t, const float *xyzm, int32_t *first, int32_t *count, int32_t *end,
                    int32_t *isleaf, float *rec, float *bblo, float *bbhi, int32_t *leaf_cell) {
    int64_t nc = t->ncell;
    memcpy(first, t->first, sizeof(int32_t) * nc);
    memcpy(count, t->count, sizeof(int32_t) * nc);
    memcpy(end, t->end, sizeof(int32_t) * nc);
    memcpy(isleaf, t->isleaf, sizeof(int32_t) * nc);
    int64_t nl = 0;
    for (int64_t c = 0; c < nc; ++c)
        if (t->isleaf[c]) leaf_cell[nl++] = (int32_t)c;
    const int64_t BIG = 1 << 18;
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t c = 0; c < nc; ++c)
        if (t->count[c] < BIG)
            cell_record(xyzm, t->first[c], (int64_t)t->first[c] + t->count[c], rec + REC * c,
                        bblo + 3 * c, bbhi + 3 * c, 0);
    for (int64_t c = 0; c < nc; ++c)
        if (t->count[c] >= BIG)
            cell_record(xyzm, t->first[c], (int64_t)t->first[c] + t->count[c], rec + REC * c,
                        bblo + 3 * c, bbhi + 3 * c, 1);
}

/* ------------------------------------------------------------------------------------------
 * Interaction lists for buckets [b0,b1) (bucket b is the leaf cell leaf_cell[b]).
 * Walk from the root in pre-order; for source cell k and sink bucket B (reading A6):
 *   k is a P-C source  iff  k != B, count[k] >= 2,
 *                           |COM_B - COM_k| > b_max,B + b_max,k / theta   and
 *                           gap(bbox_B, bbox_k) >= 2 eps;
 *   else if k is a leaf: its particles are P-P sources (including B's own particles);
 *   else k is opened.
 * Every particle is therefore covered exactly once per bucket.
 * ---------------------------------------------------------------------------------------- */
typedef struct { int32_t *v; int64_t n, cap; } ivec;
static inline void push(ivec *a, int32_t x) {
    if (a->n == a->cap) { a->cap = a->cap ? a->cap * 2 : 4096; a->v = realloc(a->v, sizeof(int32_t) * a->cap); }
    a->v[a->n++] = x;
}

typedef struct {
    int64_t b0, b1, nblk;
    int64_t blk;      /* buckets per block */
    ivec *pp, *pc;    /* per block */
    int64_t *pp_len, *pc_len; /* per bucket (b - b0) */
} tg_lists;

tg_lists *tg_lists_build(int64_t ncell, const int32_t *first, const int32_t *count, const int32_t *end,
                         const int32_t *isleaf, const float *rec, const float *bblo, const float *bbhi,
                         const int32_t *leaf_cell, int64_t b0, int64_t b1, double theta, double eps) {
    tg_lists *L = calloc(1, sizeof(tg_lists));
    L->b0 = b0; L->b1 = b1; L->blk = 512;
    L->nblk = (b1 - b0 + L->blk - 1) / L->blk;
    L->pp = calloc(L->nblk ? L->nblk : 1, sizeof(ivec));
    L->pc = calloc(L->nblk ? L->nblk : 1, sizeof(ivec));
    L->pp_len = calloc(b1 - b0 + 1, sizeof(int64_t));
    L->pc_len = calloc(b1 - b0 + 1, sizeof(int64_t));
    double gap_min2 = 4.0 * eps * eps;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t ib = 0; ib < L->nblk; ++ib) {
        ivec *pp = &L->pp[ib], *pc = &L->pc[ib];
        int64_t e1 = b0 + (ib + 1) * L->blk; if (e1 > b1) e1 = b1;
        for (int64_t b = b0 + ib * L->blk; b < e1; ++b) {
            int64_t cb = leaf_cell[b];
            const float *rb = rec + REC * cb;
            double bx = rb[0], by = rb[1], bz = rb[2], bmaxB = rb[35];
            const float *lob = bblo + 3 * cb, *hib = bbhi + 3 * cb;
            int64_t npp0 = pp->n, npc0 = pc->n;
            int64_t k = 0;
            while (k < ncell) {
                int accept = 0;
                if (k != cb && count[k] >= 2) {
                    const float *rk = rec + REC * k;
                    double dx = bx - rk[0], dy = by - rk[1], dz = bz - rk[2];
                    double d = sqrt(dx * dx + dy * dy + dz * dz);
                    if (d > bmaxB + (double)rk[35] / theta) {
                        const float *lok = bblo + 3 * k, *hik = bbhi + 3 * k;
                        double g2 = 0;
                        for (int a = 0; a < 3; ++a) {
                            double g = 0;
                            if ((double)lok[a] - hib[a] > g) g = (double)lok[a] - hib[a];
                            if ((double)lob[a] - hik[a] > g) g = (double)lob[a] - hik[a];
                            g2 += g * g;
                        }
                        accept = g2 >= gap_min2;
                    }
                }
                if (accept) { push(pc, (int32_t)k); k = end[k]; }
                else if (isleaf[k]) {
                    for (int32_t j = 0; j < count[k]; ++j) push(pp, first[k] + j);
                    k = end[k];
                } else k = k + 1;
            }
            L->pp_len[b - b0] = pp->n - npp0;
            L->pc_len[b - b0] = pc->n - npc0;
        }
    }
    return L;
}

void tg_lists_totals(const tg_lists *L, int64_t *npp, int64_t *npc) {
    int64_t a = 0, c = 0;
    for (int64_t i = 0; i < L->nblk; ++i) { a += L->pp[i].n; c += L->pc[i].n; }
    *npp = a; *npc = c;
}

/* Copy into caller-allocated CSR arrays (offsets have b1-b0+1 entries, starting at 0) and free. */
void tg_lists_export_free(tg_lists *L, int64_t *pp_off, int32_t *pp_idx, int64_t *pc_off, int32_t *pc_idx) {
    int64_t nb = L->b1 - L->b0;
    pp_off[0] = 0; pc_off[0] = 0;
    for (int64_t b = 0; b < nb; ++b) {
        pp_off[b + 1] = pp_off[b] + L->pp_len[b];
        pc_off[b + 1] = pc_off[b] + L->pc_len[b];
    }
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t ib = 0; ib < L->nblk; ++ib) {
        int64_t b = ib * L->blk;
        if (L->pp[ib].n) memcpy(pp_idx + pp_off[b], L->pp[ib].v, sizeof(int32_t) * L->pp[ib].n);
        if (L->pc[ib].n) memcpy(pc_idx + pc_off[b], L->pc[ib].v, sizeof(int32_t) * L->pc[ib].n);
        free(L->pp[ib].v); free(L->pc[ib].v);
    }
    free(L->pp); free(L->pc); free(L->pp_len); free(L->pc_len); free(L);
}

/* ------------------------------------------------------------------------------------------
 * FMM-style lists for buckets [b0,b1): four lists per
 * sink bucket B.  Walking from the root in pre-order, for source cell k:
 *   C-C  iff  k != B, count[k] >= 2, |COM_B - COM_k| > 1.5 RO_B + RO_k (RO = b_max / theta, the paper's
 *             opening radii with its deliberate factor 1.5 on the sink) and gap(bbox_B, bbox_k) >= 2 eps;
 *   P-C  else iff reading A6 accepts k (|COM_B - COM_k| > b_max,B + RO_k, gap >= 2 eps, count >= 2);
 *   else a leaf is opened into its particles j ("with RO_source = 0", L69):
 *   C-P  iff  j is not in B, |COM_B - x_j| > 1.5 RO_B and gap(bbox_B, x_j) >= 2 eps;
 *   P-P  else;
 *   else k is opened.
 * Every particle is covered exactly once per bucket by the union of the four lists.
 * ---------------------------------------------------------------------------------------- */
typedef struct {
    int64_t b0, b1, nblk, blk;
    ivec *v[4];           /* per block: 0 = P-P, 1 = P-C, 2 = C-P, 3 = C-C */
    int64_t *len[4];      /* per bucket (b - b0) */
} tg_fmm;

tg_fmm *tg_fmm_build(int64_t ncell, const int32_t *first, const int32_t *count, const int32_t *end,
                     const int32_t *isleaf, const float *rec, const float *bblo, const float *bbhi,
                     const int32_t *leaf_cell, const float *xyzm, int64_t b0, int64_t b1, double theta, double eps) {
    tg_fmm *F = calloc(1, sizeof(tg_fmm));
    F->b0 = b0; F->b1 = b1; F->blk = 512;
    F->nblk = (b1 - b0 + F->blk - 1) / F->blk;
    for (int q = 0; q < 4; ++q) {
        F->v[q] = calloc(F->nblk ? F->nblk : 1, sizeof(ivec));
        F->len[q] = calloc(b1 - b0 + 1, sizeof(int64_t));
    }
    double gap_min2 = 4.0 * eps * eps;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t ib = 0; ib < F->nblk; ++ib) {
        ivec *v[4] = {&F->v[0][ib], &F->v[1][ib], &F->v[2][ib], &F->v[3][ib]};
        int64_t e1 = b0 + (ib + 1) * F->blk; if (e1 > b1) e1 = b1;
        for (int64_t b = b0 + ib * F->blk; b < e1; ++b) {
            int64_t cb = leaf_cell[b];
            const float *rb = rec + REC * cb;
            double bx = rb[0], by = rb[1], bz = rb[2], bmaxB = rb[35];
            const float *lob = bblo + 3 * cb, *hib = bbhi + 3 * cb;
            int64_t n0[4];
            for (int q = 0; q < 4; ++q) n0[q] = v[q]->n;
            int64_t k = 0;
            while (k < ncell) {
                int kind = 0; /* 0 none, 1 P-C, 3 C-C */
                if (k != cb && count[k] >= 2) {
                    const float *rk = rec + REC * k;
                    double dx = bx - rk[0], dy = by - rk[1], dz = bz - rk[2];
                    double d = sqrt(dx * dx + dy * dy + dz * dz);
                    const float *lok = bblo + 3 * k, *hik = bbhi + 3 * k;
                    double g2 = 0;
                    for (int a = 0; a < 3; ++a) {
                        double g = 0;
                        if ((double)lok[a] - hib[a] > g) g = (double)lok[a] - hib[a];
                        if ((double)lob[a] - hik[a] > g) g = (double)lob[a] - hik[a];
                        g2 += g * g;
                    }
                    if (g2 >= gap_min2) {
                        if (d > 1.5 * bmaxB / theta + (double)rk[35] / theta) kind = 3;
                        else if (d > bmaxB + (double)rk[35] / theta) kind = 1;
                    }
                }
                if (kind) { push(v[kind], (int32_t)k); k = end[k]; }
                else if (isleaf[k]) {
                    for (int32_t t = 0; t < count[k]; ++t) {
                        int32_t j = first[k] + t;
                        int cp = 0;
                        if (k != cb) {
                            const float *xj = xyzm + 4 * (int64_t)j;
                            double dx = bx - xj[0], dy = by - xj[1], dz = bz - xj[2];
                            double d = sqrt(dx * dx + dy * dy + dz * dz);
                            double g2 = 0;
                            for (int a = 0; a < 3; ++a) {
                                double g = 0;
                                if ((double)xj[a] - hib[a] > g) g = (double)xj[a] - hib[a];
                                if ((double)lob[a] - xj[a] > g) g = (double)lob[a] - xj[a];
                                g2 += g * g;
                            }
                            cp = d > 1.5 * bmaxB / theta && g2 >= gap_min2;
                        }
                        push(v[cp ? 2 : 0], j);
                    }
                    k = end[k];
                } else k = k + 1;
            }
            for (int q = 0; q < 4; ++q) F->len[q][b - b0] = v[q]->n - n0[q];
        }
    }
    return F;
}

void tg_fmm_totals(const tg_fmm *F, int64_t *tot) {
    for (int q = 0; q < 4; ++q) {
        tot[q] = 0;
        for (int64_t i = 0; i < F->nblk; ++i) tot[q] += F->v[q][i].n;
    }
}

/* off: 4 arrays of b1-b0+1 int64; idx: 4 arrays sized by tg_fmm_totals.  Frees F. */
void tg_fmm_export_free(tg_fmm *F, int64_t **off, int32_t **idx) {
    int64_t nb = F->b1 - F->b0;
    for (int q = 0; q < 4; ++q) {
        off[q][0] = 0;
        for (int64_t b = 0; b < nb; ++b) off[q][b + 1] = off[q][b] + F->len[q][b];
#pragma omp parallel for schedule(dynamic, 1)
        for (int64_t ib = 0; ib < F->nblk; ++ib) {
            if (F->v[q][ib].n) memcpy(idx[q] + off[q][ib * F->blk], F->v[q][ib].v, sizeof(int32_t) * F->v[q][ib].n);
            free(F->v[q][ib].v);
        }
        free(F->v[q]); free(F->len[q]);
    }
    free(F);
}

/* Canonical records for stand-alone clouds (config 4): cloud c is points [c*k,(c+1)*k) of
 * pts (x,y,z,m fp32).  Same arithmetic as the tree's cell records. */
void tg_cloud_records(int64_t nclouds, int64_t k, const float *pts, float *rec) {
#pragma omp parallel for schedule(static)
    for (int64_t c = 0; c < nclouds; ++c) {
        float lo[3], hi[3];
        cell_record(pts, c * k, (c + 1) * k, rec + REC * c, lo, hi, 0);
    }
}

/* P-P lists in LEAF form (PKDG_PP_LEAVES): the tree walk adds a rejected leaf to the P-P list whole, so
 * every P-P list is a sequence of complete buckets.  map[i] = bucket of particle i (from the GLOBAL bucket
 * arrays gfirst / gcount, ng buckets); entry e is replaced by its bucket wherever e is the bucket's first
 * particle.  Two passes: count (leaf_off), then fill (leaf_idx).  Returns -1 if a list is not made of
 * whole buckets in order, else the number of references. */
int64_t tg_pp_to_leaves(int64_t n_particles, int64_t ng, const int32_t *gfirst, const int32_t *gcount, int64_t nb,
                        const int64_t *pp_off, const int32_t *pp_idx, int64_t *leaf_off, int32_t *leaf_idx) {
    int32_t *map = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n_particles > 0 ? n_particles : 1));
    if (!map) return -1;
    for (int64_t i = 0; i < n_particles; ++i) map[i] = -1;
    for (int64_t g = 0; g < ng; ++g)
        for (int32_t t = 0; t < gcount[g]; ++t) map[gfirst[g] + t] = (int32_t)g;
    int bad = 0;
    leaf_off[0] = 0;
    for (int64_t b = 0; b < nb; ++b) {     /* serial prefix: cheap next to the list build itself */
        int64_t n = 0;
        for (int64_t e = pp_off[b]; e < pp_off[b + 1];) {
            int32_t j = pp_idx[e];
            int32_t g = (j >= 0 && j < n_particles) ? map[j] : -1;
            if (g < 0 || gfirst[g] != j || e + gcount[g] > pp_off[b + 1]) { bad = 1; break; }
            for (int32_t t = 0; t < gcount[g]; ++t)
                if (pp_idx[e + t] != j + t) bad = 1;
            if (leaf_idx) leaf_idx[leaf_off[b] + n] = g;
            ++n;
            e += gcount[g];
        }
        leaf_off[b + 1] = leaf_off[b] + n;
    }
    free(map);
    return bad ? -1 : leaf_off[nb];
}

int tg_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
