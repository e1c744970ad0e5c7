/*
 * pkdg_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * A plain, slow, fp64 CPU statement of what the gravity hot path of PKDGRAV3
 * (arXiv 1609.08621, /root/reference/PAPER.md) computes: per-bucket evaluation
 * of particle-particle (P-P) and particle-cell (P-C) interaction lists.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call this file.  It shares no code, header, table
 * or constant with paper_1609_08621_b200/csrc (the CUDA path).
 *
 * The paper prints no formula for either kernel (SURVEY.md preamble); it fixes
 * the structure: PP for nearby particles, PC = "multipole expansion of the mass
 * within a more distant cell" (sec 3.1), centre of mass "always
 * the center of expansions" (L69), "4th order moments" (L71), softening 1/50 of
 * the mean separation with multipoles only for boxes >= 2 softenings apart
 * (L69), fp32 inputs and fp64 accumulation (L83).  The formulas below are the
 * DESIGN.md readings A1-A18; each function cites its own.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): spline closed forms and
 * quadrature of the spline density; brute-force pairwise sums written in
 * numpy; momentum conservation; Legendre series of an off-centre point mass;
 * (b/d)^5 convergence of a cloud's P-C field towards its direct sum; gradient
 * versus central differences; rotation covariance; trace invariance; tree +
 * lists versus direct summation; the paper's 655 -> 640 + 15 tile example; the
 * tree walk (orc_walk_lists, at the end of this file) against hand-built trees
 * on either side of every threshold and a numpy evaluation of the acceptance
 * inequality for every (sink, cell) pair.
 * No function here is "parity unpinned".
 *
 * No blocking, fusion or reordering: every loop is the definition written out.
 * OpenMP is used only to run independent buckets on several cores.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_MAXORD 12 /* highest |k| the Taylor-coefficient table can hold */
#define ORC_TDIM (ORC_MAXORD + 1)

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---------------------------------------------------------------------------
 * Softening (readings A1, A2): cubic-spline (Monaghan-Lattanzio) density of
 * support h = 2*eps; the pair force and potential of a unit mass smeared with
 * that density (Hernquist & Katz 1989 form), in units u = r/h:
 *   acceleration factor  g(u):  a_i -= m_j * d * g(u) / h^3,  d = x_i - x_j
 *   potential factor     w(u):  phi_i += m_j * w(u) / h
 * For u >= 1 both are exactly Newtonian (1/u^3, -1/u).
 * ------------------------------------------------------------------------- */
void orc_spline(double u, double *g, double *w) {
    double u2 = u * u, u3 = u2 * u;
    if (u < 0.5) {
        *g = 32.0 / 3.0 - (192.0 / 5.0) * u2 + 32.0 * u3;
        *w = (16.0 / 3.0) * u2 - (48.0 / 5.0) * u2 * u2 + (32.0 / 5.0) * u2 * u3 - 14.0 / 5.0;
    } else if (u < 1.0) {
        *g = 64.0 / 3.0 - 48.0 * u + (192.0 / 5.0) * u2 - (32.0 / 3.0) * u3 - 1.0 / (15.0 * u3);
        *w = 1.0 / (15.0 * u) + (32.0 / 3.0) * u2 - 16.0 * u3 + (48.0 / 5.0) * u2 * u2 -
             (32.0 / 15.0) * u2 * u3 - 16.0 / 5.0;
    } else {
        *g = 1.0 / u3;
        *w = -1.0 / u;
    }
}

/* One P-P interaction: contribution of a source (xs, ms) to a target at xt.
 * Adds to acc[3], pot[1].  G = 1.  ("PP interactions for nearby
 * particles"; softening L69; readings A1-A4.) */
void orc_pp_pair(const double xt[3], const double xs[3], double ms, double eps, double acc[3],
                 double *pot) {
    double h = 2.0 * eps;
    double d[3] = {xt[0] - xs[0], xt[1] - xs[1], xt[2] - xs[2]};
    double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    if (h > 0.0) {
        double g, w;
        orc_spline(r / h, &g, &w);
        double gh3 = g / (h * h * h);
        acc[0] -= ms * d[0] * gh3;
        acc[1] -= ms * d[1] * gh3;
        acc[2] -= ms * d[2] * gh3;
        *pot += ms * w / h;
    } else { /* eps == 0: pure Newtonian; coincident distinct particles are the caller's problem */
        double ir = 1.0 / r;
        acc[0] -= ms * d[0] * ir * ir * ir;
        acc[1] -= ms * d[1] * ir * ir * ir;
        acc[2] -= ms * d[2] * ir * ir * ir;
        *pot -= ms * ir;
    }
}

/* ---------------------------------------------------------------------------
 * Taylor coefficients of f(r) = 1/|r|:  t_k = (d^k f)/(a! b! c!), k = (a,b,c),
 * for all |k| <= order, by the recurrence:
 *   t_0 = 1/|r|
 *   n |r|^2 t_k + (2n-1) sum_i r_i t_{k-e_i} + (n-1) sum_i t_{k-2e_i} = 0,  n = |k| >= 1
 * (terms with a negative index are zero).  t is a dense [ORC_TDIM]^3 table,
 * entry (a,b,c) at t[(a*ORC_TDIM + b)*ORC_TDIM + c]; entries with |k| > order
 * and every index <= order + 1 are zero, the rest of the table is untouched.
 * ------------------------------------------------------------------------- */
#define TIDX(a, b, c) ((((a) * ORC_TDIM) + (b)) * ORC_TDIM + (c))

void orc_taylor_coeffs(const double r[3], int order, double *t) {
    int zmax = order + 1 < ORC_MAXORD ? order + 1 : ORC_MAXORD; /* zero what a caller may read */
    for (int a = 0; a <= zmax; ++a)
        for (int b = 0; b <= zmax; ++b)
            for (int c = 0; c <= zmax; ++c) t[TIDX(a, b, c)] = 0.0;
    double r2 = r[0] * r[0] + r[1] * r[1] + r[2] * r[2];
    t[TIDX(0, 0, 0)] = 1.0 / sqrt(r2);
    for (int n = 1; n <= order; ++n) {
        for (int a = n; a >= 0; --a) {
            for (int b = n - a; b >= 0; --b) {
                int c = n - a - b;
                double s1 = 0.0, s2 = 0.0;
                if (a >= 1) s1 += r[0] * t[TIDX(a - 1, b, c)];
                if (b >= 1) s1 += r[1] * t[TIDX(a, b - 1, c)];
                if (c >= 1) s1 += r[2] * t[TIDX(a, b, c - 1)];
                if (a >= 2) s2 += t[TIDX(a - 2, b, c)];
                if (b >= 2) s2 += t[TIDX(a, b - 2, c)];
                if (c >= 2) s2 += t[TIDX(a, b, c - 2)];
                t[TIDX(a, b, c)] = -((2.0 * n - 1.0) * s1 + (n - 1.0) * s2) / (n * r2);
            }
        }
    }
}

/* ---------------------------------------------------------------------------
 * One P-C interaction (readings A4, A5, A9, A12).
 * Canonical cell record `rec` (36 fp32):
 *   [0..2] centre of mass, [3] mass, [4..9] raw 2nd moments, [10..19] raw 3rd,
 *   [20..34] raw 4th, [35] b_max.  M_k = sum_j m_j s^a s^b s^c about the stored
 *   centre of mass; for each order n the entries run a = n..0, b = n-a..0,
 *   c = n-a-b.  The dipole is not stored and not used (A9).
 * With r = x_target - COM and t_k the Taylor coefficients of 1/|r|:
 *   phi  += - sum_{|k| in {0,2,3,4}} (-1)^{|k|} M_k t_k
 *   a_l  +=   sum_{|k| in {0,2,3,4}} (-1)^{|k|} M_k (k_l + 1) t_{k+e_l}
 * i.e. the acceleration is the exact gradient of the truncated potential.
 * ------------------------------------------------------------------------- */
void orc_pc_pair(const double xt[3], const float *rec, double acc[3], double *pot) {
    double r[3] = {xt[0] - (double)rec[0], xt[1] - (double)rec[1], xt[2] - (double)rec[2]};
    double t[ORC_TDIM * ORC_TDIM * ORC_TDIM];
    orc_taylor_coeffs(r, 5, t);
    int pos = 3; /* rec[3] is M_000 */
    for (int n = 0; n <= 4; ++n) {
        if (n == 1) continue; /* dipole about the centre of mass: dropped */
        double sign = (n % 2 == 0) ? 1.0 : -1.0;
        for (int a = n; a >= 0; --a) {
            for (int b = n - a; b >= 0; --b) {
                int c = n - a - b;
                double M = (double)rec[pos++];
                *pot -= sign * M * t[TIDX(a, b, c)];
                acc[0] += sign * M * (a + 1) * t[TIDX(a + 1, b, c)];
                acc[1] += sign * M * (b + 1) * t[TIDX(a, b + 1, c)];
                acc[2] += sign * M * (c + 1) * t[TIDX(a, b, c + 1)];
            }
        }
    }
}

/* ---------------------------------------------------------------------------
 * The whole path for a set of buckets (SURVEY.md sec 8(c) "Oracle algorithm").
 * xyzm: [n_particles][4] fp32 (x,y,z,m), tree order.  cells: [n_cells][stride]
 * fp32 canonical records.  Bucket b holds targets first[b] .. first[b]+count[b].
 * Lists are CSR: entries off[b] .. off[b+1] of idx.  A P-P source j equal to the
 * target's own index is skipped BY INDEX (A11).  Negative indices (tile padding)
 * are skipped.  If `sel` is non-NULL only the n_sel buckets sel[0..n_sel) are
 * evaluated.  out: [n_particles][4] fp64 (ax, ay, az, phi); only targets of the
 * evaluated buckets are written.
 * ------------------------------------------------------------------------- */
int orc_gravity_eval(int64_t n_particles, const float *xyzm, int64_t n_cells, const float *cells,
                     int32_t stride, int64_t n_buckets, const int32_t *first, const int32_t *count,
                     const int64_t *pp_off, const int32_t *pp_idx, const int64_t *pc_off,
                     const int32_t *pc_idx, double eps, const int64_t *sel, int64_t n_sel,
                     double *out) {
    int64_t nb = sel ? n_sel : n_buckets;
    int err = 0;
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t ib = 0; ib < nb; ++ib) {
        int64_t b = sel ? sel[ib] : ib;
        if (b < 0 || b >= n_buckets) {
#pragma omp atomic write
                err = 1;
                continue;
            }
        for (int32_t ti = 0; ti < count[b]; ++ti) {
            int64_t i = (int64_t)first[b] + ti;
            if (i < 0 || i >= n_particles) {
#pragma omp atomic write
                err = 1;
                continue;
            }
            double xt[3] = {xyzm[4 * i], xyzm[4 * i + 1], xyzm[4 * i + 2]};
            double acc[3] = {0, 0, 0}, pot = 0;
            if (pp_off) {
                for (int64_t e = pp_off[b]; e < pp_off[b + 1]; ++e) {
                    int64_t j = pp_idx[e];
                    if (j < 0 || j == i) continue;
                    if (j >= n_particles) {
#pragma omp atomic write
                err = 1;
                continue;
            }
                    double xs[3] = {xyzm[4 * j], xyzm[4 * j + 1], xyzm[4 * j + 2]};
                    orc_pp_pair(xt, xs, (double)xyzm[4 * j + 3], eps, acc, &pot);
                }
            }
            if (pc_off) {
                for (int64_t e = pc_off[b]; e < pc_off[b + 1]; ++e) {
                    int64_t c = pc_idx[e];
                    if (c < 0) continue;
                    if (c >= n_cells) {
#pragma omp atomic write
                err = 1;
                continue;
            }
                    orc_pc_pair(xt, cells + c * (int64_t)stride, acc, &pot);
                }
            }
            out[4 * i + 0] = acc[0];
            out[4 * i + 1] = acc[1];
            out[4 * i + 2] = acc[2];
            out[4 * i + 3] = pot;
        }
    }
    return err;
}

/* ---------------------------------------------------------------------------
 * Conditioning of the sum (reading A17): for each target of the
 * evaluated buckets, S_i = sum over its list entries of |a_ij| (the Euclidean norm
 * of each entry's acceleration contribution, from the same pair functions as
 * above).  kappa_i = S_i / |a_i| measures the cancellation in a_i; a relative
 * error of any finite-precision evaluation grows in proportion to it.  Diagnostic
 * only: no evaluation result depends on it.  out_abs: [n_particles] fp64.
 * ------------------------------------------------------------------------- */
static int contribution_norms_p(int64_t n_particles, const float *xyzm, int64_t n_cells, const float *cells,
                                int32_t stride, int64_t n_buckets, const int32_t *first, const int32_t *count,
                                const int64_t *pp_off, const int32_t *pp_idx, const int64_t *pc_off,
                                const int32_t *pc_idx, double eps, const int64_t *sel, int64_t n_sel,
                                double *out_abs, int squared) {
    int64_t nb = sel ? n_sel : n_buckets;
    int err = 0;
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t ib = 0; ib < nb; ++ib) {
        int64_t b = sel ? sel[ib] : ib;
        if (b < 0 || b >= n_buckets) {
#pragma omp atomic write
            err = 1;
            continue;
        }
        for (int32_t ti = 0; ti < count[b]; ++ti) {
            int64_t i = (int64_t)first[b] + ti;
            if (i < 0 || i >= n_particles) continue;
            double xt[3] = {xyzm[4 * i], xyzm[4 * i + 1], xyzm[4 * i + 2]};
            double S = 0.0;
            if (pp_off) {
                for (int64_t e = pp_off[b]; e < pp_off[b + 1]; ++e) {
                    int64_t j = pp_idx[e];
                    if (j < 0 || j == i || j >= n_particles) continue;
                    double xs[3] = {xyzm[4 * j], xyzm[4 * j + 1], xyzm[4 * j + 2]};
                    double a[3] = {0, 0, 0}, pot = 0;
                    orc_pp_pair(xt, xs, (double)xyzm[4 * j + 3], eps, a, &pot);
                    S += squared ? a[0] * a[0] + a[1] * a[1] + a[2] * a[2] : sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]);
                }
            }
            if (pc_off) {
                for (int64_t e = pc_off[b]; e < pc_off[b + 1]; ++e) {
                    int64_t c = pc_idx[e];
                    if (c < 0 || c >= n_cells) continue;
                    double a[3] = {0, 0, 0}, pot = 0;
                    orc_pc_pair(xt, cells + c * (int64_t)stride, a, &pot);
                    S += squared ? a[0] * a[0] + a[1] * a[1] + a[2] * a[2] : sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]);
                }
            }
            out_abs[i] = S;
        }
    }
    return err;
}

int orc_contribution_norms(int64_t n_particles, const float *xyzm, int64_t n_cells, const float *cells,
                           int32_t stride, int64_t n_buckets, const int32_t *first, const int32_t *count,
                           const int64_t *pp_off, const int32_t *pp_idx, const int64_t *pc_off,
                           const int32_t *pc_idx, double eps, const int64_t *sel, int64_t n_sel,
                           double *out_abs) {
    return contribution_norms_p(n_particles, xyzm, n_cells, cells, stride, n_buckets, first, count, pp_off, pp_idx,
                                pc_off, pc_idx, eps, sel, n_sel, out_abs, 0);
}

/* The same with squares: S2_i = sum over list entries of |a_ij|^2.  kappa2_i = sqrt(S2_i) / |a_i| is what the
 * error of a sum of terms with INDEPENDENT rounding errors grows with (DESIGN.md "Conditioning and the fp64
 * fix-up"); used to calibrate and to test the library's fix-up threshold.  Diagnostic only. */
int orc_contribution_norms2(int64_t n_particles, const float *xyzm, int64_t n_cells, const float *cells,
                            int32_t stride, int64_t n_buckets, const int32_t *first, const int32_t *count,
                            const int64_t *pp_off, const int32_t *pp_idx, const int64_t *pc_off,
                            const int32_t *pc_idx, double eps, const int64_t *sel, int64_t n_sel,
                            double *out_sq) {
    return contribution_norms_p(n_particles, xyzm, n_cells, cells, stride, n_buckets, first, count, pp_off, pp_idx,
                                pc_off, pc_idx, eps, sel, n_sel, out_sq, 1);
}

/* Direct summation: the plain definition the tree method approximates
 * (PAPER.md:L57).  For each listed target, the softened sum over ALL other
 * particles.  Used only to pin the oracle (north_star self-checks 1, 3, 4). */
void orc_direct_sum(int64_t n_particles, const float *xyzm, double eps, const int64_t *targets,
                    int64_t n_targets, double *out /* [n_targets][4] */) {
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t it = 0; it < n_targets; ++it) {
        int64_t i = targets ? targets[it] : it;
        double xt[3] = {xyzm[4 * i], xyzm[4 * i + 1], xyzm[4 * i + 2]};
        double acc[3] = {0, 0, 0}, pot = 0;
        for (int64_t j = 0; j < n_particles; ++j) {
            if (j == i) continue;
            double xs[3] = {xyzm[4 * j], xyzm[4 * j + 1], xyzm[4 * j + 2]};
            orc_pp_pair(xt, xs, (double)xyzm[4 * j + 3], eps, acc, &pot);
        }
        out[4 * it + 0] = acc[0];
        out[4 * it + 1] = acc[1];
        out[4 * it + 2] = acc[2];
        out[4 * it + 3] = pot;
    }
}

/* ---------------------------------------------------------------------------
 * Cell-cell and cell-particle interactions and the local expansion
 * ("FMM also considers cell-cell (CC)
 * interactions by approximating the potential landscape within a given cell (the
 * sink cell) that is induced by a sufficiently distant multipole (the source
 * cell)"; L69 fn 2 "Cell-particle interactions ... are the expansions of the
 * potential within the sink cell induced by a single source particle"; L71 "The
 * local expansion of the potential about the sink's center of mass is actually
 * done to 5th order ... accumulating the CC and CP interactions").
 *
 * The paper prints no formula (readings A20-A22).  With the notation of
 * orc_pc_pair -- t_k(r) = d^k(1/|r|)/k!, raw moments M_m of the source cell about
 * its centre z_C -- the source's potential at x is
 *     phi(x) = - sum_m (-1)^|m| M_m t_m(x - z_C).
 * Expanding about the sink's centre z_B (x = z_B + s, R = z_B - z_C):
 *     t_m(R + s) = sum_n binom(n + m, m) t_{n+m}(R) s^n      (Taylor's theorem),
 * so phi(z_B + s) = sum_n L_n s^n with
 *     L_n = - sum_m (-1)^|m| M_m binom(n + m, m) t_{n+m}(R),
 * binom(n + m, m) = prod_i (n_i + m_i)! / (n_i! m_i!).  Truncation (A20): the local
 * expansion holds |n| <= 5 and a term is kept iff |n| + |m| <= 5 (total order 5:
 * exactly the derivatives of 1/r up to 5th order that the P-C kernel uses too);
 * |m| in {0, 2, 3, 4}, the dipole about the centre of mass is dropped (A9).
 * A source PARTICLE (x_j, m_j) is the case z_C = x_j, M_0 = m_j, no higher moment:
 *     L_n += - m_j t_n(z_B - x_j),  |n| <= 5.
 * Unsoftened, like P-C (A4): the list builder accepts C-C / C-P only for boxes at
 * least two softenings apart.
 *
 * Local coefficients are stored in the order of the moments: for n = 0..5,
 * a = n..0, b = n-a..0, c = n-a-b: 56 doubles.
 * ------------------------------------------------------------------------- */
#define ORC_NLOC 56

static double binom1(int n, int m) { /* binom(n + m, m), small arguments */
    double r = 1.0;
    for (int i = 1; i <= m; ++i) r = r * (double)(n + i) / (double)i;
    return r;
}

/* L += contribution of one source cell (canonical record) to the local expansion about zB. */
void orc_cc_accumulate(const double zB[3], const float *rec, double *L) {
    double R[3] = {zB[0] - (double)rec[0], zB[1] - (double)rec[1], zB[2] - (double)rec[2]};
    double t[ORC_TDIM * ORC_TDIM * ORC_TDIM];
    orc_taylor_coeffs(R, 5, t);
    int li = 0;
    for (int n = 0; n <= 5; ++n)
        for (int na = n; na >= 0; --na)
            for (int nb = n - na; nb >= 0; --nb) {
                int nc = n - na - nb;
                double sum = 0.0;
                int pos = 3; /* rec[3] is M_000 */
                for (int m = 0; m <= 4; ++m) {
                    if (m == 1) continue;
                    double sign = (m % 2 == 0) ? 1.0 : -1.0;
                    for (int ma = m; ma >= 0; --ma)
                        for (int mb = m - ma; mb >= 0; --mb) {
                            int mc = m - ma - mb;
                            double M = (double)rec[pos++];
                            if (n + m > 5) continue;
                            sum += sign * M * binom1(na, ma) * binom1(nb, mb) * binom1(nc, mc) *
                                   t[TIDX(na + ma, nb + mb, nc + mc)];
                        }
                }
                L[li++] -= sum;
            }
}

/* L += contribution of one source particle (xs, ms) to the local expansion about zB. */
void orc_cp_accumulate(const double zB[3], const double xs[3], double ms, double *L) {
    double R[3] = {zB[0] - xs[0], zB[1] - xs[1], zB[2] - xs[2]};
    double t[ORC_TDIM * ORC_TDIM * ORC_TDIM];
    orc_taylor_coeffs(R, 5, t);
    int li = 0;
    for (int n = 0; n <= 5; ++n)
        for (int na = n; na >= 0; --na)
            for (int nb = n - na; nb >= 0; --nb) L[li++] -= ms * t[TIDX(na, nb, n - na - nb)];
}

/* Evaluate the local expansion at xt: pot += sum_n L_n s^n, acc_l -= sum_n L_n n_l s^(n - e_l), s = xt - zB
 * (the acceleration is minus the exact gradient of the polynomial). */
void orc_local_eval(const double zB[3], const double *L, const double xt[3], double acc[3], double *pot) {
    double s[3] = {xt[0] - zB[0], xt[1] - zB[1], xt[2] - zB[2]};
    double pw[3][7];
    for (int d = 0; d < 3; ++d) {
        pw[d][0] = 1.0;
        for (int e = 1; e < 7; ++e) pw[d][e] = pw[d][e - 1] * s[d];
    }
    int li = 0;
    for (int n = 0; n <= 5; ++n)
        for (int a = n; a >= 0; --a)
            for (int b = n - a; b >= 0; --b) {
                int c = n - a - b;
                double Ln = L[li++];
                *pot += Ln * pw[0][a] * pw[1][b] * pw[2][c];
                if (a >= 1) acc[0] -= Ln * a * pw[0][a - 1] * pw[1][b] * pw[2][c];
                if (b >= 1) acc[1] -= Ln * b * pw[0][a] * pw[1][b - 1] * pw[2][c];
                if (c >= 1) acc[2] -= Ln * c * pw[0][a] * pw[1][b] * pw[2][c - 1];
            }
}

/* The FMM part of the path for a set of sink buckets: for bucket b, the local expansion about the
 * bucket's centre zB[b] (fp32, widened) accumulates its C-C list (cell indices) and its C-P list
 * (particle indices), and is evaluated at every particle of the bucket.  out: [n_particles][4] fp64,
 * ADDED to (the caller sums it with the P-P / P-C part); Lout (may be NULL): [n_buckets][56]. */
int orc_fmm_eval(int64_t n_particles, const float *xyzm, int64_t n_cells, const float *cells, int32_t stride,
                 int64_t n_buckets, const int32_t *first, const int32_t *count, const float *zB,
                 const int64_t *cc_off, const int32_t *cc_idx, const int64_t *cp_off, const int32_t *cp_idx,
                 double *out, double *Lout) {
    int err = 0;
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t b = 0; b < n_buckets; ++b) {
        double z[3] = {zB[3 * b], zB[3 * b + 1], zB[3 * b + 2]};
        double L[ORC_NLOC];
        for (int i = 0; i < ORC_NLOC; ++i) L[i] = 0.0;
        if (cc_off)
            for (int64_t e = cc_off[b]; e < cc_off[b + 1]; ++e) {
                int64_t c = cc_idx[e];
                if (c < 0) continue;
                if (c >= n_cells) {
#pragma omp atomic write
                    err = 1;
                    continue;
                }
                orc_cc_accumulate(z, cells + c * (int64_t)stride, L);
            }
        if (cp_off)
            for (int64_t e = cp_off[b]; e < cp_off[b + 1]; ++e) {
                int64_t j = cp_idx[e];
                if (j < 0) continue;
                if (j >= n_particles) {
#pragma omp atomic write
                    err = 1;
                    continue;
                }
                double xs[3] = {xyzm[4 * j], xyzm[4 * j + 1], xyzm[4 * j + 2]};
                orc_cp_accumulate(z, xs, (double)xyzm[4 * j + 3], L);
            }
        if (Lout)
            for (int i = 0; i < ORC_NLOC; ++i) Lout[b * ORC_NLOC + i] = L[i];
        for (int32_t ti = 0; ti < count[b]; ++ti) {
            int64_t i = (int64_t)first[b] + ti;
            if (i < 0 || i >= n_particles) {
#pragma omp atomic write
                err = 1;
                continue;
            }
            double xt[3] = {xyzm[4 * i], xyzm[4 * i + 1], xyzm[4 * i + 2]};
            double acc[3] = {0, 0, 0}, pot = 0;
            orc_local_eval(z, L, xt, acc, &pot);
            out[4 * i + 0] += acc[0];
            out[4 * i + 1] += acc[1];
            out[4 * i + 2] += acc[2];
            out[4 * i + 3] += pot;
        }
    }
    return err;
}

/* ---------------------------------------------------------------------------
 * Integer side (SURVEY.md sec 8(c) "Integer side"; PAPER.md:L168, L188 fn 11:
 * lists are cut at warp multiples -- "655 elements ... 640 ... and 15").
 * Written spec of the packer: per bucket, tiles of 32 entries in list order,
 * the last tile padded with -1.  tile_off[b] = first tile of bucket b (int64,
 * [n_buckets+1]); tiles = [n_tiles][32] int32.  Two-call use: tiles == NULL
 * only fills tile_off and returns the tile count.
 * ------------------------------------------------------------------------- */
int64_t orc_pack_tiles(int64_t n_buckets, const int64_t *off, const int32_t *idx, int64_t *tile_off,
                       int32_t *tiles) {
    int64_t nt = 0;
    for (int64_t b = 0; b < n_buckets; ++b) {
        tile_off[b] = nt;
        int64_t len = off[b + 1] - off[b];
        nt += (len + 31) / 32;
    }
    tile_off[n_buckets] = nt;
    if (!tiles) return nt;
    for (int64_t b = 0; b < n_buckets; ++b) {
        int64_t len = off[b + 1] - off[b];
        int64_t ntile = (len + 31) / 32;
        for (int64_t k = 0; k < ntile * 32; ++k)
            tiles[tile_off[b] * 32 + k] = (k < len) ? idx[off[b] + k] : -1;
    }
    return nt;
}

/* Interaction counts: I = sum_b count[b] * len[b] (SURVEY.md sec 8 notation). */
int64_t orc_interactions(int64_t n_buckets, const int32_t *count, const int64_t *off) {
    int64_t I = 0;
    for (int64_t b = 0; b < n_buckets; ++b) I += (int64_t)count[b] * (off[b + 1] - off[b]);
    return I;
}

/* Chunk boundaries for the streamed variant: greedy fill in bucket order; a
 * chunk is closed before the bucket that would push its P-P or its P-C entry
 * count above max_entries (a single bucket longer than max_entries gets a chunk
 * of its own).  bounds[0] = 0, bounds[n_chunks] = n_buckets; returns n_chunks.
 * bounds must have room for n_buckets + 1 values. */
int64_t orc_chunk_bounds(int64_t n_buckets, const int64_t *pp_off, const int64_t *pc_off,
                         int64_t max_entries, int64_t *bounds) {
    int64_t nc = 0, b0 = 0;
    bounds[0] = 0;
    if (n_buckets == 0) return 0;
    for (int64_t b = 0; b < n_buckets; ++b) {
        int64_t pp = pp_off[b + 1] - pp_off[b0];
        int64_t pc = pc_off[b + 1] - pc_off[b0];
        if ((pp > max_entries || pc > max_entries) && b > b0) {
            bounds[++nc] = b;
            b0 = b;
        }
    }
    bounds[++nc] = n_buckets;
    return nc;
}

/* ---------------------------------------------------------------------------
 * Tree walk: which cells and particles end up on which list of a sink.
 *
 * PAPER.md:L65 (sec 3.1): the walk starts at the root with a checklist; every
 * checklist element gets a case value -- open it, put it on the PP list, on the
 * PC list, on the CC list, on the CP list, or keep it for the sink's children;
 * cells are visited node-left-right.  L69: the opening radius of a cell is
 * RO = b_max / theta; a cell-cell interaction is allowed when the centres are
 * further apart than 1.5 RO_sink + RO_source, and multipoles are only used
 * when the bounding boxes are at least two softening lengths apart; a particle
 * is a source with RO_source = 0 (fn 2); the walk for a sink stops at group
 * size g and resolves what is left into the lists.  The paper prints the CC /
 * CP radius only; readings A6 (two lists) and A22 (four lists) fix
 * the rest, and this is those readings written out as a RECURSIVE descent over
 * explicit children -- one sink at a time, no checklist inheritance, no skip
 * pointers -- so that each decision can be read off against the inequality:
 *
 *   visit(k):  if k may act on the sink as a whole (rule below) -> list it, done
 *              else if k is a leaf -> its particles go on a particle list, done
 *              else visit every child of k, left to right.
 *
 * Two lists (A6).  Cell k is a P-C source of sink cell B  iff
 *     k != B,  count[k] >= 2,
 *     |COM_B - COM_k| > b_max,B + RO_k,        RO_k = b_max,k / theta,
 *     gap(bbox_B, bbox_k) >= 2 eps.
 *   A rejected leaf's particles all go on the P-P list (B's own included; the
 *   evaluation skips i = j by index).
 * Four lists (A22).  With RO_B = b_max,B / theta:
 *     C-C  iff k != B, count[k] >= 2, gap >= 2 eps, |COM_B - COM_k| > 1.5 RO_B + RO_k
 *     P-C  else iff the two-list rule holds
 *     a rejected leaf's particles one by one (RO_source = 0):
 *     C-P  iff j is not in B, |COM_B - x_j| > 1.5 RO_B, gap(bbox_B, x_j) >= 2 eps
 *     P-P  else.
 * gap(.,.) is the Euclidean distance between two axis-aligned boxes (0 when they
 * touch or overlap), compared squared.  All arithmetic in fp64 on the fp32
 * inputs.  The tree comes as arrays in depth-first pre-order: cell k's subtree
 * is cells [k, end[k]), so its children are k + 1, end[k + 1], end[end[k + 1]],
 * ... below end[k].  The sink is ANY cell: a bucket (lists per bucket), or a
 * cell of up to g particles (lists per group, L69).
 *
 * Pins (tests/test_oracle_walk_pins.py): hand-built three-cell trees on either
 * side of every threshold (distance, 2 eps gap, count = 1, k = B, 1.5 RO_B);
 * on N ~ 500 a numpy evaluation of the inequality for every (sink, cell) pair:
 * every listed cell satisfies it, no ancestor of a listed cell or listed leaf
 * does (the list is the coarsest admissible cover), every particle is covered
 * exactly once.
 * ------------------------------------------------------------------------- */
typedef struct {
    int64_t n_cells;
    const int32_t *first, *count, *end, *isleaf;
    const float *rec;   /* canonical records, stride 36: COM at [0..2], b_max at [35] */
    const float *bblo, *bbhi;
    const float *xyzm;  /* four-list walk only */
    const int32_t *leaf_rank; /* two-list walk: non-NULL = a leaf's P-P entry is leaf_rank[k], once */
    double theta, eps;
    int64_t B;          /* the sink cell */
    int four;           /* 0: lists 0 = P-P, 1 = P-C;  1: also 2 = C-P, 3 = C-C */
    int32_t *out[4];    /* where to write (NULL = count only) */
    int64_t n[4];       /* entries so far */
} orc_walk;

static void walk_emit(orc_walk *w, int list, int32_t v) {
    if (w->out[list]) w->out[list][w->n[list]] = v;
    w->n[list]++;
}

static double box_gap2(const float *loA, const float *hiA, const float *loB, const float *hiB) {
    double g2 = 0.0;
    for (int a = 0; a < 3; ++a) {
        double g = 0.0;
        if ((double)loA[a] - (double)hiB[a] > g) g = (double)loA[a] - (double)hiB[a];   /* A lies above B */
        if ((double)loB[a] - (double)hiA[a] > g) g = (double)loB[a] - (double)hiA[a];   /* A lies below B */
        g2 += g * g;
    }
    return g2;
}

static double centre_dist(const float *a, const float *b) {
    double dx = (double)a[0] - (double)b[0], dy = (double)a[1] - (double)b[1], dz = (double)a[2] - (double)b[2];
    return sqrt(dx * dx + dy * dy + dz * dz);
}

/* 0: k may not act on the sink as a whole; 1: P-C; 3: C-C (four-list walk only) */
static int walk_cell_rule(const orc_walk *w, int64_t k) {
    if (k == w->B || w->count[k] < 2) return 0;
    const float *rB = w->rec + 36 * w->B, *rk = w->rec + 36 * k;
    const double two_eps = 2.0 * w->eps;
    if (box_gap2(w->bblo + 3 * k, w->bbhi + 3 * k, w->bblo + 3 * w->B, w->bbhi + 3 * w->B) < two_eps * two_eps) return 0;
    const double d = centre_dist(rB, rk);
    const double RO_k = (double)rk[35] / w->theta, RO_B = (double)rB[35] / w->theta;
    if (w->four && d > 1.5 * RO_B + RO_k) return 3;
    if (d > (double)rB[35] + RO_k) return 1;
    return 0;
}

static void walk_visit(orc_walk *w, int64_t k) {
    const int rule = walk_cell_rule(w, k);
    if (rule) { walk_emit(w, rule, (int32_t)k); return; }
    if (w->isleaf[k]) {
        if (!w->four && w->leaf_rank) { walk_emit(w, 0, w->leaf_rank[k]); return; }
        for (int32_t t = 0; t < w->count[k]; ++t) {
            const int32_t j = w->first[k] + t;
            int cp = 0;
            if (w->four && k != w->B) {   /* a source particle: RO_source = 0, its box is the point itself */
                const float *xj = w->xyzm + 4 * (int64_t)j, *rB = w->rec + 36 * w->B;
                const double two_eps = 2.0 * w->eps, RO_B = (double)rB[35] / w->theta;
                cp = centre_dist(rB, xj) > 1.5 * RO_B &&
                     box_gap2(xj, xj, w->bblo + 3 * w->B, w->bbhi + 3 * w->B) >= two_eps * two_eps;
            }
            walk_emit(w, cp ? 2 : 0, j);
        }
        return;
    }
    for (int64_t c = k + 1; c < w->end[k]; c = w->end[c]) walk_visit(w, c);   /* the children, left to right */
}

/* Lists of n_sinks sink cells.  off[q] = [n_sinks + 1] int64 (written), idx[q] = entries (NULL: only the offsets
 * are computed -- call once to size, once to fill).  q = 0 P-P, 1 P-C, and with four != 0 also 2 C-P, 3 C-C.
 * Returns 0, or -1 for a malformed tree (a sink or an end[] out of range). */
int orc_walk_lists(int64_t n_cells, const int32_t *first, const int32_t *count, const int32_t *end,
                   const int32_t *isleaf, const float *rec, const float *bblo, const float *bbhi,
                   const float *xyzm, const int32_t *leaf_rank, const int32_t *sink_cell, int64_t n_sinks,
                   double theta, double eps, int four, int64_t *const off[4], int32_t *const idx[4]) {
    const int nl = four ? 4 : 2;
    for (int64_t k = 0; k < n_cells; ++k)
        if (end[k] <= k || end[k] > n_cells) return -1;
    for (int q = 0; q < nl; ++q) off[q][0] = 0;
    for (int64_t s = 0; s < n_sinks; ++s) {
        if (sink_cell[s] < 0 || sink_cell[s] >= n_cells) return -1;
        orc_walk w = {n_cells, first, count, end, isleaf, rec, bblo, bbhi, xyzm, leaf_rank, theta, eps, sink_cell[s],
                      four, {0, 0, 0, 0}, {0, 0, 0, 0}};
        for (int q = 0; q < nl; ++q) w.out[q] = idx && idx[q] ? idx[q] + off[q][s] : 0;
        if (n_cells > 0) walk_visit(&w, 0);
        for (int q = 0; q < nl; ++q) off[q][s + 1] = off[q][s] + w.n[q];
    }
    return 0;
}
