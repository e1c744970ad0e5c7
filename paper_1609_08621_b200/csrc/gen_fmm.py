"""Writes pkdg_fmm_gen.cuh: the straight-line arithmetic of the cell-cell / cell-particle kernel.

    python paper_1609_08621_b200/csrc/gen_fmm.py          (rewrites the header next to this file)

What is generated (readings A20-A22):

  fmm_monomials(x, y, z, p)        p[i] = x^a y^b z^c for the 56 multi-indices |k| <= 5 in the library's order
  fmm_derivs(p, g, d)              d[i] = lambda^|k| D_k(R), D_k = d^k (1/|R|), from the monomials p of the unit
                                   vector u = R / |R| and g[n] = (lambda / |R|)^n / |R|
  fmm_fold_moments(q, sc, F)       the 22 folded moments of a cell record (see "Trace-free" below)
  fmm_m2l_cell(d, F, L)            L[n] += sum_m F[m] d[n + m],  |m| in {0, 2, 3, 4},  |n| + |m| <= 5, n and m with at most one z
  fmm_m2l_particle(d, mu0, L)      L[n] += mu0 d[n], the 36 n with at most one z
  kExp*                            the table that rebuilds all 56 coefficients from those 36
  fmm_eval(p, Lam, phi, gx, gy, gz)  polynomial sum_n Lam[n] sigma^n and its gradient from the monomials p of sigma

The derivative tensors come from the DEFINITION, not from a recurrence: D_k = N_k(x, rho) / r^(2|k|+1) with
rho = r^2 and N_0 = 1, d_i (N / r^(2n+1)) = (rho d_i N - (2n+1) x_i N) / r^(2n+3), d_i rho = 2 x_i, carried out
on polynomials with exact integer coefficients; on the unit sphere rho = 1, which leaves the few-term polynomials
emitted below (D_xx = 3 x^2 - 1, D_xxy = -(15 x^2 y - 3 y), ...).  The multi-index order is that of the canonical
cell record (include/pkdg.h): for n = 0..5, a = n..0, b = n-a..0, c = n-a-b.

With D_k = k! t_k the shift of a multipole expansion to a local one (Taylor's theorem) reads
    L_n = -(1/n!) sum_m (-1)^|m| (M_m / m!) D_{n+m}(R),      R = z_sink - z_source,
so the kernel feeds mu[m] = -(-1)^|m| M_m / (m! lambda^|m|) and divides by n! once, after the whole list.

Trace-free.  1/|R| is harmonic, so D_{k+2ex} + D_{k+2ey} + D_{k+2ez} = 0 for every k.  Two consequences, both exact:
(1) in sum_m mu[m] D_{n+m} every m with two or more z can be moved onto the m with fewer (D_{n+m0+2ez} = -D_{n+m0+2ex}
- D_{n+m0+2ey}), so only the 1 + 5 + 7 + 9 = 22 FOLDED moments F[m], m_z <= 1, are needed (linear combinations of the
record's 32, made once per cell); (2) the accumulated coefficients obey the same identity (the truncation is by the
total order |n| + |m|, so all three terms of it are always present together), hence only the 36 coefficients with
n_z <= 1 are accumulated and the other 20 are rebuilt once per bucket.  215 multiply-adds per cell instead of 336.
"""
from __future__ import annotations

import math
import os
from collections import defaultdict
from fractions import Fraction

ORDER = 5
HERE = os.path.dirname(os.path.abspath(__file__))


def multi_indices(nmax):
    return [(a, b, n - a - b) for n in range(nmax + 1) for a in range(n, -1, -1) for b in range(n - a, -1, -1)]


IDX = multi_indices(ORDER)
POS = {k: i for i, k in enumerate(IDX)}
MOM = multi_indices(4)          # record layout: 35 moments (the 3 dipole slots are absent from the record)
IND = [k for k in IDX if k[2] <= 1]                         # the 36 coefficients that are accumulated
POSI = {k: i for i, k in enumerate(IND)}
MOMF = [m for m in MOM if sum(m) != 1 and m[2] <= 1]        # the 22 folded moments
POSF = {m: i for i, m in enumerate(MOMF)}


def reduce_z(k):
    """k -> {k' with k'_z <= 1: integer coefficient}: repeated use of T[k + 2ez] = -T[k + 2ex] - T[k + 2ey]."""
    if k[2] <= 1:
        return {k: 1}
    out = defaultdict(int)
    for kk in ((k[0] + 2, k[1], k[2] - 2), (k[0], k[1] + 2, k[2] - 2)):
        for key, c in reduce_z(kk).items():
            out[key] -= c
    return {key: c for key, c in out.items() if c != 0}


# --- exact polynomial algebra in (x, y, z, rho): dict {(ex, ey, ez, erho): int} ---------------------------------
def p_add(p, q, s=1):
    r = defaultdict(int, p)
    for k, v in q.items():
        r[k] += s * v
    return {k: v for k, v in r.items() if v != 0}


def p_mul_mono(p, mono, c=1):
    return {tuple(a + b for a, b in zip(k, mono)): v * c for k, v in p.items()}


def p_diff(p, axis):
    """d/dx_axis with rho = x^2 + y^2 + z^2 kept as a symbol: d rho / dx_i = 2 x_i."""
    r = defaultdict(int)
    for k, v in p.items():
        if k[axis]:
            kk = list(k); kk[axis] -= 1
            r[tuple(kk)] += v * k[axis]
        if k[3]:
            kk = list(k); kk[3] -= 1; kk[axis] += 1
            r[tuple(kk)] += v * k[3] * 2
    return {k: v for k, v in r.items() if v != 0}


def numerators():
    """N_k with d^k (1/r) = N_k / r^(2|k|+1)."""
    N = {(0, 0, 0): {(0, 0, 0, 0): 1}}
    for k in IDX[1:]:
        axis = next(i for i in range(3) if k[i] > 0)
        prev = list(k); prev[axis] -= 1; prev = tuple(prev)
        n = sum(prev)
        e = [0, 0, 0, 0]; e[axis] = 1
        N[k] = p_add(p_mul_mono(p_diff(N[prev], axis), (0, 0, 0, 1)), p_mul_mono(N[prev], tuple(e), 2 * n + 1), -1)
    return N


def on_unit_sphere(p):
    r = defaultdict(int)
    for k, v in p.items():
        r[k[:3]] += v
    return {k: v for k, v in r.items() if v != 0}


def flit(v):
    f = float(v)
    s = repr(f)
    if "e" not in s and "." not in s:
        s += ".0"
    return s + "f"


def emit():
    N = numerators()
    out = []
    w = out.append
    w("// GENERATED by gen_fmm.py -- do not edit; see that file for the derivation.")
    w("#pragma once")
    w("namespace pkdg {")
    w("constexpr int kNLoc = %d;   // local-expansion coefficients, |n| <= 5" % len(IDX))
    w("")
    w("// p[i] = x^a y^b z^c for the 56 multi-indices (a, b, c) in the order n = 0..5, a = n..0, b = n-a..0")
    w("__device__ __forceinline__ void fmm_monomials(const float x, const float y, const float z, float (&p)[kNLoc]) {")
    w("    p[0] = 1.0f;")
    for i, k in enumerate(IDX[1:], 1):
        axis = next(a for a in range(3) if k[a] > 0)
        prev = list(k); prev[axis] -= 1
        w("    p[%d] = p[%d] * %s;" % (i, POS[tuple(prev)], "xyz"[axis]))
    w("}")
    w("")
    w("// d[i] = lambda^|k| d^k(1/|R|): p = monomials of the unit vector R/|R|, g[n] = (lambda/|R|)^n / |R|")
    w("__device__ __forceinline__ void fmm_derivs(const float (&p)[kNLoc], const float (&g)[%d], float (&d)[kNLoc]) {" % (ORDER + 1))
    nterms = 0
    for i, k in enumerate(IDX):
        if k[2] > 2:
            continue            # n and m have at most one z each: no D with three or more z is ever read
        poly = on_unit_sphere(N[k])
        terms = sorted(poly.items(), key=lambda kv: -sum(kv[0]))
        nterms += len(terms)
        expr = None
        for mono, c in terms:
            t = "%s * p[%d]" % (flit(c), POS[mono])
            expr = t if expr is None else "fmaf(%s, p[%d], %s)" % (flit(c), POS[mono], expr)
        w("    d[%d] = g[%d] * (%s);" % (i, sum(k), expr))
    w("}")
    w("")
    pairs = [(n, m) for n in IND for m in MOMF if sum(n) + sum(m) <= ORDER]
    w("// L[n] += sum_m F[m] d[n + m] over the 36 n and 22 folded m with at most one z: %d multiply-adds." % len(pairs))
    w("constexpr int kNRed = %d;   // accumulated local coefficients (n_z <= 1)" % len(IND))
    w("constexpr int kNFold = %d;  // folded moments (m_z <= 1)" % len(MOMF))
    w("__device__ __forceinline__ void fmm_m2l_cell(const float (&d)[kNLoc], const float (&F)[kNFold], float (&L)[kNRed]) {")
    for n in IND:
        for m in MOMF:
            if sum(n) + sum(m) > ORDER:
                continue
            nm = tuple(a + b for a, b in zip(n, m))
            w("    L[%d] = fmaf(F[%d], d[%d], L[%d]);" % (POSI[n], POSF[m], POS[nm], POSI[n]))
    w("}")
    w("")
    # folded moments: F[m] = sc[|m|] * sum_{m'} c(m', m) / m'! * q[rec(m')]
    def rec_of(m):
        n = sum(m)
        base = {0: 3, 2: 4, 3: 10, 4: 20}[n]
        return base + [k for k in multi_indices(n) if sum(k) == n].index(m)
    w("// F[m] = sc[|m|] * sum_m' c(m', m) q[m'] / m'!  (q = the canonical record; sc[r] = -(-1)^r / lambda^r)")
    w("__device__ __forceinline__ void fmm_fold_moments(const float (&q)[36], const float sc0, const float sc2, const float sc3,")
    w("                                                 const float sc4, float (&F)[kNFold]) {")
    nfold_terms = 0
    for m in MOMF:
        terms = []
        for mp in MOM:
            if sum(mp) != sum(m) or sum(mp) == 1:
                continue
            c = reduce_z(mp).get(m, 0)
            if c:
                terms.append((Fraction(c, math.factorial(mp[0]) * math.factorial(mp[1]) * math.factorial(mp[2])), rec_of(mp)))
        nfold_terms += len(terms)
        expr = None
        for c, r in terms:
            expr = "%s * q[%d]" % (flit(c), r) if expr is None else "fmaf(%s, q[%d], %s)" % (flit(c), r, expr)
        w("    F[%d] = sc%d * (%s);" % (POSF[m], sum(m), expr))
    w("}")
    w("")
    w("__device__ __forceinline__ void fmm_m2l_particle(const float (&d)[kNLoc], const float mu0, float (&L)[kNRed]) {")
    for n in IND:
        w("    L[%d] = fmaf(mu0, d[%d], L[%d]);" % (POSI[n], POS[n], POSI[n]))
    w("}")
    w("")
    w("// all 56 coefficients from the 36 accumulated ones: full[k] = sum_j kExpCoef[k][j] * red[kExpIdx[k][j]]")
    exp = []
    for k in IDX:
        t = sorted(reduce_z(k).items(), key=lambda kv: POSI[kv[0]])
        assert 1 <= len(t) <= 3
        t = t + [(IND[0], 0)] * (3 - len(t))
        exp.append(t)
    w("__device__ constexpr int kExpIdx[kNLoc][3] = {%s};" % ", ".join("{%s}" % ", ".join(str(POSI[n]) for n, _ in t) for t in exp))
    w("__device__ constexpr float kExpCoef[kNLoc][3] = {%s};" % ", ".join("{%s}" % ", ".join(flit(c) for _, c in t) for t in exp))
    w("")
    w("// 1 / n! of the 56 local coefficients")
    w("__device__ constexpr float kLocInvFact[kNLoc] = {%s};" % ", ".join(
        flit(Fraction(1, math.factorial(k[0]) * math.factorial(k[1]) * math.factorial(k[2]))) for k in IDX))
    w("")
    w("// phi = sum_n Lam[n] sigma^n and its gradient; p = monomials of sigma")
    w("__device__ __forceinline__ void fmm_eval(const float (&p)[kNLoc], const float* __restrict__ Lam, float& phi, float& gx,")
    w("                                         float& gy, float& gz) {")
    w("    phi = 0.0f; gx = 0.0f; gy = 0.0f; gz = 0.0f;")
    for i, k in reversed(list(enumerate(IDX))):      # small terms first
        w("    { const float l = Lam[%d];" % i)
        w("      phi = fmaf(l, p[%d], phi);" % i)
        for axis, gname in enumerate(("gx", "gy", "gz")):
            if k[axis]:
                lower = list(k); lower[axis] -= 1
                w("      %s = fmaf(%s * l, p[%d], %s);" % (gname, flit(k[axis]), POS[tuple(lower)], gname))
        w("    }")
    w("}")
    w("}  // namespace pkdg")
    return "\n".join(out) + "\n", nterms, len(pairs), nfold_terms


def main():
    text, nterms, npairs, nfold = emit()
    with open(os.path.join(HERE, "pkdg_fmm_gen.cuh"), "w") as f:
        f.write(text)
    print("pkdg_fmm_gen.cuh: %d derivative terms, %d shift multiply-adds, %d moment-folding terms" % (nterms, npairs, nfold))


if __name__ == "__main__":
    main()
