"""-m "not gpu": pins of the oracle's cell-cell / cell-particle / local-expansion functions (SURVEY.md sec
8(f) NEXT-4; readings A20-A22) against things that are NOT the oracle's own formula: the Legendre
series of a point mass, hand values, the already-pinned P-C pair (potential and its exact gradient at the sink
centre), finite differences, direct summation with the (size / distance)^6 law of a total-order-5 scheme, and
the exactly-once coverage of the four-list walk.
"""
import numpy as np
import pytest
from numpy.polynomial import legendre

import oracle
from paper_1609_08621_b200 import inputs

IDX = oracle.local_index()
POS = {k: i for i, k in enumerate(IDX)}


def _fact(k):
    import math
    return float(np.prod([math.factorial(v) for v in k]))


def _poly(L, s):
    return sum(L[i] * s[0] ** a * s[1] ** b * s[2] ** c for i, (a, b, c) in enumerate(IDX))


def test_local_index_order_matches_the_moments():
    assert len(IDX) == 56 and IDX[0] == (0, 0, 0) and IDX[1:4] == [(1, 0, 0), (0, 1, 0), (0, 0, 1)]
    assert IDX[4:10] == [(2, 0, 0), (1, 1, 0), (1, 0, 1), (0, 2, 0), (0, 1, 1), (0, 0, 2)]     # xx xy xz yy yz zz
    assert [sum(k) for k in IDX] == [0] + [1] * 3 + [2] * 6 + [3] * 10 + [4] * 15 + [5] * 21


def test_cell_particle_is_the_legendre_series_of_a_point_mass():
    """One source particle: sum_n L_n s^n is the Taylor polynomial of -m / |R + s| in s, whose degree-n part is
    -m |s|^n / |R|^(n+1) P_n(-mu) (textbook generating function of the Legendre polynomials)."""
    rng = np.random.default_rng(0)
    for _ in range(20):
        zB = rng.random(3); xs = zB + rng.standard_normal(3) * 0.7; m = rng.uniform(0.5, 2.0)
        L = oracle.cp_accumulate(zB, xs, m)
        R = zB - xs; Rn = np.linalg.norm(R)
        assert abs(L[0] + m / Rn) < 1e-15 * m / Rn                                     # L_000 = -m / |R|
        assert np.allclose(L[1:4], m * R / Rn ** 3, rtol=1e-14, atol=0)                # L_e = -m d(1/r) = m R / |R|^3
        s = rng.standard_normal(3); s *= 0.2 * Rn / np.linalg.norm(s)
        sn = np.linalg.norm(s); mu = float(R @ s) / (Rn * sn)
        want = -m * sum(sn ** n / Rn ** (n + 1) * legendre.legval(-mu, [0] * n + [1]) for n in range(6))
        acc, pot = oracle.local_eval(zB, L, zB + s)
        assert abs(pot - want) < 1e-13 * abs(want)
        assert abs(pot - _poly(L, s)) < 1e-14 * abs(pot)
        exact = -m / np.linalg.norm(R + s)
        assert abs(pot - exact) < 2.0 * 0.2 ** 6 * abs(exact)                           # remainder of order (s/R)^6
        # acceleration = minus the gradient of the polynomial (central differences)
        h = 1e-5 * Rn
        for l in range(3):
            e = np.zeros(3); e[l] = h
            fd = -(oracle.local_eval(zB, L, zB + s + e)[1] - oracle.local_eval(zB, L, zB + s - e)[1]) / (2 * h)
            assert abs(acc[l] - fd) < 1e-7 * np.linalg.norm(acc)


def test_cell_particle_coefficients_are_the_taylor_coefficients():
    rng = np.random.default_rng(1)
    zB = rng.random(3); xs = rng.random(3) + 2.0; m = 1.7
    L = oracle.cp_accumulate(zB, xs, m)
    t = oracle.taylor_coeffs(zB - xs, 5)
    for i, (a, b, c) in enumerate(IDX):
        assert L[i] == -m * t[a, b, c]
    # accumulation adds
    L2 = oracle.cp_accumulate(zB, xs + 0.3, 0.4, L.copy())
    assert np.allclose(L2 - L, oracle.cp_accumulate(zB, xs + 0.3, 0.4), rtol=1e-13, atol=0)


def _cloud_record(rng, centre, b, k=64):
    pts = np.empty((k, 4), np.float32)
    v = rng.standard_normal((k, 3)); v *= (b * rng.random(k) ** (1 / 3) / np.linalg.norm(v, axis=1))[:, None]
    pts[:, :3] = centre + v; pts[:, 3] = rng.uniform(0.5, 1.5, k) / k
    return pts, inputs.cloud_records(pts, k)[0]


def test_cell_cell_low_orders_are_the_pinned_pc_pair_at_the_sink_centre():
    """|n| = 0 keeps every moment and |n| = 1 keeps moments up to order 4: L_0 is the P-C potential at the sink
    centre and (L_x, L_y, L_z) minus its acceleration -- both from orc_pc_pair, which is pinned independently."""
    rng = np.random.default_rng(2)
    for _ in range(10):
        _, rec = _cloud_record(rng, rng.random(3), 0.05)
        zB = rec[:3].astype(np.float64) + rng.standard_normal(3) * 0.4
        L = oracle.cc_accumulate(zB, rec)
        acc, pot = oracle.pc_pair(zB, rec)
        assert abs(L[0] - pot) < 1e-14 * abs(pot)
        assert np.allclose(L[1:4], -acc, rtol=1e-13, atol=1e-16 * np.linalg.norm(acc))


def test_cell_cell_higher_orders_by_finite_differences_of_truncated_pc_pairs():
    """|n| = 2 keeps moments up to order 3, |n| = 3 up to order 2, |n| = 4, 5 the monopole only (total order <= 5).
    L_n = d^n phi_trunc / n! with phi_trunc the P-C potential of the record with the higher moments removed:
    taken as central differences of orc_pc_pair's ACCELERATION (the exact gradient), so one order of
    differencing less than the derivative."""
    rng = np.random.default_rng(3)
    _, rec = _cloud_record(rng, np.array([0.3, 0.4, 0.5]), 0.08)
    zB = rec[:3].astype(np.float64) + np.array([0.5, -0.3, 0.4])
    L = oracle.cc_accumulate(zB, rec)
    r3 = rec.copy(); r3[20:35] = 0.0          # moments up to order 3
    r2 = r3.copy(); r2[10:20] = 0.0           # up to order 2
    r0 = r2.copy(); r0[4:10] = 0.0            # monopole
    h = 2e-4
    E = np.eye(3)
    # |n| = 2: d_k d_l phi = -d_l a_k
    for k in range(3):
        for l in range(k, 3):
            fd = -(oracle.pc_pair(zB + h * E[l], r3)[0][k] - oracle.pc_pair(zB - h * E[l], r3)[0][k]) / (2 * h)
            n = tuple(int(x) for x in E[k] + E[l])
            assert abs(L[POS[n]] - fd / _fact(n)) < 1e-6 * abs(L[4:10]).max(), n
    # |n| = 3: d_j d_k d_l phi = -(second difference of a_j)
    for n in [k for k in IDX if sum(k) == 3]:
        axes = [d for d in range(3) for _ in range(n[d])]
        j, k, l = axes
        f = lambda x: oracle.pc_pair(x, r2)[0][j]
        if k == l:
            fd = -(f(zB + h * E[k]) - 2 * f(zB) + f(zB - h * E[k])) / h ** 2
        else:
            fd = -(f(zB + h * E[k] + h * E[l]) - f(zB + h * E[k] - h * E[l]) - f(zB - h * E[k] + h * E[l])
                   + f(zB - h * E[k] - h * E[l])) / (4 * h ** 2)
        assert abs(L[POS[n]] - fd / _fact(n)) < 2e-5 * abs(L[10:20]).max(), n
    # |n| = 4, 5: monopole only
    t = oracle.taylor_coeffs(zB - rec[:3].astype(np.float64), 5)
    for i, (a, b, c) in enumerate(IDX):
        if a + b + c >= 4:
            assert abs(L[i] + float(rec[3]) * t[a, b, c]) < 1e-14 * abs(L[i]) + 1e-300
    # and a record with only a monopole is a particle at the centre of mass
    Lm = oracle.cc_accumulate(zB, r0)
    assert np.allclose(Lm, oracle.cp_accumulate(zB, r0[:3].astype(np.float64), float(r0[3])), rtol=1e-14, atol=0)


def test_local_eval_is_the_polynomial_and_its_gradient():
    rng = np.random.default_rng(4)
    L = rng.standard_normal(56); zB = rng.random(3); s = 0.3 * rng.standard_normal(3)
    acc, pot = oracle.local_eval(zB, L, zB + s)
    assert abs(pot - _poly(L, s)) < 1e-13 * abs(pot)
    h = 1e-6
    for l in range(3):
        e = np.zeros(3); e[l] = h
        assert abs(acc[l] + (_poly(L, s + e) - _poly(L, s - e)) / (2 * h)) < 1e-7 * np.linalg.norm(acc)
    # a constant-plus-linear expansion is a uniform field
    L = np.zeros(56); L[0] = -2.0; L[1:4] = [0.5, -1.0, 0.25]
    acc, pot = oracle.local_eval(zB, L, zB + s)
    assert np.allclose(acc, [-0.5, 1.0, -0.25], atol=1e-15) and abs(pot - (-2.0 + L[1:4] @ s)) < 1e-14


def test_cell_cell_converges_to_the_direct_sum_with_the_sixth_power():
    """A 64-particle source cloud (radius b) and sinks within b of the sink centre: local expansion vs direct
    summation.  Total order 5 => the error falls as (b / d)^6 when the separation d doubles."""
    rng = np.random.default_rng(5)
    b = 0.02
    pts, rec = _cloud_record(rng, np.array([0.5, 0.5, 0.5]), b)
    u = np.array([0.6, -0.5, 0.62]); u /= np.linalg.norm(u)
    sv = rng.standard_normal((32, 3)); sv *= (b * rng.random(32) ** (1 / 3) / np.linalg.norm(sv, axis=1))[:, None]
    errs_a, errs_p = [], []
    for d in (4 * b, 8 * b, 16 * b):        # beyond 16 b the fp32 storage of the record (6e-8) is the floor
        zB = rec[:3].astype(np.float64) + d * u
        L = oracle.cc_accumulate(zB, rec)
        ea = ep = 0.0
        for s in sv:
            acc, pot = oracle.local_eval(zB, L, zB + s)
            da = np.zeros(3); dp = 0.0
            for q in pts:
                r = zB + s - q[:3].astype(np.float64); rn = np.linalg.norm(r)
                da -= float(q[3]) * r / rn ** 3; dp -= float(q[3]) / rn
            ea = max(ea, np.linalg.norm(acc - da) / np.linalg.norm(da)); ep = max(ep, abs(pot - dp) / abs(dp))
        errs_a.append(ea); errs_p.append(ep)
    for e in (errs_a, errs_p):
        slopes = [np.log2(e[i] / e[i + 1]) for i in range(2)]
        assert all(4.6 < sl < 7.5 for sl in slopes), (e, slopes)      # acceleration loses one order: ~5, potential ~6
    assert errs_a[0] < 1e-2 and errs_p[0] < 1e-3 and errs_a[2] < 1e-5
    slopes_p = [np.log2(errs_p[i] / errs_p[i + 1]) for i in range(2)]
    assert slopes_p[0] > 5.5 and slopes_p[1] > 4.8, slopes_p     # the second octave already feels the fp32 storage floor


@pytest.mark.parametrize("theta", [0.7, 0.5])
def test_fmm_lists_cover_every_particle_once_and_match_direct_summation(theta):
    """The four-list walk (P-P, P-C, C-P, C-C): coverage is exact; the whole path (P-P + P-C per sink, C-C + C-P
    through the local expansion) agrees with direct summation within the expansion error, which shrinks with
    theta; the local-expansion part alone is a sizeable share of the force (the lists are not empty)."""
    p = inputs.config1(2048, seed=7, theta=theta)
    F = inputs.build_fmm_lists(p, theta, p.eps)
    tr = p.tree
    for b in (0, 17, p.n_buckets // 2, p.n_buckets - 1):
        cov = np.zeros(p.n, int)
        for k in ("pp", "cp"):
            o, i = F[k]; np.add.at(cov, i[o[b]:o[b + 1]], 1)
        for k in ("pc", "cc"):
            o, i = F[k]
            for c in i[o[b]:o[b + 1]]:
                cov[tr["first"][c]:tr["first"][c] + tr["count"][c]] += 1
        assert (cov == 1).all()
        own = np.arange(p.first[b], p.first[b] + p.count[b])
        o, i = F["pp"]; assert np.isin(own, i[o[b]:o[b + 1]]).all()         # a bucket's own particles are P-P
    assert len(F["cc"][1]) > 0 and len(F["cp"][1]) > 0 and len(F["pc"][1]) > 0
    near = oracle.gravity_eval(p.xyzm, p.cells, p.first, p.count, F["pp"][0], F["pp"][1], F["pc"][0], F["pc"][1], p.eps)
    tot, L = oracle.fmm_eval(p.xyzm, p.cells, p.first, p.count, F["centre"], F["cc"][0], F["cc"][1], F["cp"][0], F["cp"][1],
                             out=near.copy(), want_L=True)
    ds = oracle.direct_sum(p.xyzm, p.eps)
    err = np.linalg.norm(tot[:, :3] - ds[:, :3], axis=1) / np.linalg.norm(ds[:, :3], axis=1)
    rms = float(np.sqrt(np.mean(err ** 2)))
    assert rms < (6e-3 if theta == 0.7 else 8e-4), rms          # falls as ~theta^6 (5e-3 at 0.7, 6e-4 at 0.5)
    # ... and is no worse than the per-sink (P-P + P-C only) lists of the same tree at the same theta, whose
    # oracle is pinned in test_oracle_pins.py: the sink-side expansion adds little to the source-side error
    bh = oracle.gravity_eval(p.xyzm, p.cells, p.first, p.count, p.pp_off, p.pp_idx, p.pc_off, p.pc_idx, p.eps)
    err_bh = np.linalg.norm(bh[:, :3] - ds[:, :3], axis=1) / np.linalg.norm(ds[:, :3], axis=1)
    assert rms < 1.25 * float(np.sqrt(np.mean(err_bh ** 2)))
    assert np.abs(tot[:, 3] - ds[:, 3]).max() < 1e-3 * np.abs(ds[:, 3]).max()
    far = tot - near
    assert np.median(np.linalg.norm(far[:, :3], axis=1) / np.linalg.norm(tot[:, :3], axis=1)) > 0.05
    assert L.shape == (p.n_buckets, 56) and np.isfinite(L).all()
