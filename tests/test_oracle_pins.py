"""Pins of the fp64 oracle against things other than itself (-m "not gpu").

The paper prints no kernel formula and no worked example (tests/golden/README.md), so the
oracle is pinned to closed forms, textbook series, quadrature, brute force and invariants,
chosen so that a dropped term, a wrong sign or index, or a transposed operand fails one of
them.  Citations: SURVEY.md sec 8(c) table "What pins each part", BASELINE.json north_star
(the four self-checks).
"""
import math
import os

import numpy as np
import pytest
from scipy import integrate, special

import oracle
from paper_1609_08621_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden")


# ----------------------------------------------------------------------------- spline (A1, A2)
def _W(u):
    """Monaghan-Lattanzio cubic-spline density of unit mass and support 1 (textbook)."""
    if u < 0.5:
        return 8 / math.pi * (1 - 6 * u * u + 6 * u ** 3)
    if u < 1.0:
        return 8 / math.pi * 2 * (1 - u) ** 3
    return 0.0


def test_spline_density_has_unit_mass():
    m, _ = integrate.quad(lambda s: 4 * math.pi * s * s * _W(s), 0, 1, points=[0.5])
    assert abs(m - 1) < 1e-12


@pytest.mark.parametrize("u", [0.05, 0.2, 0.4, 0.5, 0.6, 0.8, 0.95, 1.0, 1.7])
def test_spline_matches_quadrature_of_density(u):
    """g(u) = M(<u)/u^3, w(u) = -M(<u)/u - int_u^1 4 pi s W ds (Newton's shell theorems)."""
    menc, _ = integrate.quad(lambda s: 4 * math.pi * s * s * _W(s), 0, min(u, 1), points=[0.5] if u > 0.5 else None)
    outer, _ = integrate.quad(lambda s: 4 * math.pi * s * _W(s), min(u, 1), 1, points=[0.5] if u < 0.5 else None)
    g, w = oracle.spline(u)
    assert g == pytest.approx(menc / u ** 3, rel=1e-11)
    assert w == pytest.approx(-menc / u - outer, rel=1e-11)


def test_spline_closed_forms():
    g0, w0 = oracle.spline(0.0)
    assert g0 == pytest.approx(32 / 3, rel=1e-15)
    assert w0 == pytest.approx(-14 / 5, rel=1e-15)          # phi(0) = -1.4 m / eps
    gh, wh = oracle.spline(0.5)
    gl, wl = oracle.spline(0.5 - 1e-12)
    assert gh == pytest.approx(gl, rel=1e-9) and wh == pytest.approx(wl, rel=1e-9)
    assert wh == pytest.approx(-28 / 15, rel=1e-12)
    g1, w1 = oracle.spline(1.0)
    gl, wl = oracle.spline(1.0 - 1e-12)
    assert g1 == pytest.approx(1.0) and w1 == pytest.approx(-1.0)
    assert gl == pytest.approx(1.0, rel=1e-9) and wl == pytest.approx(-1.0, rel=1e-9)
    for u in (1.0, 2.5, 40.0):                               # exactly Newtonian beyond the support
        g, w = oracle.spline(u)
        assert g == pytest.approx(u ** -3, rel=1e-15) and w == pytest.approx(-1 / u, rel=1e-15)


@pytest.mark.parametrize("u", [0.1, 0.3, 0.49, 0.51, 0.7, 0.9, 1.3])
def test_spline_force_is_gradient_of_potential(u):
    """dw/du = u g(u)."""
    d = 1e-6
    wp = oracle.spline(u + d)[1]; wm = oracle.spline(u - d)[1]
    assert (wp - wm) / (2 * d) == pytest.approx(u * oracle.spline(u)[0], rel=1e-7)


def test_pp_pair_sign_and_scaling():
    eps = 0.05
    acc, pot = oracle.pp_pair([1.0, 0, 0], [0, 0, 0], 2.0, eps)     # r = 1 > h: Newtonian
    assert np.allclose(acc, [-2.0, 0, 0], rtol=1e-15) and pot == pytest.approx(-2.0)
    acc, pot = oracle.pp_pair([0.0, 0.03, 0], [0, 0, 0], 2.0, eps)  # u = 0.3
    g, w = oracle.spline(0.3)
    assert np.allclose(acc, [0, -2.0 * 0.03 * g / 0.1 ** 3, 0], rtol=1e-14)
    assert pot == pytest.approx(2.0 * w / 0.1, rel=1e-14)


# ----------------------------------------------------------------------------- P-P path
def _all_pairs_problem(n, seed, eps_scale):
    rng = np.random.default_rng(seed)
    xyzm = np.empty((n, 4), np.float32)
    xyzm[:, :3] = rng.random((n, 3))
    xyzm[:, 3] = rng.uniform(0.5, 1.5, n) / n
    first = np.arange(0, n, 7, dtype=np.int32)
    count = np.minimum(7, n - first).astype(np.int32)
    nb = first.size
    pp_off = np.arange(nb + 1, dtype=np.int64) * n
    pp_idx = np.tile(np.arange(n, dtype=np.int32), nb)
    return xyzm, first, count, pp_off, pp_idx


def test_pp_newtonian_against_numpy_brute_force():
    """north_star self-check 1: P-P against brute-force direct summation on tiny N (textbook
    a_i = -sum m_j d/|d|^3, phi_i = -sum m_j/|d|), written independently in numpy."""
    n = 97
    xyzm, first, count, pp_off, pp_idx = _all_pairs_problem(n, 11, 0)
    x = xyzm[:, :3].astype(np.float64); m = xyzm[:, 3].astype(np.float64)
    d = x[:, None, :] - x[None, :, :]
    r = np.sqrt((d ** 2).sum(-1)); np.fill_diagonal(r, np.inf)
    eps = 0.4 * r.min()                                           # every pair beyond h = 2 eps
    a_ref = -(m[None, :, None] * d / r[:, :, None] ** 3).sum(1)
    p_ref = -(m[None, :] / r).sum(1)
    out = oracle.gravity_eval(xyzm, None, first, count, pp_off, pp_idx, None, None, eps)
    assert np.allclose(out[:, :3], a_ref, rtol=1e-11, atol=1e-13 * np.abs(a_ref).max())
    assert np.allclose(out[:, 3], p_ref, rtol=1e-13)
    ds = oracle.direct_sum(xyzm, eps)
    assert np.allclose(ds, out, rtol=1e-11, atol=1e-13 * np.abs(a_ref).max())


def test_pp_softened_against_numpy_brute_force():
    n = 64
    xyzm, first, count, pp_off, pp_idx = _all_pairs_problem(n, 12, 0)
    x = xyzm[:, :3].astype(np.float64); m = xyzm[:, 3].astype(np.float64)
    eps = 0.1                                                     # h = 0.2: many softened pairs
    h = 2 * eps
    a_ref = np.zeros((n, 3)); p_ref = np.zeros(n)
    for i in range(n):
        for j in range(n):
            if i == j:
                continue
            d = x[i] - x[j]; r = np.linalg.norm(d)
            menc = integrate.quad(lambda s: 4 * math.pi * s * s * _W(s), 0, min(r / h, 1), points=[0.5])[0]
            outer = integrate.quad(lambda s: 4 * math.pi * s * _W(s), min(r / h, 1), 1, points=[0.5])[0]
            a_ref[i] -= m[j] * menc * d / r ** 3
            p_ref[i] += m[j] * (-menc / r - outer / h)
    out = oracle.gravity_eval(xyzm, None, first, count, pp_off, pp_idx, None, None, eps)
    assert np.allclose(out[:, :3], a_ref, rtol=1e-9, atol=1e-12)
    assert np.allclose(out[:, 3], p_ref, rtol=1e-10)


def test_pp_momentum_conservation():
    """north_star self-check 2: zero net momentum change for an isolated all-pairs system."""
    n = 200
    xyzm, first, count, pp_off, pp_idx = _all_pairs_problem(n, 13, 0)
    for eps in (1e-4, 0.05):
        out = oracle.gravity_eval(xyzm, None, first, count, pp_off, pp_idx, None, None, eps)
        m = xyzm[:, 3].astype(np.float64)
        net = (m[:, None] * out[:, :3]).sum(0)
        scale = np.abs(m[:, None] * out[:, :3]).sum(0)
        assert np.all(np.abs(net) < 1e-13 * scale)


def test_self_skipped_by_index_and_coincident_pair_interacts():
    """Reading A11: j == i skipped by index; two distinct coincident particles interact through the
    spline: a = 0, phi = w(0) m / h = -2.8 m / h."""
    xyzm = np.array([[0.5, 0.5, 0.5, 0.25], [0.5, 0.5, 0.5, 0.75]], np.float32)
    first = np.array([0], np.int32); count = np.array([2], np.int32)
    off = np.array([0, 4], np.int64); idx = np.array([0, 1, -1, -1], np.int32)   # padding is ignored
    eps = 0.01
    out = oracle.gravity_eval(xyzm, None, first, count, off, idx, None, None, eps)
    assert np.all(out[:, :3] == 0)
    assert out[0, 3] == pytest.approx(-2.8 * 0.75 / 0.02) and out[1, 3] == pytest.approx(-2.8 * 0.25 / 0.02)


# ----------------------------------------------------------------------------- Taylor coefficients
def test_taylor_low_orders_by_hand():
    r = np.array([0.3, -1.1, 0.7]); x, y, z = r; R = np.linalg.norm(r)
    t = oracle.taylor_coeffs(r, 3)
    assert t[0, 0, 0] == pytest.approx(1 / R)
    assert t[1, 0, 0] == pytest.approx(-x / R ** 3)
    assert t[0, 0, 1] == pytest.approx(-z / R ** 3)
    assert 2 * t[2, 0, 0] == pytest.approx((3 * x * x - R * R) / R ** 5)
    assert t[1, 1, 0] == pytest.approx(3 * x * y / R ** 5)
    assert t[0, 1, 1] == pytest.approx(3 * y * z / R ** 5)
    # d_xyz(1/r) = -15 xyz / r^7 ; d_xxx / 3! = (9 x r^2 - 15 x^3) / (6 r^7)
    assert t[1, 1, 1] == pytest.approx(-15 * x * y * z / R ** 7)
    assert t[3, 0, 0] == pytest.approx((9 * x * R * R - 15 * x ** 3) / (6 * R ** 7))


def test_taylor_series_reproduces_shifted_kernel():
    """sum_k t_k(r) h^k = 1/|r + h| (order 12, |h|/|r| ~ 0.07 -> remainder ~ 1e-15)."""
    r = np.array([0.9, -0.4, 1.3]); h = np.array([0.05, 0.08, -0.06])
    t = oracle.taylor_coeffs(r, 12)
    s = 0.0
    for a in range(13):
        for b in range(13 - a):
            for c in range(13 - a - b):
                s += t[a, b, c] * h[0] ** a * h[1] ** b * h[2] ** c
    assert s == pytest.approx(1 / np.linalg.norm(r + h), rel=1e-13)


def test_taylor_coefficients_are_harmonic():
    """Laplace: sum_i (k_i+2)(k_i+1) t_{k+2e_i} = 0 for every k."""
    t = oracle.taylor_coeffs([0.2, 0.5, -0.8], 6)
    for a in range(5):
        for b in range(5 - a):
            for c in range(5 - a - b):
                lap = (a + 2) * (a + 1) * t[a + 2, b, c] + (b + 2) * (b + 1) * t[a, b + 2, c] + (c + 2) * (c + 1) * t[a, b, c + 2]
                assert abs(lap) < 1e-12 * abs(t[0, 0, 0]) * 60


# ----------------------------------------------------------------------------- P-C
def _moment_order():
    ks = []
    for n in (2, 3, 4):
        for a in range(n, -1, -1):
            for b in range(n - a, -1, -1):
                ks.append((a, b, n - a - b))
    return ks


def _record(pts, m, com=None):
    """Canonical record written independently in numpy (layout: SURVEY.md sec 8(b))."""
    pts = np.asarray(pts, np.float64); m = np.asarray(m, np.float64)
    if com is None:
        com = (m[:, None] * pts).sum(0) / m.sum()
    com = np.asarray(com, np.float32)
    s = pts - com.astype(np.float64)
    rec = np.zeros(36, np.float32)
    rec[:3] = com; rec[3] = m.sum()
    for q, (a, b, c) in enumerate(_moment_order()):
        rec[4 + q] = (m * s[:, 0] ** a * s[:, 1] ** b * s[:, 2] ** c).sum()
    rec[35] = np.sqrt((s ** 2).sum(1).max())
    return rec


def test_record_layout_order():
    ks = _moment_order()
    assert ks[:6] == [(2, 0, 0), (1, 1, 0), (1, 0, 1), (0, 2, 0), (0, 1, 1), (0, 0, 2)]
    assert len(ks) == 31 and ks[6] == (3, 0, 0) and ks[16] == (4, 0, 0) and ks[-1] == (0, 0, 4)


def test_pc_point_mass_is_legendre_series_without_dipole():
    """A single point mass m at offset s from the expansion centre: the truncated series is
    -m sum_{n in {0,2,3,4}} s^n P_n(mu) / r^(n+1) (textbook Legendre generating function; the
    dipole n=1 is dropped by reading A9)."""
    c = np.array([0.5, 0.25, 0.125]); s = np.array([0.0625, -0.03125, 0.09375]); m = 0.75
    rec = _record([c + s], [m], com=c)
    xt = c + np.array([0.9, 0.5, -0.7])
    r = xt - c; R = np.linalg.norm(r); S = np.linalg.norm(s); mu = r.dot(s) / (R * S)
    phi = -m * sum(S ** n * special.eval_legendre(n, mu) / R ** (n + 1) for n in (0, 2, 3, 4))
    _, pot = oracle.pc_pair(xt, rec)
    assert pot == pytest.approx(phi, rel=1e-7)       # record is fp32


def _cloud(rng, k, centre, radius):
    v = rng.normal(size=(k, 3)); v /= np.linalg.norm(v, axis=1)[:, None]
    pts = centre + radius * rng.random(k)[:, None] ** (1 / 3) * v
    m = rng.uniform(0.5, 1.5, k) / k
    return pts.astype(np.float32).astype(np.float64), m.astype(np.float32).astype(np.float64)


def _direct(xt, pts, m):
    d = xt - pts; r = np.linalg.norm(d, axis=1)
    return -(m[:, None] * d / r[:, None] ** 3).sum(0), -(m / r).sum()


def test_pc_cloud_converges_to_direct_sum_as_fifth_power():
    """north_star self-check 3: P-C of a k-particle cell against direct summation, error falling
    as (r_cell/d)^5.  Equal power-of-two masses and a cloud centred on the origin keep the fp32
    record exact in mass and centre, so the slope is visible over four octaves; the error is the
    rms over 12 directions."""
    rng = np.random.default_rng(5)
    pts, m = _cloud(rng, 64, np.zeros(3), 0.05)
    m[:] = 2.0 ** -6
    pts = pts - (m[:, None] * pts).sum(0) / m.sum()
    rec = _record(pts, m, com=np.zeros(3))
    b = float(rec[35])
    us = rng.normal(size=(12, 3)); us /= np.linalg.norm(us, axis=1)[:, None]
    ea, ep = [], []
    for mult in (2, 4, 8, 16, 32):
        da, dp = [], []
        for u in us:
            xt = mult * b * u
            acc, pot = oracle.pc_pair(xt, rec)
            a_d, p_d = _direct(xt, pts, m)
            da.append(np.linalg.norm(acc - a_d) / np.linalg.norm(a_d)); dp.append(abs(pot - p_d) / abs(p_d))
        ea.append(np.sqrt(np.mean(np.square(da)))); ep.append(np.sqrt(np.mean(np.square(dp))))
    sa = np.log2(np.array(ea[:-1]) / np.array(ea[1:])); sp = np.log2(np.array(ep[:-1]) / np.array(ep[1:]))
    assert ea[0] < 1e-2 and ep[0] < 1e-3
    assert np.all(np.abs(sa - 5) < 0.25) and np.all(np.abs(sp - 5) < 0.25)


def test_pc_each_order_matters():
    """Zeroing any one of the orders 2, 3, 4 spoils the agreement with the direct sum: guards
    against a dropped order or a wrong sign of the odd order."""
    rng = np.random.default_rng(6)
    pts, m = _cloud(rng, 32, np.array([0.3, 0.6, 0.4]), 0.04)
    pts[:, 0] += 0.03 * (pts[:, 1] - 0.6) ** 2 / 0.04         # skew it so the octupole is not small
    rec = _record(pts, m)
    xt = rec[:3].astype(np.float64) + 5.0 * float(rec[35]) * np.array([0.48, 0.6, -0.64])
    a_d, _ = _direct(xt, pts, m)
    full = np.linalg.norm(oracle.pc_pair(xt, rec)[0] - a_d)
    for lo, hi in ((4, 10), (10, 20), (20, 35)):
        r2 = rec.copy(); r2[lo:hi] = 0
        assert np.linalg.norm(oracle.pc_pair(xt, r2)[0] - a_d) > 2 * full
        r3 = rec.copy(); r3[lo:hi] *= -1
        assert np.linalg.norm(oracle.pc_pair(xt, r3)[0] - a_d) > 2 * full


def test_pc_acceleration_is_gradient_of_truncated_potential():
    rng = np.random.default_rng(7)
    pts, m = _cloud(rng, 20, np.array([0.4, 0.4, 0.6]), 0.05)
    rec = _record(pts, m)
    xt = rec[:3].astype(np.float64) + np.array([0.11, -0.17, 0.13])
    acc, _ = oracle.pc_pair(xt, rec)
    d = 1e-5
    for ax in range(3):
        e = np.zeros(3); e[ax] = d
        g = (oracle.pc_pair(xt + e, rec)[1] - oracle.pc_pair(xt - e, rec)[1]) / (2 * d)
        assert acc[ax] == pytest.approx(-g, rel=1e-7, abs=1e-9)


def test_pc_rotation_covariance_and_axis_permutation():
    rng = np.random.default_rng(8)
    pts, m = _cloud(rng, 24, np.zeros(3), 0.0625)
    xt = np.array([0.25, -0.375, 0.5])
    acc, pot = oracle.pc_pair(xt, _record(pts, m, com=np.zeros(3)))
    # cyclic permutation (x,y,z) -> (y,z,x): exact in floating point
    P = [1, 2, 0]
    acc2, pot2 = oracle.pc_pair(xt[P], _record(pts[:, P], m, com=np.zeros(3)))
    assert np.allclose(acc2, acc[P], rtol=1e-12, atol=1e-15) and pot2 == pytest.approx(pot, rel=1e-13)
    # a general rotation
    A = rng.normal(size=(3, 3)); Q, _ = np.linalg.qr(A)
    acc3, pot3 = oracle.pc_pair(Q @ xt, _record(pts @ Q.T, m, com=np.zeros(3)))
    assert np.allclose(acc3, Q @ acc, rtol=0, atol=3e-6 * np.linalg.norm(acc))
    assert pot3 == pytest.approx(pot, rel=1e-6)


def test_pc_trace_invariance_and_linearity():
    """d^n(1/r) is trace-free: adding c*delta_ij to M^(2) changes nothing (SURVEY sec 8(c) iv)."""
    rng = np.random.default_rng(9)
    pts, m = _cloud(rng, 16, np.array([0.5, 0.5, 0.5]), 0.05)
    rec = _record(pts, m)
    xt = np.array([0.8, 0.3, 0.65])
    acc, pot = oracle.pc_pair(xt, rec)
    r2 = rec.copy(); c = np.float32(2.0 ** -10)
    r2[4] += c; r2[7] += c; r2[9] += c                          # xx, yy, zz
    acc2, pot2 = oracle.pc_pair(xt, r2)
    assert np.allclose(acc2, acc, rtol=0, atol=1e-6 * np.linalg.norm(acc)) and pot2 == pytest.approx(pot, rel=1e-6)
    r3 = rec.copy(); r3[3:35] *= np.float32(4.0)                # exact in fp32
    acc3, pot3 = oracle.pc_pair(xt, r3)
    assert np.allclose(acc3, 4 * acc, rtol=1e-14) and pot3 == pytest.approx(4 * pot, rel=1e-14)


def test_generator_records_match_numpy_records(cfg1):
    """The harness's C moment code against the independent numpy record above."""
    p = cfg1
    t = p.tree
    for c in (0, 1, 5, int(t["leaf_cell"][3]), p.cells.shape[0] - 1):
        lo = int(t["first"][c]); hi = lo + int(t["count"][c])
        rec = _record(p.xyzm[lo:hi, :3], p.xyzm[lo:hi, 3], com=p.cells[c, :3])
        ref_com = (p.xyzm[lo:hi, 3:4].astype(np.float64) * p.xyzm[lo:hi, :3]).sum(0) / p.xyzm[lo:hi, 3].astype(np.float64).sum()
        assert np.allclose(p.cells[c, :3], ref_com, rtol=1e-6)
        assert np.allclose(p.cells[c], rec, rtol=2e-6, atol=1e-12)


# ----------------------------------------------------------------------------- tree + lists + kernels
def test_lists_cover_every_particle_exactly_once(cfg1):
    """Integer coverage invariant: for every bucket, P-P particles and the
    particles of the P-C cells are all N particles exactly once; masses sum to 1."""
    p = cfg1; t = p.tree
    for b in range(0, p.n_buckets, 37):
        seen = np.zeros(p.n, np.int32)
        np.add.at(seen, p.pp_idx[p.pp_off[b]:p.pp_off[b + 1]], 1)
        for c in p.pc_idx[p.pc_off[b]:p.pc_off[b + 1]]:
            seen[t["first"][c]: t["first"][c] + t["count"][c]] += 1
        assert np.all(seen == 1)
        mass = p.xyzm[p.pp_idx[p.pp_off[b]:p.pp_off[b + 1]], 3].astype(np.float64).sum() + \
            p.cells[p.pc_idx[p.pc_off[b]:p.pc_off[b + 1]], 3].astype(np.float64).sum()
        assert mass == pytest.approx(1.0, rel=1e-5)
    assert p.first[0] == 0 and np.all(p.first[1:] == p.first[:-1] + p.count[:-1]) and p.count.max() <= 16


def test_full_tree_force_against_direct_sum_and_theta_scaling():
    """north_star self-check 4: tree + lists against direct summation within the error expected
    at the opening angle (rms 2.4e-3 / 5e-4 / 1e-4 at theta 0.7 / 0.55 / 0.4)."""
    x = inputs.particles_uniform(4096, 1)
    rms = {}
    for theta in (0.7, 0.55, 0.4):
        p = inputs.build_tree(x, "octree", 16)
        inputs.with_lists(p, theta, 0.02 * 4096 ** (-1 / 3))
        out = oracle.gravity_eval(p.xyzm, p.cells, p.first, p.count, p.pp_off, p.pp_idx, p.pc_off, p.pc_idx, p.eps)
        ds = oracle.direct_sum(p.xyzm, p.eps)
        rel = np.linalg.norm(out[:, :3] - ds[:, :3], axis=1) / np.linalg.norm(ds[:, :3], axis=1)
        rms[theta] = float(np.sqrt(np.mean(rel ** 2)))
        assert np.median(rel) < {0.7: 1.5e-3, 0.55: 5e-4, 0.4: 1.5e-4}[theta]
        assert np.abs(out[:, 3] / ds[:, 3] - 1).max() < 1e-3
    assert rms[0.7] < 5e-3 and rms[0.55] < 1.2e-3 and rms[0.4] < 3e-4
    assert rms[0.7] / rms[0.55] > 2.5 and rms[0.55] / rms[0.4] > 2.5      # ~ theta^5..6
    # the paper's accuracy statement (<0.1 % rms) is met at theta = 0.55
    assert rms[0.55] < 1e-3


def test_binary_tree_also_within_band():
    x = inputs.particles_uniform(4096, 1)
    p = inputs.build_tree(x, "binary", 16)
    inputs.with_lists(p, 0.7, 0.02 * 4096 ** (-1 / 3))
    out = oracle.gravity_eval(p.xyzm, p.cells, p.first, p.count, p.pp_off, p.pp_idx, p.pc_off, p.pc_idx, p.eps)
    ds = oracle.direct_sum(p.xyzm, p.eps)
    rel = np.linalg.norm(out[:, :3] - ds[:, :3], axis=1) / np.linalg.norm(ds[:, :3], axis=1)
    assert np.sqrt(np.mean(rel ** 2)) < 5e-3 and p.count.mean() > 9


def test_sel_evaluates_only_selected_buckets(cfg1):
    p = cfg1
    full = oracle.gravity_eval(p.xyzm, p.cells, p.first, p.count, p.pp_off, p.pp_idx, p.pc_off, p.pc_idx, p.eps)
    sel = np.array([3, 100, p.n_buckets - 1])
    part = oracle.gravity_eval(p.xyzm, p.cells, p.first, p.count, p.pp_off, p.pp_idx, p.pc_off, p.pc_idx, p.eps, sel=sel)
    mask = np.zeros(p.n, bool)
    for b in sel:
        mask[p.first[b]:p.first[b] + p.count[b]] = True
    assert np.array_equal(part[mask], full[mask]) and np.all(np.isnan(part[~mask]))


# ----------------------------------------------------------------------------- integer side
def test_packer_reproduces_paper_tile_example():
    """PAPER.md:L188 fn 11: 655 elements -> 640 in full warp tiles + 15."""
    L, W, full, n_full, tail = [int(v) for v in open(os.path.join(GOLD, "paper_tile_example.txt")).read().split("\n")[3].split()]
    off = np.array([0, L], np.int64); idx = np.arange(L, dtype=np.int32)[::-1].copy()
    tile_off, tiles = oracle.pack_tiles(off, idx)
    assert W == 32 and tiles.shape == (full + 1, 32) and list(tile_off) == [0, full + 1]
    assert np.array_equal(tiles[:full].reshape(-1), idx[:n_full])
    assert np.array_equal(tiles[full, :tail], idx[n_full:]) and np.all(tiles[full, tail:] == -1)


def test_paper_flop_convention_is_consistent():
    """Table 3 with rsqrt = 7, div = 35 (reading A14)."""
    for line in open(os.path.join(GOLD, "paper_flop_table.txt")):
        if line.startswith("#"):
            continue
        _, asm, rs, dv, fl = line.split()
        assert int(asm) + 7 * int(rs) + 35 * int(dv) == int(fl)


def test_packer_ragged_and_empty_buckets():
    lens = [0, 1, 31, 32, 33, 64, 0, 100]
    off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    idx = np.arange(off[-1], dtype=np.int32) * 3
    tile_off, tiles = oracle.pack_tiles(off, idx)
    assert list(np.diff(tile_off)) == [0, 1, 1, 1, 2, 2, 0, 4]
    flat = tiles.reshape(-1)
    assert np.array_equal(flat[flat >= 0], idx)                  # order preserved, nothing lost
    assert oracle.interactions(np.array([16] * 8, np.int32), off) == 16 * off[-1]


def test_chunk_bounds_greedy():
    pp_len = np.array([10, 10, 10, 50, 5, 5, 40, 1]); pc_len = np.array([1, 1, 30, 1, 1, 1, 1, 1])
    pp_off = np.concatenate([[0], np.cumsum(pp_len)]); pc_off = np.concatenate([[0], np.cumsum(pc_len)])
    b = oracle.chunk_bounds(pp_off, pc_off, 30)
    assert b[0] == 0 and b[-1] == 8 and np.all(np.diff(b) > 0)
    for lo, hi in zip(b[:-1], b[1:]):
        assert hi - lo == 1 or (pp_off[hi] - pp_off[lo] <= 30 and pc_off[hi] - pc_off[lo] <= 30)
        if hi < 8:                                               # greedy: one more bucket would not fit
            assert pp_off[hi + 1] - pp_off[lo] > 30 or pc_off[hi + 1] - pc_off[lo] > 30
    assert list(oracle.chunk_bounds(np.array([0]), np.array([0]), 10)) == [0]


def test_contribution_norms_diagnostic():
    """S_i = sum_j |a_ij| (conditioning diagnostic): one source -> |a|; two equal sources on opposite
    sides -> a = 0 but S = 2 |a_1|; always S >= |a|."""
    xyzm = np.array([[0.5, 0.5, 0.5, 1.0], [0.7, 0.5, 0.5, 2.0], [0.3, 0.5, 0.5, 2.0]], np.float32)
    first = np.array([0], np.int32); count = np.array([1], np.int32)
    z = np.zeros(2, np.int64); e = np.zeros(0, np.int32)
    a1 = 2.0 / np.float64(np.float32(0.7) - np.float32(0.5)) ** 2
    for idx, want_a, want_s in (([1], a1, a1), ([1, 2], None, None)):
        off = np.array([0, len(idx)], np.int64); ii = np.array(idx, np.int32)
        ref = oracle.gravity_eval(xyzm, None, first, count, off, ii, z, e, 0.0)
        S = oracle.contribution_norms(xyzm, None, first, count, off, ii, z, e, 0.0)
        an = np.linalg.norm(ref[0, :3])
        assert S[0] >= an * (1 - 1e-15) and np.isnan(S[1:]).all()
        if want_a is not None:
            assert abs(an - want_a) < 1e-12 * want_a and abs(S[0] - want_s) < 1e-12 * want_s
        else:
            d1 = np.float64(np.float32(0.7)) - 0.5; d2 = 0.5 - np.float64(np.float32(0.3))
            assert abs(S[0] - (2.0 / d1 ** 2 + 2.0 / d2 ** 2)) < 1e-12 * S[0]
            assert an < 1e-5 * S[0]
    p = inputs.config1(512, seed=5)
    ref = oracle.gravity_eval(p.xyzm, p.cells, p.first, p.count, p.pp_off, p.pp_idx, p.pc_off, p.pc_idx, p.eps)
    S = oracle.contribution_norms(p.xyzm, p.cells, p.first, p.count, p.pp_off, p.pp_idx, p.pc_off, p.pc_idx, p.eps)
    assert (S >= np.linalg.norm(ref[:, :3], axis=1) * (1 - 1e-12)).all()


def test_contribution_norms_squared_diagnostic():
    """S2_i = sum_j |a_ij|^2: two sources -> |a_1|^2 + |a_2|^2 in closed form; S2 <= S^2 <= n S2 (Cauchy-Schwarz)."""
    xyzm = np.array([[0.5, 0.5, 0.5, 1.0], [0.7, 0.5, 0.5, 2.0], [0.5, 0.25, 0.5, 3.0]], np.float32)
    first = np.array([0], np.int32); count = np.array([1], np.int32)
    z = np.zeros(2, np.int64); e = np.zeros(0, np.int32)
    off = np.array([0, 2], np.int64); ii = np.array([1, 2], np.int32)
    S2 = oracle.contribution_norms(xyzm, None, first, count, off, ii, z, e, 0.0, squared=True)
    d1 = np.float64(np.float32(0.7)) - 0.5
    want = (2.0 / d1 ** 2) ** 2 + (3.0 / 0.25 ** 2) ** 2
    assert abs(S2[0] - want) < 1e-12 * want and np.isnan(S2[1:]).all()
    p = inputs.config1(512, seed=5)
    args = (p.xyzm, p.cells, p.first, p.count, p.pp_off, p.pp_idx, p.pc_off, p.pc_idx, p.eps)
    S = oracle.contribution_norms(*args); S2 = oracle.contribution_norms(*args, squared=True)
    n = np.repeat(np.diff(p.pp_off) + np.diff(p.pc_off), p.count)
    assert (S2 <= S ** 2 * (1 + 1e-12)).all() and (S ** 2 <= n * S2 * (1 + 1e-12)).all()
