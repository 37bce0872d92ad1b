"""Pins for the oracle on a NON-UNIFORM theta grid ("logically-rectangular non-uniform";
Eq. 27-28 :438-460 with Delta theta_{j+-1/2}, Delta theta_j; :354; App. A; App. B :662-680 D-factors; DESIGN.md readings
U12 and U33).  CPU only.

  * nodes j pi/(nt+1) handed in as a "non-uniform" grid reproduce the default oracle to round-off (uniform limit);
  * flux conservation incl. the caps and dA-symmetry of L on a random monotone grid (:448);
  * the dense matrix of Eq. 28, assembled entry by entry with the printed Delta's, on 8 x 16 (brute force);
  * the theta sweep of App. B with the D-factors keyed by half-integer faces, in plain Python (brute force);
  * second order (diffusion, Y_2^1 decay) and third order (advection, App. C translation) on the smooth stretching
    theta(xi) = xi + a sin 2 xi (:480-482).
"""
import math
from fractions import Fraction as Fr

import numpy as np

from oracle.sft_oracle import ADV_OFF, ADV_WENO3, DIFF_EULER, DIFF_OFF, DIFF_RKG2, TIME_SSPRK43, Oracle

KM2 = 7.43162901307967e-9
H = Fr(1, 2)


def stretched(nt, a=0.15):
    xi = np.arange(nt + 2) * math.pi / (nt + 1)
    th = xi + a * np.sin(2 * xi)
    th[0], th[-1] = 0.0, math.pi
    return th


def random_nodes(nt, seed):
    rng = np.random.default_rng(seed)
    w = rng.uniform(0.6, 1.6, size=nt + 1)
    th = np.concatenate([[0.0], np.cumsum(w)])
    th *= math.pi / th[-1]
    th[-1] = math.pi
    return th


def areas(o, nphi):
    g = o.grid_arrays()
    dph = 2 * math.pi / nphi
    dA = np.sin(g["th"])[:, None] * g["dthc"][:, None] * dph * np.ones((1, nphi))
    dA[0, :] = g["ApoleN"] / nphi
    dA[-1, :] = g["ApoleS"] / nphi
    return dA


def caps_uniform(B):
    B[0, :], B[-1, :] = B[0, 0], B[-1, 0]
    return B


def test_uniform_nodes_reproduce_the_uniform_oracle():
    nt, nphi = 40, 64
    p = [[500.0, 212.30, -337.43, -251.67, 46.0, -46.0, 0.0]]
    a, b = Oracle(nt, nphi, p), Oracle(nt, nphi, p)
    b.set_theta_nodes(np.arange(nt + 2) * math.pi / (nt + 1) * np.ones(nt + 2))
    b_nodes = np.arange(nt + 2) * math.pi / (nt + 1)
    b_nodes[-1] = math.pi
    b.set_theta_nodes(b_nodes)
    B = caps_uniform(np.random.default_rng(0).normal(size=(nt + 2, nphi)))
    a.set_full(0, B)
    b.set_full(0, B)
    adv, dif = a.stable_dt()
    adv2, dif2 = b.stable_dt()
    assert abs(adv2 / adv - 1) < 1e-13 and abs(dif2 / dif - 1) < 1e-13
    a.step(3, 0.5 * adv)
    b.step(3, 0.5 * adv)
    assert np.abs(a.get_full(0) - b.get_full(0)).max() <= 1e-12 * np.abs(B).max()
    assert np.allclose(a.diagnostics(), b.diagnostics(), rtol=1e-12)


def test_conservation_and_symmetry_on_a_random_monotone_grid():
    nt, nphi = 24, 32
    o = Oracle(nt, nphi, [[500.0, 200.0, -300.0, -200.0, 40.0, -40.0, 10.0]])
    o.set_theta_nodes(random_nodes(nt, 3))
    dA = areas(o, nphi)
    assert abs(dA.sum() - 4 * math.pi) < 2e-2          # midpoint quadrature of the sphere
    rng = np.random.default_rng(4)
    u, v = caps_uniform(rng.normal(size=(nt + 2, nphi))), caps_uniform(rng.normal(size=(nt + 2, nphi)))
    Lu, Lv = o.diffusion_op(0, u), o.diffusion_op(0, v)
    scale = np.abs(Lu * dA).sum()
    assert abs((Lu * dA).sum()) < 1e-13 * scale                               # conservation: constants are in the left null space
    assert abs(((u * Lv - v * Lu) * dA).sum()) < 1e-13 * np.abs(u * Lv * dA).sum()   # "symmetric self-adjoint" (:448)
    assert np.abs(o.diffusion_op(0, np.ones((nt + 2, nphi)))).max() < 1e-9 * np.abs(Lu).max()
    T = o.advection_tendency(0, u, ADV_WENO3)
    assert abs((T * dA).sum()) < 1e-13 * np.abs(T * dA).sum()                 # every face flux leaves one cell and enters the next
    # a whole step keeps the signed flux
    o.set_full(0, u)
    before = o.diagnostics()[0]
    adv, dif = o.stable_dt()
    o.step(4, 0.5 * adv)
    after = o.diagnostics()[0]
    assert abs(after[0] - before[0]) < 1e-12 * before[1]


def test_dense_matrix_of_eq28_on_8x16():
    """Eq. 28 (:450-458) entry by entry with the printed Delta theta_{j+-1/2}, Delta theta_j (constant nu), rows of the caps
    from App. A (:646) with the first half-cell's own prefactor; the looped operator must be this matrix."""
    nt, nphi = 8, 16
    nu_km = 400.0
    o = Oracle(nt, nphi, [[nu_km, 0, 0, 0, 0, 0, 0]])
    th = random_nodes(nt, 7)
    o.set_theta_nodes(th)
    nu = nu_km * KM2
    thf = 0.5 * (th[:-1] + th[1:])
    dph = 2 * math.pi / nphi
    N = (nt + 2) * nphi

    def idx(j, k):
        return j * nphi + (k % nphi)

    A = np.zeros((N, N))
    for j in range(1, nt + 1):
        dth_j = thf[j] - thf[j - 1]
        for k in range(nphi):
            a_s = nu * math.sin(thf[j]) / ((th[j + 1] - th[j]) * dth_j * math.sin(th[j]))          # a_{j+1,k}
            a_n = nu * math.sin(thf[j - 1]) / ((th[j] - th[j - 1]) * dth_j * math.sin(th[j]))      # a_{j-1,k}
            a_e = nu / (dph * dph * math.sin(th[j]) ** 2)                                          # a_{j,k+1} = a_{j,k-1}
            A[idx(j, k), idx(j + 1, k)] += a_s
            A[idx(j, k), idx(j - 1, k)] += a_n
            A[idx(j, k), idx(j, k + 1)] += a_e
            A[idx(j, k), idx(j, k - 1)] += a_e
            A[idx(j, k), idx(j, k)] -= a_s + a_n + 2 * a_e
    for cap, row, x, dnode in ((0, 1, thf[0], th[1] - th[0]), (nt + 1, nt, math.pi - thf[nt], th[nt + 1] - th[nt])):
        P = math.sin(x) / (2 * math.pi * (1 - math.cos(x)))
        for k in range(nphi):                          # the cap is ONE cell stored nphi times
            for kk in range(nphi):
                A[idx(cap, k), idx(row, kk)] += P * nu / dnode * dph
            A[idx(cap, k), idx(cap, k)] -= P * nu / dnode * dph * nphi
    u = caps_uniform(np.random.default_rng(8).normal(size=(nt + 2, nphi)))
    ref = (A @ u.ravel()).reshape(nt + 2, nphi)
    got = o.diffusion_op(0, u)
    assert np.abs(got - ref).max() <= 1e-12 * np.abs(ref).max()
    # and the Euler limit is 1 / max |diagonal| (Gershgorin, reading U8)
    assert abs(o.stable_dt()[1] * np.abs(np.diag(A)).max() - 1) < 1e-12


def _weno_nu(far, near, other, eps, Dex, Da, Db, d0, d1):
    p0 = (1 + Dex) * near - Dex * far
    p1 = Da * near + Db * other
    b0 = 4 * (Dex * (near - far)) ** 2
    b1 = 4 * (Db * (other - near)) ** 2
    w0 = d0 / (eps + b0) ** 2
    w1 = d1 / (eps + b1) ** 2
    return (w0 * p0 + w1 * p1) / (w0 + w1)


def test_theta_sweep_equals_half_integer_brute_force_with_d_factors():
    """App. B on the non-uniform grid, in plain Python: cells keyed by integers, faces by half-integers, the six D-factors
    of :680 by their names (c = centre, m / p = the cell below / above, t = all three), centred as the subscript says."""
    nt, nphi = 12, 4
    o = Oracle(nt, nphi, [[0.0] * 7])
    th = random_nodes(nt, 9)
    o.set_theta_nodes(th)
    g = o.grid_arrays()
    dx = {Fr(j): g["dthc"][j] for j in range(nt + 2)}
    rng = np.random.default_rng(10)
    vt = rng.normal(size=nt + 1) * 1e-3
    o.set_flow_tables(0, vt, np.zeros(nt + 2))
    B = caps_uniform(rng.normal(size=(nt + 2, nphi)))
    T = o.advection_tendency(0, B, ADV_WENO3)

    v = {Fr(f) + H: vt[f] for f in range(nt + 1)}

    def D(kind, face):                 # D^{kind}_{face}: "centre" is the cell above the face, i = face + 1/2
        i = face + H
        c, m, p = dx[i], dx[i - 1], dx.get(i + 1, float("nan"))
        return {"c/cp": c / (c + p), "c/cm": c / (c + m), "p/t": p / (m + c + p), "m/t": m / (m + c + p),
                "cp/t": (c + p) / (m + c + p), "cm/t": (c + m) / (m + c + p)}[kind]

    def alpha(c):
        return max(abs(v[c + Fr(n, 2)]) for n in (-5, -3, -1, 1, 3, 5) if (c + Fr(n, 2)) in v)

    k = 1
    Bc = {Fr(j): B[j, k] for j in range(nt + 2)}
    LP = lambda c: 0.5 * Bc[c] * (v[c + H] - alpha(c))
    LM = lambda c: 0.5 * Bc[c] * (v[c - H] + alpha(c))
    Ft = np.zeros(nt + 1)
    for f in range(nt + 1):
        if f <= 1 or f >= nt - 1:
            vv = vt[f]
            Ft[f] = vv * B[f, k] if vv > 0 else (vv * B[f + 1, k] if vv < 0 else 0.0)
            continue
        i = Fr(f + 1)
        fm, f0 = i - Fr(3, 2), i - H                  # the faces i-3/2 and i-1/2
        eps = th[f + 1] - th[f]
        um = _weno_nu(LM(i - 2), LM(i - 1), LM(i), eps, D("c/cm", fm), D("c/cm", f0), D("c/cp", fm), D("p/t", fm), D("cm/t", fm))
        up = _weno_nu(LP(i + 1), LP(i), LP(i - 1), eps, D("c/cp", f0), D("c/cp", fm), D("c/cm", f0), D("m/t", f0), D("cp/t", f0))
        Ft[f] = up + um
    sth, st = np.sin(g["thf"]), np.sin(g["th"])
    ref = np.array([(sth[j] * Ft[j] - sth[j - 1] * Ft[j - 1]) / (st[j] * g["dthc"][j]) for j in range(1, nt + 1)])
    assert np.abs(T[1:-1, k] - ref).max() <= 1e-13 * np.abs(ref).max()
    # the D-factors are interpolation weights: both candidate polynomials and their optimal combination reproduce a LINEAR
    # cell-average profile exactly at the face (what "first-order polynomial approximation", :660, means)
    for f in range(2, nt - 1):
        i = Fr(f + 1)
        fm, f0 = i - Fr(3, 2), i - H
        xc = {c: 0.5 * (g["thf"][int(c)] + g["thf"][int(c) - 1]) for c in (i - 2, i - 1, i, i + 1)}   # cell centres
        lin = {c: 3.0 + 2.0 * x for c, x in xc.items()}
        face = g["thf"][f]
        assert abs((1 + D("c/cm", fm)) * lin[i - 1] - D("c/cm", fm) * lin[i - 2] - (3 + 2 * face)) < 1e-12
        assert abs(D("c/cm", f0) * lin[i - 1] + D("c/cp", fm) * lin[i] - (3 + 2 * face)) < 1e-12
        assert abs((1 + D("c/cp", f0)) * lin[i] - D("c/cp", f0) * lin[i + 1] - (3 + 2 * face)) < 1e-12
        assert abs(D("p/t", fm) + D("cm/t", fm) - 1) < 1e-15 and abs(D("m/t", f0) + D("cp/t", f0) - 1) < 1e-15


def _y21_decay_error(nt, nphi):
    """Y_2^1 ~ sin(theta) cos(theta) cos(phi) decays as exp(-6 nu t) (north_star closed form) on the stretched grid."""
    o = Oracle(nt, nphi, [[500.0, 0, 0, 0, 0, 0, 0]])
    th = stretched(nt)
    o.set_theta_nodes(th)
    ph = np.arange(nphi) * 2 * math.pi / nphi
    Y = np.sin(th)[:, None] * np.cos(th)[:, None] * np.cos(ph)[None, :]
    o.set_full(0, Y)
    _, dif = o.stable_dt()
    t_end = 20000.0                                  # exp(-6 nu t) = 0.64: long enough for the mode's error to dominate the
    n = math.ceil(t_end / (0.4 * dif))               # first-order truncation error of the rows next to the poles (also there
    o.step(n, t_end / n, adv_flux=ADV_OFF, diff_time=DIFF_EULER)   # on the uniform grid), which is a short-lived transient
    exact = Y * math.exp(-6 * 500.0 * KM2 * t_end)
    return np.abs(o.get_full(0) - exact).max() / np.abs(exact).max()


def test_diffusion_is_second_order_on_a_smoothly_stretched_grid():
    e = [_y21_decay_error(n, 2 * (n + 1)) for n in (15, 31, 63)]
    orders = [math.log2(e[i] / e[i + 1]) for i in range(2)]
    assert e[2] < 1e-3 and all(1.8 < q < 2.3 for q in orders), (e, orders)
    # the stretching is not cosmetic: cells differ by a factor ~1.9 in width
    g = Oracle(31, 8, [[0.0] * 7])
    g.set_theta_nodes(stretched(31))
    w = g.grid_arrays()["dthc"][1:-1]
    assert w.max() / w.min() > 1.7


def _theta_translation_error(nt):
    """App. C (:697-731): for constant v_theta, B = g(theta - v t)/sin(theta) is exact; on the stretched grid."""
    nphi = 8
    o = Oracle(nt, nphi, [[0.0] * 7])
    th1 = stretched(nt)
    o.set_theta_nodes(th1)
    v = 1.0e-3
    o.set_flow_tables(0, np.full(nt + 1, v), np.zeros(nt + 2))
    th = th1[:, None]
    sth = np.sin(th)
    sth[0], sth[-1] = 1.0, 1.0

    def sol(t):
        B = np.exp(-(th - math.pi / 4 - v * t) ** 2 / 0.03) / sth * np.ones((1, nphi))
        B[0, :], B[-1, :] = 0.0, 0.0
        return B

    o.set_full(0, sol(0.0))
    T = (math.pi / 4) / v
    adv, _ = o.stable_dt()
    n = math.ceil(T / (0.5 * adv))
    o.step(n, T / n, adv_flux=ADV_WENO3, adv_time=TIME_SSPRK43, diff_time=DIFF_OFF)
    return np.abs(o.get_full(0) - sol(T)).max()


def test_theta_advection_is_third_order_on_a_smoothly_stretched_grid():
    e = [_theta_translation_error(n) for n in (63, 127, 255)]
    orders = [math.log2(e[i] / e[i + 1]) for i in range(2)]
    assert e[2] < 3e-3 and orders[1] > 2.5 and orders[0] > 1.9, (e, orders)


def test_sts_step_on_the_stretched_grid_matches_many_small_euler_steps():
    """The super-time-stepping recurrence is grid-agnostic (it only applies L): one RKG2 step of 40 stable Euler steps' length
    must agree with the Euler integration to the scheme's second-order accuracy."""
    nt, nphi = 31, 64
    p = [[500.0, 0, 0, 0, 0, 0, 0]]
    a, b = Oracle(nt, nphi, p), Oracle(nt, nphi, p)
    for o in (a, b):
        o.set_theta_nodes(stretched(nt))
    th = stretched(nt)[:, None]
    ph = (np.arange(nphi) * 2 * math.pi / nphi)[None, :]
    B = np.sin(th) ** 2 * np.cos(2 * ph) + np.cos(th) + 0.5 * np.sin(th) * np.cos(th) * np.sin(ph)    # smooth, all of l = 1, 2
    a.set_full(0, B)
    b.set_full(0, B)
    _, dif = a.stable_dt()
    a.step(1, 40 * dif, adv_flux=ADV_OFF, diff_time=DIFF_RKG2)
    b.step(400, 0.1 * dif, adv_flux=ADV_OFF, diff_time=DIFF_EULER)
    assert np.abs(a.get_full(0) - b.get_full(0)).max() < 1e-5 * np.abs(b.get_full(0)).max()
