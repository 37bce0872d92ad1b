"""Pins for the oracle's diffusion operator and super-time-stepping (CPU only).

Each test checks oracle/sft_oracle.c against something the paper or the mathematics fixes:
printed values (tests/golden/paper_values.txt), closed forms, invariants, library special functions,
dense brute force on a tiny grid.
"""
import math

import numpy as np
import pytest
from scipy.special import eval_gegenbauer, eval_legendre

from helpers import cell_areas, golden, grid, hh_metric, soccer_ball
from oracle.sft_oracle import DIFF_EULER, DIFF_RKG2, DIFF_RKG2_TEXTBOOK, DIFF_RKL2, DIFF_RKL2_TEXTBOOK, Oracle

NU500 = [[500.0, 0, 0, 0, 0, 0, 0]]


def test_units_match_printed_constants():
    """both conversion factors, and they equal 3600/R_sun[m], 3600/R_sun[km]^2 (:292)."""
    o = Oracle(8, 16, [[1.0, 1.0, 0, 0, 0, 0, 0]])
    t = o.tables()
    assert t["nu"] == golden("km2_s_to_rs2_hr")
    assert np.all(t["om"] == golden("m_s_to_rs_hr"))
    r_m = golden("r_sun_cm") / 100.0
    assert abs(t["om"][3] / (3600.0 / r_m) - 1.0) < 1e-15
    assert abs(t["nu"] / (3600.0 / (r_m / 1e3) ** 2) - 1.0) < 1e-14


def test_rigid_rotation_speed_is_one_turn_in_672h():
    """v_phi = 1.80766 km/s sin(theta) 'corresponding to a full rotation' in 672 h."""
    o = Oracle(8, 16, [[0.0, golden("rigid_rotation_km_s") * 1e3, 0, 0, 0, 0, 0]])
    om = o.tables()["om"]
    assert abs(om[4] * golden("t_end_hours") / (2 * math.pi) - 1.0) < 2e-6


def test_grid_metric_and_polar_prefactor():
    """App. A :642-646: A_pole = 2pi(1-cos(dth/2)), P = sin(dth/2)/A_pole ~ 2/(pi dth)."""
    o = Oracle(64, 128, NU500)
    t = o.tables()
    dth = math.pi / 65
    assert abs(t["dth"] - dth) < 1e-16 and abs(t["dph"] - 2 * math.pi / 128) < 1e-16
    assert np.allclose(t["st"], np.sin(np.arange(66) * dth), rtol=0, atol=1e-15)
    assert np.allclose(t["sth"], np.sin((np.arange(65) + 0.5) * dth), rtol=0, atol=1e-15)
    assert abs(t["Apole"] / (2 * math.pi * (1 - math.cos(dth / 2))) - 1) < 1e-10
    assert abs(t["P"] * t["Apole"] / math.sin(dth / 2) - 1) < 1e-15
    assert abs(t["P"] / (2 / (math.pi * dth)) - 1) < dth ** 2


@pytest.mark.parametrize("nt,nphi", [(31, 64), (63, 128), (127, 256)])
def test_constants_in_null_space_and_flux_conserved(nt, nphi):
    o = Oracle(nt, nphi, NU500)
    assert np.abs(o.diffusion_op(0, np.full((nt + 2, nphi), 3.25))).max() == 0.0
    rng = np.random.default_rng(1)
    B = rng.normal(size=(nt + 2, nphi))
    B[0, :] = B[0, 0]
    B[-1, :] = B[-1, 0]
    L = o.diffusion_op(0, B)
    dA = cell_areas(nt, nphi)
    assert np.ptp(L[0]) == 0 and np.ptp(L[-1]) == 0
    assert abs((dA * L).sum()) < 1e-13 * (dA * np.abs(L)).sum()


def test_operator_is_symmetric_in_the_area_weighted_inner_product():
    """PAPER.md:448 'symmetric self-adjoint': <u, L v>_dA == <L u, v>_dA, caps included."""
    nt, nphi = 24, 48
    o = Oracle(nt, nphi, NU500)
    dA = cell_areas(nt, nphi)
    rng = np.random.default_rng(2)
    for _ in range(3):
        u, v = rng.normal(size=(2, nt + 2, nphi))
        for a in (u, v):
            a[0, :] = a[0, 0]
            a[-1, :] = a[-1, 0]
        lhs = (dA * u * o.diffusion_op(0, v)).sum()
        rhs = (dA * v * o.diffusion_op(0, u)).sum()
        assert abs(lhs - rhs) < 1e-12 * abs(lhs)


def _ylm_error(nt, nphi, which):
    o = Oracle(nt, nphi, NU500)
    th, ph, _, _ = grid(nt, nphi)
    if which == "y21":
        u, l = np.sin(th) * np.cos(th) * np.cos(ph), 2
    else:
        u, l = soccer_ball(th, ph), 6
    L = o.diffusion_op(0, u)
    nu = o.tables()["nu"]
    err = (L + l * (l + 1) * nu * u) / (l * (l + 1) * nu * np.abs(u).max())
    dA = cell_areas(nt, nphi)
    return math.sqrt((dA * err ** 2).sum() / dA.sum()), np.abs(err[(nt + 1) // 6:-((nt + 1) // 6)]).max(), np.abs(err).max()


@pytest.mark.parametrize("which", ["y21", "soccer"])
def test_spherical_harmonics_are_eigenfunctions_second_order(which):
    """L Y_l^m = -l(l+1) nu Y_l^m (Eq. 19 :261 decay rate 42 nu for l = 6).  The truncation error falls 4x
    per grid doubling (:482 'second-order') in the area-weighted L2 norm and pointwise at colatitudes
    30..150 degrees; at a fixed number of rows from a cap the 1/sin^2(theta) metric keeps the local error
    O(1)-to-O(h) for m != 0, which does not reduce the order of the solution (see the decay tests)."""
    e = [_ylm_error(n, 2 * (n + 1), which) for n in (31, 63, 127)]
    for q in (0, 1):
        assert e[0][q] < 0.05 and 3.5 < e[0][q] / e[1][q] < 4.5 and 3.5 < e[1][q] / e[2][q] < 4.5, (q, e)
    assert e[2][2] < e[1][2] < e[0][2]


def test_y21_decay_config0_style():
    """BASELINE config 0 check: Y_2^1 decays as exp(-6 nu t); 200 steps of 8 explicit limits, s = 8 forced."""
    for nt, nphi, tol in ((64, 128, 5e-5), (128, 256, 1.3e-5)):
        o = Oracle(nt, nphi, NU500)
        th, ph, _, _ = grid(nt, nphi)
        u = np.sin(th) * np.cos(th) * np.cos(ph)
        o.set_full(0, u)
        _, dtd = o.stable_dt()
        n = 200 if nt == 64 else 50
        o.step(n, 8 * dtd, adv_flux=0, diff_time=DIFF_RKG2, sts_stages=8)
        exact = u * math.exp(-6 * o.tables()["nu"] * n * 8 * dtd)
        assert np.abs(o.get_full(0) - exact).max() < tol


def test_euler_limit_against_printed_value_and_gershgorin():
    """PAPER.md:476 prints dt_Euler = 1.8e-4 h at 512x1024, nu = 500: our stability limit times the paper's
    unstated safety factor (~0.9-0.95, :406).  Also: the limit is the true one within the Gershgorin slack
    (checked on a small dense matrix)."""
    o = Oracle(510, 1023, NU500)
    _, dtd = o.stable_dt()
    assert 0.90 <= golden("dt_euler_hours") / dtd <= 0.96
    nt, nphi = 8, 16
    o = Oracle(nt, nphi, NU500)
    M = _dense_matrix(o, nt, nphi)
    rho = np.abs(np.linalg.eigvals(M)).max()
    _, dtd = o.stable_dt()
    assert dtd <= 2.0 / rho <= 1.3 * dtd


def _dense_matrix(o, nt, nphi):
    """Dense matrix of L over the unknowns [cap_N, rows 1..nt, cap_S], built column by column."""
    n = nt * nphi + 2

    def expand(x):
        full = np.empty((nt + 2, nphi))
        full[0, :] = x[0]
        full[1:-1] = x[1:-1].reshape(nt, nphi)
        full[-1, :] = x[-1]
        return full

    def compress(f):
        return np.concatenate([[f[0, 0]], f[1:-1].ravel(), [f[-1, 0]]])

    M = np.zeros((n, n))
    for i in range(n):
        e = np.zeros(n)
        e[i] = 1.0
        M[:, i] = compress(o.diffusion_op(0, expand(e)))
    return M


@pytest.mark.parametrize("scheme,lib_poly", [(DIFF_RKL2, "legendre"), (DIFF_RKG2, "gegenbauer")])
def test_sts_equals_shifted_orthogonal_polynomial_of_dense_matrix(scheme, lib_poly):
    """Brute force on 8x16: the staged oracle result equals R_s(dt L) Y0 with
    R_s(z) = a_s + b_s p_s(1 + w1 z), p = Legendre P_s (RKL2; Meyer et al. via :470) or normalised
    Gegenbauer C_s^(3/2)/C_s^(3/2)(1) (RKG2(3/2); Skaras et al. via :472), evaluated through the
    eigendecomposition of the dense matrix with scipy's polynomial routines."""
    nt, nphi, s = 8, 16, 11
    o = Oracle(nt, nphi, NU500)
    M = _dense_matrix(o, nt, nphi)
    rng = np.random.default_rng(5)
    y0 = rng.normal(size=nt * nphi + 2)
    full = np.empty((nt + 2, nphi))
    full[0, :], full[1:-1], full[-1, :] = y0[0], y0[1:-1].reshape(nt, nphi), y0[-1]
    _, dtd = o.stable_dt()
    dt = 0.8 * dtd * ((s * s + s - 2) / 4.0 if scheme == DIFF_RKL2 else (s * s + 3 * s - 4) / 6.0)
    o.set_full(0, full)
    assert o.step(1, dt, adv_flux=0, diff_time=scheme, sts_stages=s) == s
    got = o.get_full(0)
    lam, V = np.linalg.eig(M)
    z = dt * lam.real
    assert np.abs(lam.imag).max() < 1e-9 * np.abs(lam).max()
    if lib_poly == "legendre":
        w1 = 4.0 / (s * s + s - 2)
        b = (s * s + s - 2) / (2.0 * s * (s + 1))
        p = eval_legendre(s, 1 + w1 * z)
    else:
        w1 = 6.0 / ((s - 1) * (s + 4))
        b = 2.0 * (s - 1) * (s + 4) / (3.0 * s * (s + 3))
        p = eval_gegenbauer(s, 1.5, 1 + w1 * z) / eval_gegenbauer(s, 1.5, 1.0)
    R = (1 - b) + b * p
    want = (V @ (R * np.linalg.solve(V, y0))).real
    assert np.abs(got[0] - want[0]).max() < 1e-11
    assert np.abs(got[-1] - want[-1]).max() < 1e-11
    assert np.abs(got[1:-1].ravel() - want[1:-1]).max() < 1e-11


@pytest.mark.parametrize("scheme", [DIFF_RKL2, DIFF_RKG2])
def test_sts_scalar_polynomial_order_and_stability(scheme):
    """The coefficient tables alone: scalar recurrence -> R_s(z) = 1 + z + z^2/2 + O(z^3), |R_s| <= 1 on
    [-2/w1, 0] and blow-up beyond it."""
    o = Oracle(4, 8, NU500)
    for s in (2, 3, 8, 25, 60):
        c = o.sts_coeffs(scheme, s)

        def R(z):
            y0, y2, y1 = 1.0, 1.0, 1.0 + c["mut"][1] * z
            for j in range(2, s + 1):
                yn = (c["mu"][j] * y1 + c["nu"][j] * y2 + (1 - c["mu"][j] - c["nu"][j]) * y0
                      + c["mut"][j] * z * y1 + c["gt"][j] * z * y0)
                y2, y1 = y1, yn
            return y1

        for z in (-1e-2, -2e-2):
            assert abs(R(z) - (1 + z + z * z / 2)) < 0.6 * abs(z) ** 3
        e1, e2 = abs(R(-1e-2) - math.exp(-1e-2)), abs(R(-2e-2) - math.exp(-2e-2))
        assert 6.0 < e2 / e1 < 10.0 or e2 < 1e-13          # third-order local error
        w1 = 4.0 / (s * s + s - 2) if scheme == DIFF_RKL2 else 6.0 / ((s - 1) * (s + 4))
        zs = np.linspace(-2.0 / w1, 0.0, 2001)
        assert max(abs(R(z)) for z in zs) <= 1.0 + 1e-12
        if s >= 8:
            assert abs(R(-1.25 * 2.0 / w1)) > 1.0


def test_stage_count_rule_and_paper_time_ratio():
    """RKG2 took 0.55 s, RKL2 0.45 s for the same single 672 h step -> stage ratio ~1.22 = sqrt(6/4)."""
    o = Oracle(510, 1023, NU500)
    s_rkl, s_rkg = o.sts_stage_count(672.0, DIFF_RKL2), o.sts_stage_count(672.0, DIFF_RKG2)
    assert abs(s_rkg / s_rkl / golden("time_ratio_rkg2_rkl2") - 1) < 0.05
    _, dtd = o.stable_dt()
    for s, C in ((s_rkl, lambda q: (q * q + q - 2) / 4.0), (s_rkg, lambda q: (q * q + 3 * q - 4) / 6.0)):
        assert dtd * C(s) >= 672.0 > dtd * C(s - 1)
    o2 = Oracle(64, 128, NU500)
    assert o2.sts_stage_count(0.5 * o2.stable_dt()[1], DIFF_RKG2) == 2


@pytest.mark.slow
def test_printed_hh_errors_soccer_ball_one_672h_step():
    """diffusion only, Eq. 19, 512x1024 (= 510 x 1023 regular cells, reading U1), nu = 500,
    one 672 h step: HH = 8.0e-5 (RKL2), 6.3e-5 (RKG2).  Reproduced to the two printed digits."""
    nt, nphi = 510, 1023
    o = Oracle(nt, nphi, NU500)
    th, ph, _, _ = grid(nt, nphi)
    u = soccer_ball(th, ph)
    exact = u * math.exp(-42.0 * o.tables()["nu"] * 672.0)
    for scheme, name in ((DIFF_RKL2, "hh_rkl2_diffusion"), (DIFF_RKG2, "hh_rkg2_diffusion")):
        o.set_full(0, u)
        o.step(1, 672.0, adv_flux=0, diff_time=scheme)
        hh = hh_metric(o.get_full(0)[1:-1], exact[1:-1])
        assert abs(hh / golden(name) - 1) < 0.02, (name, hh)


def test_deviation_form_equals_textbook_form():
    """delta-form and textbook form are the same polynomial; they differ by round-off only."""
    nt, nphi = 48, 96
    o = Oracle(nt, nphi, NU500)
    rng = np.random.default_rng(7)
    B = rng.normal(size=(nt + 2, nphi)) * 50
    B[0, :], B[-1, :] = B[0, 0], B[-1, 0]
    _, dtd = o.stable_dt()
    for dev, txt in ((DIFF_RKG2, DIFF_RKG2_TEXTBOOK), (DIFF_RKL2, DIFF_RKL2_TEXTBOOK)):
        o.set_full(0, B)
        s1 = o.step(3, 300 * dtd, adv_flux=0, diff_time=dev)
        a = o.get_full(0)
        o.set_full(0, B)
        s2 = o.step(3, 300 * dtd, adv_flux=0, diff_time=txt)
        b = o.get_full(0)
        assert s1 == s2 and s1 > 30
        assert np.abs(a - b).max() < 1e-11 * np.abs(B).max()


def test_euler_diffusion_is_flux_conserving_and_unsigned_flux_nonincreasing():
    nt, nphi = 32, 64
    o = Oracle(nt, nphi, NU500)
    rng = np.random.default_rng(8)
    o.set_map(0, rng.normal(size=(nt, nphi)) * 10)
    _, dtd = o.stable_dt()
    d0 = o.diagnostics()[0]
    for _ in range(5):
        o.step(4, 0.5 * dtd, adv_flux=0, diff_time=DIFF_EULER)
        d1 = o.diagnostics()[0]
        assert abs(d1[0] - d0[0]) < 1e-13 * d0[1]
        assert d1[1] <= d0[1] * (1 + 1e-14)
        d0 = d1


def test_sts_conserves_signed_flux_to_roundoff():
    nt, nphi = 64, 128
    o = Oracle(nt, nphi, NU500)
    rng = np.random.default_rng(9)
    o.set_map(0, rng.normal(size=(nt, nphi)) * 10 + 1.0)
    before = o.diagnostics()[0]
    _, dtd = o.stable_dt()
    o.step(20, 8 * dtd, adv_flux=0, diff_time=DIFF_RKG2, sts_stages=8)
    after = o.diagnostics()[0]
    assert abs(after[0] - before[0]) < 1e-13 * before[1]
    assert after[1] < before[1]


def test_fp32_oracle_tracks_fp64():
    nt, nphi = 64, 128
    B = np.random.default_rng(10).normal(size=(nt, nphi)) * 30
    res = []
    for dt in (np.float64, np.float32):
        o = Oracle(nt, nphi, NU500, dtype=dt)
        o.set_map(0, B)
        _, dtd = o.stable_dt()
        o.step(10, 40 * dtd, adv_flux=0, diff_time=DIFF_RKG2)
        res.append(o.get_map(0).astype(np.float64))
    assert np.abs(res[0] - res[1]).max() < 2e-6 * np.abs(B).max()
