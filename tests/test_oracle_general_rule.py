"""Pins for the two parts of the oracle's advection operator that round 1 left unpinned:

(a) `advection_tendency_general` -- the sweep with face speeds that vary along the sweep (flow attenuation, Eq. 5): the
    staggering of B2 (LP_i takes v_{i+1/2}, LM_i takes v_{i-1/2}) and the alpha window of :689
    (alpha_i = max |v| over the faces i-5/2 .. i+5/2);
(b) the same alpha window in the table rule `advection_tendency`;
(c) "a latitude row under pure rotation shifts by Omega(theta) t" (north_star) with DIFFERENTIAL rotation, Eq. 3 (:78).

CPU only.  The brute force below is written from the paper with faces keyed by literal half-integers and shares nothing
with oracle/sft_oracle.c.
"""
import math
from fractions import Fraction as Fr

import numpy as np

from helpers import grid
from oracle.sft_oracle import ADV_WENO3, DIFF_OFF, TIME_SSPRK43, Oracle

H = Fr(1, 2)


def _caps_uniform(B):
    B[0, :], B[-1, :] = B[0, 0], B[-1, 0]
    return B


def _random_problem(nt, nphi, seed):
    rng = np.random.default_rng(seed)
    B = _caps_uniform(rng.normal(size=(nt + 2, nphi)))
    VT = rng.normal(size=(nt + 1, nphi)) * 1e-3
    VP = rng.normal(size=(nt + 2, nphi)) * 1e-3
    return B, VT, VP


# ---------------------------------------------------------------------------------------------------------------------
# (a)(i) phi-mirror: reflecting the field and the flow in phi must reflect the tendency bit for bit.  The reflection
# turns every right-moving split flux LM into a left-moving LP (and v into -v), so a face index that is off by one
# anywhere in the phi sweep -- v_{k+1/2} in LP, v_{k-1/2} in LM, the window of alpha -- breaks the symmetry.

def _mirror(B, VT, VP):
    nphi = B.shape[1]
    k = np.arange(nphi)
    Bm = B[:, (-k) % nphi]
    VTm = VT[:, (-k) % nphi]
    # phi-face k-1/2 lies between columns k-1 and k; under k -> -k it becomes the face between -k and -k+1 = face (1-k)-1/2
    VPm = -VP[:, (1 - k) % nphi]
    return Bm, VTm, VPm


def test_general_rule_is_mirror_symmetric_in_phi_bit_for_bit():
    nt, nphi = 12, 24
    o = Oracle(nt, nphi, [[0.0] * 7])
    B, VT, VP = _random_problem(nt, nphi, 11)
    T = o.advection_tendency_faces(B, VT, VP, ADV_WENO3)
    Bm, VTm, VPm = _mirror(B, VT, VP)
    Tm = o.advection_tendency_faces(Bm, VTm, VPm, ADV_WENO3)
    k = np.arange(nphi)
    # rows 1..nt bit for bit; the two cap values are phi-sums taken in the opposite order (round-off only)
    assert np.array_equal(Tm[1:-1], T[1:-1, (-k) % nphi])
    assert np.abs(Tm[[0, -1]] - T[[0, -1]]).max() <= 4e-16 * np.abs(T).max()
    # the test has teeth: shifting the phi-face speeds by one face breaks it
    Tbad = o.advection_tendency_faces(Bm, VTm, np.roll(VPm, 1, axis=1), ADV_WENO3)
    assert not np.array_equal(Tbad[1:-1], T[1:-1, (-k) % nphi])


# ---------------------------------------------------------------------------------------------------------------------
# (a)(ii) brute force on 8 x 16, faces keyed by half-integers, straight from App. B.

def _weno_side(far, near, other, eps):
    """App. B (:658-676) on a uniform grid: candidate polynomials at the face, smoothness = squared first differences,
    ideal weights 1/3 (far stencil) and 2/3 (central stencil), eps_w = h (:670)."""
    p0 = 1.5 * near - 0.5 * far
    p1 = 0.5 * near + 0.5 * other
    b0 = (near - far) ** 2
    b1 = (other - near) ** 2
    w0 = (1.0 / 3.0) / (eps + b0) ** 2
    w1 = (2.0 / 3.0) / (eps + b1) ** 2
    return (w0 * p0 + w1 * p1) / (w0 + w1)


def _flux_1d(Bc, v, i, eps, exists, wrap):
    """Flux at face i-1/2 of a 1-D sweep.  Bc: cell -> value; v: half-integer face -> speed; `exists(face)` clips the
    alpha window (:689) to faces that exist; `wrap` maps any cell / face key onto the stored one."""
    def alpha(c):                                   # max |v| over faces c-5/2 .. c+5/2   (:689)
        faces = [wrap(c + Fr(n, 2)) for n in (-5, -3, -1, 1, 3, 5) if exists(c + Fr(n, 2))]
        return max(abs(v[f]) for f in faces)

    def LP(c):                                      # B2 (:684): LP_i = 1/2 B_i (v_{i+1/2} - alpha_i)
        return 0.5 * Bc[wrap(c)] * (v[wrap(c + H)] - alpha(c))

    def LM(c):                                      # B2 (:684): LM_i = 1/2 B_i (v_{i-1/2} + alpha_i)
        return 0.5 * Bc[wrap(c)] * (v[wrap(c - H)] + alpha(c))

    u_minus = _weno_side(LM(i - 2), LM(i - 1), LM(i), eps)      # right-moving part, stencil i-2, i-1, i
    u_plus = _weno_side(LP(i + 1), LP(i), LP(i - 1), eps)       # left-moving part, stencil i+1, i, i-1
    return u_plus + u_minus


def _brute_tendency(B, VT, VP, nt, nphi):
    th, ph, dth, dph = grid(nt, nphi)
    st = np.sin(np.arange(nt + 2) * dth)
    sth = np.sin((np.arange(nt + 1) + 0.5) * dth)
    P = math.sin(dth / 2) / (2 * math.pi * (1 - math.cos(dth / 2)))
    Ft = np.zeros((nt + 1, nphi))                  # theta-face j+1/2 stored at index j
    Fp = np.zeros((nt + 2, nphi))                  # phi-face k-1/2 stored at index k
    for k in range(nphi):
        Bc = {Fr(j): B[j, k] for j in range(nt + 2)}
        v = {Fr(f) + H: VT[f, k] for f in range(nt + 1)}
        for f in range(nt + 1):
            face = Fr(f) + H
            if f <= 1 or f >= nt - 1:              # upwind next to the poles (:388, reading U6)
                vv = v[face]
                Ft[f, k] = vv * Bc[Fr(f)] if vv > 0 else (vv * Bc[Fr(f + 1)] if vv < 0 else 0.0)
            else:
                Ft[f, k] = _flux_1d(Bc, v, Fr(f + 1), dth, lambda x: H <= x <= Fr(nt) + H, lambda x: x)
    for j in range(1, nt + 1):
        Bc = {Fr(k): B[j, k] for k in range(nphi)}
        v = {Fr(k) - H: VP[j, k] for k in range(nphi)}

        def wrap(x):
            return x - nphi * math.floor(float(x + H) / nphi) if (x.denominator == 2) else x - nphi * math.floor(float(x) / nphi)
        # cells live on integers 0..nphi-1, faces on k-1/2 for k = 0..nphi-1, i.e. -1/2 .. nphi-3/2
        for k in range(nphi):
            Fp[j, k] = _flux_1d(Bc, v, Fr(k), dph, lambda x: True, wrap)
    T = np.zeros_like(B)
    for j in range(1, nt + 1):
        for k in range(nphi):
            T[j, k] = (sth[j] * Ft[j, k] - sth[j - 1] * Ft[j - 1, k]) / (st[j] * dth) + \
                      (Fp[j, (k + 1) % nphi] - Fp[j, k]) / (st[j] * dph)
    T[0, :] = P * dph * Ft[0].sum()
    T[-1, :] = -P * dph * Ft[nt].sum()
    return T


def test_general_rule_equals_half_integer_brute_force_on_8x16():
    nt, nphi = 8, 16
    o = Oracle(nt, nphi, [[0.0] * 7])
    for seed in (1, 2, 3):
        B, VT, VP = _random_problem(nt, nphi, seed)
        T = o.advection_tendency_faces(B, VT, VP, ADV_WENO3)
        ref = _brute_tendency(B, VT, VP, nt, nphi)
        assert np.abs(T - ref).max() <= 1e-13 * np.abs(ref).max()


# ---------------------------------------------------------------------------------------------------------------------
# (a)(iii), (b) the alpha window of :689.  The flux at face i-1/2 uses alpha of cells i-2 .. i+1, each a maximum over
# faces c-5/2 .. c+5/2: it depends on the speeds at faces i-9/2 .. i+7/2 and on no other.  A spike of |v| at ONE face must
# therefore change exactly the fluxes at the nine faces within 4 of it, i.e. the tendency of exactly ten cells.

def test_alpha_window_of_the_phi_sweep_spans_faces_minus_5_2_to_plus_5_2():
    nt, nphi = 10, 40
    o = Oracle(nt, nphi, [[0.0] * 7])
    rng = np.random.default_rng(5)
    B = _caps_uniform(rng.uniform(0.5, 1.5, size=(nt + 2, nphi)))
    VT = np.zeros((nt + 1, nphi))
    VP = rng.uniform(0.5e-3, 1.0e-3, size=(nt + 2, nphi))
    T0 = o.advection_tendency_faces(B, VT, VP, ADV_WENO3)
    q = 20                                           # the face q-1/2, between columns q-1 and q
    VPs = VP.copy()
    VPs[5, q] = 5e-3                                 # a spike larger than every other speed, in row 5 only
    T1 = o.advection_tendency_faces(B, VT, VPs, ADV_WENO3)
    rows = np.nonzero(np.abs(T1 - T0).max(axis=1) > 0)[0]
    assert list(rows) == [5]
    cols = np.nonzero(np.abs(T1[5] - T0[5]) > 0)[0]
    # faces k-1/2 with |k - q| <= 4 change; cell c touches faces c-1/2 and c+1/2: cells q-5 .. q+4
    assert list(cols) == list(range(q - 5, q + 5)), cols
    # one face further out the spike is outside every window: with the spike at face q-1/2 the flux at face (q+5)-1/2
    # uses alpha of cells q+3 .. q+6, whose windows start at face (q+3)-5/2 = q+1/2
    # (checked by the exact set above); a spike SMALLER than its neighbours changes only v itself: faces |k - q| <= 1
    VPd = VP.copy()
    VPd[5, q] = 0.1e-3
    T2 = o.advection_tendency_faces(B, VT, VPd, ADV_WENO3)
    cols2 = np.nonzero(np.abs(T2[5] - T0[5]) > 0)[0]
    # v_{q-1/2} enters LP_{q-1} and LM_q (B2).  The flux at face i-1/2 reads LM_{i-2..i} and LP_{i-1..i+1}: LM_q is read by
    # i = q, q+1, q+2 and LP_{q-1} by i = q-2, q-1, q -- faces i-1/2 for i = q-2 .. q+2, which touch cells q-3 .. q+2.
    # (v_{k+1/2} in LM or v_{k-1/2} in LP would shift this set by one.)
    assert list(cols2) == list(range(q - 3, q + 3)), cols2


def test_alpha_window_of_the_theta_table_rule_spans_faces_minus_5_2_to_plus_5_2():
    nt, nphi = 40, 8
    o = Oracle(nt, nphi, [[0.0] * 7])
    rng = np.random.default_rng(6)
    B = _caps_uniform(rng.uniform(0.5, 1.5, size=(nt + 2, nphi)))
    vt = rng.uniform(0.5, 1.0, size=nt + 1) * 1e-3           # R_sun/hr at the theta-faces, all positive
    om = np.zeros(nt + 2)
    o.set_flow_tables(0, vt, om)
    T0 = o.advection_tendency(0, B, ADV_WENO3)
    q = 20                                           # theta-face q+1/2, between rows q and q+1
    vts = vt.copy()
    vts[q] = 5e-3
    o.set_flow_tables(0, vts, om)
    T1 = o.advection_tendency(0, B, ADV_WENO3)
    rows = np.nonzero(np.abs(T1 - T0).max(axis=1) > 0)[0]
    # fluxes at faces f+1/2 with |f - q| <= 4 change; row j touches faces j-1/2 (f = j-1) and j+1/2 (f = j): rows q-4 .. q+5
    assert list(rows) == list(range(q - 4, q + 6)), rows
    # the general rule with the same speeds copied to every column agrees bit for bit (same window, same staggering)
    VT = np.repeat(vts[:, None], nphi, axis=1)
    T1g = o.advection_tendency_faces(B, VT, np.zeros((nt + 2, nphi)), ADV_WENO3)
    assert np.array_equal(T1g, T1)


# ---------------------------------------------------------------------------------------------------------------------
# (c) differential rotation: with v_theta = 0 every row is an independent 1-D advection at angular speed
# Omega_j = [d0 + d2 cos^2 + d4 cos^4](theta_j) (Eq. 3 :78 divided by sin theta): sin(m phi) on every row must arrive as
# sin(m (phi - Omega_j t)), each row with ITS OWN phase.  WENO3-CS(h) + SSPRK(4,3) is third order (:480-482): the phase
# error falls at least ~8x per doubling of n_phi (measured 16x: the leading third-order error term is dissipative).

def _phase_errors(nphi, m=2, t_end=480.0):
    nt = 9
    o = Oracle(nt, nphi, [[0.0, 212.30, -337.43, -251.67, 0, 0, 0]])     # BASELINE cfg 1 rotation (U17), no v_theta
    tab = o.tables()
    th, ph, dth, dph = grid(nt, nphi)
    B = np.sin(m * ph) * np.ones_like(th)
    B[0, :] = 0.0
    B[-1, :] = 0.0
    o.set_full(0, B)
    lim = (dph / np.abs(tab["om"][1:-1])).min()
    n = math.ceil(t_end / (0.5 * lim))
    o.step(n, t_end / n, adv_flux=ADV_WENO3, adv_time=TIME_SSPRK43, diff_time=DIFF_OFF)
    out = o.get_full(0)
    k = np.arange(nphi)
    err = []
    for j in range(1, nt + 1):
        c = (out[j] * np.exp(-1j * m * k * dph)).sum() * 2.0 / nphi      # = -i A exp(-i m Omega t) for A sin(m(phi - Omega t))
        phase = -np.angle(1j * c)                                        # = m Omega_j t  (mod 2 pi)
        want = m * tab["om"][j] * t_end
        d = (phase - want + math.pi) % (2 * math.pi) - math.pi
        err.append(abs(d))
    return np.array(err), tab["om"][1:-1] * t_end


def test_rows_under_differential_rotation_shift_by_omega_theta_t():
    e1, shift = _phase_errors(64)
    e2, _ = _phase_errors(128)
    e3, _ = _phase_errors(256)
    # the rows really move by different amounts (equator forward, high latitudes backward in the Carrington frame)
    assert shift.max() > 0.5 and shift.min() < -0.7 and np.ptp(shift) > 1.2
    assert e3.max() < 1e-6
    # (the dissipative error of the scheme is third order; its phase error is one order better on a smooth profile)
    o12, o23 = np.log2(e1.max() / e2.max()), np.log2(e2.max() / e3.max())
    assert 2.6 < o12 < 4.4 and 2.6 < o23 < 4.4, (e1.max(), e2.max(), e3.max())
    # row by row, not only in the maximum
    assert np.all(e3 <= e2 / 4.0 + 1e-9)
