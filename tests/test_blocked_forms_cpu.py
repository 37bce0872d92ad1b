"""Host-side algebra behind the temporally blocked kernels, checked on the CPU against the oracle's own stage scalars.

* reading U32 (k_sts_upipe): the zeta-form  zeta_l = zeta_{l-1} + kappa Lh zeta_{l-1} + N_l zeta_{l-2} + G_l F  with
  Pi_l = mu_l Pi_{l-1}, N_l = nu_l Pi_{l-2} / Pi_l, G_l = g_l / Pi_l, kappa = w1 dt nu_r reproduces the deviation form
  delta_l = mu_l delta_{l-1} + nu_l delta_{l-2} + a_l L delta_{l-1} + g_l F  (U20) block after block;
* reading U21 (k_sts_capseq): with phi-independent coefficients the zonal mean commutes with L, so the cap values of a block
  follow from the zonal means of rows 0..K alone.
The operator is the oracle's (diffusion_op), the stage scalars are the oracle's (sts_coeffs); nothing is taken from the CUDA
path.  numpy fp64.
"""
import math

import numpy as np
import pytest

from oracle.sft_oracle import DIFF_RKG2, DIFF_RKL2, Oracle


def _caps_uniform(B):
    B[0, :], B[-1, :] = B[0, 0], B[-1, 0]
    return B


@pytest.mark.parametrize("scheme", [DIFF_RKL2, DIFF_RKG2])
def test_zeta_form_equals_deviation_form_block_by_block(scheme):
    nt, nphi, s, K = 14, 24, 26, 8
    eta = 430.0
    o = Oracle(nt, nphi, [[eta, 0, 0, 0, 0, 0, 0]])
    o1 = Oracle(nt, nphi, [[1.0 / 7.43162901307967e-9, 0, 0, 0, 0, 0, 0]])      # nu = 1 R_sun^2/hr: the operator Lh = L / nu
    nu_r = eta * 7.43162901307967e-9
    L = lambda u: o.diffusion_op(0, u)
    Lh = lambda u: o1.diffusion_op(0, u)
    c = o.sts_coeffs(scheme, s)
    _, dif = o.stable_dt()
    dt = 0.8 * dif * ((s * s + s - 2) / 4.0 if scheme == DIFF_RKL2 else (s * s + 3 * s - 4) / 6.0)
    w1 = c["mut"][2] / c["mu"][2]
    mu, nu = c["mu"], c["nu"]
    a = c["mut"] * dt                                   # a_l = mu~_l dt
    g = np.array([0.0, 0.0] + [c["mut"][j] * c["b"][j - 1] * dt for j in range(2, s + 1)])   # g_l = mu~_l b_{l-1} dt (U20)
    Y0 = _caps_uniform(np.random.default_rng(1).normal(size=(nt + 2, nphi)))
    F = L(Y0)
    # deviation form, stage by stage
    d = [np.zeros_like(Y0), c["mut"][1] * dt * F]
    for j in range(2, s + 1):
        d.append(mu[j] * d[j - 1] + nu[j] * d[j - 2] + a[j] * L(d[j - 1]) + g[j] * F)
    # zeta-form in blocks of K from stage j0 = 1 (the first stage is un-blocked, as in the library; remainder block first)
    kappa = w1 * dt * nu_r
    cur, prev, j0 = d[1].copy(), d[0].copy(), 1
    while j0 < s:
        kb = min(K, s - j0)
        Pi = [1.0]
        z = {0: cur, -1: prev}
        for l in range(1, kb + 1):
            j = j0 + l
            Pi.append(mu[j] * Pi[l - 1])
            N = nu[j] * (Pi[l - 2] if l >= 2 else 1.0) / Pi[l]
            G = g[j] / Pi[l]
            z[l] = z[l - 1] + kappa * Lh(z[l - 1]) + N * z[l - 2] + G * F
        cur, prev = Pi[kb] * z[kb], Pi[kb - 1] * z[kb - 1]
        j0 += kb
        assert np.abs(cur - d[j0]).max() <= 1e-12 * np.abs(d[j0]).max(), j0
    assert np.abs(prev - d[s - 1]).max() <= 1e-12 * np.abs(d[s - 1]).max()
    # the result of the step is the oracle's own
    o.set_full(0, Y0)
    o.step(1, dt, adv_flux=0, diff_time=scheme, sts_stages=s)
    assert np.abs(Y0 + cur - o.get_full(0)).max() <= 1e-12 * np.abs(Y0).max()


def test_cap_values_of_a_block_follow_from_zonal_means():
    """U21: the zonal means m_j = mean_k u_jk of rows 0..K obey the recurrence without the phi term; K stages of it give the
    cap values that K full stages give."""
    nt, nphi, K = 20, 32, 8
    o = Oracle(nt, nphi, [[500.0, 0, 0, 0, 0, 0, 0]])
    L = lambda u: o.diffusion_op(0, u)
    rng = np.random.default_rng(2)
    cur, prev, F = (_caps_uniform(rng.normal(size=(nt + 2, nphi))) for _ in range(3))
    mu = rng.uniform(1.2, 2.0, K + 1); nu = -rng.uniform(0.3, 1.0, K + 1)
    _, dif = o.stable_dt()
    a = rng.uniform(0.5, 1.5, K + 1) * dif; g = rng.uniform(0.1, 0.5, K + 1) * dif
    # K full stages
    c1, p2, caps = cur, prev, []
    for l in range(1, K + 1):
        new = mu[l] * c1 + nu[l] * p2 + a[l] * L(c1) + g[l] * F
        caps.append(new[0, 0])
        c1, p2 = new, c1
    # the same from zonal means of rows 0..K: a field whose rows are constant in phi has no phi term
    zm = lambda u: _caps_uniform(np.repeat(u.mean(axis=1, keepdims=True), nphi, axis=1))
    c1, p2, Fz, capz = zm(cur), zm(prev), zm(F), []
    for l in range(1, K + 1):
        new = mu[l] * c1 + nu[l] * p2 + a[l] * L(c1) + g[l] * Fz
        capz.append(new[0, 0])
        c1, p2 = new, c1
    assert np.allclose(caps, capz, rtol=0, atol=1e-12 * np.abs(caps).max())
    # and only rows 0..K of the inputs matter for them: perturbing row K+1 changes nothing
    cur2 = cur.copy(); cur2[K + 1] += 1.0
    c1, p2, caps2 = cur2, prev, []
    for l in range(1, K + 1):
        new = mu[l] * c1 + nu[l] * p2 + a[l] * L(c1) + g[l] * F
        caps2.append(new[0, 0])
        c1, p2 = new, c1
    assert np.array_equal(caps, caps2)
