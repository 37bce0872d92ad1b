"""Pins for the oracle's assimilation blend, diagnostics, set/get and the workload recipes (CPU only)."""
import math

import numpy as np
import pytest

from helpers import cell_areas, grid
from oracle.sft_oracle import DIFF_RKG2, Oracle
from paper_2501_06377_b200 import workloads as wl


def test_diagnostics_closed_form_cos_theta():
    """:225-230 with B = cos(theta): Phi+ = pi, Phi- = -pi, signed 0, unsigned 2 pi (midpoint rule, O(h^2))."""
    errs = []
    for nt in (63, 127):
        nphi = 2 * (nt + 1)
        o = Oracle(nt, nphi, [[0.0] * 7])
        th, ph, _, _ = grid(nt, nphi)
        o.set_full(0, np.cos(th) * np.ones_like(ph))
        d = o.diagnostics()[0]
        assert abs(d[0]) < 1e-13 and abs(d[1] - (d[2] - d[3])) < 1e-14 and d[3] < 0 < d[2]
        errs.append(abs(d[1] - 2 * math.pi))
    assert errs[0] < 2e-3 and 3.5 < errs[0] / errs[1] < 4.5


def test_diagnostics_scale_with_radius_squared_and_weights_sum_to_sphere():
    nt, nphi = 30, 64
    o1, o2 = Oracle(nt, nphi, [[0.0] * 7]), Oracle(nt, nphi, [[0.0] * 7], radius_cm=6.96e10)
    B = np.ones((nt + 2, nphi))
    o1.set_full(0, B)
    o2.set_full(0, B)
    assert abs(o1.diagnostics()[0, 0] - cell_areas(nt, nphi).sum()) < 1e-13
    assert abs(o1.diagnostics()[0, 0] / (4 * math.pi) - 1) < 1e-3
    assert abs(o2.diagnostics()[0, 0] / (o1.diagnostics()[0, 0] * 6.96e10 ** 2) - 1) < 1e-15


def test_set_map_pole_cell_averaging_and_roundtrip():
    """Reading U18: caps start as the dph-weighted mean of the adjacent row; get_map returns rows 1..nt."""
    nt, nphi = 9, 20
    o = Oracle(nt, nphi, [[0.0] * 7] * 2)
    m = np.random.default_rng(0).normal(size=(nt, nphi))
    o.set_map(-1, m)
    for r in range(2):
        f = o.get_full(r)
        assert np.array_equal(f[1:-1], m) and np.array_equal(o.get_map(r), m)
        assert np.allclose(f[0], m[0].mean(), atol=1e-15) and np.allclose(f[-1], m[-1].mean(), atol=1e-15)
    th, ph, _, _ = grid(nt, nphi)
    y = (np.sin(th) * np.cos(th) * np.cos(ph))[1:-1]     # m != 0 harmonic: exact pole value 0 = that mean
    o.set_map(0, y)
    assert abs(o.get_full(0)[0, 0]) < 1e-16


def test_assimilation_blend_eq8():
    """Eq. 8 (:131): B <- F B_d + (1-F) B cell by cell; F = 0 leaves the state, F = 1 replaces it."""
    nt, nphi = 12, 24
    rng = np.random.default_rng(1)
    o = Oracle(nt, nphi, [[0.0] * 7] * 3)
    maps = rng.normal(size=(3, nt, nphi))
    for r in range(3):
        o.set_map(r, maps[r])
    obs, w = rng.normal(size=(nt, nphi)), rng.uniform(size=(nt, nphi))
    w[:, :5], w[:, 5:8] = 0.0, 1.0
    caps = [(o.get_full(r)[0, 0], o.get_full(r)[-1, 0]) for r in range(3)]
    o.assimilate(obs, w)                                   # one obs/weight map shared by all realizations
    for r in range(3):
        f = o.get_full(r)
        want = w * obs + (1 - w) * maps[r]
        assert np.abs(f[1:-1] - want).max() < 1e-15
        assert np.array_equal(f[1:-1][:, :5], maps[r][:, :5]) and np.array_equal(f[1:-1][:, 5:8], obs[:, 5:8])
        wn, ws = w[0].mean(), w[-1].mean()
        assert abs(f[0, 0] - (wn * obs[0].mean() + (1 - wn) * caps[r][0])) < 1e-15
        assert abs(f[-1, 0] - (ws * obs[-1].mean() + (1 - ws) * caps[r][1])) < 1e-15
        assert np.ptp(f[0]) == 0 and np.ptp(f[-1]) == 0
    obs3, w3 = rng.normal(size=(3, nt, nphi)), rng.uniform(size=(3, nt, nphi))
    before = [o.get_map(r) for r in range(3)]
    o.assimilate(obs3, w3)                                 # per-realization obs/weights
    for r in range(3):
        assert np.abs(o.get_map(r) - (w3[r] * obs3[r] + (1 - w3[r]) * before[r])).max() < 1e-15


def test_flux_balanced_assimilation_eq10_11():
    """Eq. 10-11 (:144-153): the scaled increment has zero net flux, keeps the sign pattern (neutral lines)
    and the ratio of scalings is |Phi+/Phi-|."""
    nt, nphi = 16, 32
    rng = np.random.default_rng(2)
    o = Oracle(nt, nphi, [[0.0] * 7])
    m = rng.normal(size=(nt, nphi))
    o.set_map(0, m)
    f0 = o.get_full(0)
    d0 = o.diagnostics()[0]
    obs, w = rng.normal(size=(nt, nphi)) + 0.7, rng.uniform(size=(nt, nphi))
    o.assimilate(obs, w, flags=1)
    f1 = o.get_full(0)
    d1 = o.diagnostics()[0]
    assert abs(d1[0] - d0[0]) < 1e-13 * d0[1]              # net flux unchanged
    raw = w * (obs - m)
    inc = (f1 - f0)[1:-1]
    assert np.all(np.sign(inc) == np.sign(raw))
    pos, neg = raw > 1e-2, raw < -1e-2               # ratio of differences: skip tiny increments
    sp, sn = (inc[pos] / raw[pos]), (inc[neg] / raw[neg])
    assert np.ptp(sp) < 1e-11 and np.ptp(sn) < 1e-11 and abs(sp[0] * sn[0] - 1) < 1e-11
    dA = cell_areas(nt, nphi)
    full_raw = np.zeros((nt + 2, nphi))
    full_raw[1:-1] = raw
    full_raw[0, :] = w[0].mean() * (obs[0].mean() - f0[0, 0])
    full_raw[-1, :] = w[-1].mean() * (obs[-1].mean() - f0[-1, 0])
    php, phm = (dA * full_raw)[full_raw > 0].sum(), (dA * full_raw)[full_raw <= 0].sum()
    assert abs(sn[0] / sp[0] - abs(php / phm)) < 1e-10 * abs(php / phm)


def test_workload_recipes_and_step_plans():
    """DESIGN.md input recipe: config parameters map onto Eq. 3/4 (reading U17) and the derived step sizes."""
    w1 = wl.config(1)
    p = w1.params[0]
    assert np.allclose(p[1:4], [212.30, -337.43, -251.67], atol=0.01)
    assert abs(p[4] / 15.0 - 16 / (3 * math.sqrt(3))) < 1e-15 and p[5] == -p[4] and p[6] == 0
    o = Oracle(w1.n_theta, w1.n_phi, w1.params)
    t = o.tables()
    lat30 = np.argmin(np.abs(np.arange(w1.n_theta + 1) + 0.5 - (w1.n_theta + 1) / 3))     # theta = 60 deg
    assert abs(abs(t["vt"][lat30]) / (15.0 * 5.172413793103448e-6) - 1) < 1e-3 and t["vt"][lat30] < 0
    dt, n, _ = wl.plan(w1, *o.stable_dt())
    assert n == 16 and abs(dt - 1.5) < 1e-12
    assert o.sts_stage_count(dt, DIFF_RKG2) == 217
    w0 = wl.config(0)
    o0 = Oracle(w0.n_theta, w0.n_phi, w0.params)
    dt0, n0, _ = wl.plan(w0, *o0.stable_dt())
    assert n0 == 200 and abs(dt0 - 8 * o0.stable_dt()[1]) < 1e-15 and abs(dt0 - 6.04) < 0.01
    w3 = wl.config(3)
    assert w3.params.shape == (64, 7) and np.all(np.abs(w3.params[:, 0] / 500 - 1) <= 0.2)
    w4 = wl.config(4)
    dt4, n4, per = wl.plan(w4, 0.7, 1e-5)
    assert per == 3 and n4 == 72 and abs(dt4 - 1.0 / 3.0) < 1e-15


def test_synthetic_maps_are_seeded_and_paper_shaped():
    w0 = wl.config(0)
    a, b = wl.initial_maps(w0).numpy(), wl.initial_maps(w0).numpy()
    assert a.shape == (1, 64, 128) and np.array_equal(a, b)
    assert 1.0 < np.abs(a).max() <= 100.0 + 1e-9
    lat = 90 - np.degrees((np.arange(1, 65) * math.pi / 65))
    assert np.abs(a[0][np.abs(lat) > 60]).max() < 1e-3 * np.abs(a).max()      # pairs live within +-40 deg
    w3 = wl.scaled(wl.config(3), 32, 64, n_real=3)
    m3 = wl.initial_maps(w3).numpy()
    assert m3.shape == (3, 32, 64) and not np.array_equal(m3[0], m3[1])
    ww = wl.assimilation_weights(wl.scaled(wl.config(4), 64, 128), 0.0).numpy()
    assert ww.max() <= 1 and ww.min() == 0 and abs(ww[32, 64] - math.sin(33 * math.pi / 65) ** 4) < 1e-12
    assert ww[32, 0] == 0
