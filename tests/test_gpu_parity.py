"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same
seeded inputs.  Tolerances (BASELINE.json north_star): fp64 relative L-inf <= 1e-12 of max|Br|, fp32 <= 1e-5
(against the oracle instantiated in float; the error against the fp64 oracle is also checked at 1e-5)."""
import math

import numpy as np
import pytest
import torch

from helpers import rel_linf
from oracle import sft_oracle as orc
from paper_2501_06377_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-12, "f32": 1e-5}
NPDT = {"f64": np.float64, "f32": np.float32}


def hft():
    from paper_2501_06377_b200 import hft as m
    return m


def make_pair(w, dtype, **opt):
    """(gpu context, oracle) with the same parameters and initial maps."""
    H = hft()
    maps = wl.initial_maps(w)                                   # fp64 CPU tensor [R][nt][np]
    maps_t = maps.to(torch.float64 if dtype == "f64" else torch.float32)
    ctx = H.Context(w.n_theta, w.n_phi, w.params, dtype=dtype, **opt)
    o = orc.Oracle(w.n_theta, w.n_phi, w.params, dtype=NPDT[dtype])
    for r in range(w.n_real):
        ctx.set_map(r, maps_t[r].contiguous().cuda())
        o.set_map(r, maps_t[r].numpy())
    return ctx, o


def compare(ctx, o, tol, what=""):
    worst = 0.0
    for r in range(o.nr):
        g = ctx.get_full(r).cpu().numpy()
        e = rel_linf(g, o.get_full(r))
        worst = max(worst, e)
        assert np.isfinite(g).all()
        assert e <= tol, (what, r, e)
    return worst


def test_set_get_roundtrip_and_pole_cell_averaging():
    H = hft()
    for dtype in ("f64", "f32"):
        w = wl.scaled(wl.config(3), 37, 200, n_real=3)           # ragged: 200 is not a multiple of 128
        ctx, o = make_pair(w, dtype)
        assert compare(ctx, o, 1e-15 if dtype == "f64" else 1e-7) >= 0.0
        allm = ctx.get_map(-1).cpu().numpy()
        for r in range(3):
            assert np.array_equal(allm[r], o.get_map(r)) and np.array_equal(ctx.get_map(r).cpu().numpy(), o.get_map(r))
        m = torch.randn(37, 200, dtype=ctx.tdtype, device="cuda")
        ctx.set_map(-1, m)
        assert all(torch.equal(ctx.get_map(r), m) for r in range(3))
        ga, gd = ctx.stable_dt()
        oa, od = o.stable_dt()
        assert abs(ga / oa - 1) < 1e-14 and abs(gd / od - 1) < 1e-14
        assert ctx.sts_stage_count(37.0 * gd) == o.sts_stage_count(37.0 * od, orc.DIFF_RKG2)
        ctx.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("block", [1, 0])
def test_config0_diffusion_only_full_length(dtype, block):
    """BASELINE config 0: 64x128, 6 pairs, eta = 500, s = 8 forced, dt = 8 dt_expl, 200 steps."""
    H = hft()
    w = wl.config(0)
    ctx, o = make_pair(w, dtype, adv_flux=H.ADV_OFF, diff_time=H.DIFF_RKG2, sts_stages=8, sts_block=block)
    dt, n, _ = wl.plan(w, *o.stable_dt())
    dg = wl.plan(w, *ctx.stable_dt())
    assert dg[1] == n and abs(dg[0] / dt - 1) < 1e-14
    before = ctx.diagnostics()
    ctx.step(n, dt)
    o.step(n, dt, adv_flux=orc.ADV_OFF, diff_time=orc.DIFF_RKG2, sts_stages=8)
    compare(ctx, o, TOL[dtype], "cfg0")
    after = ctx.diagnostics()
    cons = 1e-12 if dtype == "f64" else 2e-5
    assert abs(after[0, 0] - before[0, 0]) <= cons * before[0, 1]      # signed flux conserved
    assert np.allclose(after, o.diagnostics(), rtol=0, atol=cons * before[0, 1])
    ctx.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("block", [1, 0])
def test_y21_decay_on_gpu(dtype, block):
    H = hft()
    w = wl.config(0)
    ctx = H.Context(w.n_theta, w.n_phi, w.params, dtype=dtype, adv_flux=H.ADV_OFF, sts_stages=8, sts_block=block)
    y = wl.y21_map(w.n_theta, w.n_phi).to(ctx.tdtype).cuda()
    ctx.set_map(0, y)
    _, dtd = ctx.stable_dt()
    ctx.step(200, 8 * dtd)
    nu = 500.0 * 7.43162901307967e-9
    exact = y.double() * math.exp(-6 * nu * 200 * 8 * dtd)
    assert (ctx.get_map(0).double() - exact).abs().max().item() < 6e-5
    ctx.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("case", ["weno_ssprk43_rkg2", "upwind_euler_rkl2", "weno_ssprk33_euler", "adv_only", "diff_auto_s"])
def test_small_ragged_multi_realization(dtype, case):
    """Several tiles and a ragged tail in both directions, 3 realizations with different parameters."""
    H = hft()
    w = wl.scaled(wl.config(3), 75, 200, n_real=3)
    opts = {
        "weno_ssprk43_rkg2": dict(adv_flux=2, adv_time=4, diff_time=3),
        "upwind_euler_rkl2": dict(adv_flux=1, adv_time=1, diff_time=2),
        "weno_ssprk33_euler": dict(adv_flux=2, adv_time=3, diff_time=1),
        "adv_only": dict(adv_flux=2, adv_time=4, diff_time=0),
        "diff_auto_s": dict(adv_flux=0, adv_time=4, diff_time=3),
    }[case]
    ctx, o = make_pair(w, dtype, **opts)
    adv, dif = o.stable_dt()
    dt = {"weno_ssprk43_rkg2": 0.5 * adv, "upwind_euler_rkl2": 0.4 * adv, "weno_ssprk33_euler": 0.9 * dif,
          "adv_only": 0.5 * adv, "diff_auto_s": 300.0 * dif}[case]
    n = 6
    ctx.step(n, dt)
    s = o.step(n, dt, **opts)
    if opts["diff_time"] >= 2:
        assert s == ctx.sts_stage_count(dt)
    compare(ctx, o, TOL[dtype], case)
    # the error against the fp64 oracle (arithmetic design, reading U14)
    if dtype == "f32":
        o64 = orc.Oracle(w.n_theta, w.n_phi, w.params)
        maps = wl.initial_maps(w).to(torch.float32)
        for r in range(3):
            o64.set_map(r, maps[r].numpy().astype(np.float64))
        o64.step(n, dt, **opts)
        compare(ctx, o64, 1e-5, case + " vs fp64 oracle")
    ctx.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("block", [2, 4, 6, 8])
@pytest.mark.parametrize("s_forced", [0, 41])
@pytest.mark.parametrize("nphi", [328, 327, 329, 330])
@pytest.mark.parametrize("kern", ["pipe", "upipe", "default"])
def test_sts_block_sizes_ragged(dtype, block, s_forced, nphi, kern):
    """Both temporally blocked kernels -- k_sts_pipe (sts_kernel = 1), k_sts_upipe (2) in the state's own arithmetic, and
    the library default (fp32: k_sts_upipe with fp64 block arithmetic) -- at
    every temporal-blocking depth K of the STS kernel (hft_options.sts_block) on a grid with ragged strips, a
    phi seam inside a strip and theta segments: s = 42 -> (s-1) mod K remainder stages un-blocked; s_forced = 41
    -> (s-1) mod 8 = 0, the block that starts from delta_0 = 0.  n_phi = 327, 329, 330 are not multiples of the
    16-byte vector width (2 doubles / 4 floats): the lanes behind the seam move their columns one by one, a vector
    may straddle the seam (the paper's own grids have odd n_phi in this API: 512 x 1024 files = 510 x 1023 cells)."""
    H = hft()
    w = wl.scaled(wl.config(3), 150, nphi, n_real=2)
    kw = {"pipe": dict(sts_kernel=1, f32_arith=1), "upipe": dict(sts_kernel=2, f32_arith=1), "default": {}}[kern]
    ctx, o = make_pair(w, dtype, adv_flux=H.ADV_OFF, diff_time=H.DIFF_RKG2, sts_block=block, sts_stages=s_forced, **kw)
    _, dif = o.stable_dt()
    dt = 250.0 * dif
    s = ctx.sts_stage_count(dt)
    assert s <= 41
    ctx.step(3, dt)
    o.step(3, dt, adv_flux=orc.ADV_OFF, diff_time=orc.DIFF_RKG2, sts_stages=s_forced)
    compare(ctx, o, TOL[dtype], f"K={block}")
    ctx.close()


def _stretched_nodes(nt, a=0.2):
    xi = np.arange(nt + 2) * math.pi / (nt + 1)
    th = xi + a * np.sin(2 * xi)
    th[0], th[-1] = 0.0, math.pi
    return th


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("path", ["default", "pipe", "upipe", "unblocked", "attenuated", "nu_map"])
def test_nonuniform_theta_grid(dtype, path):
    """the non-uniform theta grid (Eq. 27-28 with the printed spacings, App. A per-cap
    prefactors, App. B D-factors; readings U12, U33) through every STS path -- both temporally blocked kernels, one launch
    per stage, nu(theta, phi) -- with WENO3 advection, flow attenuation, assimilation and all diagnostics, on a ragged
    stretched grid (cells differ by a factor 2.3 in width), 3 realizations."""
    H = hft()
    w = wl.scaled(wl.config(3), 75, 264, n_real=3)
    w.params = np.array(w.params, dtype=np.float64)
    w.params[:, 0] *= 12.0                            # eta x 12: s ~ 35 stages at CFL 0.5, enough for the blocked kernels
    kw = {"default": {}, "pipe": dict(sts_kernel=1, f32_arith=1), "upipe": dict(sts_kernel=2, f32_arith=1), "unblocked": dict(sts_block=1),
          "attenuated": dict(flow_attenuation=1), "nu_map": dict(diffusivity_map=1)}[path]
    ctx, o = make_pair(w, dtype, **kw)
    th = _stretched_nodes(w.n_theta)
    ctx.set_theta_nodes(th)
    o.set_theta_nodes(th)
    # set_map averaged the caps on the old grid: same on both sides; re-set the maps so that both start from the same state
    maps = wl.initial_maps(w).to(torch.float64 if dtype == "f64" else torch.float32)
    for r in range(w.n_real):
        ctx.set_map(r, maps[r].contiguous().cuda())
        o.set_map(r, maps[r].numpy())
    if path == "attenuated":
        ctx.set_attenuation(-1, 30.0)
        for r in range(w.n_real):
            o.set_attenuation(r, 30.0)
    if path == "nu_map":
        for r in range(w.n_real):
            m = wl.diffusivity_map(w, r)
            ctx.set_diffusivity_map(r, m)
            o.set_diffusivity_map(r, m)
    ga, gd = ctx.stable_dt()
    oa, od = o.stable_dt()
    assert abs(ga / oa - 1) < 1e-13 and abs(gd / od - 1) < 1e-13
    dt = 0.5 * ga
    s = ctx.sts_stage_count(dt)
    assert s == o.sts_stage_count(dt) and s > 20
    before = ctx.diagnostics()
    ctx.step(3, dt)
    o.step(3, dt)
    compare(ctx, o, TOL[dtype], "non-uniform " + path)
    after = ctx.diagnostics()
    assert np.all(np.abs(after[:, 0] - before[:, 0]) <= (1e-12 if dtype == "f64" else 2e-5) * before[:, 1])
    wt = wl.assimilation_weights(w, 3 * dt)
    obs = torch.from_numpy(o.get_map(0)).clone() + wl.emergence_map(w, 0).to(maps.dtype)
    ctx.assimilate(obs.contiguous().cuda(), wt.to(maps.dtype).cuda(), flags=1)
    o.assimilate(obs.numpy(), wt.to(maps.dtype).numpy(), flags=1)
    compare(ctx, o, TOL[dtype], "non-uniform assimilation")
    dg, do = ctx.diagnostics(), o.diagnostics()
    assert np.allclose(dg, do, rtol=0, atol=(1e-12 if dtype == "f64" else 1e-5) * do[:, 1].max())
    eg, eo = ctx.diagnostics_ext(55.0), o.diagnostics_ext(55.0)
    tol, bmax = (1e-12 if dtype == "f64" else 2e-5), np.abs(eo[:, 6:8]).max()
    assert np.allclose(eg[:, 0:4], eo[:, 0:4], rtol=0, atol=tol * do[:, 1].max())
    assert np.allclose(eg[:, 4:6], eo[:, 4:6], rtol=1e-13, atol=0)                    # region areas: geometry only
    assert np.allclose(eg[:, 6:13], eo[:, 6:13], rtol=0, atol=tol * bmax)
    ctx.close()


@pytest.mark.parametrize("block", [1, 0])
def test_config1_full_length(block):
    """BASELINE config 1: 512x1024, 40 pairs, flows of reading U17, eta = 500, 16 steps of 1.5 h, s = 217."""
    H = hft()
    w = wl.config(1)
    ctx, o = make_pair(w, "f64", sts_block=block)
    dt, n, _ = wl.plan(w, *ctx.stable_dt())
    assert n == 16 and abs(dt - 1.5) < 1e-12 and ctx.sts_stage_count(dt) == 217
    before = ctx.diagnostics()
    ctx.step(n, dt)
    o.step(n, dt)
    compare(ctx, o, 1e-12, "cfg1")
    after = ctx.diagnostics()
    assert abs(after[0, 0] - before[0, 0]) <= 1e-12 * before[0, 1]
    ctx.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config3_full_size_sampled_realizations(dtype):
    """BASELINE config 3 at full size (1024x2048, 64 realizations) in the launch configuration bench.py
    times, 2 steps; the oracle checks sampled realizations one by one; all 64 conserve flux."""
    H = hft()
    w = wl.config(3, dtype)
    ctx = H.Context(w.n_theta, w.n_phi, w.params, dtype=dtype)
    maps = wl.initial_maps(w, device="cuda").to(ctx.tdtype)
    for r in range(w.n_real):
        ctx.set_map(r, maps[r].contiguous())
    dt, _, _ = wl.plan(w, *ctx.stable_dt())
    before = ctx.diagnostics()
    ctx.step(2, dt)
    after = ctx.diagnostics()
    cons = 1e-12 if dtype == "f64" else 2e-5
    assert np.all(np.abs(after[:, 0] - before[:, 0]) <= cons * before[:, 1])
    for r in (0, 42) if dtype == "f64" else (21,):
        # one realization at a time, with the ensemble's dt and stage count (one s for all realizations)
        o = orc.Oracle(w.n_theta, w.n_phi, w.params[r:r + 1], dtype=NPDT[dtype])
        o.set_map(0, maps[r].cpu().numpy())
        o.step(2, dt, sts_stages=ctx.sts_stage_count(dt))
        e = rel_linf(ctx.get_full(r).cpu().numpy(), o.get_full(0))
        assert e <= TOL[dtype], (r, e)
    ctx.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("path", ["nu_map", "nu_map_stagewise", "unblocked"])
def test_config3_full_size_stage_by_stage_paths(dtype, path):
    """The nu(theta, phi) paths and the one-launch-per-stage path at BASELINE config 3's full size in the launch configurations
    bench.py times (`--nu-map`: nu(theta, phi) of workloads.diffusivity_map through the temporally blocked k_sts_mpipe with the
    polar band k_sts_mcapseq; the same with `--sts-block 1`: one launch per stage; `--sts-block 1` alone), one step; the oracle
    checks a sampled realization; all 64 conserve flux."""
    H = hft()
    w = wl.config(3, dtype)
    opt = {"nu_map": dict(diffusivity_map=1), "nu_map_stagewise": dict(diffusivity_map=1, sts_block=1), "unblocked": dict(sts_block=1)}[path]
    path = "nu_map" if path.startswith("nu_map") else path
    ctx = H.Context(w.n_theta, w.n_phi, w.params, dtype=dtype, **opt)
    maps = wl.initial_maps(w, device="cuda").to(ctx.tdtype)
    for r in range(w.n_real):
        ctx.set_map(r, maps[r].contiguous())
        if path == "nu_map":
            ctx.set_diffusivity_map(r, wl.diffusivity_map(w, r))
    dt, _, _ = wl.plan(w, *ctx.stable_dt())
    s = ctx.sts_stage_count(dt)
    before = ctx.diagnostics()
    ctx.step(1, dt)
    after = ctx.diagnostics()
    cons = 1e-12 if dtype == "f64" else 2e-5
    assert np.all(np.abs(after[:, 0] - before[:, 0]) <= cons * before[:, 1])
    r = 42 if dtype == "f64" else 21
    o = orc.Oracle(w.n_theta, w.n_phi, w.params[r:r + 1], dtype=NPDT[dtype])
    o.set_map(0, maps[r].cpu().numpy())
    if path == "nu_map":
        o.set_diffusivity_map(0, wl.diffusivity_map(w, r))
    o.step(1, dt, sts_stages=s)
    e = rel_linf(ctx.get_full(r).cpu().numpy(), o.get_full(0))
    assert e <= TOL[dtype], (r, e)
    ctx.close()


def test_config2_full_size_sampled_realizations():
    """BASELINE config 2 at full size (1024x2048, 8 realizations with eta = 250..600, v0 = 10..20, shared map),
    2 of its 31 steps; the oracle checks realizations 0 and 7 (smallest and largest diffusivity) one by one."""
    H = hft()
    w = wl.config(2)
    ctx = H.Context(w.n_theta, w.n_phi, w.params, dtype="f64")
    maps = wl.initial_maps(w, device="cuda")
    ctx.set_map(-1, maps[0].contiguous())
    dt, n, _ = wl.plan(w, *ctx.stable_dt())
    s = ctx.sts_stage_count(dt)
    assert n == 31 and 600 < s < 760, (n, s)
    before = ctx.diagnostics()
    ctx.step(2, dt)
    after = ctx.diagnostics()
    assert np.all(np.abs(after[:, 0] - before[:, 0]) <= 1e-12 * before[:, 1])
    for r in (0, 7):
        o = orc.Oracle(w.n_theta, w.n_phi, w.params[r:r + 1])
        o.set_map(0, maps[r].cpu().numpy())
        o.step(2, dt, sts_stages=s)
        e = rel_linf(ctx.get_full(r).cpu().numpy(), o.get_full(0))
        assert e <= 1e-12, (r, e)
    ctx.close()


def test_config3_full_length_sampled_realizations():
    """BASELINE config 3 at full size AND full length: 2 simulated days = 79 steps of 604 RKG2 stages + SSPRK(4,3) on all
    64 realizations, started from the same float-representable maps in every precision.  The fp64 oracle follows
    realizations 0, 21, 42, 63 (BASELINE.md section 3's plan) through all 79 steps, one by one.
      fp64                                        <= 1e-12 (measured 2.3e-15 .. 3.9e-15)
      fp32, default (fp64 block arithmetic)       <= 1e-5, north_star's gate (measured 2.0e-6 .. 2.7e-6)
      fp32, f32_arith = 1 (fp32 arithmetic)       north_star's 1e-5 is NOT met: measured 1.4e-5 .. 2.2e-5.  Every one of the
          79 x 604 stages rounds delta to 24 bits and the three-term recurrence amplifies that noise; the oracle built in
          float is itself 3.7e-5 from the fp64 oracle on this run (HFT_SLOW=1 below runs it: 7 min).  The assertion below is
          a regression bound on that known miss, not a claim of parity."""
    import os
    H = hft()
    w = wl.config(3, "f64")
    maps32 = wl.initial_maps(w, device="cuda").to(torch.float32)
    R = (0, 21, 42, 63)
    errs, refs, g42 = {}, {}, None
    for name, kw in (("f64", dict(dtype="f64")), ("f32", dict(dtype="f32")), ("f32_arith1", dict(dtype="f32", f32_arith=1))):
        ctx = H.Context(w.n_theta, w.n_phi, w.params, **kw)
        for q in range(w.n_real):
            ctx.set_map(q, maps32[q].to(ctx.tdtype).contiguous())
        dt, n, _ = wl.plan(w, *ctx.stable_dt())
        s = ctx.sts_stage_count(dt)
        assert n == 79 and s == 604, (n, s)
        before = ctx.diagnostics()
        ctx.step(n, dt)
        after = ctx.diagnostics()
        cons = 1e-12 if name == "f64" else 1e-4
        assert np.all(np.abs(after[:, 0] - before[:, 0]) <= cons * before[:, 1])
        if not refs:
            for r in R:
                o = orc.Oracle(w.n_theta, w.n_phi, w.params[r:r + 1], dtype=np.float64)
                o.set_map(0, maps32[r].double().cpu().numpy())
                o.step(n, dt, sts_stages=s)
                refs[r] = o.get_full(0)
                o.close()
        errs[name] = [rel_linf(ctx.get_full(r).cpu().numpy(), refs[r]) for r in R]
        if name == "f32_arith1":
            g42 = ctx.get_full(42).cpu().numpy()
        ctx.close()
    print("cfg3 full length (79 steps), realizations %s: rel L-inf %s" % (R, {k: ["%.2e" % e for e in v] for k, v in errs.items()}))
    assert max(errs["f64"]) <= 1e-12, errs
    assert max(errs["f32"]) <= 1e-5, errs                  # north_star's fp32 gate, met by the default fp32 path
    assert max(errs["f32_arith1"]) <= 3e-5, errs           # fp32 arithmetic: north_star NOT met (1.4e-5 .. 2.2e-5); regression bound
    if os.environ.get("HFT_SLOW") == "1":
        o = orc.Oracle(w.n_theta, w.n_phi, w.params[42:43], dtype=np.float32)
        o.set_map(0, maps32[42].cpu().numpy())
        o.step(n, dt, sts_stages=s)
        ref32 = o.get_full(0)
        e_gpu, e_orc = rel_linf(g42, ref32), rel_linf(ref32, refs[42])
        print("float oracle: cuda fp32 vs float oracle %.3e, float oracle vs fp64 oracle %.3e" % (e_gpu, e_orc))
        assert errs["f32_arith1"][2] <= e_orc and e_gpu <= 2.0 * e_orc      # the CUDA path is the more accurate of the two


def test_config2_full_length_sampled_realization():
    """BASELINE config 2 at full size and full length: 31 steps of 683 stages, 8 realizations, fp64; the oracle follows
    realization 7 (largest diffusivity and flow speed) to the end."""
    H = hft()
    w = wl.config(2)
    ctx = H.Context(w.n_theta, w.n_phi, w.params, dtype="f64")
    maps = wl.initial_maps(w, device="cuda")
    ctx.set_map(-1, maps[0].contiguous())
    dt, n, _ = wl.plan(w, *ctx.stable_dt())
    s = ctx.sts_stage_count(dt)
    assert n == 31
    ctx.step(n, dt)
    o = orc.Oracle(w.n_theta, w.n_phi, w.params[7:8])
    o.set_map(0, maps[0].cpu().numpy())
    o.step(n, dt, sts_stages=s)
    e = rel_linf(ctx.get_full(7).cpu().numpy(), o.get_full(0))
    print("cfg2 full length (31 steps), realization 7: rel L-inf %.3e" % e)
    assert e <= 1e-12, e
    ctx.close()


def test_config4_full_size_first_assimilation_hour():
    """BASELINE config 4 at full size (2048x4096, fp64): the first simulated hour (its steps at CFL 0.5, s ~ 1640
    stages each) followed by the hourly assimilation of the synthetic observation with the disc weights; element by
    element against the oracle, then diagnostics."""
    H = hft()
    w = wl.config(4)
    ctx, o = make_pair(w, "f64")
    dt, n, per = wl.plan(w, *ctx.stable_dt())
    assert n == 24 * per and abs(per * dt - 1.0) < 1e-12
    s = ctx.sts_stage_count(dt)
    assert s == o.sts_stage_count(dt) and s > 1000, s
    ctx.step(per, dt)
    o.step(per, dt)
    compare(ctx, o, 1e-12, "cfg4 hour 1")
    E = wl.emergence_map(w, 0)
    wt = wl.assimilation_weights(w, per * dt)
    obs = (torch.from_numpy(o.get_map(0)) + E).contiguous()     # "current state + emergence": the ORACLE's state, fed to both
    ctx.assimilate(obs.cuda(), wt.cuda())
    o.assimilate(obs.numpy(), wt.numpy())
    compare(ctx, o, 1e-12, "cfg4 assimilation 1")
    dg, do = ctx.diagnostics(), o.diagnostics()
    assert np.allclose(dg, do, rtol=0, atol=1e-12 * do[:, 1].max())
    ctx.close()


def test_config4_full_size_assimilation_cycle():
    """BASELINE config 4 at full size, 2048x4096 fp64: repeated hft_step <-> hft_assimilate.  By default the first 6 of the 24
    assimilation hours (18 steps of 1638 stages + 6 blends of the synthetic observation with the moving disc weights, about
    2 min of oracle time); HFT_SLOW=1 runs the full simulated day (72 steps + 24 assimilations, ~8 min).  Element by element
    at the end."""
    import os
    hours = 24 if os.environ.get("HFT_SLOW") == "1" else 6
    w = wl.config(4)
    ctx, o = make_pair(w, "f64")
    dt, n, per = wl.plan(w, *ctx.stable_dt())
    t = 0.0
    for hour in range(hours):
        ctx.step(per, dt)
        o.step(per, dt)
        t += per * dt
        obs = (torch.from_numpy(o.get_map(0)) + wl.emergence_map(w, hour)).contiguous()
        wt = wl.assimilation_weights(w, t)
        ctx.assimilate(obs.cuda(), wt.cuda())
        o.assimilate(obs.numpy(), wt.numpy())
    e = compare(ctx, o, 1e-12, "cfg4 %d hours" % hours)
    print("cfg4 (%d steps + %d assimilations): rel L-inf %.3e" % (hours * per, hours, e))
    dg, do = ctx.diagnostics(), o.diagnostics()
    assert np.allclose(dg, do, rtol=0, atol=1e-12 * do[:, 1].max())
    ctx.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("flags", [0, 1])
def test_fused_assimilation_diagnostics(dtype, flags):
    """hft_assimilate_diagnostics = hft_assimilate + hft_diagnostics in one pass over the state (north_star's fused
    assimilation/diagnostics kernel): the blended state must be bit-identical to the two-call sequence, the diagnostics equal
    to it up to summation order, and both must match the oracle; plain (Eq. 8) and flux-balanced (Eq. 10-11) blend, shared
    and per-realization observations, ragged grid."""
    H = hft()
    w = wl.scaled(wl.config(4), 61, 200, t_end_hours=3.0)
    w.params = np.repeat(w.params, 3, axis=0)
    w.params[1, 0], w.params[2, 0] = 350.0, 650.0
    w.n_real = 3
    ctx, o = make_pair(w, dtype)
    ctx2, _ = make_pair(w, dtype)
    dt, _, per = wl.plan(w, *ctx.stable_dt())
    for c in (ctx, ctx2):
        c.step(1, dt)
    o.step(1, dt)
    td = torch.float64 if dtype == "f64" else torch.float32
    wt = wl.assimilation_weights(w, dt).to(td)
    obs1 = (torch.from_numpy(o.get_map(0)) + wl.emergence_map(w, 0).to(td)).contiguous()
    dg = ctx.assimilate_diagnostics(obs1.cuda(), wt.cuda(), flags=flags)
    ctx2.assimilate(obs1.cuda(), wt.cuda(), flags=flags)
    d2 = ctx2.diagnostics()
    o.assimilate(obs1.numpy(), wt.numpy(), flags=flags)
    do = o.diagnostics()
    for r in range(w.n_real):
        assert torch.equal(ctx.get_full(r), ctx2.get_full(r))
    tol = 1e-12 if dtype == "f64" else 1e-5
    assert np.allclose(dg, d2, rtol=0, atol=1e-13 * do[:, 1].max())
    assert np.allclose(dg, do, rtol=0, atol=tol * do[:, 1].max())
    compare(ctx, o, TOL[dtype], "fused blend")
    # per-realization observations
    obsR = torch.stack([torch.from_numpy(o.get_map(r)) + wl.emergence_map(w, 1 + r).to(td) for r in range(w.n_real)]).contiguous()
    wtR = torch.stack([wl.assimilation_weights(w, dt * (2 + r)).to(td) for r in range(w.n_real)]).contiguous()
    dg = ctx.assimilate_diagnostics(obsR.cuda(), wtR.cuda(), flags=flags)
    o.assimilate(obsR.numpy(), wtR.numpy(), flags=flags)
    assert np.allclose(dg, o.diagnostics(), rtol=0, atol=tol * do[:, 1].max())
    compare(ctx, o, TOL[dtype], "fused blend, per-realization maps")
    ctx.close()
    ctx2.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_assimilation_and_diagnostics(dtype):
    """Config 4 recipe on a small grid: steps, hourly blend with disc weights, per-realization and shared
    observations, flux-balanced variant, diagnostics."""
    H = hft()
    w = wl.scaled(wl.config(4), 60, 136, t_end_hours=3.0)
    w.params = np.repeat(w.params, 2, axis=0)
    w.params[1, 0] = 350.0
    w.n_real = 2
    ctx, o = make_pair(w, dtype)
    dt, n, per = wl.plan(w, *ctx.stable_dt())
    tdt = ctx.tdtype
    t = 0.0
    for it in range(3):
        ctx.step(per, dt)
        o.step(per, dt)
        t += per * dt
        E = wl.emergence_map(w, it)
        wt = wl.assimilation_weights(w, t)
        if it == 1:            # shared observation map
            obs = (torch.from_numpy(o.get_map(0)).double() + E).to(tdt)     # the oracle's state, fed to both sides
            ctx.assimilate(obs.cuda(), wt.to(tdt).cuda())
            o.assimilate(obs.numpy(), wt.to(tdt).numpy())
        else:                  # per-realization observation = own state + emergence
            cur = torch.from_numpy(np.stack([o.get_map(q) for q in range(2)])).double()
            obs = (cur + E[None]).to(tdt).contiguous()
            wts = wt[None].expand(2, -1, -1).to(tdt).contiguous()
            ctx.assimilate(obs.cuda(), wts.cuda(), flags=H.FLAG_FLUX_BALANCE if it == 2 else 0)
            o.assimilate(obs.numpy(), wts.numpy(), flags=1 if it == 2 else 0)
        compare(ctx, o, TOL[dtype], f"assim {it}")
    dg, do = ctx.diagnostics(), o.diagnostics()
    assert np.allclose(dg, do, rtol=0, atol=(1e-12 if dtype == "f64" else 1e-5) * do[:, 1].max())
    ctx.close()


def test_custom_flow_tables_appendix_c():
    """hft_set_flow_tables: constant v_theta, the App. C solution moves without changing shape."""
    H = hft()
    nt, nphi = 127, 64
    ctx = H.Context(nt, nphi, [[0.0] * 7], diff_time=H.DIFF_OFF)
    o = orc.Oracle(nt, nphi, [[0.0] * 7])
    v_ms = 200.0
    ctx.set_flow_tables(0, np.full(nt + 1, v_ms), np.zeros(nt + 2))
    o.set_flow_tables(0, np.full(nt + 1, v_ms * 5.172413793103448e-6), np.zeros(nt + 2))
    th = wl.colatitudes(nt)[:, None]
    B = (torch.exp(-(th - math.pi / 4) ** 2 / 0.03) / torch.sin(th)).expand(-1, nphi).contiguous()
    ctx.set_map(0, B.cuda())
    o.set_map(0, B.numpy())
    adv, _ = ctx.stable_dt()
    assert abs(adv / o.stable_dt()[0] - 1) < 1e-14
    ctx.step(40, 0.5 * adv)
    o.step(40, 0.5 * adv, diff_time=orc.DIFF_OFF)
    compare(ctx, o, 1e-12, "appendix C")
    v = v_ms * 5.172413793103448e-6
    exact = torch.exp(-(th - math.pi / 4 - v * 20 * adv) ** 2 / 0.03) / torch.sin(th)
    assert (ctx.get_map(0).cpu()[:, 0:1] - exact).abs().max().item() < 2e-2
    ctx.close()


def test_errors_are_reported():
    H = hft()
    ctx = H.Context(64, 128, [[500.0, 0, 0, 0, 0, 0, 0]], adv_flux=H.ADV_OFF, sts_stages=2)
    _, dtd = ctx.stable_dt()
    with pytest.raises(H.HftError, match="unstable"):
        ctx.step(1, 50 * dtd)                    # s = 2 forced is too few stages for this dt
    with pytest.raises(H.HftError):
        ctx.step(1, -1.0)
    assert ctx.launch_count() >= 0
    ctx.step(1, dtd)
    ctx.synchronize()                            # where an asynchronous kernel fault of that step would be reported
    ctx.close()
    # hft_create rejects what would fail later with a generic launch error or run anti-diffusion silently
    for bad in ([[float("nan"), 0, 0, 0, 0, 0, 0]], [[-1.0, 0, 0, 0, 0, 0, 0]], [[500.0, float("inf"), 0, 0, 0, 0, 0]]):
        with pytest.raises(H.HftError, match="invalid argument"):
            H.Context(64, 128, bad)
    with pytest.raises(H.HftError, match="invalid argument"):
        H.workspace_bytes(65534, 128, 1, "f64", None)          # n_theta + 2 rows ride in gridDim.y (16 bits)
    with pytest.raises(H.HftError, match="invalid argument"):
        H.workspace_bytes(64, 128, 65536, "f64", None)         # realizations ride in gridDim.z


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_strang_splitting(dtype):
    """Eq. 22 with S omitted, A(dt/2) D(dt) A(dt/2), at the doubled step it allows (:326)."""
    H = hft()
    w = wl.scaled(wl.config(3), 70, 264, n_real=3)
    ctx, o = make_pair(w, dtype, strang=1)
    adv, _ = ctx.stable_dt()
    dt = 0.9 * adv                                   # each half advection step runs at CFL 0.45 of the Eq. 26 limit
    ctx.step(3, dt)
    o.step(3, dt, strang=True)
    compare(ctx, o, TOL[dtype], "strang")
    ctx.close()
    # and it differs from the un-split sequence by the O(dt) splitting error, far above the tolerance
    if dtype == "f64":
        ctx2, _ = make_pair(w, dtype, strang=0)
        ctx2.step(3, dt)
        assert rel_linf(ctx2.get_full(0).cpu().numpy(), o.get_full(0)) > 1e4 * TOL[dtype]
        ctx2.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_run_history_diagnostics(dtype):
    """polar fluxes / areas, min / max / min|Br| and the dipoles of Eq. 16-17 (:230-242) after
    a few steps, on a ragged grid with several realizations and a physical radius."""
    H = hft()
    w = wl.scaled(wl.config(3), 45, 200, n_real=3)
    maps = wl.initial_maps(w).to(torch.float64 if dtype == "f64" else torch.float32)
    ctx = H.Context(w.n_theta, w.n_phi, w.params, dtype=dtype, radius_cm=6.96e10)
    o = orc.Oracle(w.n_theta, w.n_phi, w.params, dtype=NPDT[dtype], radius_cm=6.96e10)
    for r in range(w.n_real):
        ctx.set_map(r, maps[r].contiguous().cuda())
        o.set_map(r, maps[r].numpy())
    dt, _, _ = wl.plan(w, *ctx.stable_dt())
    ctx.step(2, dt)
    o.step(2, dt)
    for lat in (60.0, 33.3, 90.0, 0.0):
        g, e = ctx.diagnostics_ext(lat), o.diagnostics_ext(lat)
        tol = 1e-12 if dtype == "f64" else 2e-5
        flux_scale = o.diagnostics()[:, 1].max()
        assert np.allclose(g[:, 0:4], e[:, 0:4], rtol=0, atol=tol * flux_scale), lat
        assert np.allclose(g[:, 4:6], e[:, 4:6], rtol=1e-13, atol=0), lat            # areas: geometry only
        bmax = np.abs(e[:, 6:8]).max()
        assert np.allclose(g[:, 6:9], e[:, 6:9], rtol=0, atol=tol * bmax), lat
        assert np.allclose(g[:, 9:13], e[:, 9:13], rtol=0, atol=tol * bmax), lat
    assert np.all(g[:, 4] > 0) and abs(g[0, 4] + g[0, 5] - cell_sum(w) * 6.96e10 ** 2) < 1e-9 * g[0, 4]   # lat 0: both hemispheres
    ctx.close()


def cell_sum(w):
    from helpers import cell_areas
    return cell_areas(w.n_theta, w.n_phi).sum()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("case", ["weno", "upwind", "strang"])
@pytest.mark.parametrize("nphi", [200, 345, 40])
def test_flow_attenuation(dtype, case, nphi):
    """flow attenuation Eq. 5 (:100), per-realization B0 (one realization off), strong active regions
    (|Br| up to ~3 B0) on a ragged grid; WENO3 + SSPRK(4,3) + STS, upwind + Euler, and inside a Strang step.  n_phi = 345:
    k_adv_stage_att_u (28 columns per warp) and the other stage kernels (31) use different numbers of CTAs along phi, hence
    of polar partial sums; n_phi = 40: a warp's 32 columns wrap around the seam onto themselves."""
    H = hft()
    w = wl.scaled(wl.config(3), 52, nphi, n_real=3)
    maps = torch.stack([wl.bipolar_map(w.n_theta, w.n_phi, 8, 50 + r, amp=(100.0, 1500.0), sigma_deg=8.0) for r in range(3)])
    maps_t = maps.to(torch.float64 if dtype == "f64" else torch.float32)
    opt = dict(adv_flux=H.ADV_UPWIND, adv_time=H.TIME_EULER) if case == "upwind" else {}
    ctx = H.Context(w.n_theta, w.n_phi, w.params, dtype=dtype, flow_attenuation=1, strang=int(case == "strang"), **opt)
    o = orc.Oracle(w.n_theta, w.n_phi, w.params, dtype=NPDT[dtype])
    for r, b0 in enumerate((500.0, 0.0, 120.0)):
        ctx.set_attenuation(r, b0)
        o.set_attenuation(r, b0)
        ctx.set_map(r, maps_t[r].contiguous().cuda())
        o.set_map(r, maps_t[r].numpy())
    adv, _ = ctx.stable_dt()
    dt = (0.9 if case == "strang" else 0.5) * adv
    before = ctx.diagnostics()
    ctx.step(3, dt)
    if case == "upwind":
        o.step(3, dt, adv_flux=orc.ADV_UPWIND, adv_time=orc.TIME_EULER)
    else:
        o.step(3, dt, strang=(case == "strang"))
    compare(ctx, o, TOL[dtype], "attenuation " + case)
    after = ctx.diagnostics()
    assert np.all(np.abs(after[:, 0] - before[:, 0]) <= (1e-12 if dtype == "f64" else 2e-5) * before[:, 1])
    # the attenuated realizations really moved differently from an un-attenuated run
    if dtype == "f64" and case == "weno":
        ctx0 = H.Context(w.n_theta, w.n_phi, w.params, dtype=dtype)
        ctx0.set_map(0, maps_t[0].contiguous().cuda())
        ctx0.step(3, dt)
        assert rel_linf(ctx0.get_full(0).cpu().numpy(), o.get_full(0)) > 1e-6
        ctx0.close()
    with pytest.raises(H.HftError):
        H.Context(16, 32, [[0.0] * 7]).set_attenuation(0, 500.0)           # workspace was not reserved for it
    ctx.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("model", [1, 2])
def test_random_flux_emergence(dtype, model):
    """source term of Sec. 2.4.  The two balanced source maps element by element (the per-cell normals
    come from the same counter-based generator on both sides), then steps with A, D and S in the Eq. 21 order across two
    map rotations, then a Strang step (Eq. 22)."""
    H = hft()
    w = wl.scaled(wl.config(3), 41, 136, n_real=2)
    flux, tau, seed = 100e21, 0.7, 0x1234567890ABCDEF
    for strang in (0, 1):
        ctx = H.Context(w.n_theta, w.n_phi, w.params, dtype=dtype, radius_cm=6.96e10, rfe=1, strang=strang)
        o = orc.Oracle(w.n_theta, w.n_phi, w.params, dtype=NPDT[dtype], radius_cm=6.96e10)
        maps = wl.initial_maps(w).to(ctx.tdtype)
        for r in range(w.n_real):
            ctx.set_map(r, maps[r].contiguous().cuda())
            o.set_map(r, maps[r].numpy())
        ctx.set_rfe(model, flux, tau, seed)
        o.set_rfe(model, flux, tau, seed)
        for r in range(w.n_real):
            s1, s2 = o.get_rfe_maps(r)
            scale = np.abs(s1).max()
            for which, s in ((0, s1), (1, s2)):
                g = ctx.get_rfe_map(r, which).cpu().numpy()
                assert np.abs(g - s[1:-1]).max() <= (1e-12 if dtype == "f64" else 1e-5) * scale, (r, which)
        dt = 0.3
        ctx.step(6, dt)                       # t = 0 .. 1.8 h: rotations at 0.7 and 1.4 h
        o.step(6, dt, strang=bool(strang))
        compare(ctx, o, TOL[dtype], f"rfe model {model} strang {strang}")
        g1 = ctx.get_rfe_map(0, 0).cpu().numpy()
        assert np.abs(g1 - o.get_rfe_maps(0)[0][1:-1]).max() <= (1e-12 if dtype == "f64" else 1e-5) * np.abs(g1).max()
        ctx.close()
    with pytest.raises(H.HftError):
        H.Context(16, 32, [[0.0] * 7]).set_rfe(2, 1.0e21, 1.0, 1)          # workspace was not reserved for it


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("block", [1, 0])
def test_latitude_dependent_diffusivity(dtype, block):
    """SURVEY.md 8(f)-4 (phi-independent part): nu(theta) profiles per realization and the grid-based nu_g of Eq. 7, through
    both STS paths (the zonal-mean cap recurrence of the blocked kernel only needs phi-independent coefficients), with
    advection on; then the map-smoother use (:586): diffusion only, one large step."""
    H = hft()
    w = wl.scaled(wl.config(3), 72, 264, n_real=3)
    ctx, o = make_pair(w, dtype, sts_block=block)
    rng = np.random.default_rng(12)
    thf = (np.arange(w.n_theta + 1) + 0.5) * math.pi / (w.n_theta + 1)
    prof = [300.0 * (1 + 0.8 * np.cos(thf) ** 2), None, 200.0 + 400.0 * rng.random(w.n_theta + 1)]
    for r, p in enumerate(prof):
        if p is not None:
            ctx.set_diffusivity_profile(r, p)
            o.set_diffusivity_profile(r, p)
    ga, gd = ctx.stable_dt()
    oa, od = o.stable_dt()
    assert abs(gd / od - 1) < 1e-14
    dt, _, _ = wl.plan(w, ga, gd)
    assert ctx.sts_stage_count(dt) == o.sts_stage_count(dt)
    before = ctx.diagnostics()
    ctx.step(3, dt)
    o.step(3, dt)
    compare(ctx, o, TOL[dtype], "nu(theta)")
    after = ctx.diagnostics()
    assert np.all(np.abs(after[:, 0] - before[:, 0]) <= (1e-12 if dtype == "f64" else 2e-5) * before[:, 1])
    ctx.close()
    # smoother: grid-based diffusivity, diffusion only
    ctx = H.Context(w.n_theta, w.n_phi, w.params[:1], dtype=dtype, adv_flux=H.ADV_OFF, sts_block=block)
    o = orc.Oracle(w.n_theta, w.n_phi, w.params[:1], dtype=NPDT[dtype])
    m = (wl.bipolar_map(w.n_theta, w.n_phi, 12, 77) + torch.from_numpy(rng.normal(0, 5.0, (w.n_theta, w.n_phi)))).to(ctx.tdtype)
    ctx.set_grid_diffusivity(0, 2.0e6)
    o.set_grid_diffusivity(0, 2.0e6)
    ctx.set_map(0, m.contiguous().cuda())
    o.set_map(0, m.numpy())
    _, gd = ctx.stable_dt()
    assert abs(gd / o.stable_dt()[1] - 1) < 1e-14
    ctx.step(1, 150 * gd)
    o.step(1, 150 * gd, adv_flux=orc.ADV_OFF)
    compare(ctx, o, TOL[dtype], "smoother")
    ctx.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_diffusivity_map_tall_grid_segments(dtype):
    """k_sts_mpipe keeps the row metric of a CTA's theta segment in a shared-memory table of 1024 rows: a grid of 1500 rows
    cannot be one segment, whatever the occupancy says (the host skips segment counts whose table would not fit), and its
    segments meet at rows that are not multiples of anything.  nu(theta, phi) rough in both directions; diffusion only."""
    H = hft()
    nphi = 64 if dtype == "f64" else 128                         # one strip of 32 lanes x C columns, halo wrapping onto itself
    w = wl.scaled(wl.config(3), 1500, nphi, n_real=2)
    ctx, o = make_pair(w, dtype, diffusivity_map=1, adv_flux=H.ADV_OFF)
    rng = np.random.default_rng(77)
    for r in range(2):
        m = 200.0 + 400.0 * rng.random((w.n_theta + 1, w.n_phi))
        ctx.set_diffusivity_map(r, m); o.set_diffusivity_map(r, m)
    _, gd = ctx.stable_dt()
    dt = 40.0 * gd
    s = ctx.sts_stage_count(dt)
    assert s > 8 and s == o.sts_stage_count(dt, orc.DIFF_RKG2)
    n0 = ctx.launch_count()
    ctx.step(2, dt); o.step(2, dt, adv_flux=orc.ADV_OFF)
    assert ctx.launch_count() - n0 < 2 * s                       # blocked: about s / 2 launches per step, not s
    compare(ctx, o, TOL[dtype], "nu(theta,phi) tall grid")
    ctx.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("case", ["rkg2_adv", "rkl2", "euler"])
@pytest.mark.parametrize("nphi", [264, 263])
@pytest.mark.parametrize("block", [0, 1])
def test_diffusivity_map_theta_phi(dtype, case, nphi, block):
    """nu(theta, phi) on the half-half grid (Eq. 27-28): realization 0 a smooth map, 1 keeps its scalar
    value, 2 a rough random map; ragged grids: 264 columns take the temporally blocked k_sts_mpipe + polar band k_sts_mcapseq
    (block = 0, when the step has more than 8 stages) or the 16-byte-vector kernel k_sts_stage_mapv one stage per launch
    (block = 1; part-filled
    warps, 75 + 2 rows = 4 row blocks + tail), 263 columns the one-column-per-thread kernel k_sts_stage_map.  Then the
    gpu fp32 result against the fp64 oracle, a map replaced by a profile, and the constant map against the table path."""
    H = hft()
    w = wl.scaled(wl.config(3), 75, nphi, n_real=3)
    opt = dict(diffusivity_map=1, sts_block=block)
    kw = {}
    if case == "rkl2":
        opt.update(adv_flux=H.ADV_OFF, diff_time=H.DIFF_RKL2); kw.update(adv_flux=orc.ADV_OFF, diff_time=orc.DIFF_RKL2)
    if case == "euler":
        opt.update(adv_flux=H.ADV_OFF, diff_time=H.DIFF_EULER); kw.update(adv_flux=orc.ADV_OFF, diff_time=orc.DIFF_EULER)
    ctx, o = make_pair(w, dtype, **opt)
    o64 = orc.Oracle(w.n_theta, w.n_phi, w.params, dtype=np.float64)
    for r in range(3):
        o64.set_full(r, o.get_full(r).astype(np.float64))
    rng = np.random.default_rng(31)
    thf = ((np.arange(w.n_theta + 1) + 0.5) * math.pi / (w.n_theta + 1))[:, None]
    phf = ((np.arange(w.n_phi) + 0.5) * 2 * math.pi / w.n_phi)[None, :]
    maps = {0: 400.0 * (1 + 0.5 * np.sin(thf) * np.cos(phf) + 0.3 * np.cos(thf) ** 2 * np.sin(3 * phf)),
            2: 100.0 + 500.0 * rng.random((w.n_theta + 1, w.n_phi))}
    for r, m in maps.items():
        ctx.set_diffusivity_map(r, m); o.set_diffusivity_map(r, m); o64.set_diffusivity_map(r, m)
    ga, gd = ctx.stable_dt()
    oa, od = o.stable_dt()
    assert abs(gd / od - 1) < 1e-13
    if case == "euler":
        dt, n = 0.9 * gd, 25
    else:
        dt, n = (wl.plan(w, ga, gd)[0] if case == "rkg2_adv" else 300.0 * gd), 3
        assert ctx.sts_stage_count(dt) == o.sts_stage_count(dt, kw.get("diff_time", orc.DIFF_RKG2))
    before = ctx.diagnostics()
    ctx.step(n, dt); o.step(n, dt, **kw); o64.step(n, dt, **kw)
    compare(ctx, o, TOL[dtype], "nu(theta,phi) " + case)
    compare(ctx, o64, TOL[dtype], "nu(theta,phi) vs fp64 oracle " + case)
    after = ctx.diagnostics()
    assert np.all(np.abs(after[:, 0] - before[:, 0]) <= (1e-12 if dtype == "f64" else 2e-5) * before[:, 1])
    # realization 2 leaves its map for a profile; realization 0 keeps its map
    prof = 200.0 + 300.0 * rng.random(w.n_theta + 1)
    ctx.set_diffusivity_profile(2, prof); o.set_diffusivity_map(2, None); o.set_diffusivity_profile(2, prof)
    assert abs(ctx.stable_dt()[1] / o.stable_dt()[1] - 1) < 1e-13
    ctx.step(1, dt); o.step(1, dt, **kw)
    compare(ctx, o, TOL[dtype], "map then profile " + case)
    ctx.close()
    # a constant map is the table path (blocked kernel) up to round-off
    if case == "rkl2":
        a, oa_ = make_pair(w, dtype, adv_flux=H.ADV_OFF, diff_time=H.DIFF_RKL2)
        b, _ = make_pair(w, dtype, diffusivity_map=1, adv_flux=H.ADV_OFF, diff_time=H.DIFF_RKL2)
        for r in range(3):
            b.set_diffusivity_map(r, np.full((w.n_theta + 1, w.n_phi), w.params[r][0]))
        assert abs(a.stable_dt()[1] / b.stable_dt()[1] - 1) < 1e-13
        dt = 300.0 * a.stable_dt()[1]
        a.step(2, dt); b.step(2, dt)
        for r in range(3):
            assert rel_linf(b.get_full(r).cpu().numpy(), a.get_full(r).cpu().numpy()) <= TOL[dtype]
        a.close(); b.close()
    # the option is required
    c = H.Context(16, 32, w.params[:1], dtype=dtype)
    with pytest.raises(H.HftError):
        c.set_diffusivity_map(0, np.ones((17, 32)))
    c.close()


@pytest.mark.parametrize("scheme,name", [("rkl2", "hh_rkl2_diffusion"), ("rkg2", "hh_rkg2_diffusion")])
@pytest.mark.parametrize("nphi", [1023, 1024])
def test_paper_printed_hh_errors_on_the_gpu(scheme, name, nphi):
    """diffusion only, Eq. 19 field, 512x1024 file grid (= 510 x 1023 regular cells), nu = 500 km^2/s, ONE 672 h
    super-time step: HH (Eq. 18) against the analytic decay = 8.0e-5 (RKL2), 6.3e-5 (RKG2).  The CUDA path reproduces the
    two printed digits on the paper's grid (odd n_phi: one-column kernels, one launch per stage) and, within 2 %, on
    510 x 1024 (temporally blocked kernel, ~4.7 k stages in one step)."""
    from helpers import golden, grid, hh_metric, soccer_ball
    H = hft()
    nt = 510
    th, ph, _, _ = grid(nt, nphi)
    u = soccer_ball(th, ph)
    ctx = H.Context(nt, nphi, [[500.0, 0, 0, 0, 0, 0, 0]], dtype="f64", adv_flux=H.ADV_OFF,
                    diff_time=H.DIFF_RKL2 if scheme == "rkl2" else H.DIFF_RKG2)
    ctx.set_full(0, torch.from_numpy(np.ascontiguousarray(u)).cuda())
    s = ctx.sts_stage_count(672.0)
    assert 3500 < s < 5200
    ctx.step(1, 672.0)
    got = ctx.get_full(0).cpu().numpy()
    exact = u * math.exp(-42.0 * 500.0 * golden("km2_s_to_rs2_hr") * 672.0)
    hh = hh_metric(got[1:-1], exact[1:-1])
    assert abs(hh / golden(name) - 1) < 0.02, (name, nphi, hh)
    ctx.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_degenerate_sizes_and_calls(dtype):
    """Edge cases: the smallest grid the ABI accepts (8 x 8) and an odd ragged one (9 x 17, below every vector width, so
    all stages take the un-blocked kernels); zero steps is a no-op; a zero map stays zero; a constant map is a fixed point
    of diffusion."""
    H = hft()
    for nt, nphi in ((8, 8), (9, 17)):
        w = wl.scaled(wl.config(1), nt, nphi)
        rng = np.random.default_rng(nt)
        m = torch.from_numpy(rng.normal(0, 10.0, (nt, nphi)))
        ctx = H.Context(nt, nphi, w.params, dtype=dtype)
        o = orc.Oracle(nt, nphi, w.params, dtype=NPDT[dtype])
        ctx.set_map(0, m.to(ctx.tdtype).cuda())
        o.set_map(0, m.to(ctx.tdtype).numpy())
        ctx.step(0, 1.0)
        compare(ctx, o, 1e-15 if dtype == "f64" else 1e-7, "zero steps")   # caps = row means: summation order
        dt, _, _ = wl.plan(w, *ctx.stable_dt())
        ctx.step(3, dt)
        o.step(3, dt)
        compare(ctx, o, TOL[dtype], f"{nt}x{nphi}")
        z = torch.zeros(nt, nphi, dtype=ctx.tdtype, device="cuda")
        ctx.set_map(0, z)
        ctx.step(2, dt)
        assert torch.equal(ctx.get_map(0), z)
        ctx.close()
        ctx = H.Context(nt, nphi, w.params, dtype=dtype, adv_flux=H.ADV_OFF)
        cst = torch.full((nt, nphi), 3.25, dtype=ctx.tdtype, device="cuda")
        ctx.set_map(0, cst)
        ctx.step(2, dt)
        assert (ctx.get_full(0) - 3.25).abs().max().item() <= (1e-13 if dtype == "f64" else 1e-5)
        ctx.close()
    with pytest.raises(H.HftError):
        H.Context(7, 8, [[0.0] * 7])


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("nt,nphi,opt", [(37, 256, {}), (37, 250, {}), (21, 131, {}), (40, 512, {"sts_block": 1}),
                                          (37, 256, {"flow_attenuation": 1}), (37, 256, {"rfe": 1}), (24, 128, {"diffusivity_map": 1}),
                                          (1024, 2048, {"n_real": 64})])
def test_no_write_outside_caller_buffers(dtype, nt, nphi, opt):
    """Every buffer is caller-owned (include/hft.h).  The workspace and the output of hft_get_map sit inside poisoned
    allocations; after the whole path has run (set_map, advection + blocked / stage-by-stage STS with a remainder block,
    both assimilation variants, both diagnostics, get_map) every guard byte on either side is untouched.  (compute-sanitizer
    is not available on the GPU boxes; this is the bounds check that is.)"""
    H = hft()
    opt = dict(opt)
    w = wl.scaled(wl.config(3), nt, nphi, n_real=opt.pop("n_real", 3))      # the last case is cfg 3 itself, as bench.py launches it
    tdt = torch.float64 if dtype == "f64" else torch.float32
    o = H.hft_options(H.ADV_WENO3, H.TIME_SSPRK43, H.DIFF_RKG2, 0, opt.get("sts_block", 0), opt.get("rfe", 0), 0,
                      opt.get("flow_attenuation", 0), opt.get("diffusivity_map", 0))
    need = H.workspace_bytes(nt, nphi, w.n_real, dtype, o)
    G = 1 << 16
    big = torch.full((G + need + G,), 0xA5, dtype=torch.uint8, device="cuda")
    ctx = H.Context(nt, nphi, w.params, dtype=dtype, radius_cm=6.96e10, workspace=big[G:G + need], **opt)
    if opt.get("flow_attenuation"):
        ctx.set_attenuation(-1, 300.0)
    if opt.get("diffusivity_map"):
        th = (np.arange(nt + 1)[:, None] + 0.5) * math.pi / (nt + 1)
        ph = (np.arange(nphi)[None, :] + 0.5) * 2 * math.pi / nphi
        ctx.set_diffusivity_map(1, 400.0 * (1 + 0.3 * np.sin(th) * np.cos(ph)))
    rng = torch.Generator(device="cuda").manual_seed(5)
    maps = 50.0 * torch.randn((w.n_real, nt, nphi), generator=rng, device="cuda", dtype=tdt)
    for r in range(w.n_real):
        ctx.set_map(r, maps[r].contiguous())
    if opt.get("rfe"):
        ctx.set_rfe(1, 100e21, 0.3, 7)
    dt, _, _ = wl.plan(w, *ctx.stable_dt())
    for dt_k in (dt, 0.37 * dt):                      # two stage counts: different remainders of the K = 8 blocks
        ctx.step(1 if nt >= 1024 else 2, dt_k)
    obs = (maps + torch.randn(maps.shape, generator=rng, device="cuda", dtype=tdt)).contiguous()
    wts = torch.rand(maps.shape, generator=rng, device="cuda", dtype=tdt).contiguous()
    ctx.assimilate(obs, wts, 0)
    ctx.assimilate(obs, wts, 1)
    ctx.step(1, dt)
    ctx.diagnostics()
    ctx.diagnostics_ext(60.0)
    cells = w.n_real * nt * nphi
    outbig = torch.full((G + cells * maps.element_size() + G,), 0x5A, dtype=torch.uint8, device="cuda")
    out = outbig[G:G + cells * maps.element_size()].view(tdt).view(w.n_real, nt, nphi)
    ctx.get_map(-1, out)
    torch.cuda.synchronize()
    assert torch.isfinite(out).all()
    assert bool((big[:G] == 0xA5).all()) and bool((big[G + need:] == 0xA5).all()), "write outside the workspace"
    assert bool((outbig[:G] == 0x5A).all()) and bool((outbig[-G:] == 0x5A).all()), "write outside the get_map buffer"
    ctx.close()


def test_fma_rate_probe():
    """hft_probe_fma_rate (the denominator of bench.py's "alu" roofline): sane on a B200 -- fp64 near 64 lanes per clock and SM,
    fp32 near 128, and three register operands per DFMA slower than a shared or constant operand."""
    H = hft()
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    r64 = [H.probe_fma_rate("f64", p) for p in (0, 1, 2)]
    r32 = [H.probe_fma_rate("f32", p) for p in (0, 1, 2)]
    per_clk = lambda r: r / sms / 1.965e9                        # lanes per clock and SM at the maximum SM clock
    assert 40 < per_clk(r64[0]) < 70 and 40 < per_clk(r64[2]) < 70, r64
    assert 80 < per_clk(r32[0]) < 140, r32
    assert r64[1] < 0.9 * r64[2], r64
    with pytest.raises(Exception):
        H.probe_fma_rate("f64", 3)


def test_interleaved_contexts_share_the_constant_table():
    """k_sts_upipe (the default for fp64 states and for fp32 states with fp64 block arithmetic) reads its coefficient table
    from the constant bank, which is process-wide state per device: contexts take turns, the library tracks the owner and
    re-uploads on a change.  Three contexts -- two fp64 grids of different size and one fp32 -- stepped in turn, one step
    at a time, must each end where their oracle does."""
    H = hft()
    cases = [("f64", wl.scaled(wl.config(3), 90, 200, n_real=2)), ("f64", wl.scaled(wl.config(2), 61, 136, n_real=3)),
             ("f32", wl.scaled(wl.config(3), 75, 264, n_real=2))]
    pairs, dts = [], []
    for dtype, w in cases:
        ctx, o = make_pair(w, dtype, adv_flux=H.ADV_OFF)
        _, dif = o.stable_dt()
        dt = 120.0 * dif
        assert ctx.sts_stage_count(dt) > 10                      # blocked path
        pairs.append((dtype, ctx, o)); dts.append(dt)
    for step in range(3):
        for (dtype, ctx, o), dt in zip(pairs, dts):
            ctx.step(1, dt)
    for (dtype, ctx, o), dt in zip(pairs, dts):
        o.step(3, dt, adv_flux=orc.ADV_OFF)
        compare(ctx, o, TOL[dtype], "interleaved contexts")
        ctx.close()
