#!/usr/bin/env python
"""bench.py -- throughput of the HipFT time-stepping hot path on B200 (contract: see DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3] [--dtype f64|f32]

A "step" is one pass of the whole hot path -- hft_step(1, dt): SSPRK(4,3) WENO3 advection + s RKG2 super-time-step
stages + polar caps -- over all realizations of the workload.  metric = cell-updates/s =
realizations x n_theta x n_phi x steps / seconds (BASELINE.json), inputs resident in HBM; `e2e` is the same
metric through the C ABI with HOST buffers (pinned H2D of the maps and D2H of the result inside the timed
region).  Multi-GPU (torchrun): realizations are independent, every rank advances its own
ensemble shard with no data-path collective ("scaling": "weak"); time = max over ranks.
"""
import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

import numpy as np
import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2501_06377_b200 import ensemble as ens  # noqa: E402
from paper_2501_06377_b200 import workloads as wl  # noqa: E402


# FMA-class lane-operations per second measured on this pool's B200 with a register-only loop
# (profiles/r01_pipe_cfg3_gen2.md): 64 DFMA lanes per clock per SM; fp32: 128 lanes per clock per SM (FFMA2 or dual issue)
ALU_PEAK_FMA_PER_S = {"f64": 1.70e13, "f32": 3.53e13}


def kernel_source_hash():
    """sha1 over the blocked-STS kernel sources: ties a stored ncu traffic figure to the code it was measured on."""
    import hashlib
    h = hashlib.sha1()
    d = os.path.join(ROOT, "paper_2501_06377_b200", "csrc")
    for f in ("hft_sts_blocked.cuh", "hft_sts_pipe.cuh", "hft_sts_upipe.cuh", "hft_sts_mpipe.cuh"):
        with open(os.path.join(d, f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:12]


def record_traffic(csv_path, profile, config):
    """bench.py --record-traffic raw.csv --traffic-profile profiles/x.md: read an `ncu -i x.ncu-rep --page raw --csv` export
    and store the mean dram__bytes_read.sum + dram__bytes_write.sum per launch of every blocked STS kernel in
    profiles/traffic.json, stamped with the commit and the hash of the kernel sources.  No GPU needed."""
    import csv
    import re
    rows = list(csv.reader(open(csv_path)))
    hdr, units, data = rows[0], rows[1], rows[2:]
    ix = {h: i for i, h in enumerate(hdr)}
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
    acc = {}
    for r in data:
        m = re.search(r"(k_sts_[um]?pipe)<(double|float), (?:(double|float), )?(?:\(int\))?(\d+)", r[ix["Kernel Name"]])
        if not m:
            continue
        name = "%s<%s,%s>" % (m.group(1), ",".join(x for x in (m.group(2), m.group(3)) if x), m.group(4))
        tot = sum(float(r[ix[c]]) * scale[units[ix[c]]] for c in ("dram__bytes_read.sum", "dram__bytes_write.sum"))
        acc.setdefault(name, []).append(tot)
    try:
        head = subprocess.run(["git", "rev-parse", "--short", "HEAD"], cwd=ROOT, capture_output=True, text=True).stdout.strip()
    except OSError:
        head = ""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    doc = json.load(open(p)) if os.path.exists(p) else {"kernels": []}
    for name, v in acc.items():
        doc["kernels"] = [e for e in doc["kernels"] if not (e["kernel"] == name and e["config"] == config)]
        doc["kernels"].append({"kernel": name, "config": config, "dram_bytes_per_launch": sum(v) / len(v), "launches": len(v),
                               "git_head": head, "source_sha1": kernel_source_hash(), "profile": profile})
    json.dump(doc, open(p, "w"), indent=1)
    print(json.dumps(doc["kernels"], indent=1))


def ncu_traffic(kernel, config):
    """Per-launch DRAM bytes of `kernel` from profiles/traffic.json (written next to each ncu --set full summary), or None."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    if not os.path.exists(p):
        return None
    for e in json.load(open(p)).get("kernels", []):
        if e["kernel"] == kernel and e["config"] == config:
            return e
    return None


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json, torch copy)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap,power.draw,power.limit")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(self.index)], stdout=subprocess.PIPE, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        self.th.join(timeout=2)
        sm = [float(r[0]) for r in self.rows if len(r) >= 6 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 6 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) >= 6 and r[2 + i].lower().startswith("active") for r in self.rows)]
        def col(i):
            out = []
            for r in self.rows:
                try:
                    out.append(float(r[i]))
                except (IndexError, ValueError):
                    pass
            return out
        pw, pl = col(6), col(7)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm),
                # board power during the timed region: the blocked kernels run AT the power limit (sw_power_cap), see DESIGN.md 6
                "power_w": float(np.median(pw)) if pw else None, "power_limit_w": max(pl) if pl else None}


def oracle_sample(w, dtype, n_steps, dt, s):
    """The CPU oracle, as it stands, on ONE realization of the workload for n_steps steps."""
    from oracle import sft_oracle as orc
    npdt = np.float64 if dtype == "f64" else np.float32
    o = orc.Oracle(w.n_theta, w.n_phi, w.params[:1], dtype=npdt)
    m = wl.bipolar_map(w.n_theta, w.n_phi, w.n_pairs, w.map_seed + 1000, background_g=w.background_g)
    o.set_map(0, m.numpy().astype(npdt))
    if dt is None:
        dt, _, _ = wl.plan(w, *o.stable_dt())
        s = 0
    t0 = time.perf_counter()
    o.step(n_steps, dt, sts_stages=s)
    el = time.perf_counter() - t0
    return w.n_theta * w.n_phi * n_steps / el, el, orc.threads()


def run_reference(args, w):
    """--impl reference: the oracle timed on the host cores; each step = one realization, one time step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import sft_oracle as orc
    npdt = np.float64 if args.dtype == "f64" else np.float32
    o = orc.Oracle(w.n_theta, w.n_phi, w.params, dtype=npdt)      # all realizations -> the ensemble's dt and s
    dt, _, _ = wl.plan(w, *o.stable_dt())
    s = o.sts_stage_count(dt)
    o.close()
    steps, warm = max(1, args.steps), max(0, min(args.warmup, 1))
    if warm:
        oracle_sample(w, args.dtype, 1, dt, s)
    rate, el, thr = oracle_sample(w, args.dtype, steps, dt, s)
    sample = f"1 of {w.n_real} realizations x {steps} step(s) of the full grid, s={s} stages/step"
    print(json.dumps({
        "impl": "reference", "metric": "cell-updates/s", "value": rate, "unit": "cell-updates/s", "n_gpus": args.gpus,
        "steps": steps, "warmup": warm, "ms_per_step": 1e3 * el / steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": args.dtype, "data": "synthetic",
        "config": {"workload": w.name, "grid": [w.n_theta, w.n_phi], "realizations_timed": 1, "dt_hours": dt, "sts_stages": s},
        "cpu_baseline": {"value": rate, "unit": "cell-updates/s", "cores": thr, "kind": "oracle", "sample": sample},
        "e2e": {"value": rate, "unit": "cell-updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def run_paper_case(args):
    """The two validation runs the paper prints wall times for (RTX 3090 Ti), on this GPU:
    `diffusion`: Eq. 19 field, nu = 500 km^2/s, 512x1024 file grid, ONE 672 h step of RKG2(3/2) (0.55 s, HH 6.3e-5);
    `advdiff`:   the same field with rigid rotation v_phi = 1.80766 km/s sin(theta), WENO3 + SSPRK(4,3) + RKG2, dt = 0.62 h
                 over 672 h (Table 1 :337-344: 21.1 s, HH 4.8e-5).
    Context lines, not the bench metric: another machine's numbers, the paper's grid (510 x 1023 regular cells, odd n_phi)."""
    from paper_2501_06377_b200 import hft
    torch.cuda.set_device(0)
    nt, nphi = (510, 1023) if not args.paper_grid_even else (510, 1024)
    u = wl.soccer_ball_full(nt, nphi)
    rot = 1.80766e3 if args.paper_case == "advdiff" else 0.0
    ctx = hft.Context(nt, nphi, [[500.0, rot, 0, 0, 0, 0, 0]], dtype=args.dtype,
                      adv_flux=hft.ADV_WENO3 if rot else hft.ADV_OFF, sts_block=args.sts_block, sts_kernel=args.sts_kernel)
    ut = torch.from_numpy(u).to(ctx.tdtype).cuda().contiguous()
    n = round(672.0 / 0.62) if rot else 1
    dt = 672.0 / n
    s = ctx.sts_stage_count(dt)
    times = []
    for rep in range(1 + max(1, args.steps)):          # first repetition = warm-up
        ctx.set_full(0, ut)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        l0 = ctx.launch_count()
        e0.record()
        ctx.step(n, dt)
        e1.record()
        torch.cuda.synchronize()
        times.append(e0.elapsed_time(e1) * 1e-3)
        launches = ctx.launch_count() - l0
    got = ctx.get_full(0).double().cpu().numpy()
    exact = u * math.exp(-42.0 * 500.0 * 7.43162901307967e-9 * 672.0)      # l(l+1) = 42, nu in R_sun^2/hr
    hh = math.sqrt(((got[1:-1] - exact[1:-1]) ** 2).sum() / (np.abs(got[1:-1]) * np.abs(exact[1:-1])).sum())   # Eq. 18 (:246)
    ctx.close()
    paper = {"diffusion": {"seconds": 0.55, "hh": 6.3e-5, "hardware": "RTX 3090 Ti", "cite": "PAPER.md:476"},
             "advdiff": {"seconds": 21.1, "hh": 4.8e-5, "hardware": "RTX 3090 Ti", "cite": "PAPER.md:337-344 (Table 1)"}}[args.paper_case]
    print(json.dumps({"paper_case": args.paper_case, "metric": "seconds per run", "value": min(times[1:]), "unit": "s",
                      "higher_is_better": False, "dtype": args.dtype, "grid": [nt, nphi], "steps_per_run": n, "dt_hours": dt,
                      "sts_stages": s, "gpu_launches": launches, "hh_error_vs_analytic": hh, "runs_timed": len(times) - 1,
                      "paper": paper, "note": "context only: the paper's number is another machine's"}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=4)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"])
    ap.add_argument("--sts-block", type=int, default=0)
    ap.add_argument("--sts-kernel", type=int, default=0, help="hft_options.sts_kernel: 0 library default, 1 k_sts_pipe, 2 k_sts_upipe")
    ap.add_argument("--f32-fast", action="store_true", help="hft_options.f32_arith = 1: fp32 arithmetic throughout (default: fp64 block arithmetic)")
    ap.add_argument("--attenuation", type=float, default=0.0, help="B0 in Gauss: time the step with flow attenuation (Eq. 5) on")
    ap.add_argument("--nu-map", action="store_true",
                    help="time the step with a spatially varying diffusivity nu(theta, phi) (Eq. 27-28): one launch per STS stage")
    ap.add_argument("--paper-case", choices=["diffusion", "advdiff"], default=None,
                    help="time one of the two validation runs the paper prints wall times for (context, not the bench metric)")
    ap.add_argument("--paper-grid-even", action="store_true", help="--paper-case on 510 x 1024 instead of the paper's 510 x 1023")
    ap.add_argument("--alu-probe", action="store_true", help="print the FMA issue rates hft_probe_fma_rate measures on this GPU and exit")
    ap.add_argument("--record-traffic", default=None, metavar="RAW_CSV", help="no GPU: store the per-launch DRAM bytes of an ncu raw-page export in profiles/traffic.json")
    ap.add_argument("--traffic-profile", default="", help="with --record-traffic: the profiles/*.md summary the capture belongs to")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--also-f32", action="store_true", help="add a second timed run in fp32 to the JSON line (default in the full report)")
    ap.add_argument("--no-also-f32", action="store_true", help="full report without the fp32 leg")
    args = ap.parse_args()
    if args.record_traffic:
        record_traffic(args.record_traffic, args.traffic_profile, args.config)
        return
    if args.alu_probe:
        # the denominators of the "alu" roofline, re-measured: FMA lane-operations per second per operand pattern (hft.h)
        from paper_2501_06377_b200 import hft
        torch.cuda.set_device(0)
        names = {0: "two_shared_operands", 1: "three_register_operands", 2: "constant_bank_operand"}
        out = {"alu_probe_fma_per_s": {dt: {names[p]: hft.probe_fma_rate(dt, p) for p in (0, 1, 2)} for dt in ("f64", "f32")},
               "used_as_peak": ALU_PEAK_FMA_PER_S}
        print(json.dumps(out))
        return
    if args.paper_case:
        run_paper_case(args)
        return
    w = wl.config(args.config, args.dtype)
    args.warmup = max(args.warmup, 3)            # timing rule: at least 3 untimed warm-up steps; the JSON line reports the count run
    if args.impl == "reference":
        run_reference(args, w)
        return

    from paper_2501_06377_b200 import hft
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1 or "TORCHELASTIC_RUN_ID" in os.environ:     # under torchrun, also with one rank: same code path at every N
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def timed_run(dtype, with_extras, f32_arith=None):
        # rank k owns realizations [k R, (k+1) R) of the weak-scaled ensemble; one clock for the whole ensemble
        wd = ens.shard(args.config, dtype, rank, world)
        def make_ctx(**kw):
            c = hft.Context(wd.n_theta, wd.n_phi, wd.params, dtype=dtype, sts_block=args.sts_block, sts_kernel=args.sts_kernel,
                            f32_arith=int(args.f32_fast if f32_arith is None else f32_arith), flow_attenuation=int(args.attenuation > 0), diffusivity_map=int(args.nu_map), device=f"cuda:{local}", **kw)
            if args.attenuation > 0:
                c.set_attenuation(-1, args.attenuation)
            if args.nu_map:      # nu_r (1 + 0.3 sin(theta) cos(phi)) on the half-half grid, per realization (workloads.diffusivity_map)
                for r in range(wd.n_real):
                    c.set_diffusivity_map(r, wl.diffusivity_map(wd, r))
            return c
        ctx = make_ctx()
        maps = ens.shard_maps(wd, device=f"cuda:{local}").to(ctx.tdtype).contiguous()
        ctx.set_map(-1, maps[0]) if not wd.per_real_maps else [ctx.set_map(r, maps[r]) for r in range(wd.n_real)]
        dt, n_cfg, per = wl.plan(wd, *ens.global_limits(*ctx.stable_dt()))
        s = int(ens.max_over_ranks(float(ctx.sts_stage_count(dt))))
        if s != ctx.sts_stage_count(dt):          # another rank's realizations need more stages: force the same s
            ctx.close()
            ctx = make_ctx(sts_stages=s)
            ctx.set_map(-1, maps[0]) if not wd.per_real_maps else [ctx.set_map(r, maps[r]) for r in range(wd.n_real)]
        cells = wd.n_real * wd.n_theta * wd.n_phi
        for _ in range(args.warmup):
            ctx.step(1, dt)
        barrier()
        sampler = ClockSampler(local)
        if rank == 0 and with_extras:
            sampler.start()
        ctx.profile_kernels(1)
        l0 = ctx.launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.steps):
            ctx.step(1, dt)
        e1.record()
        barrier()
        ms = e0.elapsed_time(e1)
        launches = ctx.launch_count() - l0
        kms, kn, kst = ctx.kernel_time()
        ctx.profile_kernels(0)
        clocks = sampler.stop() if (rank == 0 and with_extras) else None
        ms = ens.max_over_ranks(ms)
        res = dict(ms=ms, value=world * cells * args.steps / (ms * 1e-3), launches=launches, dt=dt, s=s, cells=cells, dtype=dtype,
                   f32_arith=int(args.f32_fast if f32_arith is None else f32_arith),
                   kernel_ms=(kms / kn if kn else None), kernel_samples=kn, kernel_stages=(kst / kn if kn else None), clocks=clocks, wd=wd)
        # ---- end-to-end through the C ABI with host buffers
        if with_extras and not args.no_e2e:
            host_in = maps.cpu().pin_memory()
            host_out = torch.empty_like(host_in).pin_memory()
            dev_in = [torch.empty_like(maps), torch.empty_like(maps)]
            dev_out = [torch.empty_like(maps), torch.empty_like(maps)]
            n_e2e = max(1, args.steps)
            # three streams, as a user of the C ABI would drive it: step i+1's maps come up and step i-1's result goes
            # down while step i computes (PCIe is full duplex); every copy, the first host-to-device and the last
            # device-to-host included, is inside the timed region
            main, up, side = torch.cuda.current_stream(), torch.cuda.Stream(), torch.cuda.Stream()
            barrier()
            t0 = torch.cuda.Event(enable_timing=True); t1 = torch.cuda.Event(enable_timing=True)
            t0.record()
            up.wait_stream(main)

            consumed, copied = [None, None], [None, None]

            def upload(i):
                with torch.cuda.stream(up):
                    if consumed[i % 2] is not None:
                        up.wait_event(consumed[i % 2])      # set_map of step i-2 has read this buffer
                    dev_in[i % 2].copy_(host_in, non_blocking=True)
                    ev = torch.cuda.Event()
                    ev.record(up)
                return ev

            arrived = upload(0)
            for i in range(n_e2e):
                main.wait_event(arrived)
                for r in range(wd.n_real):
                    ctx.set_map(r, dev_in[i % 2][r])
                consumed[i % 2] = torch.cuda.Event()
                consumed[i % 2].record(main)
                if i + 1 < n_e2e:
                    arrived = upload(i + 1)          # into the other input buffer
                ctx.step(1, dt)
                if copied[i % 2] is not None:
                    main.wait_event(copied[i % 2])    # the result of step i-2 has left this buffer
                ctx.get_map(-1, out=dev_out[i % 2])
                done = torch.cuda.Event()
                done.record(main)
                with torch.cuda.stream(side):
                    side.wait_event(done)
                    host_out.copy_(dev_out[i % 2], non_blocking=True)
                    copied[i % 2] = torch.cuda.Event()
                    copied[i % 2].record(side)
            main.wait_stream(side)
            t1.record()
            barrier()
            ems = t0.elapsed_time(t1)
            ems = ens.max_over_ranks(ems)
            res["e2e"] = {"value": world * cells * n_e2e / (ems * 1e-3), "unit": "cell-updates/s",
                          "h2d_bytes_per_step": host_in.numel() * host_in.element_size(),
                          "d2h_bytes_per_step": host_out.numel() * host_out.element_size(), "steps": n_e2e}
            assert torch.isfinite(host_out).all()
        ctx.close()
        return res

    res = timed_run(args.dtype, True)
    wd = res["wd"]
    wbytes = 8 if args.dtype == "f64" else 4
    peak, peak_src = peaks()
    # algorithmic bytes: 4 array passes per STS stage, 9 per SSPRK(4,3) advection step
    # (with nu(theta, phi) a stage also reads the nu array once: 5 passes)
    stage_passes = 5 if args.nu_map else 4

    def b_alg(r, w):
        return (9 + stage_passes * r["s"]) * w

    def traffic_keys(kern):
        """Per-launch DRAM bytes of the last committed ncu --set full capture of `kern` (profiles/traffic.json), or traffic = None."""
        t = ncu_traffic(kern, args.config)
        if not t:
            return {"traffic": None}
        return {"traffic": t["dram_bytes_per_launch"], "traffic_source": t["profile"], "traffic_head": t["git_head"],
                "traffic_stale": t["source_sha1"] != kernel_source_hash()}   # true: the kernel sources changed since that capture

    def roofline_of(r):
        """The dominant kernel's distance from its roofs, from the CUDA-event samples of this run."""
        if not r["kernel_ms"]:
            return None
        dtype, w = r["dtype"], (8 if r["dtype"] == "f64" else 4)
        spl = r["kernel_stages"]                        # STS stages per sampled launch
        cells_launch = wd.n_real * (wd.n_theta + 2) * wd.n_phi
        field_bytes = cells_launch * w
        sec = r["kernel_ms"] * 1e-3
        alg_gbs = stage_passes * field_bytes * spl / sec / 1e9      # 4 passes per stage, as a stage-by-stage code moves
        if spl <= 1:
            kern = "k_sts_stage_mapv<MAP=true>" if args.nu_map else "k_sts_stage_mapv<MAP=false>"
            return {"bound": "hbm", "achieved": alg_gbs, "peak": peak, "unit": "GB/s", "frac": alg_gbs / peak, "traffic": None,
                    "kernel": kern, "stages_per_launch": spl, "avg_launch_ms": r["kernel_ms"], "sampled_launches": r["kernel_samples"],
                    "peak_source": peak_src}
        # K stages per launch: the kernel moves 5 array passes per K stages, not 4 K, so it is NOT bound by HBM; what it
        # saturates first is the FP pipe of its arithmetic type (fp64: DFMA 64 lanes/clk/SM; ncu: the pipe is the busiest
        # unit, then the issue slots).  "alu": useful FP instruction slots per second -- 7 per cell and stage (1 add, 1 mul,
        # 5 fma; halo recomputation and k_sts_upipe's 8th operation are NOT counted as useful) -- against the measured FMA
        # issue rate of that type, both in FMA-equivalent TFLOP/s (2 flops per slot).
        if args.nu_map:     # k_sts_mpipe: 4 stages per launch, 14 FP operations per cell and stage (10 for Eq. 27 with the face
            # conductances, 4 for the recurrence), 6 array passes per launch (3 fields + nu in, 2 out), 4 halo columns per side
            cols = 32 * (2 if dtype == "f64" else 4)
            useful = 14 * spl * cells_launch / sec
            alu_peak = ALU_PEAK_FMA_PER_S[dtype]
            return {"bound": "alu", "achieved": 2 * useful / 1e12, "peak": 2 * alu_peak / 1e12, "unit": "TFLOP/s", "frac": useful / alu_peak,
                    "kernel": "k_sts_mpipe<%s,4>" % ("double" if dtype == "f64" else "float"), "stages_per_launch": spl,
                    "avg_launch_ms": r["kernel_ms"], "sampled_launches": r["kernel_samples"],
                    "frac_with_halo": useful * cols / (cols - 8) / alu_peak, **traffic_keys("k_sts_mpipe<%s,4>" % ("double" if dtype == "f64" else "float")),
                    "hbm_algorithmic": {"achieved": alg_gbs, "peak": peak, "unit": "GB/s", "frac": alg_gbs / peak, "peak_source": peak_src,
                                        "meaning": "speed-up over the HBM roofline of one launch per stage (5 passes per stage with nu(theta, phi))"},
                    "dram": {"achieved": 6 * field_bytes / sec / 1e9, "peak": peak, "unit": "GB/s", "frac": 6 * field_bytes / sec / 1e9 / peak,
                             "meaning": "the 6 array passes per launch this kernel moves (3 fields + nu in, 2 out) / time"}}
        mixed = dtype == "f32" and r["f32_arith"] == 0
        upipe = mixed or args.sts_kernel == 2 or (dtype == "f64" and args.sts_kernel == 0)   # the library's choice (hft.h: sts_kernel)
        arith = "f64" if (dtype == "f64" or mixed) else "f32"
        kern = ("k_sts_upipe<%s,%s,8>" % ("float" if dtype == "f32" else "double", "double" if arith == "f64" else "float")) if upipe \
            else "k_sts_pipe<%s,8>" % ("double" if dtype == "f64" else "float")
        alu_peak = ALU_PEAK_FMA_PER_S[arith]
        useful = 7 * spl * cells_launch / sec
        cols = 32 * (2 if arith == "f64" else 4)        # columns per warp strip; 8 invalid columns per side
        executed = (8 if upipe else 7) * spl * cells_launch * cols / (cols - 16) / sec
        out = {"bound": "alu", "achieved": 2 * useful / 1e12, "peak": 2 * alu_peak / 1e12, "unit": "TFLOP/s", "frac": useful / alu_peak,
               "traffic": None, "kernel": kern, "stages_per_launch": spl, "avg_launch_ms": r["kernel_ms"],
               "sampled_launches": r["kernel_samples"],
               "peak_source": "FP%s FMA issue rate: 64 (fp64) / 128 (fp32) lanes per clock and SM x 148 SMs x the clock under the power "
                              "cap, as measured with the library's register-only loop (hft_probe_fma_rate; bench.py --alu-probe), x 2 flops" % arith[1:],
               "frac_with_halo_and_extra_ops": executed / alu_peak,
               # context, not distances to a roof of this kernel: the rate expressed in the bytes a stage-by-stage code would
               # move (SURVEY 8(d) B_alg) over the measured copy bandwidth -- how much faster than ANY such code could be
               "hbm_algorithmic": {"achieved": alg_gbs, "peak": peak, "unit": "GB/s", "frac": alg_gbs / peak, "peak_source": peak_src,
                                   "meaning": "speed-up over the HBM roofline of one launch per stage (4 passes per stage); > 1 because 8 stages stay on chip"},
               "dram": {"achieved": 5 * field_bytes / sec / 1e9, "peak": peak, "unit": "GB/s", "frac": 5 * field_bytes / sec / 1e9 / peak,
                        "meaning": "the 5 array passes per launch this kernel actually moves (3 in, 2 out) / time"}}
        if spl > 7:
            out.update(traffic_keys(kern))
        return out

    frac_step = res["value"] / world * b_alg(res, wbytes) / (peak * 1e9)
    out = {
        "metric": "cell-updates/s", "value": res["value"], "unit": "cell-updates/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": res["ms"] / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": args.dtype, "data": "synthetic",
        "config": {"workload": wd.name, "grid": [wd.n_theta, wd.n_phi], "realizations_per_gpu": wd.n_real,
                   "dt_hours": res["dt"], "sts_stages": res["s"], "adv": "WENO3-CS(h)+SSPRK(4,3)", "diff": "RKG2(3/2)",
                   "l2": "inputs larger than L2 (arrays of %.0f MiB each)" % (wd.n_real * (wd.n_theta + 2) * wd.n_phi * wbytes / 2**20),
                   "sts_block": args.sts_block, "sts_kernel": args.sts_kernel, "f32_arith": res["f32_arith"] if args.dtype == "f32" else None,
                   "flow_attenuation_b0": args.attenuation, "nu_map": bool(args.nu_map),
                   "b_alg_bytes_per_cell_update": b_alg(res, wbytes), "hbm_roofline_frac_whole_step": frac_step},
        "gpu_launches": res["launches"],
        "clocks": res["clocks"],
    }
    if res.get("e2e"):
        out["e2e"] = res["e2e"]
    rf = roofline_of(res)
    if rf:
        out["roofline"] = rf
    # BASELINE.json's metric is quoted "(fp64, fp32)": the full report (no --no-e2e / --no-cpu-baseline, i.e. not a profiling
    # run) carries the fp32 record of the same workload beside the fp64 line -- the default fp32 path (fp64 block arithmetic,
    # meets north_star's 1e-5) with its own clocks, roofline and end-to-end figure, and the fp32-arithmetic path (f32_arith = 1)
    full_report = not (args.no_e2e or args.no_cpu_baseline or args.no_also_f32)
    if (args.also_f32 or full_report) and args.dtype == "f64":
        def f32_record(r, parity):
            d = {"value": r["value"], "ms_per_step": r["ms"] / args.steps, "sts_stages": r["s"], "f32_arith": r["f32_arith"],
                 "gpu_launches": r["launches"], "parity_cfg3_full_length_vs_fp64_oracle": parity,
                 "hbm_roofline_frac_whole_step": r["value"] / world * b_alg(r, 4) / (peak * 1e9)}
            if r.get("clocks"):
                d["clocks"] = r["clocks"]
            if r.get("e2e"):
                d["e2e"] = r["e2e"]
            rr = roofline_of(r)
            if rr:
                d["roofline"] = rr
            return d
        r32 = timed_run("f32", True, 0)
        out["also_f32"] = f32_record(r32, "2.0e-6 .. 2.7e-6 (north_star 1e-5 met; tests/test_gpu_parity.py)")
        r32f = timed_run("f32", False, 1)
        out["also_f32"]["fp32_arithmetic"] = f32_record(r32f, "1.4e-5 .. 2.2e-5 (north_star 1e-5 NOT met)")
    if rank == 0:
        if not args.no_cpu_baseline:
            # ~10-30 s of oracle work on the box's host cores (the float build of the oracle runs ~12x slower per step than
            # the double build on this workload -- subnormal operands, no flush-to-zero -- so its sample is shorter)
            n_or = (24 if args.dtype == "f64" else 3) if wd.n_theta >= 1024 else 200
            rate, el, thr = oracle_sample(wd, args.dtype, n_or, res["dt"], res["s"])
            out["cpu_baseline"] = {"value": rate, "unit": "cell-updates/s", "cores": thr, "kind": "oracle",
                                   "sample": f"1 of {wd.n_real} realizations x {n_or} steps of the full grid ({el:.1f} s)"}
        print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
