"""Seeded synthetic inputs for the five BASELINE.json configurations.

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the method's
arithmetic: it only draws parameters, builds initial / observed maps and assimilation weights, and
states each configuration's stepping recipe (CFL number, simulated time).  Time-step limits are an
input here (each side computes them with its own helper and passes them to `plan`).

The paper's workloads are HMI Carrington maps and MagMAP assimilation sequences,
which are not available offline; the maps below take their shape (theta x phi maps in Gauss, bipolar
active regions over a weak background) and stand in for them.  Recipe: DESIGN.md
"Input recipe".

User-facing maps are dense [n_theta][n_phi]: row i (0-based) is at colatitude (i+1)*pi/(n_theta+1),
column k at longitude 2*pi*k/n_phi.
"""
import math
from dataclasses import dataclass, field

import numpy as np
import torch

R_SUN_M = 6.96e8
DEG_PER_DAY_TO_M_S = math.pi / 180.0 / 86400.0 * R_SUN_M   # 140.596 m/s at the equator
CARRINGTON_DEG_PER_DAY = 13.2                      # BASELINE.json config 1
K_MERID = 16.0 / (3.0 * math.sqrt(3.0))            # -v0 sin(2 lat) cos^2(lat) normalised to peak v0


@dataclass
class Workload:
    name: str
    n_theta: int
    n_phi: int
    n_real: int
    dtype: str                      # "f64" or "f32"
    params: np.ndarray              # [n_real][7]: eta_km2_s, d0, d2, d4, m1, m3, m5 (Eq. 3, 4, 6)
    t_end_hours: float
    cfl: float = 0.5                # multiplies the Eq. 26 advective limit
    advect: bool = True
    sts_stages: int = 0             # 0 = auto
    dt_in_dt_expl: float = 0.0      # >0: dt = this many explicit diffusion limits (config 0)
    n_steps_fixed: int = 0
    assim_every_hours: float = 0.0
    n_pairs: int = 0
    map_seed: int = 0
    per_real_maps: bool = False
    background_g: float = 0.0
    extra: dict = field(default_factory=dict)


def flow_params(eta, v0, a_deg=14.71, b_deg=-2.40, c_deg=-1.79):
    """Map BASELINE config-1 flow description onto the paper's Eq. 3 / Eq. 4 parameters (m/s)."""
    d0 = (a_deg - CARRINGTON_DEG_PER_DAY) * DEG_PER_DAY_TO_M_S
    d2 = b_deg * DEG_PER_DAY_TO_M_S
    d4 = c_deg * DEG_PER_DAY_TO_M_S
    return [eta, d0, d2, d4, K_MERID * v0, -K_MERID * v0, 0.0]


def ensemble_params(idx: int, n_real: int) -> np.ndarray:
    """[n_real][7] parameters of the first n_real realizations of configuration idx's ensemble.  Realization r
    has the same parameters whatever n_real is (draws are consumed row by row), so an ensemble can be extended
    over more GPUs without changing the realizations already there (ensemble.shard)."""
    if idx == 0:
        return np.tile(np.array([[500.0, 0, 0, 0, 0, 0, 0]]), (n_real, 1))
    if idx in (1, 4):
        return np.tile(np.array([flow_params(500.0, 15.0)]), (n_real, 1))
    if idx == 2:      # reading U16: eta = 250 + 50 r, v0 = 10 + (10/7) r, r = 0..7 (repeats beyond 8)
        return np.array([flow_params(250.0 + 50.0 * (r % 8), 10.0 + (10.0 / 7.0) * (r % 8)) for r in range(n_real)])
    if idx == 3:      # reading U16: eta, v0, (A - 13.2), B, C each x (1 + 0.2 u), u ~ U(-1, 1), seed 3
        rng = np.random.default_rng(3)
        u = rng.uniform(-1.0, 1.0, size=(n_real, 5))
        p = []
        for r in range(n_real):
            f = 1.0 + 0.2 * u[r]
            eta, v0 = 500.0 * f[0], 15.0 * f[1]
            a = CARRINGTON_DEG_PER_DAY + (14.71 - CARRINGTON_DEG_PER_DAY) * f[2]
            p.append(flow_params(eta, v0, a, -2.40 * f[3], -1.79 * f[4]))
        return np.array(p)
    raise ValueError(idx)


def config(idx: int, dtype: str = "f64") -> Workload:
    if idx == 0:
        return Workload("cfg0_64x128_r1_diffusion", 64, 128, 1, "f64", ensemble_params(0, 1),
                        t_end_hours=0.0, advect=False, sts_stages=8, dt_in_dt_expl=8.0, n_steps_fixed=200,
                        n_pairs=6, map_seed=0)
    if idx == 1:
        return Workload("cfg1_512x1024_r1", 512, 1024, 1, "f64", ensemble_params(1, 1),
                        t_end_hours=24.0, n_pairs=40, map_seed=1)
    if idx == 2:
        return Workload("cfg2_1024x2048_r8", 1024, 2048, 8, "f64", ensemble_params(2, 8), t_end_hours=24.0,
                        n_pairs=120, map_seed=2, background_g=2.0)
    if idx == 3:
        return Workload("cfg3_1024x2048_r64_" + dtype, 1024, 2048, 64, dtype, ensemble_params(3, 64),
                        t_end_hours=48.0, n_pairs=120, map_seed=3, per_real_maps=True)
    if idx == 4:
        return Workload("cfg4_2048x4096_r1_assim", 2048, 4096, 1, "f64", ensemble_params(4, 1),
                        t_end_hours=24.0, n_pairs=120, map_seed=4, assim_every_hours=1.0)
    raise ValueError(idx)


def scaled(w: Workload, n_theta: int, n_phi: int, n_real: int = None, t_end_hours: float = None) -> Workload:
    """Same recipe on a smaller grid / fewer realizations (parity-test sizes)."""
    import copy
    q = copy.deepcopy(w)
    q.n_theta, q.n_phi = n_theta, n_phi
    if n_real is not None:
        q.n_real = n_real
        q.params = q.params[:n_real].copy()
    if t_end_hours is not None:
        q.t_end_hours = t_end_hours
    q.name = f"{w.name}_scaled_{n_theta}x{n_phi}_r{q.n_real}"
    return q


def plan(w: Workload, dt_adv_limit: float, dt_diff_expl: float):
    """Step size and count from the caller-supplied limits: (dt_hours, n_steps, steps_per_assim)."""
    if w.dt_in_dt_expl > 0.0:
        return w.dt_in_dt_expl * dt_diff_expl, w.n_steps_fixed, 0
    span = w.assim_every_hours if w.assim_every_hours > 0.0 else w.t_end_hours
    dt = w.cfl * dt_adv_limit if w.advect and math.isfinite(dt_adv_limit) else span
    n = max(1, math.ceil(span / dt - 1e-12))
    dt = span / n
    if w.assim_every_hours > 0.0:
        return dt, n * int(round(w.t_end_hours / span)), n
    return dt, n, 0


def diffusivity_map(w: Workload, r: int):
    """Synthetic spatially varying diffusivity of realization r on the half-half grid [n_theta+1][n_phi], km^2/s
    (bench.py --nu-map and the full-size parity test): eta_r (1 + 0.3 sin(theta) cos(phi)) -- smooth, phi-dependent,
    positive; entry [f][k] at colatitude (f+1/2) dtheta, longitude (k+1/2) dphi.  numpy float64."""
    thf = ((np.arange(w.n_theta + 1) + 0.5) * math.pi / (w.n_theta + 1))[:, None]
    phf = ((np.arange(w.n_phi) + 0.5) * 2.0 * math.pi / w.n_phi)[None, :]
    return float(w.params[r][0]) * (1.0 + 0.3 * np.sin(thf) * np.cos(phf))


def soccer_ball_full(n_theta, n_phi):
    """The paper's validation field, Eq. 19: Y_6^0 + sqrt(14/11) Y_6^5 (real harmonics), scaled to
    max |.| = 1, on the internal grid incl. the two pole rows: numpy float64 [n_theta+2][n_phi].  An l = 6 eigenfunction
    of the surface Laplacian: under diffusion alone it decays as exp(-42 nu t)."""
    from scipy.special import sph_harm_y
    th = (np.arange(n_theta + 2) * math.pi / (n_theta + 1))[:, None]
    ph = (np.arange(n_phi) * 2.0 * math.pi / n_phi)[None, :]
    u = sph_harm_y(6, 0, th, ph).real + math.sqrt(14.0 / 11.0) * math.sqrt(2.0) * sph_harm_y(6, 5, th, ph).real
    return np.ascontiguousarray(u / np.abs(u).max())


def colatitudes(n_theta, device="cpu"):
    return torch.arange(1, n_theta + 1, dtype=torch.float64, device=device) * (math.pi / (n_theta + 1))


def longitudes(n_phi, device="cpu"):
    return torch.arange(n_phi, dtype=torch.float64, device=device) * (2.0 * math.pi / n_phi)


def bipolar_map(n_theta, n_phi, n_pairs, seed, amp=(1.0, 100.0), sigma_deg=3.0, lat_deg=40.0,
                background_g=0.0, noise_g=0.0, device="cpu"):
    """Sum of n_pairs bipolar Gaussian spot pairs (+A / -A, separated by 3 sigma in longitude)."""
    rng = np.random.default_rng(seed)
    A = rng.uniform(amp[0], amp[1], n_pairs)
    lat = np.deg2rad(rng.uniform(-lat_deg, lat_deg, n_pairs))
    lon = np.deg2rad(rng.uniform(0.0, 360.0, n_pairs))
    sig = math.radians(sigma_deg)
    th = colatitudes(n_theta, device)[:, None]
    ph = longitudes(n_phi, device)[None, :]
    sin_l, cos_l = torch.cos(th), torch.sin(th)          # latitude = pi/2 - colatitude
    out = torch.zeros((n_theta, n_phi), dtype=torch.float64, device=device)
    for a, lc, pc in zip(A, lat, lon):
        for sgn in (+1.0, -1.0):
            p0 = pc - sgn * 1.5 * sig
            cd = sin_l * math.sin(lc) + cos_l * math.cos(lc) * torch.cos(ph - p0)
            d = torch.acos(torch.clamp(cd, -1.0, 1.0))
            out += (sgn * a) * torch.exp(-(d * d) / (2.0 * sig * sig))
    if background_g > 0.0:
        out += torch.from_numpy(rng.uniform(-background_g, background_g, (n_theta, n_phi))).to(device)
    if noise_g > 0.0:
        out += torch.from_numpy(rng.normal(0.0, noise_g, (n_theta, n_phi))).to(device)
    return out


def initial_maps(w: Workload, device="cpu"):
    """[n_real][n_theta][n_phi] fp64 tensor (realizations share one map unless per_real_maps)."""
    if w.per_real_maps:
        return torch.stack([bipolar_map(w.n_theta, w.n_phi, w.n_pairs, w.map_seed + 1000 * (r + 1),
                                        background_g=w.background_g, device=device) for r in range(w.n_real)])
    m = bipolar_map(w.n_theta, w.n_phi, w.n_pairs, w.map_seed, background_g=w.background_g, device=device)
    return m[None].expand(w.n_real, -1, -1).contiguous()


def y21_map(n_theta, n_phi, device="cpu"):
    """Real spherical harmonic l=2, m=1 (unnormalised): sin(theta) cos(theta) cos(phi)."""
    th = colatitudes(n_theta, device)[:, None]
    ph = longitudes(n_phi, device)[None, :]
    return torch.sin(th) * torch.cos(th) * torch.cos(ph)


def emergence_map(w: Workload, n: int, device="cpu"):
    """Config 4: the n-th observed increment E_n (10 new pairs of 50-500 G + 1 G Gaussian noise)."""
    return bipolar_map(w.n_theta, w.n_phi, 10, 40000 + n, amp=(50.0, 500.0), noise_g=1.0, device=device)


def assimilation_weights(w: Workload, t_hours: float, device="cpu"):
    """Config 4: w = mu^4 inside a 60-degree disc around the sub-observer point (equator, longitude
    180 deg + 13.2 deg/day * t), 0 outside; mu = sin(theta) cos(phi - phi_obs)  (Eq. 9 with
    alpha_mu = 4, mu_lim = cos 60 deg, no latitude limit)."""
    th = colatitudes(w.n_theta, device)[:, None]
    ph = longitudes(w.n_phi, device)[None, :]
    phi_obs = math.radians(180.0 + CARRINGTON_DEG_PER_DAY * t_hours / 24.0)
    mu = torch.sin(th) * torch.cos(ph - phi_obs)
    return torch.where(mu > math.cos(math.radians(60.0)), mu ** 4, torch.zeros_like(mu))
