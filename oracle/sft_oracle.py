"""ctypes front-end of the CPU oracle (oracle/sft_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It never imports the CUDA package, and the CUDA package never imports it.
All the arithmetic lives in sft_oracle.c; this file only marshals numpy arrays.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

ADV_OFF, ADV_UPWIND, ADV_WENO3, ADV_WENO3_EPS12 = 0, 1, 2, 3
TIME_EULER, TIME_SSPRK33, TIME_SSPRK43 = 1, 3, 4
DIFF_OFF, DIFF_EULER, DIFF_RKL2, DIFF_RKG2, DIFF_RKL2_TEXTBOOK, DIFF_RKG2_TEXTBOOK = 0, 1, 2, 3, 12, 13

_libs = {}


def _lib(fp32: bool):
    if fp32 not in _libs:
        _build.build()
        _libs[fp32] = C.CDLL(_build.lib_path(fp32))
    return _libs[fp32]


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


class Oracle:
    """One oracle context: nr realizations on an nt x np grid (rows 1..nt; caps are internal)."""

    def __init__(self, n_theta, n_phi, params, dtype=np.float64, radius_cm=1.0):
        self.nt, self.np_, self.dtype = int(n_theta), int(n_phi), np.dtype(dtype)
        assert self.dtype in (np.dtype(np.float64), np.dtype(np.float32))
        self.fp32 = self.dtype == np.dtype(np.float32)
        self.suf = "_f32" if self.fp32 else "_f64"
        self.lib = _lib(self.fp32)
        p = np.ascontiguousarray(np.asarray(params, dtype=np.float64).reshape(-1, 7))
        self.nr = p.shape[0]
        f = self._f("sft_oracle_create")
        f.restype = C.c_void_p
        f.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(C.c_double), C.c_double]
        self.h = C.c_void_p(f(self.nt, self.np_, self.nr, _dp(p), float(radius_cm)))

    def _f(self, name):
        return getattr(self.lib, name + self.suf)

    def _rp(self, a):
        return a.ctypes.data_as(C.c_void_p)

    def close(self):
        if self.h:
            f = self._f("sft_oracle_destroy")
            f.restype = None
            f.argtypes = [C.c_void_p]
            f(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- tables -----------------------------------------------------------------------------
    def tables(self, r=0):
        st, sth = np.zeros(self.nt + 2), np.zeros(self.nt + 1)
        vt, om, sc = np.zeros(self.nt + 1), np.zeros(self.nt + 2), np.zeros(5)
        f = self._f("sft_oracle_get_tables")
        f.restype = None
        f.argtypes = [C.c_void_p, C.c_int] + [C.POINTER(C.c_double)] * 5
        f(self.h, r, _dp(st), _dp(sth), _dp(vt), _dp(om), _dp(sc))
        return dict(st=st, sth=sth, vt=vt, om=om, dth=sc[0], dph=sc[1], P=sc[2], Apole=sc[3], nu=sc[4])

    def set_flow_tables(self, r, vt, om):
        vt = np.ascontiguousarray(vt, dtype=np.float64)
        om = np.ascontiguousarray(om, dtype=np.float64)
        assert vt.shape == (self.nt + 1,) and om.shape == (self.nt + 2,)
        f = self._f("sft_oracle_set_flow_tables")
        f.restype = None
        f.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        f(self.h, r, _dp(vt), _dp(om))

    def set_theta_nodes(self, theta):
        """Non-uniform theta grid: theta[nt+2] = the B_r nodes, theta[0] = 0, theta[-1] = pi, increasing."""
        a = np.ascontiguousarray(theta, dtype=np.float64)
        assert a.shape == (self.nt + 2,) and a[0] == 0.0 and abs(a[-1] - np.pi) < 1e-15 and np.all(np.diff(a) > 0)
        f = self._f("sft_oracle_set_theta_nodes")
        f.restype = None
        f.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
        f(self.h, _dp(a))

    def grid_arrays(self):
        th, thf, dthc, dthf, caps = np.zeros(self.nt + 2), np.zeros(self.nt + 1), np.zeros(self.nt + 2), np.zeros(self.nt + 1), np.zeros(4)
        f = self._f("sft_oracle_get_grid")
        f.restype = None
        f.argtypes = [C.c_void_p] + [C.POINTER(C.c_double)] * 5
        f(self.h, _dp(th), _dp(thf), _dp(dthc), _dp(dthf), _dp(caps))
        return dict(th=th, thf=thf, dthc=dthc, dthf=dthf, PN=caps[0], PS=caps[1], ApoleN=caps[2], ApoleS=caps[3])

    # -- state ------------------------------------------------------------------------------
    def set_diffusivity_profile(self, r, nu_face_km2_s):
        """nu(theta) at the theta-faces f+1/2, f = 0..nt, km^2/s (Eq. 6 with a latitude-dependent diffusivity)."""
        a = np.ascontiguousarray(nu_face_km2_s, dtype=np.float64)
        assert a.shape == (self.nt + 1,)
        f = self._f("sft_oracle_set_diffusivity_profile")
        f.restype = None
        f.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_double)]
        f(self.h, int(r), _dp(a))

    def set_diffusivity_map(self, r, nu_hh_km2_s):
        """nu(theta, phi) on the half-half grid [nt+1][np] in km^2/s (Eq. 27-28), or None to switch the map off."""
        f = self._f("sft_oracle_set_diffusivity_map")
        f.restype = None
        f.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_double)]
        if nu_hh_km2_s is None:
            f(self.h, r, None)
            return
        a = np.ascontiguousarray(nu_hh_km2_s, dtype=np.float64)
        assert a.shape == (self.nt + 1, self.np_)
        f(self.h, r, _dp(a))

    def set_grid_diffusivity(self, r, alpha_nu):
        """Eq. 7 (:121): nu_g = alpha_nu [dth^2 + (dph sin(theta))^2], alpha_nu in km^2/s per rad^2."""
        f = self._f("sft_oracle_set_grid_diffusivity")
        f.restype = None
        f.argtypes = [C.c_void_p, C.c_int, C.c_double]
        f(self.h, int(r), float(alpha_nu))

    def set_attenuation(self, r, b0_gauss):
        """Flow attenuation Eq. 5 (:100): saturation field B0 in Gauss for realization r (-1: all); <= 0 off."""
        f = self._f("sft_oracle_set_attenuation")
        f.restype = None
        f.argtypes = [C.c_void_p, C.c_int, C.c_double]
        f(self.h, int(r), float(b0_gauss))

    def advection_tendency_general(self, r, a, flux_mode=ADV_WENO3, b0_gauss=float("inf")):
        """F_A through the variable-face-speed rule with speeds attenuated by B0 (inf: factor exactly 1)."""
        a = np.ascontiguousarray(a, dtype=self.dtype)
        out = np.zeros_like(a)
        f = self._f("sft_oracle_advection_tendency_general")
        f.restype = None
        f.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_int, C.c_double]
        f(self.h, int(r), self._rp(a), self._rp(out), flux_mode, float(b0_gauss))
        return out

    def advection_tendency_faces(self, a, vt_faces, vp_faces, flux_mode=ADV_WENO3):
        """F_A through the variable-face-speed rule with ARBITRARY face speeds (test hook): vt_faces [nt+1][np] at the
        theta-faces f+1/2, vp_faces [nt+2][np] at the phi-faces k-1/2 (rows 1..nt used), both in R_sun/hr."""
        a = np.ascontiguousarray(a, dtype=self.dtype)
        vt = np.ascontiguousarray(vt_faces, dtype=self.dtype)
        vp = np.ascontiguousarray(vp_faces, dtype=self.dtype)
        assert a.shape == (self.nt + 2, self.np_) and vt.shape == (self.nt + 1, self.np_) and vp.shape == (self.nt + 2, self.np_)
        out = np.zeros_like(a)
        f = self._f("sft_oracle_advection_tendency_faces")
        f.restype = None
        f.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
        f(self.h, self._rp(a), self._rp(out), flux_mode, self._rp(vt), self._rp(vp))
        return out

    def set_rfe(self, model, flux_per_hr, tau_hours=float("inf"), seed=0):
        """Random flux emergence (Sec. 2.4): model 0 off / 1 Eq. 13 / 2 Eq. 14; flux_per_hr in G radius_cm^2 / hr."""
        f = self._f("sft_oracle_set_rfe")
        f.restype = None
        f.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_double, C.c_uint64]
        f(self.h, int(model), float(flux_per_hr), float(tau_hours), int(seed))

    def get_rfe_maps(self, r):
        s1 = np.empty((self.nt + 2, self.np_), dtype=self.dtype)
        s2 = np.empty_like(s1)
        f = self._f("sft_oracle_get_rfe_maps")
        f.restype = None
        f.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
        f(self.h, int(r), self._rp(s1), self._rp(s2))
        return s1, s2

    def philox(self, ctr, key):
        c = (C.c_uint32 * 4)(*ctr); k = (C.c_uint32 * 2)(*key); out = (C.c_uint32 * 4)()
        f = self._f("sft_oracle_philox")
        f.restype = None
        f.argtypes = [C.POINTER(C.c_uint32)] * 3
        f(c, k, out)
        return list(out)

    def set_map(self, r, m):
        m = np.ascontiguousarray(m, dtype=self.dtype)
        assert m.shape == (self.nt, self.np_)
        f = self._f("sft_oracle_set_map")
        f.restype = None
        f.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        f(self.h, r, self._rp(m))

    def get_map(self, r):
        out = np.empty((self.nt, self.np_), dtype=self.dtype)
        f = self._f("sft_oracle_get_map")
        f.restype = None
        f.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        f(self.h, r, self._rp(out))
        return out

    def get_full(self, r):
        out = np.empty((self.nt + 2, self.np_), dtype=self.dtype)
        f = self._f("sft_oracle_get_full")
        f.restype = None
        f.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        f(self.h, r, self._rp(out))
        return out

    def set_full(self, r, a):
        a = np.ascontiguousarray(a, dtype=self.dtype)
        assert a.shape == (self.nt + 2, self.np_)
        f = self._f("sft_oracle_set_full")
        f.restype = None
        f.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        f(self.h, r, self._rp(a))

    # -- operators --------------------------------------------------------------------------
    def diffusion_op(self, r, a):
        a = np.ascontiguousarray(a, dtype=self.dtype)
        assert a.shape == (self.nt + 2, self.np_)
        out = np.empty_like(a)
        f = self._f("sft_oracle_diffusion_op")
        f.restype = None
        f.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
        f(self.h, r, self._rp(a), self._rp(out))
        return out

    def advection_tendency(self, r, a, flux_mode=ADV_WENO3):
        a = np.ascontiguousarray(a, dtype=self.dtype)
        assert a.shape == (self.nt + 2, self.np_)
        out = np.empty_like(a)
        f = self._f("sft_oracle_advection_tendency")
        f.restype = None
        f.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_int]
        f(self.h, r, self._rp(a), self._rp(out), flux_mode)
        return out

    def sts_coeffs(self, scheme, s):
        arrs = [np.zeros(s + 1) for _ in range(5)]
        f = self._f("sft_oracle_sts_coeffs")
        f.restype = None
        f.argtypes = [C.c_int, C.c_int] + [C.POINTER(C.c_double)] * 5
        f(scheme, s, *[_dp(a) for a in arrs])
        return dict(zip(("mu", "nu", "mut", "gt", "b"), arrs))

    def stable_dt(self):
        a, b = C.c_double(), C.c_double()
        f = self._f("sft_oracle_stable_dt")
        f.restype = None
        f.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        f(self.h, C.byref(a), C.byref(b))
        return a.value, b.value

    def sts_stage_count(self, dt, scheme=DIFF_RKG2):
        f = self._f("sft_oracle_sts_stage_count")
        f.restype = C.c_int
        f.argtypes = [C.c_void_p, C.c_double, C.c_int]
        return f(self.h, float(dt), scheme)

    def step(self, n_steps, dt, adv_flux=ADV_WENO3, adv_time=TIME_SSPRK43, diff_time=DIFF_RKG2, sts_stages=0, strang=False):
        """Eq. 21 (A then D) per step; strang=True: Eq. 22 with S omitted, A(dt/2) D(dt) A(dt/2)."""
        f = self._f("sft_oracle_step_ex")
        f.restype = C.c_int
        f.argtypes = [C.c_void_p, C.c_int, C.c_double] + [C.c_int] * 5
        s = f(self.h, n_steps, float(dt), adv_flux, adv_time, diff_time, sts_stages, int(bool(strang)))
        if s < 0:
            raise ValueError("oracle step: invalid STS stage count")
        return s

    def assimilate(self, obs, w, flags=0):
        obs = np.ascontiguousarray(obs, dtype=self.dtype)
        w = np.ascontiguousarray(w, dtype=self.dtype)
        shared = obs.ndim == 2 or obs.shape[0] == 1 and self.nr > 1
        assert obs.shape == w.shape and obs.shape[-2:] == (self.nt, self.np_)
        if not shared:
            assert obs.shape[0] == self.nr
        f = self._f("sft_oracle_assimilate")
        f.restype = None
        f.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int]
        f(self.h, self._rp(obs), self._rp(w), int(shared), int(flags))

    def diagnostics(self):
        out = np.zeros((self.nr, 4))
        f = self._f("sft_oracle_diagnostics")
        f.restype = None
        f.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
        f(self.h, _dp(out))
        return out

    def diagnostics_ext(self, lat_cut_deg=60.0):
        """[nr][13]: polar Phi+-, polar areas, min / max / min|B|, H, D, h1, h2 (see sft_oracle.c)."""
        out = np.zeros((self.nr, 13))
        f = self._f("sft_oracle_diagnostics_ext")
        f.restype = None
        f.argtypes = [C.c_void_p, C.c_double, C.POINTER(C.c_double)]
        f(self.h, float(lat_cut_deg), _dp(out))
        return out


def threads() -> int:
    """Number of host threads the oracle's OpenMP loops will use."""
    n = os.environ.get("OMP_NUM_THREADS")
    if n:
        return int(n)
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1
