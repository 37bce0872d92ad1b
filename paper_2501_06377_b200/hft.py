"""Thin ctypes binding of the C-ABI library libhft.so (include/hft.h) -- argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels; PyTorch is used for device memory and
streams.  There is no CPU fallback: importing this module without the built library raises, and creating
a context without a CUDA device raises.
"""
import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libhft.so")

if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2501_06377_b200.build` "
                      "(the CUDA extension is required; there is no CPU fallback)")
_lib = C.CDLL(LIB_PATH)

EXPORTS = ["hft_workspace_bytes", "hft_create", "hft_destroy", "hft_set_theta_nodes", "hft_set_flow_tables", "hft_set_diffusivity_profile", "hft_set_grid_diffusivity", "hft_set_diffusivity_map", "hft_set_attenuation", "hft_set_rfe", "hft_get_rfe_map", "hft_set_map", "hft_get_map",
           "hft_get_full", "hft_set_full", "hft_step", "hft_assimilate", "hft_assimilate_diagnostics", "hft_diagnostics", "hft_diagnostics_noalloc", "hft_diagnostics_ext", "hft_stable_dt",
           "hft_sts_stage_count", "hft_synchronize", "hft_launch_count", "hft_profile_kernels", "hft_kernel_time", "hft_probe_fma_rate", "hft_error_string",
           "hft_last_cuda_error"]

ADV_OFF, ADV_UPWIND, ADV_WENO3 = 0, 1, 2
TIME_EULER, TIME_SSPRK33, TIME_SSPRK43 = 1, 3, 4
DIFF_OFF, DIFF_EULER, DIFF_RKL2, DIFF_RKG2 = 0, 1, 2, 3
FLAG_FLUX_BALANCE = 1


class hft_grid(C.Structure):
    _fields_ = [("n_theta", C.c_int32), ("n_phi", C.c_int32), ("dtype", C.c_int32), ("reserved", C.c_int32),
                ("radius_cm", C.c_double)]


class hft_params(C.Structure):
    _fields_ = [("eta_km2_s", C.c_double), ("d0", C.c_double), ("d2", C.c_double), ("d4", C.c_double),
                ("m1", C.c_double), ("m3", C.c_double), ("m5", C.c_double)]


class hft_options(C.Structure):
    _fields_ = [("adv_flux", C.c_int32), ("adv_time", C.c_int32), ("diff_time", C.c_int32), ("sts_stages", C.c_int32),
                ("sts_block", C.c_int32), ("rfe", C.c_int32), ("strang", C.c_int32), ("flow_attenuation", C.c_int32),
                ("diffusivity_map", C.c_int32), ("f32_arith", C.c_int32), ("sts_kernel", C.c_int32)]


_lib.hft_workspace_bytes.argtypes = [C.POINTER(hft_grid), C.c_int32, C.POINTER(hft_options), C.POINTER(C.c_size_t)]
_lib.hft_create.argtypes = [C.POINTER(hft_grid), C.c_int32, C.POINTER(hft_params), C.POINTER(hft_options), C.c_void_p,
                            C.c_size_t, C.c_void_p, C.POINTER(C.c_void_p)]
_lib.hft_destroy.argtypes = [C.c_void_p]
_lib.hft_destroy.restype = None
_lib.hft_set_flow_tables.argtypes = [C.c_void_p, C.c_int32, C.POINTER(C.c_double), C.POINTER(C.c_double)]
_lib.hft_set_theta_nodes.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
_lib.hft_set_diffusivity_profile.argtypes = [C.c_void_p, C.c_int32, C.POINTER(C.c_double)]
_lib.hft_set_grid_diffusivity.argtypes = [C.c_void_p, C.c_int32, C.c_double]
_lib.hft_set_diffusivity_map.argtypes = [C.c_void_p, C.c_int32, C.POINTER(C.c_double)]
_lib.hft_set_attenuation.argtypes = [C.c_void_p, C.c_int32, C.c_double]
_lib.hft_set_rfe.argtypes = [C.c_void_p, C.c_int32, C.c_double, C.c_double, C.c_uint64]
_lib.hft_get_rfe_map.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_void_p]
_lib.hft_set_map.argtypes = [C.c_void_p, C.c_int32, C.c_void_p]
_lib.hft_get_map.argtypes = [C.c_void_p, C.c_int32, C.c_void_p]
_lib.hft_get_full.argtypes = [C.c_void_p, C.c_int32, C.c_void_p]
_lib.hft_set_full.argtypes = [C.c_void_p, C.c_int32, C.c_void_p]
_lib.hft_step.argtypes = [C.c_void_p, C.c_int32, C.c_double]
_lib.hft_assimilate.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_int32]
_lib.hft_assimilate_diagnostics.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.POINTER(C.c_double)]
_lib.hft_diagnostics.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
_lib.hft_diagnostics_noalloc.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
_lib.hft_diagnostics_ext.argtypes = [C.c_void_p, C.c_double, C.POINTER(C.c_double)]
_lib.hft_stable_dt.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double)]
_lib.hft_sts_stage_count.argtypes = [C.c_void_p, C.c_double, C.POINTER(C.c_int32)]
_lib.hft_launch_count.argtypes = [C.c_void_p, C.POINTER(C.c_int64)]
_lib.hft_synchronize.argtypes = [C.c_void_p]
_lib.hft_profile_kernels.argtypes = [C.c_void_p, C.c_int32]
_lib.hft_kernel_time.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
_lib.hft_probe_fma_rate.argtypes = [C.c_int32, C.c_int32, C.POINTER(C.c_double)]
_lib.hft_error_string.argtypes = [C.c_int]
_lib.hft_error_string.restype = C.c_char_p
_lib.hft_last_cuda_error.argtypes = [C.c_void_p]
_lib.hft_last_cuda_error.restype = C.c_char_p


class HftError(RuntimeError):
    pass


def error_string(code: int) -> str:
    return _lib.hft_error_string(int(code)).decode()


def probe_fma_rate(dtype="f64", pattern=0) -> float:
    """FMA lane-operations per second of the current device (hft.h: hft_probe_fma_rate)."""
    out = C.c_double()
    rc = _lib.hft_probe_fma_rate(1 if dtype == "f64" else 0, int(pattern), C.byref(out))
    if rc != 0:
        raise HftError(f"hft_probe_fma_rate: {error_string(rc)}")
    return out.value


def workspace_bytes(n_theta, n_phi, n_real, dtype="f64", opt=None) -> int:
    g = hft_grid(int(n_theta), int(n_phi), 1 if dtype == "f64" else 0, 0, 1.0)
    out = C.c_size_t()
    rc = _lib.hft_workspace_bytes(C.byref(g), int(n_real), C.byref(opt) if opt is not None else None, C.byref(out))
    if rc != 0:
        raise HftError(error_string(rc))
    return out.value


class Context:
    """hft_create ... hft_destroy.  Maps are torch CUDA tensors [n_theta][n_phi] of the context dtype."""

    def __init__(self, n_theta, n_phi, params, dtype="f64", radius_cm=1.0, adv_flux=ADV_WENO3, adv_time=TIME_SSPRK43,
                 diff_time=DIFF_RKG2, sts_stages=0, sts_block=0, rfe=0, strang=0, flow_attenuation=0, diffusivity_map=0, f32_arith=0, sts_kernel=0,
                 device="cuda:0", stream=None, workspace=None):
        if not torch.cuda.is_available():
            raise HftError("no CUDA device: the hot path has no CPU fallback")
        self.device = torch.device(device)
        self.n_theta, self.n_phi = int(n_theta), int(n_phi)
        self.dtype = dtype
        self.tdtype = torch.float64 if dtype == "f64" else torch.float32
        p = np.ascontiguousarray(np.asarray(params, dtype=np.float64).reshape(-1, 7))
        self.n_real = p.shape[0]
        self._h = C.c_void_p()
        with torch.cuda.device(self.device):
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            opt = hft_options(adv_flux, adv_time, diff_time, sts_stages, sts_block, int(rfe), int(strang), int(flow_attenuation),
                              int(diffusivity_map), int(f32_arith), int(sts_kernel))
            nbytes = workspace_bytes(n_theta, n_phi, self.n_real, dtype, opt)
            if workspace is None:
                workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            # caller-owned device memory (include/hft.h): a contiguous uint8 CUDA tensor of >= hft_workspace_bytes
            assert workspace.is_cuda and workspace.dtype == torch.uint8 and workspace.is_contiguous()
            self.workspace = workspace
            nbytes = workspace.numel()
            grid = hft_grid(self.n_theta, self.n_phi, 1 if dtype == "f64" else 0, 0, float(radius_cm))
            pa = (hft_params * self.n_real)(*[hft_params(*row) for row in p])
            rc = _lib.hft_create(C.byref(grid), self.n_real, pa, C.byref(opt), C.c_void_p(self.workspace.data_ptr()),
                                 nbytes, C.c_void_p(self.stream.cuda_stream), C.byref(self._h))
        if rc != 0:
            raise HftError(f"hft_create: {error_string(rc)}")

    # -- helpers ---------------------------------------------------------------------------
    def _ck(self, rc, what):
        if rc != 0:
            detail = _lib.hft_last_cuda_error(self._h).decode() if self._h else ""
            raise HftError(f"{what}: {error_string(rc)} {detail}")

    def _map_ptr(self, t, lead=None):
        assert t.is_cuda and t.dtype == self.tdtype and t.is_contiguous(), "maps must be contiguous CUDA tensors of the context dtype"
        assert tuple(t.shape[-2:]) == (self.n_theta, self.n_phi)
        if lead is not None:
            assert t.numel() == lead * self.n_theta * self.n_phi
        return C.c_void_p(t.data_ptr())

    def close(self):
        if self._h:
            torch.cuda.synchronize(self.device)
            _lib.hft_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- C-ABI calls (same names) ----------------------------------------------------------
    def set_theta_nodes(self, theta):
        a = np.ascontiguousarray(theta, dtype=np.float64)
        assert a.shape == (self.n_theta + 2,)
        self._ck(_lib.hft_set_theta_nodes(self._h, a.ctypes.data_as(C.POINTER(C.c_double))), "hft_set_theta_nodes")

    def set_flow_tables(self, r, vtheta_m_s, omega_m_s):
        vt = np.ascontiguousarray(vtheta_m_s, dtype=np.float64)
        om = np.ascontiguousarray(omega_m_s, dtype=np.float64)
        assert vt.shape == (self.n_theta + 1,) and om.shape == (self.n_theta + 2,)
        self._ck(_lib.hft_set_flow_tables(self._h, r, vt.ctypes.data_as(C.POINTER(C.c_double)),
                                          om.ctypes.data_as(C.POINTER(C.c_double))), "hft_set_flow_tables")

    def set_diffusivity_profile(self, r, nu_face_km2_s):
        a = np.ascontiguousarray(nu_face_km2_s, dtype=np.float64)
        assert a.shape == (self.n_theta + 1,)
        self._ck(_lib.hft_set_diffusivity_profile(self._h, int(r), a.ctypes.data_as(C.POINTER(C.c_double))),
                 "hft_set_diffusivity_profile")

    def set_diffusivity_map(self, r, nu_hh_km2_s):
        a = np.ascontiguousarray(nu_hh_km2_s, dtype=np.float64)
        assert a.shape == (self.n_theta + 1, self.n_phi)
        self._ck(_lib.hft_set_diffusivity_map(self._h, int(r), a.ctypes.data_as(C.POINTER(C.c_double))),
                 "hft_set_diffusivity_map")

    def set_grid_diffusivity(self, r, alpha_nu):
        self._ck(_lib.hft_set_grid_diffusivity(self._h, int(r), float(alpha_nu)), "hft_set_grid_diffusivity")

    def set_attenuation(self, r, b0_gauss):
        self._ck(_lib.hft_set_attenuation(self._h, int(r), float(b0_gauss)), "hft_set_attenuation")

    def set_rfe(self, model, flux_per_hr, tau_hours=float("inf"), seed=0):
        self._ck(_lib.hft_set_rfe(self._h, int(model), float(flux_per_hr), float(tau_hours), int(seed)), "hft_set_rfe")

    def get_rfe_map(self, r, which):
        out = torch.empty((self.n_theta, self.n_phi), dtype=self.tdtype, device=self.device)
        self._ck(_lib.hft_get_rfe_map(self._h, int(r), int(which), C.c_void_p(out.data_ptr())), "hft_get_rfe_map")
        return out

    def set_map(self, r, t):
        self._ck(_lib.hft_set_map(self._h, int(r), self._map_ptr(t, 1)), "hft_set_map")

    def get_map(self, r=-1, out=None):
        n = self.n_real if r < 0 else 1
        if out is None:
            out = torch.empty((n, self.n_theta, self.n_phi) if r < 0 else (self.n_theta, self.n_phi),
                              dtype=self.tdtype, device=self.device)
        self._ck(_lib.hft_get_map(self._h, int(r), self._map_ptr(out, n)), "hft_get_map")
        return out

    def get_full(self, r):
        out = torch.empty((self.n_theta + 2, self.n_phi), dtype=self.tdtype, device=self.device)
        self._ck(_lib.hft_get_full(self._h, int(r), C.c_void_p(out.data_ptr())), "hft_get_full")
        return out

    def set_full(self, r, t):
        assert t.is_cuda and t.dtype == self.tdtype and t.is_contiguous() and tuple(t.shape) == (self.n_theta + 2, self.n_phi)
        self._ck(_lib.hft_set_full(self._h, int(r), C.c_void_p(t.data_ptr())), "hft_set_full")

    def step(self, n_steps, dt_hours):
        self._ck(_lib.hft_step(self._h, int(n_steps), float(dt_hours)), "hft_step")

    def assimilate(self, obs, weights, flags=0):
        shared = obs.dim() == 2 or (obs.shape[0] == 1 and self.n_real > 1)
        lead = 1 if shared else self.n_real
        self._ck(_lib.hft_assimilate(self._h, self._map_ptr(obs, lead), self._map_ptr(weights, lead), int(shared),
                                     int(flags)), "hft_assimilate")

    def assimilate_diagnostics(self, obs, weights, flags=0):
        shared = obs.dim() == 2 or (obs.shape[0] == 1 and self.n_real > 1)
        lead = 1 if shared else self.n_real
        out = np.zeros((self.n_real, 4))
        self._ck(_lib.hft_assimilate_diagnostics(self._h, self._map_ptr(obs, lead), self._map_ptr(weights, lead), int(shared),
                                                 int(flags), out.ctypes.data_as(C.POINTER(C.c_double))), "hft_assimilate_diagnostics")
        return out

    def diagnostics(self):
        out = np.zeros((self.n_real, 4))
        self._ck(_lib.hft_diagnostics(self._h, out.ctypes.data_as(C.POINTER(C.c_double))), "hft_diagnostics")
        return out

    def diagnostics_noalloc(self, field: torch.Tensor, out: torch.Tensor) -> None:
        """hft_diagnostics of a caller-held field [n_real][n_theta+2][n_phi] into a caller-held device tensor out[n_real][4]
        (float64); allocates nothing, asynchronous (hft.h: hft_diagnostics_noalloc)."""
        assert field.is_cuda and field.dtype == self.tdtype and field.is_contiguous()
        assert tuple(field.shape) == (self.n_real, self.n_theta + 2, self.n_phi)
        assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and tuple(out.shape) == (self.n_real, 4)
        self._ck(_lib.hft_diagnostics_noalloc(self._h, C.c_void_p(field.data_ptr()), C.c_void_p(out.data_ptr())), "hft_diagnostics_noalloc")

    def diagnostics_ext(self, polar_lat_deg=60.0):
        out = np.zeros((self.n_real, 13))
        self._ck(_lib.hft_diagnostics_ext(self._h, float(polar_lat_deg), out.ctypes.data_as(C.POINTER(C.c_double))),
                 "hft_diagnostics_ext")
        return out

    def stable_dt(self):
        a, b = C.c_double(), C.c_double()
        self._ck(_lib.hft_stable_dt(self._h, C.byref(a), C.byref(b)), "hft_stable_dt")
        return a.value, b.value

    def sts_stage_count(self, dt_hours):
        s = C.c_int32()
        self._ck(_lib.hft_sts_stage_count(self._h, float(dt_hours), C.byref(s)), "hft_sts_stage_count")
        return s.value

    def synchronize(self):
        self._ck(_lib.hft_synchronize(self._h), "hft_synchronize")

    def launch_count(self):
        n = C.c_int64()
        self._ck(_lib.hft_launch_count(self._h, C.byref(n)), "hft_launch_count")
        return n.value

    def profile_kernels(self, which):
        self._ck(_lib.hft_profile_kernels(self._h, int(which)), "hft_profile_kernels")

    def kernel_time(self):
        ms, n, st = C.c_double(), C.c_int64(), C.c_int64()
        self._ck(_lib.hft_kernel_time(self._h, C.byref(ms), C.byref(n), C.byref(st)), "hft_kernel_time")
        return ms.value, n.value, st.value
