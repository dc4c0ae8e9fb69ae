"""Thin Python binding of libnuma_b200.so (include/numa_b200.h): argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels; PyTorch is used for device
memory and streams.  There is no CPU fallback: if the shared library is missing (and cannot
be built) or no CUDA device is present, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

from . import build as _build

_LIB = None

STATUS = {0: "NUMA_OK", 1: "NUMA_ERR_ARG", 2: "NUMA_ERR_UNSUPPORTED", 3: "NUMA_ERR_CUDA",
          4: "NUMA_ERR_NEG_JACOBIAN", 5: "NUMA_ERR_WORKSPACE", 6: "NUMA_ERR_NOT_CONVERGED"}

# product ABI (include/numa_b200.h) and measurement ABI (include/numa_b200_measure.h)
EXPORTS = ["numa_workspace_bytes", "numa_step_scratch_bytes", "numa_init_geometry", "numa_rhs",
           "numa_dss_or_flux", "numa_apply_sources", "numa_rk_stage", "numa_step_rk3",
           "numa_step_rk3_graph", "numa_step_rk3_host", "numa_step_rk3_static",
           "numa_static_scratch_bytes", "numa_copy_table", "numa_destroy",
           "numa_last_error", "numa_ri_workspace_bytes", "numa_ri_init", "numa_ri_velocity",
           "numa_ri_destroy", "numa_hd_workspace_bytes", "numa_hd_init", "numa_hyperdiffusion",
           "numa_imex_workspace_bytes", "numa_imex_init", "numa_linear_operator", "numa_step_ark2"]
MEASURE_EXPORTS = ["numa_profile_enable", "numa_profile_read", "numa_kernel_name",
                   "numa_kernel_count", "numa_launch_count", "numa_measure_fp64_peak"]


class NumaParams(C.Structure):
    _fields_ = [("N", C.c_int32), ("method", C.c_int32), ("eqn_set", C.c_int32),
                ("reserved", C.c_int32), ("n_elem", C.c_int64), ("n_global", C.c_int64),
                ("g", C.c_double), ("p_a", C.c_double), ("R_gas", C.c_double),
                ("c_p", C.c_double), ("c_v", C.c_double), ("f_cor", C.c_double)]


class NumaError(RuntimeError):
    def __init__(self, status, text):
        super().__init__("%s: %s" % (STATUS.get(status, status), text))
        self.status = status


def load_library(path: str | None = None):
    """dlopen libnuma_b200.so (building it in-tree first if it is stale or absent)."""
    global _LIB
    if _LIB is not None and path is None:
        return _LIB
    libpath = path or _build.LIB
    if path is None and not os.path.exists(libpath):
        libpath = _build.build()
    if not os.path.exists(libpath):
        raise ImportError("libnuma_b200.so is missing and could not be built; there is no "
                          "fallback path (run python -m paper_2504_08157_b200.build)")
    L = C.CDLL(libpath)
    vp, dp = C.c_void_p, C.c_void_p
    L.numa_workspace_bytes.argtypes = [C.POINTER(NumaParams)]
    L.numa_workspace_bytes.restype = C.c_size_t
    L.numa_step_scratch_bytes.argtypes = [C.POINTER(NumaParams)]
    L.numa_step_scratch_bytes.restype = C.c_size_t
    L.numa_init_geometry.argtypes = [C.POINTER(NumaParams), dp, dp, dp, dp, dp, vp, C.c_size_t,
                                     vp, C.POINTER(vp)]
    L.numa_rhs.argtypes = [vp, dp, dp, vp]
    L.numa_dss_or_flux.argtypes = [vp, dp, vp]
    L.numa_apply_sources.argtypes = [vp, dp, dp, dp, vp]
    L.numa_rk_stage.argtypes = [vp, C.c_double, C.c_double, C.c_double, dp, dp, dp, dp, vp]
    L.numa_step_rk3.argtypes = [vp, dp, vp, dp, C.c_double, C.c_int32, vp]
    L.numa_step_rk3_graph.argtypes = [vp, dp, vp, dp, C.c_double, C.c_int32, vp]
    L.numa_step_rk3_host.argtypes = [vp, dp, dp, dp, dp, vp, C.c_double, C.c_int32, vp]
    L.numa_step_rk3_static.argtypes = [vp, dp, dp, C.c_double, C.c_int32, vp]
    L.numa_static_scratch_bytes.argtypes = []
    L.numa_static_scratch_bytes.restype = C.c_size_t
    L.numa_copy_table.argtypes = [vp, C.c_int32, dp, vp]
    L.numa_imex_workspace_bytes.argtypes = [C.POINTER(NumaParams), C.c_int32]
    L.numa_imex_workspace_bytes.restype = C.c_size_t
    L.numa_imex_init.argtypes = [vp, C.c_int32, vp, C.c_size_t, vp]
    L.numa_linear_operator.argtypes = [vp, dp, dp, vp]
    L.numa_step_ark2.argtypes = [vp, dp, dp, C.c_double, C.c_int32, C.c_double, C.c_int32,
                                 C.POINTER(C.c_int64), C.POINTER(C.c_double), vp]
    L.numa_hd_workspace_bytes.argtypes = [C.POINTER(NumaParams)]
    L.numa_hd_workspace_bytes.restype = C.c_size_t
    L.numa_hd_init.argtypes = [vp, C.POINTER(C.c_double), C.c_double, vp, C.c_size_t, vp]
    L.numa_hyperdiffusion.argtypes = [vp, dp, dp, vp]
    L.numa_ri_workspace_bytes.argtypes = [C.POINTER(NumaParams), C.c_int32, C.c_int32]
    L.numa_ri_workspace_bytes.restype = C.c_size_t
    L.numa_ri_init.argtypes = [vp, dp, dp, C.c_int32, C.c_int32, C.c_double, vp, C.c_size_t, vp,
                               C.POINTER(vp)]
    L.numa_ri_velocity.argtypes = [vp, dp, dp, dp, dp, dp, vp]
    L.numa_ri_destroy.argtypes = [vp]
    L.numa_profile_enable.argtypes = [vp, C.c_int32]
    L.numa_profile_enable.restype = C.c_int
    L.numa_profile_read.argtypes = [vp, C.c_int32, C.POINTER(C.c_double), C.POINTER(C.c_int64)]
    L.numa_profile_read.restype = C.c_int
    L.numa_kernel_name.argtypes = [C.c_int32]
    L.numa_kernel_name.restype = C.c_char_p
    L.numa_kernel_count.argtypes = []
    L.numa_kernel_count.restype = C.c_int32
    L.numa_measure_fp64_peak.argtypes = [C.c_int32, C.POINTER(C.c_double), vp]
    L.numa_measure_fp64_peak.restype = C.c_int
    L.numa_launch_count.argtypes = [vp]
    L.numa_launch_count.restype = C.c_int64
    L.numa_destroy.argtypes = [vp]
    L.numa_last_error.argtypes = [vp]
    L.numa_last_error.restype = C.c_char_p
    for f in ("numa_init_geometry", "numa_rhs", "numa_dss_or_flux", "numa_apply_sources",
              "numa_rk_stage", "numa_step_rk3", "numa_step_rk3_graph", "numa_step_rk3_host",
              "numa_step_rk3_static", "numa_copy_table", "numa_ri_init", "numa_ri_velocity", "numa_ri_destroy",
              "numa_hd_init", "numa_hyperdiffusion", "numa_imex_init", "numa_linear_operator",
              "numa_step_ark2", "numa_destroy"):
        getattr(L, f).restype = C.c_int
    if path is None:
        _LIB = L
    return L


def make_params(N, n_elem, n_global, constants, f_cor=0.0, method=0, eqn_set=0) -> NumaParams:
    return NumaParams(N=N, method=method, eqn_set=eqn_set, reserved=0, n_elem=n_elem,
                      n_global=n_global, g=constants["g"], p_a=constants["p_a"],
                      R_gas=constants["R_gas"], c_p=constants["c_p"], c_v=constants["c_v"],
                      f_cor=f_cor)


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _dev(a, dtype, device):
    """numpy array / torch tensor -> contiguous device tensor of the given dtype."""
    if a is None:
        return None
    t = torch.as_tensor(a)
    return t.to(device=device, dtype=dtype).contiguous()


class Numa:
    """One numa_ctx plus the torch tensors (workspace, scratch) that back it.

    Methods mirror the C ABI one to one: rhs, dss_or_flux, apply_sources, rk_stage,
    step_rk3, step_rk3_host.  Arrays are torch CUDA float64 tensors [5][Ne][Mn] / [Ne][Mn].
    """

    def __init__(self, N, xyz, intma_cg, n_global, face_bc, ref, constants, f_cor=0.0,
                 sponge=None, device="cuda:0", method=0, eqn_set=0):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2504_08157_b200 needs a CUDA device; there is no CPU fallback")
        self.lib = load_library()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        xyz_d = _dev(xyz, torch.float64, self.device)
        self.n_elem = int(xyz_d.shape[1])
        self.Mn = (N + 1) ** 3
        self.N = N
        self.NL = self.n_elem * self.Mn
        self.params = make_params(N, self.n_elem, int(n_global), constants, f_cor, method, eqn_set)
        cg_d = _dev(intma_cg, torch.int32, self.device)
        bc_d = _dev(face_bc, torch.uint8, self.device)
        ref_d = _dev(ref, torch.float64, self.device)
        sp_d = _dev(sponge, torch.float64, self.device)
        nbytes = self.lib.numa_workspace_bytes(C.byref(self.params))
        if nbytes == 0 and method == 0 and eqn_set == 0:
            raise NumaError(1, "numa_workspace_bytes: parameters out of range")
        self.workspace = torch.empty(max(nbytes, 256), dtype=torch.uint8, device=self.device)
        self._scratch = None
        self.ctx = C.c_void_p()
        st = self.lib.numa_init_geometry(C.byref(self.params), _ptr(xyz_d), _ptr(cg_d), _ptr(bc_d),
                                         _ptr(ref_d), _ptr(sp_d), _ptr(self.workspace),
                                         self.workspace.numel(), _stream(), C.byref(self.ctx))
        if st != 0:
            raise NumaError(st, self.lib.numa_last_error(None).decode())

    @classmethod
    def from_workload(cls, wl, device="cuda:0"):
        m = wl.mesh
        return cls(m.N, m.xyz, m.intma_cg, m.n_global, m.face_bc, wl.ref, wl.constants,
                   f_cor=wl.f_cor, sponge=wl.sponge, device=device)

    # -- helpers ------------------------------------------------------------------------
    def _check(self, st):
        if st != 0:
            raise NumaError(st, self.lib.numa_last_error(self.ctx).decode())

    def state(self, a):
        """Host array -> device state tensor [5][Ne][Mn]."""
        return _dev(a, torch.float64, self.device)

    def scratch(self):
        if self._scratch is None:
            n = self.lib.numa_step_scratch_bytes(C.byref(self.params))
            self._scratch = torch.empty(n, dtype=torch.uint8, device=self.device)
        return self._scratch

    def table(self, which):
        """Copy of a table built by A0: 0 met[9][NL], 1 omega[NL], 2 p0[NL], 3 D[Nq*Nq], 4 w[Nq]."""
        Nq = self.N + 1
        n = {0: 9 * self.NL, 1: self.NL, 2: self.NL, 3: Nq * Nq, 4: Nq}[which]
        out = torch.empty(n, dtype=torch.float64, device=self.device)
        self._check(self.lib.numa_copy_table(self.ctx, which, _ptr(out), _stream()))
        return out

    # -- the C ABI ------------------------------------------------------------------------
    def rhs(self, q, out=None):
        out = torch.empty_like(q) if out is None else out
        self._check(self.lib.numa_rhs(self.ctx, _ptr(q), _ptr(out), _stream()))
        return out

    def dss_or_flux(self, r):
        self._check(self.lib.numa_dss_or_flux(self.ctx, _ptr(r), _stream()))
        return r

    def apply_sources(self, q, heating, r):
        self._check(self.lib.numa_apply_sources(self.ctx, _ptr(q), _ptr(heating), _ptr(r), _stream()))
        return r

    def rk_stage(self, a0, a1, b_dt, q0, qs, r, out):
        self._check(self.lib.numa_rk_stage(self.ctx, a0, a1, b_dt, _ptr(q0), _ptr(qs), _ptr(r),
                                           _ptr(out), _stream()))
        return out

    def step_rk3(self, q, dt, heating=None, n_steps=1, graph=False):
        fn = self.lib.numa_step_rk3_graph if graph else self.lib.numa_step_rk3
        self._check(fn(self.ctx, _ptr(q), _ptr(self.scratch()), _ptr(heating), dt, n_steps, _stream()))
        return q

    def step_rk3_static(self, q, dt, heating=None, n_steps=1):
        """numa_step_rk3_static: step_rk3 on the library's built-in scratch array, for callers that
        cannot allocate device memory (no torch scratch tensor is created; meshes beyond
        numa_static_scratch_bytes() raise NUMA_ERR_WORKSPACE)."""
        self._check(self.lib.numa_step_rk3_static(self.ctx, _ptr(q), _ptr(heating), dt, n_steps, _stream()))
        return q

    def step_rk3_host(self, q_host, dt, heating_host=None, n_steps=1, d_q=None, d_heating=None):
        """q_host / heating_host: (pinned) CPU float64 tensors; staged through d_q / d_heating."""
        if d_q is None:
            d_q = torch.empty(q_host.shape, dtype=torch.float64, device=self.device)
        if heating_host is not None and d_heating is None:
            d_heating = torch.empty(heating_host.shape, dtype=torch.float64, device=self.device)
        # heating_host None with d_heating given: the heating resident in d_heating is reused
        self._check(self.lib.numa_step_rk3_host(self.ctx, _ptr(q_host), _ptr(heating_host),
                                                _ptr(d_q), _ptr(d_heating), _ptr(self.scratch()),
                                                dt, n_steps, _stream()))
        return q_host

    # -- IMEX: linear operator, ARK2 + GMRES (numa_imex_*, numa_step_ark2) ---------------------
    def imex_init(self, m=20):
        n = self.lib.numa_imex_workspace_bytes(C.byref(self.params), m)
        if n == 0:
            raise NumaError(1, "numa_imex_workspace_bytes: parameters out of range")
        self._imex_ws = torch.empty(n, dtype=torch.uint8, device=self.device)
        self._check(self.lib.numa_imex_init(self.ctx, m, _ptr(self._imex_ws), n, _stream()))

    def linear_operator(self, q, out=None):
        out = torch.empty_like(q) if out is None else out
        self._check(self.lib.numa_linear_operator(self.ctx, _ptr(q), _ptr(out), _stream()))
        return out

    def step_ark2(self, q, dt, heating=None, n_steps=1, tol=1e-10, max_restarts=10):
        """numa_step_ark2 -> (total GMRES iterations, largest final relative residual)."""
        its = C.c_int64(0); rel = C.c_double(0.0)
        self._check(self.lib.numa_step_ark2(self.ctx, _ptr(q), _ptr(heating), dt, n_steps, tol, max_restarts,
                                            C.byref(its), C.byref(rel), _stream()))
        return its.value, rel.value

    def hd_init(self, c3, dt_ref):
        """numa_hd_init: tensor hyper-diffusion (Eq. 14-16) on; c3 = (c_1, c_2, c_3)."""
        n = self.lib.numa_hd_workspace_bytes(C.byref(self.params))
        self._hd_ws = torch.empty(n, dtype=torch.uint8, device=self.device)
        self._hd = True
        c = (C.c_double * 3)(*[float(x) for x in c3])
        self._check(self.lib.numa_hd_init(self.ctx, c, float(dt_ref), _ptr(self._hd_ws), n, _stream()))

    def hyperdiffusion(self, q, r):
        self._check(self.lib.numa_hyperdiffusion(self.ctx, _ptr(q), _ptr(r), _stream()))
        return r

    def full_rhs(self, q, heating=None):
        """Convenience: the separate calls that form L(q) (with H_q when hd_init was called)."""
        r = self.rhs(q)
        self.dss_or_flux(r)
        if getattr(self, "_hd", False):
            self.hyperdiffusion(q, r)
        self.apply_sources(q, heating, r)
        return r

    # -- RI-velocity diagnostic (numa_ri_*) ---------------------------------------------------
    def ri_init(self, xyz, level, n_levels, r_max, n_strips=50):
        """numa_ri_init: area weights and level-sorted lists into a torch workspace."""
        xyz_d = _dev(xyz, torch.float64, self.device)
        lev_d = _dev(level, torch.int32, self.device)
        n = self.lib.numa_ri_workspace_bytes(C.byref(self.params), n_levels, n_strips)
        if n == 0:
            raise NumaError(1, "numa_ri_workspace_bytes: parameters out of range")
        self._ri_ws = torch.empty(n, dtype=torch.uint8, device=self.device)
        self._ri = C.c_void_p()
        self._ri_shape = (int(n_levels), int(n_strips))
        self._check(self.lib.numa_ri_init(self.ctx, _ptr(xyz_d), _ptr(lev_d), n_levels, n_strips,
                                          float(r_max), _ptr(self._ri_ws), n, _stream(),
                                          C.byref(self._ri)))

    def ri_velocity(self, q):
        """numa_ri_velocity -> (ubar[n_lev][n_strip], count, centroid[3*n_lev], scalars[3]) on the device."""
        nl, ns = self._ri_shape
        ubar = torch.empty((nl, ns), dtype=torch.float64, device=self.device)
        count = torch.empty((nl, ns), dtype=torch.int32, device=self.device)
        cen = torch.empty(3 * nl, dtype=torch.float64, device=self.device)
        sc = torch.empty(3, dtype=torch.float64, device=self.device)
        self._check(self.lib.numa_ri_velocity(self._ri, _ptr(q), _ptr(ubar), _ptr(count), _ptr(cen),
                                              _ptr(sc), _stream()))
        return ubar, count, cen, sc

    def profile(self, enable=True):
        self._check(self.lib.numa_profile_enable(self.ctx, 1 if enable else 0))

    def profile_read(self):
        """{kernel name: (total device ms, launches)} accumulated since profile(True)."""
        out = {}
        for kid in range(self.lib.numa_kernel_count()):
            ms = C.c_double(); n = C.c_int64()
            self._check(self.lib.numa_profile_read(self.ctx, kid, C.byref(ms), C.byref(n)))
            if n.value:
                out[self.lib.numa_kernel_name(kid).decode()] = (ms.value, n.value)
        return out

    def fp64_peak_tflops(self, repeats=5):
        """Measured DFMA ceiling of the current device (numa_measure_fp64_peak)."""
        v = C.c_double()
        st = self.lib.numa_measure_fp64_peak(repeats, C.byref(v), _stream())
        if st != 0:
            raise NumaError(st, "numa_measure_fp64_peak")
        return v.value

    @property
    def launch_count(self):
        return int(self.lib.numa_launch_count(self.ctx))

    def close(self):
        if getattr(self, "_ri", None) is not None and self._ri.value:
            self.lib.numa_ri_destroy(self._ri)
            self._ri = C.c_void_p()
        if getattr(self, "ctx", None) is not None and self.ctx.value:
            self.lib.numa_destroy(self.ctx)
            self.ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
