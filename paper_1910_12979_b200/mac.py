"""Thin ctypes binding of include/maestro_mac.h (argument marshalling only).

Every step of the path runs in the CUDA library `libmaestro_mac.so`; there is no CPU fallback.
PyTorch is used for device memory and streams only.  Importing this module does not need a GPU
(the library loads and exports its symbols on a CPU box); calling it does.
"""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmaestro_mac.so")

PERIODIC, WALL, OUTFLOW = 0, 1, 2
PLANAR, SPHERICAL = 0, 1
OK, NOT_CONVERGED = 0, 1
ERR_ARG, ERR_UNSUPPORTED, ERR_WORKSPACE, ERR_CUDA, ERR_NONFINITE = -1, -2, -3, -4, -5
ARR_PHI, ARR_RHS, ARR_BX, ARR_BY, ARR_BZ = 0, 1, 2, 3, 4

EXPORTS = [
    "maestro_mac_default_desc", "maestro_mac_setup", "maestro_mac_project",
    "maestro_mac_project_host", "maestro_mac_project_host_seq", "maestro_mac_free", "maestro_mac_num_levels",
    "maestro_mac_level_dims", "maestro_mac_level_get", "maestro_mac_level_set",
    "maestro_mac_step_coefficients", "maestro_mac_step_rhs", "maestro_mac_step_smooth",
    "maestro_mac_step_residual_restrict", "maestro_mac_step_prolong", "maestro_mac_step_bottom",
    "maestro_mac_step_vcycle", "maestro_mac_step_residual_norm", "maestro_mac_step_correct",
    "maestro_mac_base_state", "maestro_mac_set_dpdt_term", "maestro_mac_lateral_average",
    "maestro_mac_lateral_average_noalloc",
    "maestro_mac_status", "maestro_mac_level_plan", "maestro_mac_plan_query",
    "maestro_mac_nodal_project", "maestro_mac_nodal_level_get", "maestro_mac_nodal_level_set",
    "maestro_mac_nodal_step_sigma", "maestro_mac_nodal_step_rhs", "maestro_mac_nodal_step_smooth",
    "maestro_mac_nodal_step_residual_restrict", "maestro_mac_nodal_step_prolong", "maestro_mac_nodal_step_bottom",
    "maestro_mac_nodal_step_vcycle", "maestro_mac_nodal_step_residual_norm", "maestro_mac_nodal_step_correct",
]
NODAL_PHI, NODAL_RHS, NODAL_SIGMA = 0, 1, 2


class Desc(C.Structure):
    _fields_ = [("struct_bytes", C.c_int), ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("dx", C.c_double * 3), ("bc_lo", C.c_int * 3), ("bc_hi", C.c_int * 3),
                ("geometry", C.c_int), ("nr", C.c_int), ("dr", C.c_double),
                ("center", C.c_double * 3), ("nu_pre", C.c_int), ("nu_post", C.c_int),
                ("max_cycles", C.c_int), ("rel_tol", C.c_double), ("coarsest_n", C.c_int),
                ("bottom_max_iter", C.c_int), ("bottom_rel_tol", C.c_double),
                ("prolongation", C.c_int), ("host_staging", C.c_int), ("smoother", C.c_int),
                ("stop_test", C.c_int), ("rho_mean", C.c_int), ("timing", C.c_int), ("nodal", C.c_int)]


class Stats(C.Structure):
    _fields_ = [("cycles", C.c_int), ("bottom_iters_total", C.c_int), ("singular", C.c_int),
                ("levels", C.c_int), ("rhs_norm_inf", C.c_double), ("res_norm_inf", C.c_double),
                ("rhs_mean_removed", C.c_double), ("res_history", C.c_double * 128),
                ("ms_setup_kernels", C.c_float), ("ms_vcycles", C.c_float),
                ("ms_correct", C.c_float), ("gpu_launches", C.c_int),
                ("ms_smooth0", C.c_float), ("smooth0_launches", C.c_int), ("smooth0_timed", C.c_int),
                ("smooth0_sweeps_timed", C.c_int)]

    def as_dict(self):
        return dict(cycles=self.cycles, bottom_iters_total=self.bottom_iters_total,
                    singular=self.singular, levels=self.levels, rhs_norm_inf=self.rhs_norm_inf,
                    res_norm_inf=self.res_norm_inf, rhs_mean_removed=self.rhs_mean_removed,
                    res_history=list(self.res_history[:min(self.cycles, 128)]),
                    ms_setup_kernels=self.ms_setup_kernels, ms_vcycles=self.ms_vcycles,
                    ms_correct=self.ms_correct, gpu_launches=self.gpu_launches,
                    ms_smooth0=self.ms_smooth0, smooth0_launches=self.smooth0_launches,
                    smooth0_timed=self.smooth0_timed, smooth0_sweeps_timed=self.smooth0_sweeps_timed)


_lib = None
_VP = C.c_void_p


def lib():
    """Load the CUDA library.  Fails loudly if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_1910_12979_b200.build` "
                               "(the MAC projection has no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.maestro_mac_default_desc.argtypes = [C.POINTER(Desc)]
        L.maestro_mac_default_desc.restype = None
        L.maestro_mac_setup.argtypes = [C.POINTER(Desc), _VP, C.c_size_t, C.POINTER(C.c_size_t), C.POINTER(_VP)]
        proj = [_VP, _VP, _VP, _VP, _VP, _VP, _VP, _VP, _VP, C.POINTER(Stats), _VP]
        L.maestro_mac_project.argtypes = proj
        L.maestro_mac_project_host.argtypes = proj
        L.maestro_mac_project_host_seq.argtypes = [_VP, C.c_int, _VP, _VP, _VP, _VP, _VP, _VP, _VP, _VP, _VP, _VP, _VP,
                                                   C.POINTER(Stats), _VP]
        L.maestro_mac_free.argtypes = [_VP]
        L.maestro_mac_num_levels.argtypes = [_VP]
        L.maestro_mac_level_dims.argtypes = [_VP, C.c_int, C.POINTER(C.c_int * 3), C.POINTER(C.c_double * 3)]
        L.maestro_mac_level_get.argtypes = [_VP, C.c_int, C.c_int, _VP, _VP]
        L.maestro_mac_level_set.argtypes = [_VP, C.c_int, C.c_int, _VP, _VP]
        L.maestro_mac_step_coefficients.argtypes = [_VP, _VP, _VP, _VP, _VP]
        L.maestro_mac_step_rhs.argtypes = [_VP, _VP, _VP, _VP, _VP, _VP, C.POINTER(C.c_double), C.POINTER(C.c_double), _VP]
        L.maestro_mac_step_smooth.argtypes = [_VP, C.c_int, C.c_int, _VP]
        L.maestro_mac_step_residual_restrict.argtypes = [_VP, C.c_int, _VP]
        L.maestro_mac_step_prolong.argtypes = [_VP, C.c_int, _VP]
        L.maestro_mac_step_bottom.argtypes = [_VP, _VP]
        L.maestro_mac_step_vcycle.argtypes = [_VP, _VP]
        L.maestro_mac_step_residual_norm.argtypes = [_VP, C.c_int, C.POINTER(C.c_double), _VP]
        L.maestro_mac_step_correct.argtypes = [_VP, _VP, _VP, _VP, _VP, _VP, _VP]
        L.maestro_mac_base_state.argtypes = [C.c_int, _VP, _VP, _VP, _VP, _VP, _VP, _VP]
        L.maestro_mac_set_dpdt_term.argtypes = [_VP, _VP]
        L.maestro_mac_lateral_average.argtypes = [_VP, _VP, _VP, _VP]
        L.maestro_mac_lateral_average_noalloc.argtypes = [C.POINTER(Desc), _VP, _VP, _VP]
        L.maestro_mac_status.argtypes = [_VP, C.POINTER(Stats), _VP]
        L.maestro_mac_level_plan.argtypes = [_VP, C.c_int, C.POINTER(C.c_int * 8)]
        L.maestro_mac_plan_query.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int * 8)]
        L.maestro_mac_nodal_project.argtypes = proj
        L.maestro_mac_nodal_level_get.argtypes = [_VP, C.c_int, C.c_int, _VP, _VP]
        L.maestro_mac_nodal_level_set.argtypes = [_VP, C.c_int, C.c_int, _VP, _VP]
        L.maestro_mac_nodal_step_sigma.argtypes = [_VP, _VP, _VP, _VP, _VP]
        L.maestro_mac_nodal_step_rhs.argtypes = [_VP, _VP, _VP, _VP, _VP, C.POINTER(C.c_double), C.POINTER(C.c_double), _VP]
        L.maestro_mac_nodal_step_smooth.argtypes = [_VP, C.c_int, C.c_int, _VP]
        L.maestro_mac_nodal_step_residual_restrict.argtypes = [_VP, C.c_int, _VP]
        L.maestro_mac_nodal_step_prolong.argtypes = [_VP, C.c_int, _VP]
        L.maestro_mac_nodal_step_bottom.argtypes = [_VP, _VP]
        L.maestro_mac_nodal_step_vcycle.argtypes = [_VP, _VP]
        L.maestro_mac_nodal_step_residual_norm.argtypes = [_VP, C.c_int, C.POINTER(C.c_double), _VP]
        L.maestro_mac_nodal_step_correct.argtypes = [_VP, _VP, _VP, _VP, _VP, _VP, _VP]
        for name in EXPORTS:
            if name != "maestro_mac_default_desc":
                getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


class MacError(RuntimeError):
    def __init__(self, code, where):
        super().__init__(f"{where} failed with code {code}")
        self.code = code


def make_desc(n, dx, bc_lo, bc_hi, geometry=PLANAR, nr=None, dr=None, center=(0.0, 0.0, 0.0),
              nu_pre=2, nu_post=2, max_cycles=100, rel_tol=1e-10, coarsest_n=4,
              bottom_max_iter=100, bottom_rel_tol=1e-8, prolongation=0, host_staging=0,
              smoother=0, stop_test=0, rho_mean=0, timing=0, nodal=0) -> Desc:
    d = Desc()
    lib().maestro_mac_default_desc(C.byref(d))
    d.nx, d.ny, d.nz = (int(x) for x in n)
    for a in range(3):
        d.dx[a], d.bc_lo[a], d.bc_hi[a], d.center[a] = float(dx[a]), int(bc_lo[a]), int(bc_hi[a]), float(center[a])
    d.geometry = int(geometry)
    d.nr = int(nr if nr is not None else n[2])
    d.dr = float(dr if dr is not None else dx[2])
    d.nu_pre, d.nu_post, d.max_cycles, d.rel_tol = int(nu_pre), int(nu_post), int(max_cycles), float(rel_tol)
    d.coarsest_n, d.bottom_max_iter, d.bottom_rel_tol = int(coarsest_n), int(bottom_max_iter), float(bottom_rel_tol)
    d.prolongation, d.host_staging, d.smoother = int(prolongation), int(host_staging), int(smoother)
    d.stop_test = int(stop_test)
    d.rho_mean = int(rho_mean)
    d.timing = int(timing)
    d.nodal = int(nodal)
    return d


def desc_from_workload(wl, **over) -> Desc:
    kw = dict(n=wl.n, dx=wl.dx, bc_lo=wl.bc_lo, bc_hi=wl.bc_hi, geometry=wl.geometry, nr=wl.nr,
              dr=wl.dr, center=wl.center, nu_pre=wl.nu_pre, nu_post=wl.nu_post,
              max_cycles=wl.max_cycles, rel_tol=wl.rel_tol, rho_mean=wl.meta.get("rho_mean", 0))
    kw.update(over)
    return make_desc(**kw)


def plan_query(which, nx, ny, nz, sms):
    """Launch plan of the two-sweep smoother (which = 0) or the nodal march (1) as pure host arithmetic (no GPU needed)."""
    info = (C.c_int * 8)()
    rc = lib().maestro_mac_plan_query(which, nx, ny, nz, sms, C.byref(info))
    if rc != OK:
        raise MacError(rc, "plan_query")
    return dict(tiles_x=info[0], tiles=info[1], nfull=info[2], nsplit=info[3], zchunk=info[4], ncta=info[5])


NOALLOC_MAX_NR = 2048          # MAESTRO_MAC_NOALLOC_MAX_NR


def lateral_average_noalloc(desc: Desc, rho, out):
    """rho0 = lateral average of rho into the caller's tensor `out` [nr] (maestro_mac_lateral_average_noalloc: no handle,
    no workspace, no device allocation; scratch is a static device array for nr <= NOALLOC_MAX_NR).  Returns the status."""
    return lib().maestro_mac_lateral_average_noalloc(C.byref(desc), _ptr(rho), _ptr(out), _stream())


def workspace_bytes(desc: Desc) -> int:
    need = C.c_size_t(0)
    out = _VP()
    rc = lib().maestro_mac_setup(C.byref(desc), None, 0, C.byref(need), C.byref(out))
    if rc != ERR_WORKSPACE:
        raise MacError(rc, "maestro_mac_setup(size query)")
    return int(need.value)


def _ptr(t):
    """Device (or pinned host) pointer of a contiguous float64 torch tensor, or NULL."""
    if t is None:
        return None
    import torch
    assert isinstance(t, torch.Tensor) and t.dtype == torch.float64 and t.is_contiguous()
    return _VP(t.data_ptr())


def _stream():
    import torch
    return _VP(torch.cuda.current_stream().cuda_stream)


class MacProjector:
    """Owns a handle and its workspace tensor (device memory allocated through PyTorch)."""

    def __init__(self, desc: Desc, device="cuda:0"):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("MacProjector needs a CUDA device (no CPU fallback)")
        self.desc = desc
        self.device = torch.device(device)
        nbytes = workspace_bytes(desc)
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = self.workspace.data_ptr()
        aligned = (base + 255) // 256 * 256
        self._h = _VP()
        need = C.c_size_t(0)
        rc = lib().maestro_mac_setup(C.byref(desc), _VP(aligned), nbytes, C.byref(need), C.byref(self._h))
        if rc != OK:
            raise MacError(rc, "maestro_mac_setup")
        self.workspace_bytes = nbytes

    def close(self):
        if getattr(self, "_h", None):
            lib().maestro_mac_free(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the hot path -----------------------------------------------------------------------
    def project(self, beta0, rho0, rho, u, v, w, S=None, phi=None, want_stats=True):
        """Device tensors; u, v, w corrected in place.  Returns (status, stats dict | None)."""
        st = Stats()
        rc = lib().maestro_mac_project(self._h, _ptr(beta0), _ptr(rho0), _ptr(rho), _ptr(u), _ptr(v),
                                       _ptr(w), _ptr(S), _ptr(phi), C.byref(st) if want_stats else None,
                                       _stream())
        return rc, (st.as_dict() if want_stats else None)

    def status(self, want_stats=True):
        """Completes an asynchronous project call (rel_tol == 0, want_stats=False).  Returns (status, stats | None)."""
        st = Stats()
        rc = lib().maestro_mac_status(self._h, C.byref(st) if want_stats else None, _stream())
        return rc, (st.as_dict() if want_stats else None)

    def project_host(self, beta0, rho0, rho, u, v, w, S=None, phi=None, want_stats=True):
        """Host (pinned) tensors; includes the host<->device copies."""
        st = Stats()
        rc = lib().maestro_mac_project_host(self._h, _ptr(beta0), _ptr(rho0), _ptr(rho), _ptr(u),
                                            _ptr(v), _ptr(w), _ptr(S), _ptr(phi),
                                            C.byref(st) if want_stats else None, _stream())
        return rc, (st.as_dict() if want_stats else None)

    def project_host_seq(self, beta0, rho0, rho, S, u_in, v_in, w_in, u_out, v_out, w_out, phi_out=None, want_stats=True):
        """len(u_in) consecutive projections with host (pinned) tensors, transfers overlapped with the neighbouring
        steps (maestro_mac_project_host_seq; needs host_staging=2).  u_in ... phi_out are lists of host tensors."""
        n = len(u_in)
        def arr(ts):
            return (C.c_void_p * n)(*[_ptr(t) for t in ts]) if ts is not None else None
        st = (Stats * n)() if want_stats else None
        rc = lib().maestro_mac_project_host_seq(self._h, n, _ptr(beta0), _ptr(rho0), _ptr(rho), _ptr(S), arr(u_in), arr(v_in),
                                                arr(w_in), arr(u_out), arr(v_out), arr(w_out), arr(phi_out), st, _stream())
        return rc, ([x.as_dict() for x in st] if want_stats else None)

    # ---- step API ---------------------------------------------------------------------------
    def _ck(self, rc, where):
        if rc != OK:
            raise MacError(rc, where)

    @property
    def num_levels(self):
        return lib().maestro_mac_num_levels(self._h)

    def level_dims(self, level):
        n, h = (C.c_int * 3)(), (C.c_double * 3)()
        self._ck(lib().maestro_mac_level_dims(self._h, level, C.byref(n), C.byref(h)), "level_dims")
        return tuple(n), tuple(h)

    KERNELS = ("color", "fused", "tma", "t2", "tail", "bottom", "cluster")

    def level_plan(self, level):
        """Launch plan of the smoother on a level (maestro_mac_level_plan)."""
        info = (C.c_int * 8)()
        self._ck(lib().maestro_mac_level_plan(self._h, level, C.byref(info)), "level_plan")
        return dict(kernel=self.KERNELS[info[0]], tiles=info[1], nfull=info[2], nsplit=info[3], zchunk=info[4],
                    ncta=info[5], gx=info[6], gy=info[7])

    def level_shape(self, level, which):
        (nx, ny, nz), _ = self.level_dims(level)
        return {ARR_PHI: (nz, ny, nx), ARR_RHS: (nz, ny, nx), ARR_BX: (nz, ny, nx + 1),
                ARR_BY: (nz, ny + 1, nx), ARR_BZ: (nz + 1, ny, nx)}[which]

    def level_get(self, level, which):
        import torch
        out = torch.empty(self.level_shape(level, which), dtype=torch.float64, device=self.device)
        self._ck(lib().maestro_mac_level_get(self._h, level, which, _ptr(out), _stream()), "level_get")
        return out

    def level_set(self, level, which, src):
        assert tuple(src.shape) == self.level_shape(level, which)
        self._ck(lib().maestro_mac_level_set(self._h, level, which, _ptr(src), _stream()), "level_set")

    def step_coefficients(self, beta0, rho0, rho):
        self._ck(lib().maestro_mac_step_coefficients(self._h, _ptr(beta0), _ptr(rho0), _ptr(rho), _stream()), "step_coefficients")

    def step_rhs(self, beta0, u, v, w, S=None):
        nrm, mean = C.c_double(0), C.c_double(0)
        self._ck(lib().maestro_mac_step_rhs(self._h, _ptr(beta0), _ptr(u), _ptr(v), _ptr(w), _ptr(S),
                                            C.byref(nrm), C.byref(mean), _stream()), "step_rhs")
        return nrm.value, mean.value

    def step_smooth(self, level, nsweeps=1):
        self._ck(lib().maestro_mac_step_smooth(self._h, level, nsweeps, _stream()), "step_smooth")

    def step_residual_restrict(self, level):
        self._ck(lib().maestro_mac_step_residual_restrict(self._h, level, _stream()), "step_residual_restrict")

    def step_prolong(self, level):
        self._ck(lib().maestro_mac_step_prolong(self._h, level, _stream()), "step_prolong")

    def step_bottom(self):
        self._ck(lib().maestro_mac_step_bottom(self._h, _stream()), "step_bottom")

    def step_vcycle(self):
        self._ck(lib().maestro_mac_step_vcycle(self._h, _stream()), "step_vcycle")

    def step_residual_norm(self, level=0):
        nrm = C.c_double(0)
        self._ck(lib().maestro_mac_step_residual_norm(self._h, level, C.byref(nrm), _stream()), "step_residual_norm")
        return nrm.value

    def lateral_average(self, rho):
        """rho0[nr] = lateral average of rho as a device tensor."""
        import torch
        out = torch.empty(self.desc.nr, dtype=torch.float64, device=rho.device)
        self._ck(lib().maestro_mac_lateral_average(self._h, _ptr(rho), _ptr(out), _stream()), "lateral_average")
        return out

    def set_dpdt_term(self, q):
        """Register (or clear, q = None) the profile (1/(Gamma1bar p0)) dp0/dt of PAPER.md:49 Eq. 6."""
        self._dpdt_keepalive = q
        self._ck(lib().maestro_mac_set_dpdt_term(self._h, _ptr(q)), "set_dpdt_term")

    # ---- nodal (end-of-step) projection: desc.nodal = 1 ----------------------------------------
    def nodal_project(self, beta0, rho0, rho, uc, vc, wc, S=None, phi=None, want_stats=True):
        """Device tensors; uc, vc, wc (CELL arrays) corrected in place; phi: node array or None."""
        st = Stats()
        rc = lib().maestro_mac_nodal_project(self._h, _ptr(beta0), _ptr(rho0), _ptr(rho), _ptr(uc), _ptr(vc), _ptr(wc),
                                             _ptr(S), _ptr(phi), C.byref(st) if want_stats else None, _stream())
        return rc, (st.as_dict() if want_stats else None)

    def nodal_shape(self, level, which):
        (nx, ny, nz), _ = self.level_dims(level)
        return (nz, ny, nx) if which == NODAL_SIGMA else (nz + 1, ny + 1, nx + 1)

    def nodal_get(self, level, which):
        import torch
        out = torch.empty(self.nodal_shape(level, which), dtype=torch.float64, device=self.device)
        self._ck(lib().maestro_mac_nodal_level_get(self._h, level, which, _ptr(out), _stream()), "nodal_level_get")
        return out

    def nodal_set(self, level, which, src):
        assert tuple(src.shape) == self.nodal_shape(level, which)
        self._ck(lib().maestro_mac_nodal_level_set(self._h, level, which, _ptr(src), _stream()), "nodal_level_set")

    def nodal_step_sigma(self, beta0, rho0, rho):
        self._ck(lib().maestro_mac_nodal_step_sigma(self._h, _ptr(beta0), _ptr(rho0), _ptr(rho), _stream()), "nodal_step_sigma")

    def nodal_step_rhs(self, uc, vc, wc, S=None):
        nrm, mean = C.c_double(0), C.c_double(0)
        self._ck(lib().maestro_mac_nodal_step_rhs(self._h, _ptr(uc), _ptr(vc), _ptr(wc), _ptr(S), C.byref(nrm), C.byref(mean),
                                                  _stream()), "nodal_step_rhs")
        return nrm.value, mean.value

    def nodal_step_smooth(self, level, nsweeps=1):
        self._ck(lib().maestro_mac_nodal_step_smooth(self._h, level, nsweeps, _stream()), "nodal_step_smooth")

    def nodal_step_residual_restrict(self, level):
        self._ck(lib().maestro_mac_nodal_step_residual_restrict(self._h, level, _stream()), "nodal_step_residual_restrict")

    def nodal_step_prolong(self, level):
        self._ck(lib().maestro_mac_nodal_step_prolong(self._h, level, _stream()), "nodal_step_prolong")

    def nodal_step_bottom(self):
        self._ck(lib().maestro_mac_nodal_step_bottom(self._h, _stream()), "nodal_step_bottom")

    def nodal_step_vcycle(self):
        self._ck(lib().maestro_mac_nodal_step_vcycle(self._h, _stream()), "nodal_step_vcycle")

    def nodal_step_residual_norm(self, level=0):
        nrm = C.c_double(0)
        self._ck(lib().maestro_mac_nodal_step_residual_norm(self._h, level, C.byref(nrm), _stream()), "nodal_step_residual_norm")
        return nrm.value

    def nodal_step_correct(self, rho0, rho, uc, vc, wc):
        self._ck(lib().maestro_mac_nodal_step_correct(self._h, _ptr(rho0), _ptr(rho), _ptr(uc), _ptr(vc), _ptr(wc), _stream()),
                 "nodal_step_correct")

    def step_correct(self, rho0, rho, u, v, w):
        self._ck(lib().maestro_mac_step_correct(self._h, _ptr(rho0), _ptr(rho), _ptr(u), _ptr(v), _ptr(w), _stream()), "step_correct")


def base_state(rho0, p0, gamma1bar, dp0dt=None):
    """maestro_mac_base_state: (beta0, dpdt_term or None) as device tensors from device profiles (Eq. 5,
    PAPER.md:49 Eq. 6)."""
    import torch
    beta0 = torch.empty_like(rho0)
    q = torch.empty_like(rho0) if dp0dt is not None else None
    rc = lib().maestro_mac_base_state(int(rho0.numel()), _ptr(rho0), _ptr(p0), _ptr(gamma1bar), _ptr(dp0dt), _ptr(beta0),
                                      _ptr(q), _stream())
    if rc != 0:
        raise MacError(rc, "maestro_mac_base_state")
    return beta0, q


def to_device(wl, device="cuda:0"):
    """Workload (numpy) -> dict of device tensors."""
    import torch
    dev = torch.device(device)
    f = lambda a: None if a is None else torch.from_numpy(a).to(dev)
    return dict(beta0=f(wl.beta0), rho0=f(wl.rho0), rho=f(wl.rho), u=f(wl.u), v=f(wl.v), w=f(wl.w), S=f(wl.S))
