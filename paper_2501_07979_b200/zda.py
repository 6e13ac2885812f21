"""Thin ctypes binding of libzda (include/zda.h): argument marshalling only.

Every step of the hot path (grid tables, density map, H/E updates with CPML, source, running DFT,
adjoint-source build, gradient) runs inside ``libzda.so``.  PyTorch is used for device memory
(the workspace and the output tensors) and for the stream.  There is no CPU fallback: if the
shared library is missing or CUDA is unavailable, the calls raise.

The module-level ``zda_*`` functions mirror the C ABI one to one (same names, same argument
order; pointers are ``int`` addresses or objects with ``data_ptr()``).  ``Zone`` is a convenience
wrapper that takes a ``workloads.ZoneInputs`` and converts its (r, phi, z)-ordered NumPy arrays
to the ABI's [k][j][i] layout and back.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libzda.so")

ZDA_OK, ZDA_E_BADARG, ZDA_E_CFL, ZDA_E_NOMEM, ZDA_E_CUDA, ZDA_E_STATE, ZDA_E_NAN = 0, -1, -2, -3, -4, -5, -6
ZDA_ER, ZDA_EPHI, ZDA_EZ, ZDA_HR, ZDA_HPHI, ZDA_HZ = range(6)
ZDA_FWD, ZDA_ADJ = 0, 1
ZDA_DESIGN, ZDA_MONITOR = 0, 1
ZDA_OBJ_MONITOR_ENERGY, ZDA_OBJ_FOCAL_INTENSITY = 0, 1
ZDA_KERNEL_AUTO, ZDA_KERNEL_SPLIT, ZDA_KERNEL_FUSED, ZDA_KERNEL_FUSED2, ZDA_KERNEL_PERSIST = 0, 1, 2, 3, 4
ZDA_OPT_KERNEL, ZDA_OPT_ADJ_MONITOR_DFT = 0, 1
ZDA_OPT_FUSED_TJ, ZDA_OPT_FUSED_CHUNK, ZDA_OPT_FUSED_CLUSTER, ZDA_OPT_DFT_PERIOD, ZDA_OPT_SPLIT_GRAPH, ZDA_OPT_CHECK_EVERY = 2, 3, 4, 5, 6, 7
ZDA_MAX_FREQ, ZDA_MAX_TERMS = 8, 16

EXPORTS = (
    "zda_last_error", "zda_zone_workspace_bytes", "zda_zone_create", "zda_zone_destroy", "zda_set_option",
    "zda_set_design_eps", "zda_set_eps_volume", "zda_set_density", "zda_set_density_conic", "zda_set_source", "zda_set_focal_weights", "zda_build_focal_weights", "zda_get_focal_sums", "zda_run_forward", "zda_build_adjoint_source",
    "zda_run_adjoint", "zda_pair_run_forward", "zda_pair_run_adjoint", "zda_get_dft", "zda_get_field", "zda_gradient", "zda_density_vjp_static", "zda_check_finite", "zda_schedule_bytes", "zda_launch_count",
    "zda_kernel_name", "zda_lens_gradient", "zda_lens_focal_gradient",
)


class ZdaError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"libzda error {code}: {text}")
        self.code = code


class zda_zone_desc(ctypes.Structure):
    _fields_ = [
        ("Nr", ctypes.c_int), ("Nphi", ctypes.c_int), ("Nz", ctypes.c_int),
        ("dr", ctypes.c_double), ("dphi", ctypes.c_double), ("dz", ctypes.c_double),
        ("r_in", ctypes.c_double), ("dt", ctypes.c_double),
        ("n_fold", ctypes.c_int),
        ("phase_re", ctypes.c_double), ("phase_im", ctypes.c_double),
        ("complex_fields", ctypes.c_int), ("has_axis", ctypes.c_int),
        ("npml_r_lo", ctypes.c_int), ("npml_r_hi", ctypes.c_int),
        ("npml_z_lo", ctypes.c_int), ("npml_z_hi", ctypes.c_int),
        ("cpml_p", ctypes.c_double), ("cpml_sigma_max_r", ctypes.c_double),
        ("cpml_sigma_max_z", ctypes.c_double), ("cpml_kappa_max", ctypes.c_double),
        ("cpml_alpha_max", ctypes.c_double),
        ("design_i0", ctypes.c_int), ("design_i1", ctypes.c_int),
        ("design_k0", ctypes.c_int), ("design_k1", ctypes.c_int),
        ("monitor_k", ctypes.c_int), ("source_k", ctypes.c_int),
        ("n_freq", ctypes.c_int), ("omega", ctypes.POINTER(ctypes.c_double)),
        ("precision", ctypes.c_int),
        ("rpml_exact", ctypes.c_int),
        ("eps_volume", ctypes.c_int),
    ]


_lib = None


def load_library(build_if_missing: bool = True) -> ctypes.CDLL:
    """Loads ``libzda.so`` from the package directory (building it with nvcc when it is missing or
    stale and nvcc is present).  Raises if it cannot be had: there is no fallback path."""
    global _lib
    if _lib is not None:
        return _lib
    if build_if_missing:
        from . import _build
        if _build.needs_build():
            try:
                _build.build()
            except Exception as e:  # stale but present is still an error: never run old kernels silently
                raise RuntimeError(f"libzda.so is missing or stale and could not be built: {e}") from e
    if not os.path.exists(_LIB_PATH):
        raise RuntimeError(f"{_LIB_PATH} not found: build it with `python -m paper_2501_07979_b200._build`")
    lib = ctypes.CDLL(_LIB_PATH)
    vp, ci, cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
    dp = ctypes.POINTER(ctypes.c_double)
    descp = ctypes.POINTER(zda_zone_desc)
    sig = {
        "zda_last_error": (ctypes.c_char_p, []),
        "zda_zone_workspace_bytes": (ctypes.c_size_t, [descp, ci]),
        "zda_zone_create": (ci, [descp, dp, ci, vp, ctypes.c_size_t, vp, ctypes.POINTER(vp)]),
        "zda_zone_destroy": (ci, [vp]),
        "zda_set_option": (ci, [vp, ci, ci]),
        "zda_set_design_eps": (ci, [vp, vp, ci]),
        "zda_set_eps_volume": (ci, [vp, vp, ci]),
        "zda_set_density": (ci, [vp, vp, ci, cd, cd, cd, cd, cd]),
        "zda_set_density_conic": (ci, [vp, vp, ci, cd, cd, cd, cd, cd]),
        "zda_set_source": (ci, [vp, ci, vp, vp, ci, dp, ci]),
        "zda_set_focal_weights": (ci, [vp, vp, dp, ci]),
        "zda_build_focal_weights": (ci, [vp, cd, dp]),
        "zda_get_focal_sums": (ci, [vp, dp]),
        "zda_run_forward": (ci, [vp, ci]),
        "zda_build_adjoint_source": (ci, [vp, ci, cd, cd, ci, dp]),
        "zda_run_adjoint": (ci, [vp, ci]),
        "zda_pair_run_forward": (ci, [vp, vp, ci]),
        "zda_pair_run_adjoint": (ci, [vp, vp, ci]),
        "zda_get_dft": (ci, [vp, ci, ci, ci, ci, vp, ci]),
        "zda_get_field": (ci, [vp, ci, vp, ci]),
        "zda_gradient": (ci, [vp, vp, vp, vp, ci]),
        "zda_check_finite": (ci, [vp]),
        "zda_density_vjp_static": (ci, [ci, ci, ci, vp, vp, vp, cd, cd, cd, cd, cd, vp]),
        "zda_schedule_bytes": (ci, [vp, ci, dp]),
        "zda_launch_count": (ctypes.c_longlong, [vp]),
        "zda_kernel_name": (ctypes.c_char_p, [vp]),
        "zda_lens_gradient": (ci, [ctypes.POINTER(vp), ci, ctypes.POINTER(ci), ctypes.POINTER(ci), dp, dp, dp,
                                   ctypes.POINTER(vp), ctypes.POINTER(vp)]),
        "zda_lens_focal_gradient": (ci, [ctypes.POINTER(vp), ci, ctypes.POINTER(ci), ctypes.POINTER(ci), dp, dp, dp, dp, dp,
                                         ctypes.POINTER(vp), ctypes.POINTER(vp)]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)   # AttributeError if the symbol is not exported
        fn.restype, fn.argtypes = res, args
    _lib = lib
    return lib


def _check(rc: int) -> int:
    if rc != ZDA_OK:
        raise ZdaError(rc, load_library().zda_last_error().decode(errors="replace"))
    return rc


def _addr(x) -> Optional[int]:
    if x is None:
        return None
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    if isinstance(x, np.ndarray):
        return x.ctypes.data
    return int(x)


def _dptr(a: Optional[np.ndarray]):
    if a is None:
        return None
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


# ------------------------------------------------------------------------------------------------
# the C ABI, one Python function per entry point (same names)
# ------------------------------------------------------------------------------------------------
def zda_last_error() -> str:
    return load_library().zda_last_error().decode(errors="replace")


def zda_zone_workspace_bytes(desc: zda_zone_desc, max_steps: int) -> int:
    n = load_library().zda_zone_workspace_bytes(ctypes.byref(desc), max_steps)
    if n == 0:
        raise ZdaError(ZDA_E_BADARG, zda_last_error())
    return n


def zda_zone_create(desc: zda_zone_desc, eps_bg_z: Optional[np.ndarray], max_steps: int, workspace, nbytes: int,
                    stream: int) -> int:
    """Returns the opaque zone handle (an address)."""
    out = ctypes.c_void_p()
    bg = None if eps_bg_z is None else np.ascontiguousarray(eps_bg_z, dtype=np.float64)
    _check(load_library().zda_zone_create(ctypes.byref(desc), _dptr(bg), max_steps, _addr(workspace), nbytes,
                                          stream or None, ctypes.byref(out)))
    return out.value


def zda_zone_destroy(zone: int) -> None:
    _check(load_library().zda_zone_destroy(zone))


def zda_set_option(zone: int, option: int, value: int) -> None:
    _check(load_library().zda_set_option(zone, option, value))


def zda_set_design_eps(zone: int, eps_design, on_host: int) -> None:
    _check(load_library().zda_set_design_eps(zone, _addr(eps_design), on_host))


def zda_set_eps_volume(zone: int, eps, on_host: int) -> None:
    _check(load_library().zda_set_eps_volume(zone, _addr(eps), on_host))


def zda_set_density(zone: int, rho2d, on_host: int, eps0: float, eps_h: float, filt_sigma: float, beta: float,
                    eta: float) -> None:
    _check(load_library().zda_set_density(zone, _addr(rho2d), on_host, eps0, eps_h, filt_sigma, beta, eta))


def zda_set_density_conic(zone: int, rho2d, on_host: int, eps0: float, eps_h: float, radius: float, beta: float,
                          eta: float) -> None:
    _check(load_library().zda_set_density_conic(zone, _addr(rho2d), on_host, eps0, eps_h, radius, beta, eta))


def zda_set_source(zone: int, n_terms: int, A_r, A_phi, on_host: int, s_table: np.ndarray, Nt: int) -> None:
    tab = np.ascontiguousarray(s_table, dtype=np.float64)
    _check(load_library().zda_set_source(zone, n_terms, _addr(A_r), _addr(A_phi), on_host, _dptr(tab), Nt))


def zda_set_focal_weights(zone: int, g, u: Optional[np.ndarray], on_host: int) -> None:
    u = None if u is None else np.ascontiguousarray(u, dtype=np.float64)
    _check(load_library().zda_set_focal_weights(zone, _addr(g), _dptr(u), on_host))


def zda_build_focal_weights(zone: int, focal_dz: float, u: Optional[np.ndarray]) -> None:
    u = None if u is None else np.ascontiguousarray(u, dtype=np.float64)
    _check(load_library().zda_build_focal_weights(zone, focal_dz, _dptr(u)))


def zda_get_focal_sums(zone: int, n_freq: int) -> np.ndarray:
    S = np.zeros(2 * n_freq, dtype=np.float64)
    _check(load_library().zda_get_focal_sums(zone, _dptr(S)))
    return S[0::2] + 1j * S[1::2]


def zda_run_forward(zone: int, n_steps: int) -> None:
    _check(load_library().zda_run_forward(zone, n_steps))


def zda_build_adjoint_source(zone: int, objective: int, t0: float, sigma_t: float, n_steps: int,
                             want_F: bool = True) -> Optional[float]:
    F = ctypes.c_double(0.0)
    _check(load_library().zda_build_adjoint_source(zone, objective, t0, sigma_t, n_steps,
                                                   ctypes.byref(F) if want_F else None))
    return F.value if want_F else None


def zda_run_adjoint(zone: int, n_steps: int) -> None:
    _check(load_library().zda_run_adjoint(zone, n_steps))


def zda_pair_run_forward(a: int, b: int, n_steps: int) -> None:
    _check(load_library().zda_pair_run_forward(a, b, n_steps))


def zda_pair_run_adjoint(a: int, b: int, n_steps: int) -> None:
    _check(load_library().zda_pair_run_adjoint(a, b, n_steps))


def zda_get_dft(zone: int, which: int, region: int, comp: int, freq: int, out, on_host: int) -> None:
    _check(load_library().zda_get_dft(zone, which, region, comp, freq, _addr(out), on_host))


def zda_get_field(zone: int, comp: int, out, on_host: int) -> None:
    _check(load_library().zda_get_field(zone, comp, _addr(out), on_host))


def zda_gradient(zone: int, dF_deps, dF_deps_zsum, dF_drho, on_host: int) -> None:
    _check(load_library().zda_gradient(zone, _addr(dF_deps), _addr(dF_deps_zsum), _addr(dF_drho), on_host))


def zda_density_vjp_static(precision: int, Nr_d: int, Nphi: int, rho2d, dF_deps_zsum, dF_drho, eps0: float, eps_h: float,
                           filt_sigma: float, beta: float, eta: float, stream=None) -> None:
    """Device tensors / addresses in, nothing allocated (include/zda.h): the scratch is the library's static array."""
    _check(load_library().zda_density_vjp_static(precision, Nr_d, Nphi, _addr(rho2d), _addr(dF_deps_zsum), _addr(dF_drho),
                                                 eps0, eps_h, filt_sigma, beta, eta,
                                                 None if stream is None else int(getattr(stream, "cuda_stream", stream))))


def zda_check_finite(zone: int) -> None:
    _check(load_library().zda_check_finite(zone))


def zda_schedule_bytes(zone: int, which: int) -> dict:
    out = np.zeros(5, dtype=np.float64)
    _check(load_library().zda_schedule_bytes(zone, which, _dptr(out)))
    return dict(zip(("fields", "psi", "eps", "dft", "halo_if_no_l2_reuse"), out.tolist()))


def zda_launch_count(zone: int) -> int:
    return int(load_library().zda_launch_count(zone))


def zda_kernel_name(zone: int) -> str:
    return load_library().zda_kernel_name(zone).decode()


def zda_lens_gradient(zones: Sequence[int], n_steps_fwd: Sequence[int], n_steps_adj: Sequence[int],
                      adj_t0: Sequence[float], adj_sigma_t: Sequence[float], dF_deps_zsum=None, dF_drho=None):
    """Returns the per-zone objective values F (host)."""
    n = len(zones)
    vp = ctypes.c_void_p
    zs = (vp * n)(*zones)
    nf = (ctypes.c_int * n)(*n_steps_fwd)
    na = (ctypes.c_int * n)(*n_steps_adj)
    t0 = np.ascontiguousarray(adj_t0, dtype=np.float64)
    sg = np.ascontiguousarray(adj_sigma_t, dtype=np.float64)
    F = np.zeros(n, dtype=np.float64)
    gz = (vp * n)(*[_addr(x) for x in dF_deps_zsum]) if dF_deps_zsum is not None else None
    gr = (vp * n)(*[_addr(x) for x in dF_drho]) if dF_drho is not None else None
    _check(load_library().zda_lens_gradient(zs, n, nf, na, _dptr(t0), _dptr(sg), _dptr(F), gz, gr))
    return F


def zda_lens_focal_gradient(zones: Sequence[int], n_steps_fwd: Sequence[int], n_steps_adj: Sequence[int],
                            adj_t0: Sequence[float], adj_sigma_t: Sequence[float], u=None, n_freq: int = ZDA_MAX_FREQ,
                            dF_deps_zsum=None, dF_drho=None):
    """Returns (F, S_total[:n_freq]) of the coherent lens objective (host)."""
    n = len(zones)
    vp = ctypes.c_void_p
    zs = (vp * n)(*zones)
    nf = (ctypes.c_int * n)(*n_steps_fwd)
    na = (ctypes.c_int * n)(*n_steps_adj)
    t0 = np.ascontiguousarray(adj_t0, dtype=np.float64)
    sg = np.ascontiguousarray(adj_sigma_t, dtype=np.float64)
    uu = None if u is None else np.ascontiguousarray(u, dtype=np.float64)
    F = np.zeros(1, dtype=np.float64)
    S = np.zeros(2 * ZDA_MAX_FREQ, dtype=np.float64)
    gz = (vp * n)(*[_addr(x) for x in dF_deps_zsum]) if dF_deps_zsum is not None else None
    gr = (vp * n)(*[_addr(x) for x in dF_drho]) if dF_drho is not None else None
    _check(load_library().zda_lens_focal_gradient(zs, n, nf, na, _dptr(t0), _dptr(sg), _dptr(uu), _dptr(F), _dptr(S), gz, gr))
    return float(F[0]), (S[0::2] + 1j * S[1::2])[:n_freq]


# ------------------------------------------------------------------------------------------------
# convenience wrapper over a workloads.ZoneInputs (layout conversion + buffer ownership only)
# ------------------------------------------------------------------------------------------------
def desc_from_inputs(inp, precision: int = 32):
    """zda_zone_desc for a ``workloads.ZoneInputs``; returns (desc, omega_array_to_keep_alive)."""
    omega = np.ascontiguousarray(inp.omega, dtype=np.float64)
    ph = complex(inp.phase)
    d = zda_zone_desc(
        Nr=inp.Nr, Nphi=inp.Nphi, Nz=inp.Nz, dr=inp.dr, dphi=inp.dphi, dz=inp.dz, r_in=inp.r_in, dt=inp.dt,
        n_fold=inp.n_fold, phase_re=ph.real, phase_im=ph.imag, complex_fields=int(bool(inp.complex_fields)),
        has_axis=int(bool(inp.has_axis)), npml_r_lo=inp.npml_r_lo, npml_r_hi=inp.npml_r_hi,
        npml_z_lo=inp.npml_z_lo, npml_z_hi=inp.npml_z_hi, cpml_p=inp.cpml_p,
        cpml_sigma_max_r=inp.cpml_sigma_max_r, cpml_sigma_max_z=inp.cpml_sigma_max_z,
        cpml_kappa_max=inp.cpml_kappa_max, cpml_alpha_max=inp.cpml_alpha_max,
        design_i0=inp.design_i0, design_i1=inp.design_i1, design_k0=inp.design_k0, design_k1=inp.design_k1,
        monitor_k=inp.monitor_k, source_k=inp.source_k, n_freq=len(omega), omega=_dptr(omega),
        precision=precision, rpml_exact=int(getattr(inp, "rpml_exact", 0)), eps_volume=int(getattr(inp, "eps_volume", None) is not None))
    return d, omega


def table_to_abi(table: np.ndarray, complex_fields: bool) -> np.ndarray:
    """(n_terms, Nt) real or complex -> host doubles, interleaved (re, im) when complex."""
    t = np.asarray(table)
    if complex_fields:
        t = np.ascontiguousarray(t, dtype=np.complex128)
        return t.view(np.float64).reshape(t.shape[0], -1)
    return np.ascontiguousarray(t.real if np.iscomplexobj(t) else t, dtype=np.float64)


class Zone:
    """One zone on the current CUDA device.  Owns the workspace tensor and the library handle."""

    def __init__(self, inp, precision: int = 32, max_steps: Optional[int] = None, stream=None, kernel: int = ZDA_KERNEL_AUTO,
                 load_inputs: bool = True, workspace=None, options=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("libzda needs a CUDA device; there is no CPU path")
        self.torch = torch
        self.inp = inp
        self.precision = precision
        self.rdtype = np.float32 if precision == 32 else np.float64
        self.cdtype = np.complex64 if precision == 32 else np.complex128
        self.fdtype = self.cdtype if inp.complex_fields else self.rdtype
        self.max_steps = int(max_steps or max(inp.n_steps, inp.n_steps_adjoint, 1))
        self.desc, self._omega = desc_from_inputs(inp, precision)
        self.stream = stream if stream is not None else torch.cuda.current_stream()
        self.nbytes = zda_zone_workspace_bytes(self.desc, self.max_steps)
        if workspace is not None:        # a caller-owned buffer shared by zones that are solved one after the other
            if workspace.numel() * workspace.element_size() < self.nbytes:
                raise ValueError("shared workspace too small for this zone")
            self.workspace = workspace
        else:
            self.workspace = torch.empty(self.nbytes, dtype=torch.uint8, device="cuda")
        self.handle = zda_zone_create(self.desc, inp.eps_bg_z, self.max_steps, self.workspace, self.nbytes,
                                      self.stream.cuda_stream)
        self.objective = ZDA_OBJ_MONITOR_ENERGY
        if kernel != ZDA_KERNEL_AUTO:
            zda_set_option(self.handle, ZDA_OPT_KERNEL, kernel)
        for opt, val in (options or {}).items():
            zda_set_option(self.handle, opt, val)
        if load_inputs:
            self.load_inputs()

    # -- inputs -------------------------------------------------------------------------------
    def host_inputs(self):
        """The inputs in ABI layout as host arrays: dict with eps_design | rho, A_r, A_phi, table."""
        inp = self.inp
        out = {}
        if getattr(inp, "eps_volume", None) is not None:
            out["eps_volume"] = np.ascontiguousarray(np.asarray(inp.eps_volume).transpose(2, 1, 0), dtype=self.rdtype)  # [k][j][i]
        if inp.density is not None:
            out["rho"] = np.ascontiguousarray(np.asarray(inp.density.rho).T, dtype=self.rdtype)          # [j][id]
        elif inp.eps_design is not None:
            out["eps_design"] = np.ascontiguousarray(np.asarray(inp.eps_design).transpose(2, 1, 0), dtype=self.rdtype)
        if inp.src_A_r is not None:
            out["A_r"] = np.ascontiguousarray(np.asarray(inp.src_A_r).transpose(0, 2, 1), dtype=self.fdtype)  # [q][j][i]
            out["A_phi"] = np.ascontiguousarray(np.asarray(inp.src_A_phi).transpose(0, 2, 1), dtype=self.fdtype)
            out["table"] = table_to_abi(inp.src_table, inp.complex_fields)
        if getattr(inp, "focal_g", None) is not None:
            out["focal_g"] = np.ascontiguousarray(np.asarray(inp.focal_g).transpose(0, 1, 3, 2), dtype=self.cdtype)  # [f][c][j][i]
        return out

    def load_inputs(self, host=None, on_host: int = 1):
        """Hands the materials and the forward source to the library (host arrays, or device tensors
        with on_host=0)."""
        inp = self.inp
        host = self.host_inputs() if host is None else host
        if "eps_volume" in host:
            zda_set_eps_volume(self.handle, host["eps_volume"], on_host)
        if "rho" in host:
            dm = inp.density
            if dm.conic_radius > 0:
                zda_set_density_conic(self.handle, host["rho"], on_host, dm.eps0, dm.eps_h, dm.conic_radius, dm.beta, dm.eta)
            else:
                zda_set_density(self.handle, host["rho"], on_host, dm.eps0, dm.eps_h, dm.filt_sigma, dm.beta, dm.eta)
        elif "eps_design" in host:
            zda_set_design_eps(self.handle, host["eps_design"], on_host)
        if "A_r" in host:
            tab = host["table"]
            zda_set_source(self.handle, int(host["A_r"].shape[0]), host["A_r"], host["A_phi"], on_host, tab,
                           int(np.asarray(inp.src_table).shape[1]))
        if "focal_g" in host:
            zda_set_focal_weights(self.handle, host["focal_g"], inp.focal_u, on_host)
            self.objective = ZDA_OBJ_FOCAL_INTENSITY
        elif getattr(inp, "focal_dz", None) is not None:
            zda_build_focal_weights(self.handle, float(inp.focal_dz), inp.focal_u)
            self.objective = ZDA_OBJ_FOCAL_INTENSITY

    def set_design_eps(self, eps_design_rpz: np.ndarray):
        a = np.ascontiguousarray(np.asarray(eps_design_rpz).transpose(2, 1, 0), dtype=self.rdtype)
        zda_set_design_eps(self.handle, a, 1)

    # -- runs ---------------------------------------------------------------------------------
    def run_forward(self, n_steps=None):
        zda_run_forward(self.handle, int(self.inp.n_steps if n_steps is None else n_steps))

    def build_adjoint_source(self, n_steps=None, want_F=True):
        inp = self.inp
        n = int((inp.n_steps_adjoint or inp.n_steps) if n_steps is None else n_steps)
        return zda_build_adjoint_source(self.handle, self.objective, inp.adj_t0, inp.adj_sigma_t, n, want_F)

    def run_adjoint(self, n_steps=None):
        inp = self.inp
        zda_run_adjoint(self.handle, int((inp.n_steps_adjoint or inp.n_steps) if n_steps is None else n_steps))

    # -- outputs, converted back to (r, phi, z) order -------------------------------------------
    def get_field(self, comp: int) -> np.ndarray:
        inp = self.inp
        out = np.empty((inp.Nz, inp.Nphi, inp.Nr), dtype=self.fdtype)
        zda_get_field(self.handle, comp, out, 1)
        return out.transpose(2, 1, 0)

    def get_field_window(self, comp: int, i_lo, i_hi, j_lo, j_hi, k_lo, k_hi) -> np.ndarray:
        """A sub-block of a field component: the library writes the whole component into a device tensor
        (on_host = 0) and only the block crosses to the host.  For zones too big to copy whole."""
        torch, inp = self.torch, self.inp
        tdt = {np.float32: torch.float32, np.float64: torch.float64, np.complex64: torch.complex64,
               np.complex128: torch.complex128}[self.fdtype]
        if getattr(self, "_scratch_field", None) is None:
            self._scratch_field = torch.empty((inp.Nz, inp.Nphi, inp.Nr), dtype=tdt, device="cuda")
        zda_get_field(self.handle, comp, self._scratch_field, 0)
        self.stream.synchronize()
        return self._scratch_field[k_lo:k_hi, j_lo:j_hi, i_lo:i_hi].cpu().numpy().transpose(2, 1, 0)

    def get_dft_design_window(self, which: int, comp: int, freq: int, id_lo, id_hi, j_lo, j_hi, kd_lo, kd_hi) -> np.ndarray:
        """A sub-block (design-box indices) of one DFT accumulator, through a device tensor."""
        torch = self.torch
        nr, nphi, ld = self.inp.design_shape
        tdt = torch.complex64 if self.precision == 32 else torch.complex128
        if getattr(self, "_scratch_dft", None) is None:
            self._scratch_dft = torch.empty((ld, nphi, nr), dtype=tdt, device="cuda")
        zda_get_dft(self.handle, which, ZDA_DESIGN, comp, freq, self._scratch_dft, 0)
        self.stream.synchronize()
        return self._scratch_dft[kd_lo:kd_hi, j_lo:j_hi, id_lo:id_hi].cpu().numpy().transpose(2, 1, 0)

    def get_dft(self, which: int, region: int, comp: int, freq: int) -> np.ndarray:
        inp = self.inp
        if region == ZDA_DESIGN:
            nr, nphi, ld = inp.design_shape
            out = np.empty((ld, nphi, nr), dtype=self.cdtype)
            zda_get_dft(self.handle, which, region, comp, freq, out, 1)
            return out.transpose(2, 1, 0)
        out = np.empty((inp.Nphi, inp.Nr), dtype=self.cdtype)
        zda_get_dft(self.handle, which, region, comp, freq, out, 1)
        return out.T

    def dft(self, which: int, region: int) -> np.ndarray:
        """All frequencies and components: (F, 3, ...) like the oracle's accumulators."""
        F = self.inp.n_freq
        return np.stack([np.stack([self.get_dft(which, region, c, f) for c in range(3)]) for f in range(F)])

    def gradient(self, want_box=True, want_zsum=True, want_drho=False):
        nr, nphi, ld = self.inp.design_shape
        box = np.empty((ld, nphi, nr), dtype=self.rdtype) if want_box else None
        zs = np.empty((nphi, nr), dtype=self.rdtype) if want_zsum else None
        dr = np.empty((nphi, nr), dtype=self.rdtype) if want_drho else None
        zda_gradient(self.handle, box, zs, dr, 1)
        return (None if box is None else box.transpose(2, 1, 0),
                None if zs is None else zs.T,
                None if dr is None else dr.T)

    def check_finite(self):
        zda_check_finite(self.handle)

    @property
    def launch_count(self) -> int:
        return zda_launch_count(self.handle)

    @property
    def kernel_name(self) -> str:
        return zda_kernel_name(self.handle)

    def close(self):
        if getattr(self, "handle", None):
            self.torch.cuda.synchronize()
            zda_zone_destroy(self.handle)
            self.handle = None
            self.workspace = None
            self._scratch_field = self._scratch_dft = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
