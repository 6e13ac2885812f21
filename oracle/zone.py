"""ORACLE (test infrastructure, not product code): float64 CPU solve of one ZDA zone.

Follows SURVEY.md 8(c) Steps 0-10 in order, which are the discrete reading of
PAPER.md:53-68 (Eq. 3-5; Yee/leap-frog; r = 0 loop integral; CPML in r, z;
Bloch-periodic phi; DTFT of all frequencies from one run; hybrid
time/frequency adjoint).  Readings where the paper is silent are listed in
DESIGN.md ("Readings").  The voxel loops are in ``zda_oracle_core.c``; the
O(N)-sized host arithmetic (coefficients, DFT accumulate, objective, adjoint
source, gradient) is NumPy float64 below.

Shares no code with ``paper_2501_07979_b200``; never imported by it.
Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline /
``--impl reference`` legs may import this package.

Pins (tests/test_oracle_*.py, all ``-m "not gpu"``): coax-TEM Yee dispersion
(exact), leap-frog energy conservation, Bessel-zero cavity resonances
(TM010/020/030 and TE111 against tests/golden/bessel_zeros.txt),
CPML reflection in z and in r for BOTH polarisations (all eight psi arrays:
TEM/TM pulses pin psi_Hphi_z, psi_Er_z, psi_Hphi_r, psi_Ez_r; TE pulses pin
psi_Hr_z, psi_Ephi_z, psi_Hz_r, psi_Ephi_r), running DFT vs direct sum, adjoint-source DTFT identity,
adjoint gradient vs central finite differences, m <-> -m conjugation,
complex(p=1) == real.
"""
from __future__ import annotations

import ctypes
import math

import numpy as np

from . import _build

_c_double_p = ctypes.POINTER(ctypes.c_double)


class _Grid(ctypes.Structure):
    _fields_ = [
        ("Nr", ctypes.c_int), ("Nphi", ctypes.c_int), ("Nz", ctypes.c_int),
        ("has_axis", ctypes.c_int),
        ("dt", ctypes.c_double), ("inv_dr", ctypes.c_double), ("inv_dz", ctypes.c_double),
        ("phase_re", ctypes.c_double), ("phase_im", ctypes.c_double),
    ] + [(n, _c_double_p) for n in (
        "inv_rdphi_int", "inv_rdphi_half", "ca", "cb", "cc", "cd",
        "br_i", "cr_i", "ikr_i", "br_h", "cr_h", "ikr_h",
        "bz_i", "cz_i", "ikz_i", "bz_h", "cz_h", "ikz_h")] + [
        ("rpml_exact", ctypes.c_int), ("npml_r_lo", ctypes.c_int), ("npml_r_hi", ctypes.c_int),
    ] + [(n, _c_double_p) for n in ("bq_i", "cq_i", "bq_h", "cq_h", "hir_i", "hir_h")]


def _ptr(a):
    return a.ctypes.data_as(ctypes.c_void_p)


# ---------------------------------------------------------------------------
# Step a1: grid / coefficient builder
# ---------------------------------------------------------------------------
def radial_coefficients(Nr, r_in, dr, dphi):
    """Per-r metric coefficients of the cylindrical curl (Eq. 5's 1/r factors,
    PAPER.md:61), in the conservative radial form of SURVEY 8(c) Steps 3-4."""
    i = np.arange(Nr, dtype=np.float64)
    r_int = r_in + i * dr              # r_i
    r_half = r_int + 0.5 * dr          # r_{i+1/2}
    r_mhalf = r_int - 0.5 * dr         # r_{i-1/2}
    with np.errstate(divide="ignore", invalid="ignore"):
        inv_rdphi_int = np.where(r_int > 0, 1.0 / (r_int * dphi), 0.0)
        cc = np.where(r_int > 0, r_half / (r_int * dr), 0.0)
        cd = np.where(r_int > 0, r_mhalf / (r_int * dr), 0.0)
    inv_rdphi_half = 1.0 / (r_half * dphi)
    ca = (r_int + dr) / (r_half * dr)  # r_{i+1}/(r_{i+1/2} dr)
    cb = r_int / (r_half * dr)         # r_i/(r_{i+1/2} dr)
    return dict(r_int=r_int, r_half=r_half, inv_rdphi_int=inv_rdphi_int,
                inv_rdphi_half=inv_rdphi_half, ca=ca, cb=cb, cc=cc, cd=cd)


def cpml_profile(N, npml_lo, npml_hi, dt, p, sigma_max, kappa_max, alpha_max):
    """Step 2: CFS-CPML coefficients b, c, 1/kappa along one axis of N cells, at
    integer positions q = 0..N-1 and half positions q = i + 1/2.

    depth x in [0,1]: low slab x = (npml - q)/npml for q < npml;
    high slab x = (q - (N - npml))/npml for q > N - npml; x = 0 elsewhere.
    sigma = sigma_max x^p, kappa = 1 + (kappa_max-1) x^p, alpha = alpha_max (1-x),
    b = exp(-(sigma/kappa + alpha) dt), c = sigma (b-1)/(sigma kappa + kappa^2 alpha),
    c = 0 where sigma = 0.
    """
    out = {}
    for tag, off in (("i", 0.0), ("h", 0.5)):
        q = np.arange(N, dtype=np.float64) + off
        x = np.zeros(N)
        if npml_lo > 0:
            lo = q < npml_lo
            x[lo] = (npml_lo - q[lo]) / npml_lo
        if npml_hi > 0:
            hi = q > N - npml_hi
            x[hi] = (q[hi] - (N - npml_hi)) / npml_hi
        sigma = sigma_max * x ** p
        kappa = 1.0 + (kappa_max - 1.0) * x ** p
        alpha = alpha_max * (1.0 - x)
        b = np.exp(-(sigma / kappa + alpha) * dt)
        den = sigma * kappa + kappa * kappa * alpha
        c = np.zeros(N)
        nz = sigma > 0
        c[nz] = sigma[nz] * (b[nz] - 1.0) / den[nz]
        # outside the slabs psi stays identically 0 (c = 0); b is irrelevant there
        b[~nz] = 0.0
        out["b_" + tag], out["c_" + tag], out["ik_" + tag] = b, c, 1.0 / kappa
    return out


def rpml_exact_profile(Nr, npml_hi, r_in, dr, dt, p, sigma_max, alpha_max):
    """R25 ("r' = r + i zeta_r / omega ... regularised"): coefficients of the second recursive-convolution
    operator Q that realises 1/r~ = (1/r) / (1 + i zeta/(omega r)) inside the OUTER r-slab, at integer positions q = i and
    half positions q = i + 1/2:
        zeta(q) = sigma_max d x^(p+1) / (p + 1)   (the integral of sigma = sigma_max x^p from the slab's interface; d = npml dr
                  the slab thickness, x the depth in [0, 1]),
        sigma~  = zeta / r(q),   alpha~ = alpha_max (1 - x)   (the same frequency shift as the slab's own CFS term),
        bq = exp(-(sigma~ + alpha~) dt),   cq = sigma~ (bq - 1) / (sigma~ + alpha~);   0 where x = 0.
    Also hir = 1 / (2 r(q)) for the averaged F/r term.  The inner (concave) slab is left in the quasi form: there zeta < 0
    and the exact form is unstable whatever the regularisation tried (R25)."""
    out = {}
    for tag, off in (("i", 0.0), ("h", 0.5)):
        q = np.arange(Nr, dtype=np.float64) + off
        r = r_in + q * dr
        x = np.zeros(Nr)
        if npml_hi > 0:
            hi = q > Nr - npml_hi
            x[hi] = (q[hi] - (Nr - npml_hi)) / npml_hi
        zeta = sigma_max * (npml_hi * dr) * x ** (p + 1.0) / (p + 1.0)
        with np.errstate(divide="ignore", invalid="ignore"):
            sig = np.where(r > 0, zeta / r, 0.0)
            hir = np.where(r > 0, 1.0 / (2.0 * r), 0.0)
        alpha = alpha_max * (1.0 - x)
        b = np.exp(-(sig + alpha) * dt)
        c = np.zeros(Nr)
        nz = sig > 0
        c[nz] = sig[nz] * (b[nz] - 1.0) / (sig[nz] + alpha[nz])
        b[~nz] = 0.0
        out["bq_" + tag], out["cq_" + tag], out["hir_" + tag] = b, c, hir
    return out


def cfl_limit(dr, dz, dphi, r_in, has_axis, Nphi=None, phase=1.0):
    """A10: dt <= 1/sqrt(1/dr^2 + 1/dz^2 + 1/(r_min dphi)^2), r_min = r_in or dr/2 (c = 1).
    R21 (one phi cell, the paper's continuously axisymmetric first zone): the phi difference has the
    single eigenvalue (p - 1)/(r dphi), K = |p - 1|/dphi ~ |m|, so the phi term is (K^2 + 1/2 [axis]) / (2 r_min)^2;
    the 1/2 covers the 4/dr loop-integral update of Ez(0) (measured threshold, tests/test_oracle_modes.py)."""
    r_min = 0.5 * dr if has_axis else r_in
    if Nphi == 1:
        K = abs(complex(phase) - 1.0) / dphi
        phi_term = (K * K + (0.5 if has_axis else 0.0)) / (2.0 * r_min) ** 2
    else:
        phi_term = 1.0 / (r_min * dphi) ** 2
    return 1.0 / math.sqrt(1.0 / dr ** 2 + 1.0 / dz ** 2 + phi_term)


class OracleZone:
    """One zone: fields, CPML state, DFT accumulators; forward / adjoint runs; gradient."""

    def __init__(self, inp, eps_design=None):
        self.inp = inp
        self.lib = _build.load()
        self.cplx = bool(inp.complex_fields)
        self.dtype = np.complex128 if self.cplx else np.float64
        if not self.cplx and abs(complex(inp.phase).imag) != 0.0:
            raise ValueError("real fields need a real phi-boundary phase")
        if inp.has_axis and inp.r_in != 0.0:
            raise ValueError("has_axis needs r_in == 0")
        lim = cfl_limit(inp.dr, inp.dz, inp.dphi, inp.r_in, inp.has_axis, inp.Nphi, inp.phase)
        if inp.dt > lim:
            raise ValueError(f"dt={inp.dt} above the cylindrical CFL limit {lim}")
        Nr, Nphi, Nz = inp.Nr, inp.Nphi, inp.Nz
        self.shape = (Nr, Nphi, Nz)
        self.rc = radial_coefficients(Nr, inp.r_in, inp.dr, inp.dphi)
        self.pr = cpml_profile(Nr, inp.npml_r_lo, inp.npml_r_hi, inp.dt, inp.cpml_p,
                               inp.cpml_sigma_max_r, inp.cpml_kappa_max, inp.cpml_alpha_max)
        self.pz = cpml_profile(Nz, inp.npml_z_lo, inp.npml_z_hi, inp.dt, inp.cpml_p,
                               inp.cpml_sigma_max_z, inp.cpml_kappa_max, inp.cpml_alpha_max)
        self.exact = bool(getattr(inp, "rpml_exact", 0))
        self.pq = rpml_exact_profile(Nr, inp.npml_r_hi, inp.r_in, inp.dr, inp.dt, inp.cpml_p,
                                     inp.cpml_sigma_max_r, inp.cpml_alpha_max)
        self._keep = []  # keep coefficient arrays alive for the C struct

        def cptr(a):
            a = np.ascontiguousarray(a, dtype=np.float64)
            self._keep.append(a)
            return a.ctypes.data_as(_c_double_p)

        self.grid = _Grid(
            Nr=Nr, Nphi=Nphi, Nz=Nz, has_axis=int(inp.has_axis),
            dt=inp.dt, inv_dr=1.0 / inp.dr, inv_dz=1.0 / inp.dz,
            phase_re=complex(inp.phase).real, phase_im=complex(inp.phase).imag,
            inv_rdphi_int=cptr(self.rc["inv_rdphi_int"]), inv_rdphi_half=cptr(self.rc["inv_rdphi_half"]),
            ca=cptr(self.rc["ca"]), cb=cptr(self.rc["cb"]), cc=cptr(self.rc["cc"]), cd=cptr(self.rc["cd"]),
            br_i=cptr(self.pr["b_i"]), cr_i=cptr(self.pr["c_i"]), ikr_i=cptr(self.pr["ik_i"]),
            br_h=cptr(self.pr["b_h"]), cr_h=cptr(self.pr["c_h"]), ikr_h=cptr(self.pr["ik_h"]),
            bz_i=cptr(self.pz["b_i"]), cz_i=cptr(self.pz["c_i"]), ikz_i=cptr(self.pz["ik_i"]),
            bz_h=cptr(self.pz["b_h"]), cz_h=cptr(self.pz["c_h"]), ikz_h=cptr(self.pz["ik_h"]),
            rpml_exact=int(self.exact), npml_r_lo=inp.npml_r_lo, npml_r_hi=inp.npml_r_hi,
            bq_i=cptr(self.pq["bq_i"]), cq_i=cptr(self.pq["cq_i"]), bq_h=cptr(self.pq["bq_h"]), cq_h=cptr(self.pq["cq_h"]),
            hir_i=cptr(self.pq["hir_i"]), hir_h=cptr(self.pq["hir_h"]),
        )
        sfx = "_cx" if self.cplx else "_re"
        self._update_H = getattr(self.lib, "zo_update_H" + sfx)
        self._update_E = getattr(self.lib, "zo_update_E" + sfx)
        self._update_H.restype = None
        self._update_E.restype = None
        # gradient weights W_c(i) (Step 8/10): the radius of each component's own position
        self.W = np.stack([self.rc["r_half"], self.rc["r_int"], self.rc["r_int"]]).copy()
        if inp.has_axis:
            self.W[2, 0] = inp.dr / 8.0   # replicated on-axis Ez (Step 10)
        self.set_eps(eps_design if eps_design is not None else inp.eps_design)
        self.reset()
        self.dft_fwd = None
        self.dft_adj = None
        self.adj_source = None

    # -- materials ----------------------------------------------------------
    def set_eps(self, eps_design):
        """Assemble per-voxel eps: 1-D background eps(z) -- or the caller's per-voxel volume (north_star "per-voxel
        eps") -- with the design box overwritten (A3)."""
        inp = self.inp
        eps_bg = np.ones(inp.Nz) if inp.eps_bg_z is None else np.asarray(inp.eps_bg_z, np.float64)
        eps = np.empty(self.shape)
        eps[:] = eps_bg[None, None, :]
        if getattr(inp, "eps_volume", None) is not None:
            eps[:] = np.asarray(inp.eps_volume, np.float64)
        if eps_design is not None:
            eps[inp.design_i0:inp.design_i1, :, inp.design_k0:inp.design_k1] = eps_design
        self.eps = eps
        self.cE = inp.dt / eps                              # cE = dt/eps, once per voxel
        self.cE_axis = inp.dt / eps[0].mean(axis=0)         # dt/eps0[k], eps0 = mean_j eps[0,j,k]

    # -- state ----------------------------------------------------------------
    def reset(self):
        z = lambda: np.zeros(self.shape, dtype=self.dtype)
        self.E = [z(), z(), z()]      # Er, Ephi, Ez   at t = n dt
        self.H = [z(), z(), z()]      # Hr, Hphi, Hz   at t = (n + 1/2) dt
        self.psiH = [z(), z(), z(), z()]   # Hr_z, Hphi_z, Hphi_r, Hz_r
        self.psiE = [z(), z(), z(), z()]   # Er_z, Ephi_z, Ephi_r, Ez_r
        # R25 auxiliaries of the 1/r~ operator (exact complex-r PML); unused (and tiny) otherwise
        zx = z if self.exact else (lambda: np.zeros(1, dtype=self.dtype))
        self.chiH = [zx(), zx()]           # Hr, Hz
        self.chiE = [zx(), zx()]           # Er, Ez
        self.n = 0

    def _new_dft(self):
        inp = self.inp
        F = inp.n_freq
        return dict(design=np.zeros((F, 3) + inp.design_shape, np.complex128),
                    monitor=np.zeros((F, 3, inp.Nr, inp.Nphi), np.complex128))

    # -- one leap-frog step (Steps 3-7) --------------------------------------
    def step(self, J_r=None, J_phi=None, source_k=-1, dft=None):
        g = ctypes.byref(self.grid)
        E, H = self.E, self.H
        self._update_H(g, _ptr(H[0]), _ptr(H[1]), _ptr(H[2]),
                       _ptr(E[0]), _ptr(E[1]), _ptr(E[2]),
                       *[_ptr(a) for a in self.psiH], *[_ptr(a) for a in self.chiH])
        jr = _ptr(J_r) if J_r is not None else None
        jp = _ptr(J_phi) if J_phi is not None else None
        self._update_E(g, _ptr(E[0]), _ptr(E[1]), _ptr(E[2]),
                       _ptr(H[0]), _ptr(H[1]), _ptr(H[2]),
                       _ptr(self.cE), _ptr(self.cE_axis), jr, jp, ctypes.c_int(source_k),
                       *[_ptr(a) for a in self.psiE], *[_ptr(a) for a in self.chiE])
        self.n += 1
        if dft is not None:
            self._dft_accumulate(dft)

    def _dft_accumulate(self, dft):
        """Step 7: after the E update of step n (fields now at (n+1) dt; self.n == n+1):
        Ehat_{c,f} += dt exp(+i omega_f (n+1) dt) E_c^{n+1} on the design box and the monitor plane."""
        inp = self.inp
        for f, w in enumerate(inp.omega):
            tw = inp.dt * np.exp(1j * w * (self.n * inp.dt))
            for c in range(3):
                dft["design"][f, c] += tw * self.E[c][inp.design_i0:inp.design_i1, :, inp.design_k0:inp.design_k1]
                dft["monitor"][f, c] += tw * self.E[c][:, :, inp.monitor_k]

    def _run(self, n_steps, A_r, A_phi, table, source_k, dft):
        """Time loop with a sheet source J_c = sum_q A_c,q(i,j) s_q[n] (Step 6)."""
        for n in range(n_steps):
            J_r = J_phi = None
            if A_r is not None and n < table.shape[1]:
                s = table[:, n]
                J_r = np.ascontiguousarray(np.tensordot(s, A_r, axes=(0, 0)), dtype=self.dtype)
                J_phi = np.ascontiguousarray(np.tensordot(s, A_phi, axes=(0, 0)), dtype=self.dtype)
            self.step(J_r, J_phi, source_k, dft)

    # -- forward run (call stack 2) ------------------------------------------
    def run_forward(self, n_steps=None):
        inp = self.inp
        n_steps = inp.n_steps if n_steps is None else n_steps
        self.reset()
        self.dft_fwd = self._new_dft()
        self._run(n_steps, inp.src_A_r, inp.src_A_phi, np.asarray(inp.src_table), inp.source_k, self.dft_fwd)
        return self.dft_fwd

    # -- Step 8: objective ------------------------------------------------------
    def objective_mask(self):
        inp = self.inp
        m = np.zeros(inp.Nr, bool)
        m[inp.npml_r_lo:inp.Nr - inp.npml_r_hi] = True
        return m

    def focal_sums(self):
        """S_f = sum_{c in r,phi} sum_{i outside r-PML, j} g_{c,f}(i,j) Ehat_{c,f}(i,j,k_m): the field at the
        focal point as a linear functional of the monitor-plane field (R20)."""
        mon = self.dft_fwd["monitor"]
        m = self.objective_mask()
        g = self.focal_g()
        return np.array([np.sum(g[f][:, m, :] * mon[f, :2][:, m, :]) for f in range(self.inp.n_freq)])

    def focal_g(self):
        """The near-to-far weights: the caller's (R20), or built by the first Rayleigh-Sommerfeld integral to the on-axis
        point inp.focal_dz above the monitor plane (oracle/farfield.py; R24)."""
        if self.inp.focal_g is not None:
            return np.asarray(self.inp.focal_g, dtype=np.complex128)
        from .farfield import focal_weights
        return focal_weights(self.inp, float(self.inp.focal_dz))

    def focal_u(self):
        u = self.inp.focal_u
        return np.ones(self.inp.n_freq) if u is None else np.asarray(u, dtype=np.float64)

    def objective(self, kind="monitor_energy"):
        """kind = "monitor_energy": F = sum_f sum_{c in r,phi} sum_{i,j outside r-PML} W_c(i) |Ehat_{c,f}(i,j,k_m)|^2;
        kind = "focal_intensity": F = sum_f u_f |S_f|^2 (Eq. 7's focal intensity per frequency, weighted)."""
        if kind == "focal_intensity":
            return float(np.sum(self.focal_u() * np.abs(self.focal_sums()) ** 2))
        mon = self.dft_fwd["monitor"]
        m = self.objective_mask()
        F = 0.0
        for c in (0, 1):
            F += float(np.sum(self.W[c][None, m, None] * np.abs(mon[:, c][:, m, :]) ** 2))
        return F

    # -- Step 9: adjoint source -----------------------------------------------------
    def adjoint_pulses(self, n_steps):
        """q_f(t_{n+1/2}), shape (F, n_steps), and its half-step DTFT
        qhat_f(w) = dt sum_n q_f(t_{n+1/2}) exp(i w t_{n+1/2})."""
        inp = self.inp
        t = (np.arange(n_steps) + 0.5) * inp.dt
        env = np.exp(-((t - inp.adj_t0) ** 2) / (2.0 * inp.adj_sigma_t ** 2))
        q = env[None, :] * np.exp(-1j * inp.omega[:, None] * (t[None, :] - inp.adj_t0))

        def qhat(w):  # -> (F,)
            return inp.dt * (q * np.exp(1j * w * t)[None, :]).sum(axis=1)
        return q, qhat

    def build_adjoint_source(self, n_steps=None, kind="monitor_energy", S_total=None):
        """beta_{c,f}(i,j) such that the half-step DTFT of the adjoint current at every design
        frequency w_f' equals a_{c,f'}(i,j) = (dF/dEhat_{c,f'}(i,j,k_m)) / W_c(i) inside the objective mask,
        c in {r,phi}: conj(Ehat^fwd) for the monitor energy, u_f conj(S_f) g_{c,f} / W_c for the focal
        intensity; returns the (A_r, A_phi, table) triple of the sheet source.
        S_total (focal intensity only): the coherent focal field of the whole lens, sum over zones (and over the
        m = +-1 members of a pair) of their S_f, when the objective is F = sum_f u_f |sum_zones S_f|^2
        (``lens_focal_objective``; "a normally incident plane wave can be decomposed into m = +-1
        components"): dF/dEhat of THIS zone is then u_f conj(S_total_f) g, with this zone's own g."""
        inp = self.inp
        n_steps = (inp.n_steps_adjoint or inp.n_steps) if n_steps is None else n_steps
        F = inp.n_freq
        q, qhat = self.adjoint_pulses(n_steps)
        m = self.objective_mask()
        if kind == "focal_intensity":
            S = self.focal_sums() if S_total is None else np.asarray(S_total, dtype=np.complex128)
            g = self.focal_g()
            W = self.W[:2]                                         # (2, Nr): radius of each component's position
            with np.errstate(divide="ignore", invalid="ignore"):
                invW = np.where(W > 0, 1.0 / W, 0.0)
            a = (self.focal_u() * np.conj(S))[:, None, None, None] * g * invW[None, :, :, None]
        else:
            a = np.conj(self.dft_fwd["monitor"][:, :2]).copy()   # (F, 2, Nr, Nphi)
        a[:, :, ~m, :] = 0.0
        V = np.stack([qhat(w) for w in inp.omega])                 # V[f', f] = qhat_f(w_f')
        if self.cplx:
            # J = sum_f beta_f q_f(t):  a_f' = sum_f V[f',f] beta_f
            beta = np.linalg.solve(V, a.reshape(F, -1)).reshape(a.shape)
            A = beta                                               # terms: A_q = beta_f, s_q = q_f
            table = q
        else:
            # J = Re[sum_f beta_f q_f(t)]:
            # a_f' = 1/2 sum_f [ beta_f qhat_f(w_f') + conj(beta_f) conj(qhat_f(-w_f')) ]
            Vm = np.stack([np.conj(qhat(-w)) for w in inp.omega])  # Vm[f', f] = conj(qhat_f(-w_f'))
            P, M = 0.5 * (V + Vm), 0.5 * (V - Vm)                  # a = P Re(beta) + i M Im(beta)
            S = np.block([[P.real, -M.imag], [P.imag, M.real]])    # 2F x 2F real system
            rhs = np.concatenate([a.real.reshape(F, -1), a.imag.reshape(F, -1)])
            sol = np.linalg.solve(S, rhs)
            bre = sol[:F].reshape(a.shape)
            bim = sol[F:].reshape(a.shape)
            beta = bre + 1j * bim
            # Re[beta q] = Re(beta) Re(q) - Im(beta) Im(q): 2F real terms
            A = np.concatenate([bre, bim])
            table = np.concatenate([q.real, -q.imag])
        self.beta = beta
        self.adj_source = (np.ascontiguousarray(A[:, 0]), np.ascontiguousarray(A[:, 1]), table)
        return self.adj_source

    def run_adjoint(self, n_steps=None):
        """Same stepping with the conjugate phi phase (A12), state reset, source on the monitor
        plane, DFT on the design box."""
        inp = self.inp
        n_steps = (inp.n_steps_adjoint or inp.n_steps) if n_steps is None else n_steps
        if self.adj_source is None:
            self.build_adjoint_source(n_steps)
        A_r, A_phi, table = self.adj_source
        self.reset()
        self.grid.phase_im = -complex(inp.phase).imag
        try:
            self.dft_adj = self._new_dft()
            self._run(n_steps, A_r, A_phi, table, inp.monitor_k, self.dft_adj)
        finally:
            self.grid.phase_im = complex(inp.phase).imag
        return self.dft_adj

    # -- Step 10: gradient -----------------------------------------------------------
    def gradient(self):
        """dF/deps(i,j,k) = sum_f sum_c 2 Re[(-i Omega_f) W_c(i) Ehat^fwd_{c,f} Ehat^adj_{c,f}],
        Omega_f = (2/dt) sin(omega_f dt / 2), on the design box."""
        inp = self.inp
        Wd = self.W[:, inp.design_i0:inp.design_i1]
        g = np.zeros(inp.design_shape)
        for f, w in enumerate(inp.omega):
            Om = (2.0 / inp.dt) * math.sin(w * inp.dt / 2.0)
            for c in range(3):
                g += 2.0 * np.real((-1j * Om) * Wd[c][:, None, None]
                                   * self.dft_fwd["design"][f, c] * self.dft_adj["design"][f, c])
        return g

    # -- diagnostics used by the pins ---------------------------------------------
    def energy(self, H_prev):
        """W-weighted leap-frog energy (A1): 1/2 sum W eps |E^n|^2 + 1/2 sum W Re(H^{n+1/2} conj H^{n-1/2})."""
        W = self.W
        WH = np.stack([self.rc["r_int"], self.rc["r_half"], self.rc["r_half"]])
        if self.inp.has_axis:
            W = W.copy()
        e = 0.0
        for c in range(3):
            e += 0.5 * float(np.sum(W[c][:, None, None] * self.eps * np.abs(self.E[c]) ** 2))
            e += 0.5 * float(np.sum(WH[c][:, None, None] * np.real(self.H[c] * np.conj(H_prev[c]))))
        return e


def lens_focal_objective(zones, u=None):
    """F = sum_f u_f |sum_zones S_f^(zone)|^2: the focal intensity of a lens whose zones (and the m = +1 / m = -1
    members of each pair) add coherently at the focal point.  Returns (F, S_total)."""
    S = sum(z.focal_sums() for z in zones)
    u = np.ones(len(S)) if u is None else np.asarray(u, dtype=np.float64)
    return float(np.sum(u * np.abs(S) ** 2)), S
