"""Plain-data description of one ZDA zone problem.

This module is shared by the oracle (``oracle/``) and the CUDA binding
(``paper_2501_07979_b200/``).  It holds *inputs only*: no update equation,
no CPML formula, no DFT, no adjoint arithmetic lives here (each side has its
own).  Index conventions (both sides): cells (i, j, k), 0 <= i < Nr,
0 <= j < Nphi, 0 <= k < Nz; boxes are half-open ``[i0, i1) x [all j] x [k0, k1)``.
Arrays in this dataclass are NumPy, C order, shape ``(..., Nr, Nphi[, Nz])``
(the paper-notation order r, phi, z); each side converts to its own layout.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np


@dataclass
class DensityMap:
    """Parameters of the density -> eps map (PAPER.md:72-76 Eq. 6, :83 filters;
    SURVEY.md 8(c) A13).  ``rho`` has shape (Nr_d, Nphi)."""
    rho: np.ndarray
    eps0: float
    eps_h: float
    filt_sigma: float = 3.0
    beta: float = 8.0
    eta: float = 0.5
    # conic filter in the physical (r, r phi) metric ("conic filter with a radius of 0.08 lambda";
    # DESIGN.md R22): conic_radius > 0 selects it instead of the Gaussian; the metric needs the radius of the first
    # design cell's centre and the cell sizes, which the workload builder copies from the zone
    conic_radius: float = 0.0
    r_first: float = 0.0          # r_in + (design_i0 + 1/2) dr
    dr: float = 1.0
    dphi: float = 0.0


@dataclass
class ZoneInputs:
    name: str
    # grid (Fig. 2: annular wedge of angle 2 pi / n_fold)
    Nr: int
    Nphi: int
    Nz: int
    dr: float
    dphi: float
    dz: float
    r_in: float
    dt: float
    n_fold: int
    phase: complex = 1.0 + 0.0j      # phi-boundary Bloch phase p = exp(i 2 pi m / n)
    complex_fields: bool = False     # True => complex (Bloch) fields
    has_axis: bool = False           # r_in == 0 zone
    # CPML (SURVEY 8(c) Step 2 / A5)
    npml_r_lo: int = 0
    npml_r_hi: int = 0
    npml_z_lo: int = 0
    npml_z_hi: int = 0
    cpml_p: float = 3.0
    cpml_sigma_max_r: float = 0.0
    cpml_sigma_max_z: float = 0.0
    cpml_kappa_max: float = 1.0
    cpml_alpha_max: float = 0.05
    rpml_exact: int = 0              # 1: exact cylindrical PML in r (complex radius r~ = r + i zeta/omega, R25)
    # design box, monitor and source planes
    design_i0: int = 0
    design_i1: int = 0
    design_k0: int = 0
    design_k1: int = 0
    monitor_k: int = 0
    source_k: int = 0
    # design frequencies (angular, c = 1)
    omega: np.ndarray = field(default_factory=lambda: np.zeros(0))
    # materials: 1-D background eps(z) and per-voxel eps on the design box
    eps_bg_z: Optional[np.ndarray] = None            # (Nz,)
    eps_design: Optional[np.ndarray] = None          # (Nr_d, Nphi, L_d)
    density: Optional[DensityMap] = None             # alternative to eps_design
    eps_volume: Optional[np.ndarray] = None          # (Nr, Nphi, Nz): per-voxel eps over the whole zone; replaces eps_bg_z
                                                     # everywhere, the design box is then overwritten by eps_design / density
    # forward source (SURVEY 8(c) Step 6): J_c(i,j) = sum_q A_c,q(i,j) s_q[n]
    src_A_r: Optional[np.ndarray] = None             # (n_terms, Nr, Nphi)
    src_A_phi: Optional[np.ndarray] = None           # (n_terms, Nr, Nphi)
    src_table: Optional[np.ndarray] = None           # (n_terms, n_steps), sampled at (n + 1/2) dt
    n_steps: int = 0
    n_steps_adjoint: int = 0
    # adjoint basis pulses q_f(t) = exp(-(t-t0)^2 / 2 sigma_t^2) exp(-i omega_f (t-t0))
    adj_t0: float = 0.0
    adj_sigma_t: float = 1.0
    seed: int = 0
    # focal-intensity objective (Eq. 7): F = sum_f u_f |S_f|^2,
    # S_f = sum_{c in r,phi} sum_{i outside r-PML, j} g_{c,f}(i,j) Ehat_{c,f}(i,j,k_m); the near-to-far
    # weights g are an INPUT (the caller's propagator from the monitor plane to the focal point)
    focal_g: Optional[np.ndarray] = None             # (F, 2, Nr, Nphi) complex
    focal_u: Optional[np.ndarray] = None             # (F,) real, default all ones
    # alternative to focal_g: the weights are BUILT by the method's own near-to-far transform (first Rayleigh-Sommerfeld
    # integral to the on-axis point focal_dz above the monitor plane; R24)
    focal_dz: Optional[float] = None

    @property
    def n_freq(self) -> int:
        return int(len(self.omega))

    @property
    def n_voxels(self) -> int:
        return self.Nr * self.Nphi * self.Nz

    @property
    def design_shape(self):
        return (self.design_i1 - self.design_i0, self.Nphi, self.design_k1 - self.design_k0)
