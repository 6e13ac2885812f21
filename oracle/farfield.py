"""ORACLE (test infrastructure, not product code): the near-to-far transform of the focal-intensity objective.

PAPER.md:76-81 (Eq. 7-8) optimises the focal intensity I(p, omega_i) of an x-polarised, normally incident plane wave
("decomposed into m = +-1 components", :76) but does not give its near-to-far transform.  Reading R24:

  * the half-space above the monitor plane z = z_m is homogeneous (eps_m = eps_bg_z[monitor_k]), so the field there
    follows from the tangential E on the plane alone (equivalence principle with a PEC-backed aperture, Smythe's
    formula); each Cartesian tangential component then obeys the first Rayleigh-Sommerfeld integral
        E_x(r) = -(1 / 2 pi)  Int  E_x(r')  d/dz [ exp(i k R) / R ]  dS',    R = |r - r'|,  k = omega sqrt(eps_m)
    (e^{-i omega t} convention: exp(+i k R) is outgoing);
  * the focal point sits ON THE AXIS, a height dz above the plane:  R = sqrt(rho'^2 + dz^2),
        h(rho') = -(1 / 2 pi) (i k - 1 / R) exp(i k R) dz / R^2 ;
  * E_x = E_r cos(phi) - E_phi sin(phi) at each component's own Yee position: E_r at (r_{i+1/2}, phi_j), E_phi at
    (r_i, phi_{j+1/2}); midpoint quadrature dS = r dr dphi at that position; the aperture is the zone's annulus outside
    its r-PML (the objective mask), the rest of the plane belongs to other zones (they add coherently, R23) or is dark;
  * the zone is one wedge of n_fold: the other wedges carry the Bloch-continued field E(phi + w tau) = p^w E(phi), so
        cos(phi)  ->  C_r(phi)   = sum_{w=0}^{n-1} p^w cos(phi + w tau),
        sin(phi)  ->  C_phi(phi) = sum_{w=0}^{n-1} p^w sin(phi + w tau)
    (written out as the sums; they vanish unless m = +-1 mod n: only those Bloch orders reach an on-axis x-polarised
    focus, which is the paper's m = +-1 decomposition).  n_fold = 0 (a cut wedge) counts as the one wedge.

Result: g[f, 0, i, j] = h_f(r_{i+1/2}) C_r(phi_j) r_{i+1/2} dr dphi,  g[f, 1, i, j] = -h_f(r_i) C_phi(phi_{j+1/2}) r_i dr dphi,
so that S_f = sum g Ehat(monitor) = E_x(focal point; omega_f) (``OracleZone.focal_sums``).

Pins (tests/test_oracle_farfield.py): the closed-form on-axis field of a uniformly illuminated annular aperture,
E0 [ (dz / R1) exp(i k R1) - (dz / R2) exp(i k R2) ], second order in dr and dphi; half of it for the m = +1 circular
component; exactly zero for m = 0 and m = 2; a brute-force sum over all n wedges of an explicitly continued field.
Shares no code with paper_2501_07979_b200."""
from __future__ import annotations

import math

import numpy as np


def wedge_sums(inp):
    """C_r(phi_j), C_phi(phi_{j+1/2}): the x-polarisation factors summed over the n_fold Bloch-continued wedges."""
    n = max(int(inp.n_fold), 1)
    tau = inp.Nphi * inp.dphi
    p = complex(inp.phase)
    phi_int = np.arange(inp.Nphi) * inp.dphi
    phi_half = phi_int + 0.5 * inp.dphi
    C_r = np.zeros(inp.Nphi, dtype=np.complex128)
    C_p = np.zeros(inp.Nphi, dtype=np.complex128)
    pw = 1.0 + 0.0j
    for w in range(n):
        C_r += pw * np.cos(phi_int + w * tau)
        C_p += pw * np.sin(phi_half + w * tau)
        pw *= p
    return C_r, C_p


def rs_kernel(omega, eps_m, rho, dz):
    """h(rho) = -(1 / 2 pi) (i k - 1 / R) exp(i k R) dz / R^2 (first Rayleigh-Sommerfeld integral, on-axis point)."""
    k = omega * math.sqrt(eps_m)
    R = np.sqrt(rho ** 2 + dz ** 2)
    return -(1.0 / (2.0 * math.pi)) * (1j * k - 1.0 / R) * np.exp(1j * k * R) * dz / R ** 2


def focal_weights(inp, focal_dz):
    """g[f, c, i, j] (F, 2, Nr, Nphi) complex128 for the on-axis focal point focal_dz above the monitor plane."""
    eps_m = 1.0 if inp.eps_bg_z is None else float(np.asarray(inp.eps_bg_z)[inp.monitor_k])
    i = np.arange(inp.Nr, dtype=np.float64)
    r_int = inp.r_in + i * inp.dr
    r_half = r_int + 0.5 * inp.dr
    C_r, C_p = wedge_sums(inp)
    dA = inp.dr * inp.dphi
    g = np.zeros((inp.n_freq, 2, inp.Nr, inp.Nphi), dtype=np.complex128)
    for f, w in enumerate(np.asarray(inp.omega, dtype=np.float64)):
        g[f, 0] = (rs_kernel(w, eps_m, r_half, focal_dz) * r_half * dA)[:, None] * C_r[None, :]
        g[f, 1] = -(rs_kernel(w, eps_m, r_int, focal_dz) * r_int * dA)[:, None] * C_p[None, :]
    return g
