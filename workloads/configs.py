"""Seeded synthetic zone problems shaped like BASELINE.json's configs 1-5.

Inputs only (see ``zone_inputs.py``): geometry numbers, material stacks,
seeded random design patterns and source tables.  The paper's own optimised
permittivity files are not available; these stand in for
them (recipe in DESIGN.md "Input recipe", numbers from SURVEY.md 8(d)).
Units: c = 1, dr = dz = 1 cell.
"""
from __future__ import annotations

import math
from dataclasses import replace

import numpy as np

from .zone_inputs import DensityMap, ZoneInputs

TWO_PI = 2.0 * math.pi


def courant_dt(dr, dz, dphi, r_min, courant=0.5, safety=0.99):
    """dt = min(courant * dr, safety * limit) with the cylindrical CFL limit."""
    lim = 1.0 / math.sqrt(1.0 / dr ** 2 + 1.0 / dz ** 2 + 1.0 / (r_min * dphi) ** 2)
    return min(courant * dr, safety * lim)


def courant_dt_one_phi_cell(dr, dz, dphi, r_min, phase, has_axis, courant=0.5, safety=0.99):
    """The same for a zone with ONE phi cell (R21): the phi term of the limit is
    (K^2 + 1/2 [axis]) / (2 r_min)^2 with K = |p - 1| / dphi."""
    K = abs(complex(phase) - 1.0) / dphi
    lim = 1.0 / math.sqrt(1.0 / dr ** 2 + 1.0 / dz ** 2 + (K * K + (0.5 if has_axis else 0.0)) / (2.0 * r_min) ** 2)
    return min(courant * dr, safety * lim)


def cpml_sigma_max(p, cell, eps_bg=1.0):
    """SURVEY A5 default: sigma_max = 0.8 (p+1) / (cell sqrt(eps_bg))."""
    return 0.8 * (p + 1.0) / (cell * math.sqrt(eps_bg))


def plane_wave_sheet(Nr, Nphi, dphi, complex_fields, m=1):
    """'x-polarised plane wave' sheet amplitudes on the (r, phi) plane.
    real:  A_r = cos(phi_j), A_phi = -sin(phi_{j+1/2});
    Bloch m=+1: A_r = 1/2 exp(i m phi_j), A_phi = (i/2) exp(i m phi_{j+1/2})."""
    phi_int = np.arange(Nphi) * dphi
    phi_half = phi_int + 0.5 * dphi
    if complex_fields:
        a_r = 0.5 * np.exp(1j * m * phi_int)
        a_p = 0.5j * np.exp(1j * m * phi_half)
        dt = np.complex128
    else:
        a_r = np.cos(phi_int)
        a_p = -np.sin(phi_half)
        dt = np.float64
    A_r = np.broadcast_to(a_r[None, None, :], (1, Nr, Nphi)).astype(dt).copy()
    A_p = np.broadcast_to(a_p[None, None, :], (1, Nr, Nphi)).astype(dt).copy()
    return A_r, A_p


def gaussian_pulse_table(n_steps, dt, omega_c, sigma_t, t0, complex_fields):
    """s(t) = exp(-(t-t0)^2 / 2 sigma_t^2) cos(omega_c (t-t0))   [real fields]
                                          exp(-i omega_c (t-t0)) [complex fields],
    sampled at t = (n + 1/2) dt (SURVEY Step 6)."""
    t = (np.arange(n_steps) + 0.5) * dt
    env = np.exp(-((t - t0) ** 2) / (2.0 * sigma_t ** 2))
    if complex_fields:
        return (env * np.exp(-1j * omega_c * (t - t0)))[None, :]
    return (env * np.cos(omega_c * (t - t0)))[None, :]


def focal_point_weights(inp, focal_length=60.0, seed=7):
    """Synthetic near-to-far weights for the focal-intensity objective (R20; an INPUT of the method):
    a smooth spherical-wave propagator g = exp(i w R) / R from the monitor-plane point at radius r to the
    on-axis point focal_length beyond the plane, R = sqrt(r^2 + focal_length^2), times the x-polarisation
    factor of each component (cos phi_j for r, -sin phi_{j+1/2} for phi) and a seeded amplitude per (f, c).
    Shape (F, 2, Nr, Nphi) complex128."""
    rng = np.random.default_rng(seed)
    r = inp.r_in + np.arange(inp.Nr) * inp.dr
    phi = np.arange(inp.Nphi) * inp.dphi
    g = np.zeros((inp.n_freq, 2, inp.Nr, inp.Nphi), dtype=np.complex128)
    for f, w in enumerate(inp.omega):
        R = np.sqrt(r ** 2 + focal_length ** 2)
        base = np.exp(1j * w * R) / R
        g[f, 0] = base[:, None] * np.cos(phi)[None, :] * (1.0 + 0.1 * rng.standard_normal())
        g[f, 1] = -base[:, None] * np.sin(phi + 0.5 * inp.dphi)[None, :] * (1.0 + 0.1 * rng.standard_normal())
    return g


def _smooth_density(rng, n_r, n_phi):
    return rng.uniform(0.0, 1.0, size=(n_r, n_phi))


# ---------------------------------------------------------------------------
def config1(seed=1, n_steps=600):
    """Tiny zone: 48 x 16 x 64, n = 8, r_in = 20, lambda = 20 cells, Courant 0.5,
    8-cell CPML in r and z, real periodic fields, Bernoulli(0.5) eps in {1, 11.7}
    on the design box i = 8..39, k = 24..29 (2-D pattern extruded in z)."""
    Nr, Nphi, Nz, n = 48, 16, 64, 8
    dr = dz = 1.0
    r_in = 20.0
    dphi = TWO_PI / (n * Nphi)
    dt = courant_dt(dr, dz, dphi, r_in)
    lam = 20.0
    rng = np.random.default_rng(seed)
    i0, i1, k0, k1 = 8, 40, 24, 30
    pat = rng.random((i1 - i0, Nphi)) < 0.5
    eps2d = np.where(pat, 11.7, 1.0)
    eps_design = np.repeat(eps2d[:, :, None], k1 - k0, axis=2)
    A_r, A_p = plane_wave_sheet(Nr, Nphi, dphi, False)
    omega_c = TWO_PI / lam
    table = gaussian_pulse_table(n_steps, dt, omega_c, 20.0, 75.0, False)
    p = 3.0
    return ZoneInputs(
        name="config1-tiny", Nr=Nr, Nphi=Nphi, Nz=Nz, dr=dr, dphi=dphi, dz=dz, r_in=r_in, dt=dt,
        n_fold=n, phase=1.0 + 0j, complex_fields=False, has_axis=False,
        npml_r_lo=8, npml_r_hi=8, npml_z_lo=8, npml_z_hi=8, cpml_p=p,
        cpml_sigma_max_r=cpml_sigma_max(p, dr), cpml_sigma_max_z=cpml_sigma_max(p, dz),
        cpml_kappa_max=1.0, cpml_alpha_max=0.05,
        design_i0=i0, design_i1=i1, design_k0=k0, design_k1=k1, monitor_k=50, source_k=12,
        omega=np.array([omega_c]), eps_bg_z=np.ones(Nz), eps_design=eps_design,
        src_A_r=A_r, src_A_phi=A_p, src_table=table, n_steps=n_steps, n_steps_adjoint=n_steps,
        adj_t0=75.0, adj_sigma_t=20.0, seed=seed)


def _layered_zone(name, seed, Nr, Nphi, Nz, r_in, n, npml, k_sub, eps_sub, k_d0, k_d1,
                  eps0, eps_h, source_k, monitor_k, lambdas, n_steps, adjoint,
                  complex_fields=False, m=1, has_axis=False, density_shape=None, conic_radius=0.0):
    dr = dz = 1.0
    dphi = TWO_PI / (n * Nphi)
    r_min = 0.5 * dr if has_axis else r_in
    dt = courant_dt(dr, dz, dphi, r_min)
    rng = np.random.default_rng(seed)
    npr_lo = 0 if has_axis else npml
    i0, i1 = npr_lo, Nr - npml
    rho = _smooth_density(rng, i1 - i0, Nphi)
    eps_bg = np.ones(Nz)
    eps_bg[:k_sub] = eps_sub
    omega = TWO_PI / np.asarray(lambdas, dtype=np.float64)
    omega_c = float(omega.mean())
    if len(lambdas) > 1:
        sigma_w = 0.5 * float(omega.max() - omega.min())
    else:
        sigma_w = omega_c / 8.0
    sigma_t = 1.0 / sigma_w
    t0 = 4.0 * sigma_t
    A_r, A_p = plane_wave_sheet(Nr, Nphi, dphi, complex_fields, m)
    table = gaussian_pulse_table(n_steps, dt, omega_c, sigma_t, t0, complex_fields)
    # adjoint basis pulses: narrow enough in frequency to separate the design lines
    if len(lambdas) > 1:
        dw = float(np.min(np.abs(np.diff(np.sort(omega)))))
        adj_sigma_t = 1.0 / dw
    else:
        adj_sigma_t = sigma_t
    p = 3.0
    phase = complex(np.exp(1j * TWO_PI * m / n)) if complex_fields else 1.0 + 0j
    return ZoneInputs(
        name=name, Nr=Nr, Nphi=Nphi, Nz=Nz, dr=dr, dphi=dphi, dz=dz, r_in=r_in, dt=dt, n_fold=n,
        phase=phase, complex_fields=complex_fields, has_axis=has_axis,
        npml_r_lo=npr_lo, npml_r_hi=npml, npml_z_lo=npml, npml_z_hi=npml, cpml_p=p,
        cpml_sigma_max_r=cpml_sigma_max(p, dr),
        cpml_sigma_max_z=cpml_sigma_max(p, dz, math.sqrt(eps_sub)),  # geometric mean of substrate and air
        cpml_kappa_max=1.0, cpml_alpha_max=0.05,
        design_i0=i0, design_i1=i1, design_k0=k_d0, design_k1=k_d1,
        monitor_k=monitor_k, source_k=source_k, omega=omega, eps_bg_z=eps_bg,
        density=DensityMap(rho=rho, eps0=eps0, eps_h=eps_h, filt_sigma=3.0, beta=8.0, eta=0.5,
                           conic_radius=conic_radius, r_first=r_in + (i0 + 0.5) * dr, dr=dr, dphi=dphi),
        src_A_r=A_r, src_A_phi=A_p, src_table=table, n_steps=n_steps,
        n_steps_adjoint=n_steps if adjoint else 0, adj_t0=4.0 * adj_sigma_t, adj_sigma_t=adj_sigma_t,
        seed=seed)


def config2(seed=2, Nr=800, Nphi=800, Nz=160, n_steps=4000):
    """LWIR monochromatic zone, forward only: r_in = 2000, n = 22, Si (11.7) below k = 40,
    design k = 40..59 with eps = 1 + 10.7 rho_bar, 12-cell CPML, lambda = 20 cells."""
    return _layered_zone("config2-lwir", seed, Nr, Nphi, Nz, 2000.0, _n_for(2000.0, Nr, Nphi), 12,
                         40, 11.7, 40, 60, 1.0, 11.7, 20, 130, [20.0], n_steps, adjoint=False)


def config3(seed=3, Nr=1200, Nphi=1200, Nz=200, n_steps=6000):
    """RGB zone, forward + adjoint, complex Bloch fields m = 1: SiO2 (2.13) below k = 60,
    TiO2 design (1..6.25) k = 60..89, lambdas 24 / 29.33 / 34.67 cells."""
    lam = [24.0, 24.0 * 550.0 / 450.0, 24.0 * 650.0 / 450.0]
    return _layered_zone("config3-rgb", seed, Nr, Nphi, Nz, 3000.0, _n_for(3000.0, Nr, Nphi), 12,
                         60, 2.13, 60, 90, 1.0, 6.25, 30, 170, lam, n_steps, adjoint=True,
                         complex_fields=True, m=1)


def config4(seed=4, Nr=2000, Nphi=2000, Nz=250, n_steps=8000):
    """6-wavelength zone, forward + adjoint, real periodic: same stack as config 3,
    design k = 70..99, lambdas 20..35 cells (400..700 nm at lambda_min/20)."""
    lam = [20.0 * w / 400.0 for w in (400.0, 460.0, 520.0, 580.0, 640.0, 700.0)]
    return _layered_zone("config4-6wl", seed, Nr, Nphi, Nz, 5000.0, _n_for(5000.0, Nr, Nphi), 12,
                         70, 2.13, 70, 100, 1.0, 6.25, 30, 220, lam, n_steps, adjoint=True)


def _n_for(r_in, Nr, Nphi):
    """n such that the outer arc r_out * tau_phi is about Nphi cells (r_out dphi ~ 1)."""
    return max(1, round(TWO_PI * (r_in + Nr) / Nphi))


def config5_zones(seed=5, n_zones=24, n_steps=5000, Nz=200, scale=1.0):
    """Full-lens pass: 24 annular zones of width 1109.3 cells (+12-cell CPML each side overlapping
    the neighbours), zone 0 with the r = 0 axis (n = 1, Nphi = 8), n_l ~ r_out so the outer arc is
    ~ 1386.7 cells; per-zone dt from the CFL limit.  ``scale`` < 1 shrinks every zone (tests)."""
    lam = [24.0, 24.0 * 550.0 / 450.0, 24.0 * 650.0 / 450.0]
    width = 1109.3 * scale
    arc = 1386.7 * scale
    npml = 12
    zones = []
    for l in range(n_zones):
        if l == 0:
            Nr = int(math.ceil(width)) + npml
            z = _layered_zone(f"config5-zone{l}", seed + l, Nr, 8, Nz, 0.0, 1, npml, 60, 2.13, 60, 90,
                              1.0, 6.25, 30, 170, lam, n_steps, adjoint=True, has_axis=True)
        else:
            r_in = width * l - npml
            Nr = int(math.ceil(width)) + 2 * npml
            r_out = r_in + Nr
            n = max(1, round(TWO_PI * r_out / arc))
            Nphi = int(math.ceil(TWO_PI / n * r_out))
            z = _layered_zone(f"config5-zone{l}", seed + l, Nr, Nphi, Nz, r_in, n, npml, 60, 2.13, 60, 90,
                              1.0, 6.25, 30, 170, lam, n_steps, adjoint=True)
        zones.append(z)
    return zones


def config6_thin_wedge(seed=6, ell=8, n_steps=4000, lam=50.0, Nz=160):
    """A zone shaped like the paper's LWIR lens zones: radial width 25 lambda at
    dr = dz = lambda/50 (1250 cells + 12-cell CPML each side), zone number ell = 2..16 with azimuthal period
    tau_phi = 2 pi / (720 ell), r dphi < 0.021 lambda => Nphi = 11 cells, complex Bloch fields m = 1 (the phase
    p = exp(2 pi i / n) is not real at these n), Si substrate and 0.6 lambda Si design layer, F = 1,
    forward + adjoint; density through the paper's conic filter, radius 0.08 lambda (R22)."""
    npml = 12
    width = int(round(25 * lam))
    r_in = width * (ell - 1) - npml
    Nr = width + 2 * npml
    n = 720 * ell
    r_out = r_in + Nr
    Nphi = int(math.ceil(TWO_PI / n * r_out / (0.021 * lam)))
    k_d1 = 40 + int(round(0.6 * lam))
    return _layered_zone(f"config6-wedge{ell}", seed, Nr, Nphi, Nz, float(r_in), n, npml, 40, 11.7, 40, k_d1,
                         1.0, 11.7, 20, Nz - npml - 18, [lam], n_steps, adjoint=True, complex_fields=True, m=1,
                         conic_radius=0.08 * lam)


def config7_first_zone(seed=7, n_steps=4000, lam=50.0, Nz=160, m=1, n_fold=720):
    """The paper's continuously axisymmetric first zone (n -> infinity): ONE phi cell, complex fields
    with the wrap phase p = exp(i m dphi) (R2: (p - 1)/dphi -> i m), the r = 0 axis, outer r-CPML only, radial width
    25 lambda at lambda/50; same stack as config 6.  dt from the one-phi-cell limit (R21).  The value of dphi only
    sets how close (p - 1)/dphi is to i m (second order)."""
    npml = 12
    Nr = int(round(25 * lam)) + npml
    dphi = TWO_PI / n_fold
    phase = complex(np.exp(1j * m * dphi))
    z = _layered_zone("config7-first-zone", seed, Nr, 1, Nz, 0.0, n_fold, npml, 40, 11.7, 40,
                      40 + int(round(0.6 * lam)), 1.0, 11.7, 20, Nz - npml - 18, [lam], n_steps, adjoint=True,
                      complex_fields=True, m=m, has_axis=True, conic_radius=0.08 * lam)
    dt = courant_dt_one_phi_cell(z.dr, z.dz, dphi, 0.5 * z.dr, phase, True)
    sigma_t = 8.0 / float(z.omega[0])
    return replace(z, dt=dt, src_table=gaussian_pulse_table(n_steps, dt, float(z.omega[0]), sigma_t, 4.0 * sigma_t, True))


def cut_down(inp: ZoneInputs, Nr=None, Nphi=None, n_steps=None, seed=None):
    """A cut-down copy of a big config for oracle-sized parity: same r_in, dphi,
    stack, CPML, source, frequencies; fewer radial cells and phi cells (dphi is unchanged, so the
    wedge gets narrower and is no longer an integer fraction of the circle: n_fold = 0), shorter run."""
    Nr = Nr or inp.Nr
    Nphi = Nphi or inp.Nphi
    n_steps = n_steps or inp.n_steps
    rng = np.random.default_rng(inp.seed if seed is None else seed)
    npr_lo = inp.npml_r_lo
    i0, i1 = npr_lo, Nr - inp.npml_r_hi
    A_r, A_p = plane_wave_sheet(Nr, Nphi, inp.dphi, inp.complex_fields)
    table = np.asarray(inp.src_table)[:, :n_steps]
    dens = None
    if inp.density is not None:
        dens = replace(inp.density, rho=_smooth_density(rng, i1 - i0, Nphi))
    # keep dphi: the wedge angle shrinks, so the Bloch phase over the wedge is p^(Nphi_new/Nphi_old)
    phase = inp.phase
    if inp.complex_fields:
        phase = complex(np.exp(1j * np.angle(inp.phase) * Nphi / inp.Nphi))
    n_fold = inp.n_fold if Nphi == inp.Nphi else 0
    return replace(inp, name=inp.name + f"-cut{Nr}x{Nphi}", Nr=Nr, Nphi=Nphi, n_fold=n_fold, design_i0=i0, design_i1=i1,
                   density=dens, eps_design=None, src_A_r=A_r, src_A_phi=A_p, src_table=table,
                   n_steps=n_steps, n_steps_adjoint=(n_steps if inp.n_steps_adjoint else 0), phase=phase)


def window(inp: ZoneInputs, eps_design_full, i_lo, i_hi, j_lo, j_hi, k_lo, k_hi, n_steps):
    """The sub-block [i_lo, i_hi) x [j_lo, j_hi) x [k_lo, k_hi) of a zone as a zone problem of its own
    (inputs only: slices and shifted indices).  Used for parity at sizes the oracle cannot finish: after
    n explicit steps a field value depends only on data within n cells of it, so the oracle run on the
    window reproduces the big zone's fields at every point further than n + 1 cells from a CUT face.
    A face that coincides with the zone's own boundary is not a cut: the window keeps that CPML slab
    (same thickness and parameters, hence the same coefficients).  A cut face must stay clear of the
    slabs.  ``eps_design_full`` is the per-voxel eps of the big zone's design box, (Nr_d, Nphi, L_d).
    A window that spans all of phi keeps the zone's phi-boundary phase; otherwise the wedge is cut
    (n_fold = 0) and the phase at the cut is irrelevant."""
    npr_lo = inp.npml_r_lo if i_lo == 0 else 0
    npr_hi = inp.npml_r_hi if i_hi == inp.Nr else 0
    npz_lo = inp.npml_z_lo if k_lo == 0 else 0
    npz_hi = inp.npml_z_hi if k_hi == inp.Nz else 0
    assert i_lo == 0 or i_lo >= inp.npml_r_lo
    assert i_hi == inp.Nr or i_hi <= inp.Nr - inp.npml_r_hi
    assert k_lo == 0 or k_lo >= inp.npml_z_lo
    assert k_hi == inp.Nz or k_hi <= inp.Nz - inp.npml_z_hi
    full_phi = (j_lo == 0 and j_hi == inp.Nphi)
    di0, di1 = max(inp.design_i0, i_lo), min(inp.design_i1, i_hi)
    dk0, dk1 = max(inp.design_k0, k_lo), min(inp.design_k1, k_hi)
    assert di0 < di1 and dk0 < dk1, "the window must meet the design box"
    assert k_lo <= inp.source_k < k_hi, "the window must contain the source plane"
    eps = np.asarray(eps_design_full)[di0 - inp.design_i0:di1 - inp.design_i0, j_lo:j_hi,
                                      dk0 - inp.design_k0:dk1 - inp.design_k0].copy()
    bg = np.ones(inp.Nz) if inp.eps_bg_z is None else np.asarray(inp.eps_bg_z)
    return replace(
        inp, name=inp.name + "-window", Nr=i_hi - i_lo, Nphi=j_hi - j_lo, Nz=k_hi - k_lo,
        r_in=inp.r_in + i_lo * inp.dr, n_fold=(inp.n_fold if full_phi else 0),
        npml_r_lo=npr_lo, npml_r_hi=npr_hi, npml_z_lo=npz_lo, npml_z_hi=npz_hi,
        design_i0=di0 - i_lo, design_i1=di1 - i_lo, design_k0=dk0 - k_lo, design_k1=dk1 - k_lo,
        source_k=inp.source_k - k_lo, monitor_k=min(max(inp.monitor_k - k_lo, 0), k_hi - k_lo - 1),
        eps_bg_z=bg[k_lo:k_hi].copy(), eps_design=eps, density=None,
        src_A_r=np.asarray(inp.src_A_r)[:, i_lo:i_hi, j_lo:j_hi].copy(),
        src_A_phi=np.asarray(inp.src_A_phi)[:, i_lo:i_hi, j_lo:j_hi].copy(),
        src_table=np.asarray(inp.src_table)[:, :n_steps].copy(), n_steps=n_steps, n_steps_adjoint=0)
