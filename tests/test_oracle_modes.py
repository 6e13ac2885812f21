"""Pins of the oracle against closed forms: Yee dispersion (exact coax TEM eigenmode),
the Cartesian 3-D Yee dispersion in the r_in >> Nr limit, and Bessel-zero cavity resonances
(BASELINE.json north_star; SURVEY.md 8(c) pins 1 and 3)."""
import math

import numpy as np
import pytest
from scipy import special

from helpers import freq_from_complex_series, freq_from_series, make_zone
from oracle import OracleZone, cfl_limit


def _golden_zeros():
    """tests/golden/bessel_zeros.txt: the 4-digit textbook zeros north_star and SURVEY 8(c) pin 3 quote."""
    import os
    vals = {}
    for line in open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "bessel_zeros.txt")):
        if line.strip() and not line.startswith("#"):
            k, v = line.split()
            vals[k] = float(v)
    return vals


@pytest.mark.parametrize("eps", [1.0, 2.25])
def test_coax_tem_is_exact_yee_eigenmode(eps):
    """Er = sin(kz)/r cos(wt) between PEC cylinders is an exact discrete eigenmode with
    sin(w dt/2)/dt = sin(k dz/2)/(dz sqrt(eps))  (1-D Yee dispersion)."""
    Nr, Nphi, Nz = 6, 3, 40
    inp = make_zone(Nr, Nphi, Nz, r_in=7.0, n_fold=5, courant=0.9, eps_bg_z=np.full(Nz, eps))
    z = OracleZone(inp)
    mz = 3
    kap = math.pi * mz / (Nz * inp.dz)
    w = 2.0 / inp.dt * math.asin(inp.dt / inp.dz * math.sin(kap * inp.dz / 2) / math.sqrt(eps))
    r_half = inp.r_in + (np.arange(Nr) + 0.5) * inp.dr
    zk = np.arange(Nz) * inp.dz
    zh = zk + 0.5 * inp.dz
    B = -(inp.dt / inp.dz) * math.sin(kap * inp.dz / 2) / math.sin(w * inp.dt / 2)
    shape_E = (np.sin(kap * zk)[None, None, :] / r_half[:, None, None]) * np.ones((1, Nphi, 1))
    shape_H = (np.cos(kap * zh)[None, None, :] / r_half[:, None, None]) * np.ones((1, Nphi, 1))
    z.E[0][:] = shape_E                                   # Er^0
    z.H[1][:] = B * shape_H * math.sin(w * (-0.5) * inp.dt)  # Hphi^{-1/2}
    worst = 0.0
    for n in range(1, 2001):
        z.step()
        worst = max(worst, np.abs(z.E[0] - shape_E * math.cos(w * n * inp.dt)).max()
                    / np.abs(shape_E).max())
        worst = max(worst, np.abs(z.H[1] - B * shape_H * math.sin(w * (n - 0.5) * inp.dt)).max()
                    / np.abs(B * shape_H).max())
    assert worst < 2e-12
    for a in (z.E[1], z.E[2], z.H[0], z.H[2]):
        assert np.abs(a).max() < 1e-13


def test_cartesian_limit_3d_yee_dispersion():
    """r_in >> Nr: the grid is Cartesian to O(Nr/r_in).  A TM-like box mode with variation in
    r, phi and z must oscillate at sin^2(w dt/2)/dt^2 = sum_a sin^2(k_a d_a/2)/d_a^2.  Pins the
    r and phi difference terms, their coefficients and the phi wrap."""
    Nr, Nphi, Nz = 12, 8, 10
    r_in = 1.0e6
    n_fold = int(round(2 * math.pi * r_in / Nphi))   # r dphi ~ 1
    inp = make_zone(Nr, Nphi, Nz, r_in=r_in, n_fold=n_fold, courant=0.8)
    z = OracleZone(inp)
    dy = r_in * inp.dphi
    kx = math.pi * 1 / (Nr * inp.dr)
    ky = 2 * math.pi * 1 / (Nphi * dy)
    kz = math.pi * 1 / (Nz * inp.dz)
    s2 = (math.sin(kx / 2) ** 2 + (math.sin(ky * dy / 2) / dy) ** 2 + math.sin(kz / 2) ** 2)
    w_exact = 2.0 / inp.dt * math.asin(inp.dt * math.sqrt(s2))
    # TM-to-z box mode: Ez ~ sin(kx x) cos(ky y) cos(kz z') on its own nodes, started from Ez only
    x = np.arange(Nr) * inp.dr
    y = np.arange(Nphi) * dy
    zz = (np.arange(Nz) + 0.5) * inp.dz
    z.E[2][:] = np.sin(kx * x)[:, None, None] * np.cos(ky * y)[None, :, None] * np.cos(kz * zz)[None, None, :]
    # complete the mode so that div E = 0 (discrete): Ex, Ey from the TM relations
    xh = x + 0.5 * inp.dr
    yh = y + 0.5 * dy
    zi = np.arange(Nz) * inp.dz
    kc2 = (2 * math.sin(kx / 2)) ** 2 + (2 * math.sin(ky * dy / 2) / dy) ** 2
    Kx, Ky, Kz = 2 * math.sin(kx / 2), 2 * math.sin(ky * dy / 2) / dy, 2 * math.sin(kz / 2)
    z.E[0][:] = (-Kx * Kz / kc2) * (np.cos(kx * xh)[:, None, None] * np.cos(ky * y)[None, :, None]
                                     * np.sin(kz * zi)[None, None, :])
    z.E[1][:] = (Ky * Kz / kc2) * (np.sin(kx * x)[:, None, None] * np.sin(ky * yh)[None, :, None]
                                    * np.sin(kz * zi)[None, None, :])
    series = []
    for n in range(600):
        z.step()
        series.append(z.E[2][Nr // 3, 1, Nz // 3])
    w_num = freq_from_series(series, inp.dt)
    assert abs(w_num / w_exact - 1.0) < 5e-5       # O(Nr / r_in) = 1.2e-5


def _tm0n0_error(R_cells, n=1):
    """Relative error of the oracle's TM0n0 frequency against x_0n / R with x_0n READ FROM THE GOLDEN FILE (the value
    the paper's target quotes, 4 digits); the mode is started from J0(x r / R) with scipy's full-precision zero so that
    no neighbouring mode is excited."""
    Nr, Nphi, Nz = R_cells, 4, 2
    inp = make_zone(Nr, Nphi, Nz, r_in=0.0, n_fold=1, has_axis=True, courant=0.9)
    z = OracleZone(inp)
    x_file = _golden_zeros()["j0_zero_%d" % n]
    x0n = special.jn_zeros(0, n)[n - 1]
    assert abs(x0n - x_file) < 5e-4          # the file's 4 digits
    R = Nr * inp.dr
    r = np.arange(Nr) * inp.dr
    z.E[2][:] = special.j0(x0n * r / R)[:, None, None]
    series = []
    for _ in range(4000):
        z.step()
        series.append(z.E[2][Nr // 4, 0, 0])
    w = freq_from_series(series, inp.dt)
    return w / (x_file / R) - 1.0


def test_tm010_bessel_zero_second_order():
    """TM010 of a PEC cylinder (axis zone): w = 2.405/R, error O(dr^2) (-2.6e-3 -> -6.8e-4)."""
    e10, e20 = _tm0n0_error(10), _tm0n0_error(20)
    assert abs(e20) < 1.0e-3
    assert abs(e10) < 4.0e-3
    assert 3.0 < e10 / e20 < 5.0


@pytest.mark.parametrize("n", [2, 3])
def test_tm0n0_higher_bessel_zeros_second_order(n):
    """TM020 / TM030 (5.520 / R, 8.654 / R; north_star "TM0n0 resonant frequencies from Bessel zeros", SURVEY 8(c)
    pin 3): the radial operator and the r = 0 loop integral at shorter radial wavelengths.  Error O((x dr / R)^2):
    fourfold smaller from R = 20 to R = 40 cells, and about (x_0n / x_01)^2 times TM010's at equal R."""
    e20, e40 = _tm0n0_error(20, n), _tm0n0_error(40, n)
    print("TM0%d0 error at R = 20 / 40 cells: %.3e / %.3e" % (n, e20, e40))
    scale = (_golden_zeros()["j0_zero_%d" % n] / _golden_zeros()["j0_zero_1"]) ** 2
    assert abs(e20) < 1.0e-3 * scale * 1.3
    assert 3.3 < e20 / e40 < 4.7


def _te111_error(R_cells, Nphi, L_cells=12):
    Nr, Nz = R_cells, L_cells
    inp = make_zone(Nr, Nphi, Nz, r_in=0.0, n_fold=1, has_axis=True, courant=0.9)
    z = OracleZone(inp)
    xp = special.jnp_zeros(1, 1)[0]
    assert abs(xp - _golden_zeros()["j1p_zero_1"]) < 5e-4
    R, L = Nr * inp.dr, Nz * inp.dz
    kc, beta = xp / R, math.pi / L
    w_exact = math.sqrt(kc ** 2 + beta ** 2)
    ri = np.arange(Nr) * inp.dr
    rh = ri + 0.5 * inp.dr
    ph = np.arange(Nphi) * inp.dphi
    phh = ph + 0.5 * inp.dphi
    zk = np.arange(Nz) * inp.dz
    # E_r = (1/r) J1(kc r) sin(phi) sin(beta z),  E_phi = kc J1'(kc r) cos(phi) sin(beta z)
    z.E[0][:] = ((special.jv(1, kc * rh) / rh)[:, None, None] * np.sin(ph)[None, :, None]
                 * np.sin(beta * zk)[None, None, :])
    z.E[1][:] = ((kc * special.jvp(1, kc * ri))[:, None, None] * np.cos(phh)[None, :, None]
                 * np.sin(beta * zk)[None, None, :])
    z.E[1][0] = 0.0     # Ephi[0] is held at 0 on the axis (Step 5)
    series = []
    for n in range(6000):
        z.step()
        series.append(z.H[2][Nr // 2, 0, Nz // 2])
    w = freq_from_series(series, inp.dt)
    return w / w_exact - 1.0


def test_te111_crosses_axis():
    """TE111 (transverse field crossing the axis; x'_11 = 1.841): converges in dphi to the O(dr^2)
    floor."""
    e8, e16, e32 = (_te111_error(10, n) for n in (8, 16, 32))
    assert abs(e16) < 8e-3 and abs(e32) < 6e-3
    d1, d2 = abs(e8 - e16), abs(e16 - e32)
    assert d2 < d1 and 2.5 < d1 / d2 < 6.0


def _bor_te111_error(R_cells, n_fold, m=1, L_cells=12, T=300.0):
    """Continuous-axisymmetric first zone as the paper runs it: ONE phi cell,
    complex fields, wrap phase p = exp(i m dphi), axis at i = 0 with Ez(0) = 0 for m != 0.  TE111 of a PEC cylinder:
    H_z = J_1(kc r) e^{i m phi} sin-profile in z.  Returns w / w_ref - 1 with w_ref the Yee dispersion in z and t of
    the exact radial eigenvalue kc = x'_11 / R, so that what is left is the radial + azimuthal discretisation."""
    Nr, Nz = R_cells, L_cells
    dphi = 2.0 * math.pi / n_fold
    dt = 0.9 * cfl_limit(1.0, 1.0, dphi, 0.0, True, 1, np.exp(1j * m * dphi))      # R21
    inp = make_zone(Nr, 1, Nz, r_in=0.0, n_fold=n_fold, has_axis=True, dt=dt, complex_fields=True, m=m)
    z = OracleZone(inp)
    xp = special.jnp_zeros(1, 1)[0]
    R, L = Nr * inp.dr, Nz * inp.dz
    kc, beta = xp / R, math.pi / L
    bz = 2.0 / inp.dz * math.sin(beta * inp.dz / 2.0)
    w_ref = 2.0 / inp.dt * math.asin(inp.dt / 2.0 * math.sqrt(kc ** 2 + bz ** 2))
    ri = np.arange(Nr) * inp.dr
    rh = ri + 0.5 * inp.dr
    zk = np.arange(Nz) * inp.dz
    # E_r = (i m / r) J1(kc r) e^{i m phi_0},  E_phi = -kc J1'(kc r) e^{i m phi_{1/2}}
    z.E[0][:] = (1j * m * special.jv(1, kc * rh) / rh)[:, None, None] * np.sin(beta * zk)[None, None, :]
    z.E[1][:] = ((-kc * special.jvp(1, kc * ri))[:, None, None] * np.exp(0.5j * m * inp.dphi)
                 * np.sin(beta * zk)[None, None, :])
    z.E[1][0] = 0.0
    series = []
    for n in range(int(T / inp.dt)):
        z.step()
        series.append(z.H[2][Nr // 2, 0, Nz // 2])
    return freq_from_complex_series(series, inp.dt, w_ref) / w_ref - 1.0


def test_bor_first_zone_te111_one_phi_cell():
    """Pins the Nphi = 1 Bloch reading of the axisymmetric first zone (R2, R4, R21): second order in dphi
    ((p - 1)/dphi -> i m), a radial error below 5e-5 at 10 cells once dphi is small, and m = -1 degenerate with m = +1.
    A wrong sign of the wrap phase relative to the half-cell phi offset, a non-zero on-axis Ez for m != 0 or a
    non-conservative radial difference at i = 1/2 moves the frequency by far more than these bounds."""
    e8, e16, e256 = (_bor_te111_error(10, n) for n in (8, 16, 256))
    assert abs(e256) < 5e-5
    assert 3.0 < e8 / e16 < 5.0 and e8 < 0
    assert abs(_bor_te111_error(20, 256, T=200.0)) < 1e-5
    assert _bor_te111_error(10, 16, m=-1) == pytest.approx(e16, rel=1e-6)


def _bor_growth(m, dz, factor, steps=3000):
    """max |E| after `steps` steps from random data, relative to the start, for a one-phi-cell axis zone run at
    `factor` times the R21 limit (the constructor's own check is bypassed for factor > 1)."""
    import oracle.zone as oz
    n_fold = 1024
    dphi = 2.0 * math.pi / n_fold
    p = np.exp(1j * m * dphi)
    dt = factor * cfl_limit(1.0, dz, dphi, 0.0, True, 1, p)
    saved = oz.cfl_limit
    oz.cfl_limit = lambda *a, **k: float("inf")
    try:
        z = OracleZone(make_zone(16, 1, 8, r_in=0.0, n_fold=n_fold, has_axis=True, dt=dt, dz=dz,
                                 complex_fields=True, m=m))
    finally:
        oz.cfl_limit = saved
    rng = np.random.default_rng(0)
    for c in range(3):
        z.E[c][:] = rng.standard_normal(z.E[c].shape) + 1j * rng.standard_normal(z.E[c].shape)
    z.E[1][0] = 0.0
    z.E[2][0] = 0.0
    e0 = max(np.abs(e).max() for e in z.E)
    for n in range(steps):
        z.step()
        if n % 100 == 0 and max(np.abs(e).max() for e in z.E) > 1e8 * e0:
            break
    return max(np.abs(e).max() for e in z.E) / e0


@pytest.mark.parametrize("m", [0, 1, 2, 3])
@pytest.mark.parametrize("dz", [1.0, 0.5])
def test_one_phi_cell_cfl_limit_is_stable_and_tight(m, dz):
    """R21: with Nphi = 1 the phi term of the CFL limit is (K^2 + 1/2 [axis]) / (2 r_min)^2, K = |p - 1|/dphi, not
    1/(r_min dphi)^2 (which would shrink dt with the arbitrary dphi of a continuously axisymmetric zone).  At the
    limit random data stay bounded over 3000 steps; 25 % above it they blow up, so the limit is not slack."""
    assert _bor_growth(m, dz, 1.0) < 50.0
    assert _bor_growth(m, dz, 1.25) > 1e6
