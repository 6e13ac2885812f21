"""Pins of the oracle's near-to-far transform (oracle/farfield.py; Eq. 7-8; R24) against the
closed-form on-axis field of a uniformly illuminated annular aperture (first Rayleigh-Sommerfeld integral, exact):
E_x(0, 0, dz) = E0 [ (dz / R1) exp(i k R1) - (dz / R2) exp(i k R2) ],  R_i = sqrt(a_i^2 + dz^2)."""
import math

import numpy as np
import pytest

from helpers import make_zone
from oracle.farfield import focal_weights, wedge_sums


def _closed_form_one(k, a1, a2, dz):
    R1, R2 = math.hypot(a1, dz), math.hypot(a2, dz)
    return dz / R1 * np.exp(1j * k * R1) - dz / R2 * np.exp(1j * k * R2)


def _closed_form(k, a1, a2, dz, dr=0.0):
    """Uniform x-polarised illumination: E_r carries the cos^2 half of the integrand on its cells [r_i, r_i + dr], i.e. the
    annulus [a1, a2]; E_phi carries the sin^2 half on ITS cells [r_i - dr/2, r_i + dr/2] (the Yee staggering), i.e. the
    annulus shifted inwards by dr/2.  Each half is the exact closed form of its own annulus."""
    return 0.5 * _closed_form_one(k, a1, a2, dz) + 0.5 * _closed_form_one(k, a1 - 0.5 * dr, a2 - 0.5 * dr, dz)


def _S(inp, Er, Ephi, dz):
    """The linear functional written out: S_f = sum_{c, i outside r-PML, j} g E (as OracleZone.focal_sums does)."""
    g = focal_weights(inp, dz)
    m = np.zeros(inp.Nr, bool)
    m[inp.npml_r_lo:inp.Nr - inp.npml_r_hi] = True
    return np.array([np.sum(g[f, 0][m] * Er[m]) + np.sum(g[f, 1][m] * Ephi[m]) for f in range(inp.n_freq)])


def _x_polarised(inp, cplx_m=None):
    """Unit x-polarised field on the Yee positions: E_r = cos(phi_j), E_phi = -sin(phi_{j+1/2}); or its m = +-1 part."""
    phi = np.arange(inp.Nphi) * inp.dphi
    ph2 = phi + 0.5 * inp.dphi
    if cplx_m is None:
        er, ep = np.cos(phi), -np.sin(ph2)
    else:
        s = float(cplx_m)
        er, ep = 0.5 * np.exp(1j * s * phi), 0.5j * s * np.exp(1j * s * ph2)
    return np.ones((inp.Nr, 1)) * er[None, :], np.ones((inp.Nr, 1)) * ep[None, :]


def _annulus(scale, Nphi=64, n_fold=1, cplx=False, m=1, dz=180.0, lam=(20.0, 31.0)):
    """The annulus 40 <= rho < 160 (length units) at dr = 1 / scale, no PML, two frequencies."""
    dr = 1.0 / scale
    inp = make_zone(int(120 * scale), Nphi, 4, r_in=40.0, n_fold=n_fold, dr=dr, dz=1.0, dt=0.01, complex_fields=cplx, m=m,
                    omega=[2 * math.pi / l for l in lam])
    inp.monitor_k = 2
    return inp, dz


def test_uniform_annular_aperture_closed_form_second_order():
    """Full circle (n = 1), real fields.  Pins the kernel h (sign, the 1/R term, dz / R^2), k = omega sqrt(eps), the radii
    of the two staggered components, the r dr dphi quadrature and the cos / -sin projection; error O(dr^2) + O(dphi^2)."""
    errs = []
    for scale, nphi in ((1, 48), (2, 96)):
        inp, dz = _annulus(scale, Nphi=nphi)
        Er, Ep = _x_polarised(inp)
        S = _S(inp, Er, Ep, dz)
        ref = np.array([_closed_form(w, 40.0, 160.0, dz, inp.dr) for w in inp.omega])
        errs.append(np.abs(S - ref).max() / np.abs(ref).max())
    print("near-to-far vs closed form: %.3e (dr = 1, 48 cells of phi), %.3e (dr = 1/2, 96)" % tuple(errs))
    assert errs[0] < 4e-3 and errs[1] < 1e-3
    assert 3.0 < errs[0] / errs[1] < 5.0


def test_background_permittivity_enters_the_wavenumber():
    inp, dz = _annulus(2, Nphi=96)
    inp.eps_bg_z = np.full(inp.Nz, 2.13)
    Er, Ep = _x_polarised(inp)
    S = _S(inp, Er, Ep, dz)
    ref = np.array([_closed_form(w * math.sqrt(2.13), 40.0, 160.0, dz, inp.dr) for w in inp.omega])
    assert np.abs(S - ref).max() / np.abs(ref).max() < 2e-3


@pytest.mark.parametrize("m", [+1, -1])
def test_bloch_wedge_m_pm1_carries_half_of_the_x_polarised_wave(m):
    """n = 8 wedge, complex fields, p = exp(i m tau): the m = +-1 circular component of x-hat focuses to HALF the closed
    form (the plane wave is the sum of its m = +1 and m = -1 components)."""
    inp, dz = _annulus(2, Nphi=12, n_fold=8, cplx=True, m=m)
    Er, Ep = _x_polarised(inp, cplx_m=m)
    S = _S(inp, Er, Ep, dz)
    ref = 0.5 * np.array([_closed_form(w, 40.0, 160.0, dz, inp.dr) for w in inp.omega])
    assert np.abs(S - ref).max() / np.abs(ref).max() < 1e-3


@pytest.mark.parametrize("m", [0, 2, 3])
def test_other_bloch_orders_do_not_reach_the_axis(m):
    """Selection rule: sum_w p^w cos(phi + w tau) = 0 unless m = +-1 (mod n)."""
    inp, dz = _annulus(1, Nphi=12, n_fold=8, cplx=True, m=m)
    C_r, C_p = wedge_sums(inp)
    assert np.abs(C_r).max() < 1e-12 and np.abs(C_p).max() < 1e-12
    g = focal_weights(inp, dz)
    assert np.abs(g).max() < 1e-13


def test_wedge_sum_equals_explicit_continuation_over_the_full_circle():
    """Brute force: continue a random wedge field over all n wedges with the Bloch phase, build a FULL-circle zone (n = 1)
    with it, and compare the two focal sums (pins the direction of the phase and the wedge angle tau = Nphi dphi)."""
    n, Nphi = 5, 6
    inp, dz = _annulus(1, Nphi=Nphi, n_fold=n, cplx=True, m=1)
    rng = np.random.default_rng(3)
    Er = rng.standard_normal((inp.Nr, Nphi)) + 1j * rng.standard_normal((inp.Nr, Nphi))
    Ep = rng.standard_normal((inp.Nr, Nphi)) + 1j * rng.standard_normal((inp.Nr, Nphi))
    S_wedge = _S(inp, Er, Ep, dz)
    full, _ = _annulus(1, Nphi=n * Nphi, n_fold=1, cplx=True, m=0)
    p = complex(inp.phase)
    Er_full = np.concatenate([p ** w * Er for w in range(n)], axis=1)
    Ep_full = np.concatenate([p ** w * Ep for w in range(n)], axis=1)
    S_full = _S(full, Er_full, Ep_full, dz)
    assert np.abs(S_wedge - S_full).max() <= 1e-12 * np.abs(S_full).max()
