"""Pins of the oracle against invariants: the W-weighted leap-frog energy in a lossless PEC box
(SURVEY A1 / pin 2), m <-> -m conjugation and complex(p=1) == real (pin 6), the running DFT against
its plain definition and against numpy's FFT (Step 7 / A8), CPML coefficient closed forms (Step 2)."""
import math

import numpy as np
import pytest

from helpers import make_zone
from oracle import OracleZone, cpml_profile


def _pec(z):
    z.E[0][:, :, 0] = 0
    z.E[1][:, :, 0] = 0
    z.E[1][0] = 0
    z.E[2][0] = 0


def _random_state(z, rng):
    inp = z.inp
    for c in range(3):
        a = rng.standard_normal(z.shape)
        if z.cplx:
            a = a + 1j * rng.standard_normal(z.shape)
        z.E[c][:] = a
    _pec(z)   # PEC zeros (Step 1) and the axis rules (Step 5)
    if inp.has_axis and not z.cplx:
        z.E[2][0] = rng.standard_normal(inp.Nz)[None, :]   # replicated over j


@pytest.mark.parametrize("case", ["annulus-real", "annulus-bloch", "axis-real", "axis-bloch-Ez0held"])
def test_energy_conserved(case):
    """1/2 sum W eps |E^n|^2 + 1/2 sum W Re(H^{n+1/2} conj H^{n-1/2}) is constant (PEC box, any eps >= 1,
    any phase, with or without the axis) <=> curl_H is the exact W-weighted transpose of curl_E."""
    rng = np.random.default_rng(7)
    cplx = "bloch" in case
    axis = "axis" in case
    Nr, Nphi, Nz = 9, 6, 7
    if axis:
        inp = make_zone(Nr, Nphi, Nz, r_in=0.0, n_fold=(3 if cplx else 1), has_axis=True, courant=0.9,
                        complex_fields=cplx, m=1)
    else:
        inp = make_zone(Nr, Nphi, Nz, r_in=4.0, n_fold=5, courant=0.9, complex_fields=cplx, m=2)
    eps_design = 1.0 + 10.0 * rng.random((Nr, Nphi, Nz))
    if axis:
        eps_design[0] = eps_design[0].mean(axis=0)[None, :]   # one eps per axis cell
    inp.design_i0, inp.design_i1, inp.design_k0, inp.design_k1 = 0, Nr, 0, Nz
    z = OracleZone(inp, eps_design=eps_design)
    _random_state(z, rng)
    hist = []            # (E^n, H^{n-1/2}) for n = 1, 2, ...
    for n in range(300):
        z.step()
        hist.append(([e.copy() for e in z.E], [h.copy() for h in z.H]))
    vals = []
    for n in range(len(hist) - 1):
        E_n, H_nm = hist[n]
        H_np = hist[n + 1][1]
        z.E, z.H = E_n, H_np
        vals.append(z.energy(H_nm))
    vals = np.array(vals)
    assert vals.min() > 0
    assert np.abs(vals / vals[0] - 1.0).max() < 1e-12


def test_m_and_minus_m_are_conjugates():
    outs = []
    for m in (+1, -1):
        inp = make_zone(10, 5, 8, r_in=6.0, n_fold=7, courant=0.9, complex_fields=True, m=m,
                        npml_r=(3, 3), npml_z=(3, 3))
        z = OracleZone(inp)
        rs = np.random.default_rng(11)
        for c in range(3):
            a = rs.standard_normal(z.shape) + 1j * rs.standard_normal(z.shape)
            z.E[c][:] = a if m == 1 else np.conj(a)
        _pec(z)
        for n in range(50):
            z.step()
        outs.append([e.copy() for e in z.E] + [h.copy() for h in z.H])
    for a, b in zip(*outs):
        assert np.abs(a - np.conj(b)).max() <= 1e-13 * np.abs(a).max()


def test_complex_mode_with_p_one_equals_real_mode():
    res = []
    for cplx in (False, True):
        inp = make_zone(10, 5, 12, r_in=6.0, n_fold=7, courant=0.9, complex_fields=cplx, m=0,
                        npml_r=(3, 3), npml_z=(3, 3))
        z = OracleZone(inp)
        rs = np.random.default_rng(5)
        for c in range(3):
            z.E[c][:] = rs.standard_normal(z.shape)
        _pec(z)
        for n in range(60):
            z.step()
        res.append([np.array(e) for e in z.E])
    for a, b in zip(*res):
        assert np.abs(b.imag).max() == 0.0
        assert np.array_equal(a, b.real)


def test_running_dft_equals_definition_and_fft():
    """Ehat = dt sum_{n=1..Nt} E^n exp(+i w n dt) (A8).  For w on an FFT bin, w = 2 pi q/(Nt dt),
    this is dt * Nt * ifft(x)[q] with x[n mod Nt] = E^n."""
    Nt, q = 256, 9
    inp = make_zone(8, 4, 10, r_in=5.0, n_fold=6, courant=0.9)
    w_bin = 2 * math.pi * q / (Nt * inp.dt)
    inp.omega = np.array([w_bin, 0.37])
    inp.design_i0, inp.design_i1, inp.design_k0, inp.design_k1 = 2, 6, 3, 7
    inp.monitor_k = 8
    z = OracleZone(inp)
    rs = np.random.default_rng(2)
    for c in range(3):
        z.E[c][:] = rs.standard_normal(z.shape)
    _pec(z)
    dft = z._new_dft()
    rec_d, rec_m = [], []
    for n in range(Nt):
        z.step(dft=dft)
        rec_d.append(z.E[1][3, 2, 4])      # design-box voxel (1, 2, 1), component phi
        rec_m.append(z.E[0][5, 1, 8])      # monitor point, component r
    rec_d, rec_m = np.array(rec_d), np.array(rec_m)
    n = np.arange(1, Nt + 1)
    for f, w in enumerate(inp.omega):
        direct_d = inp.dt * np.sum(rec_d * np.exp(1j * w * n * inp.dt))
        direct_m = inp.dt * np.sum(rec_m * np.exp(1j * w * n * inp.dt))
        assert abs(dft["design"][f, 1, 1, 2, 1] - direct_d) < 1e-12 * abs(direct_d)
        assert abs(dft["monitor"][f, 0, 5, 1] - direct_m) < 1e-12 * abs(direct_m)
    x = np.roll(rec_d, 1)   # x[n mod Nt] = E^n, n = 1..Nt  ->  x[0] = E^Nt
    fft_val = inp.dt * Nt * np.fft.ifft(x)[q]
    assert abs(dft["design"][0, 1, 1, 2, 1] - fft_val) < 1e-11 * abs(fft_val)


def test_cpml_coefficients_closed_forms():
    dt, p, smax, amax = 0.5, 3.0, 3.2, 0.05
    pr = cpml_profile(40, 8, 8, dt, p, smax, 1.0, amax)
    # wall node q = 0: x = 1 -> sigma = sigma_max, alpha = 0, kappa = 1: b = exp(-sigma dt), c = b - 1
    assert pr["b_i"][0] == pytest.approx(math.exp(-smax * dt), rel=1e-15)
    assert pr["c_i"][0] == pytest.approx(math.exp(-smax * dt) - 1.0, rel=1e-14)
    # half node q = 7.5: x = 1/16
    x = 0.5 / 8
    s, a = smax * x ** 3, amax * (1 - x)
    b = math.exp(-(s + a) * dt)
    assert pr["b_h"][7] == pytest.approx(b, rel=1e-15)
    assert pr["c_h"][7] == pytest.approx(s * (b - 1) / (s + a), rel=1e-14)
    # mirror symmetry: integer q = N - d  <->  q = d ; half q = N - 1/2 - d <-> 1/2 + d
    assert np.allclose(pr["c_i"][1:8], pr["c_i"][:-8:-1], rtol=1e-14)
    assert np.allclose(pr["c_h"][:8], pr["c_h"][::-1][:8], rtol=1e-14)
    # interior: psi stays 0 and 1/kappa = 1
    assert np.all(pr["c_i"][8:33] == 0) and np.all(pr["c_h"][8:32] == 0)
    assert np.all(pr["ik_i"] == 1.0)
    # kappa grading
    pk = cpml_profile(40, 8, 0, dt, p, smax, 5.0, amax)
    assert pk["ik_i"][0] == pytest.approx(1 / 5.0)
    assert np.all(pk["c_i"][8:] == 0)
