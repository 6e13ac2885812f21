"""Small zone builders for the oracle pins (inputs only; no method arithmetic)."""
import math

import numpy as np

from workloads import ZoneInputs, cpml_sigma_max


def make_zone(Nr, Nphi, Nz, r_in, n_fold=1, dt=None, courant=0.9, dr=1.0, dz=1.0, complex_fields=False,
              m=0, has_axis=False, npml_r=(0, 0), npml_z=(0, 0), omega=(), **kw):
    dphi = 2.0 * math.pi / (n_fold * Nphi)
    r_min = 0.5 * dr if has_axis else r_in
    lim = 1.0 / math.sqrt(1 / dr ** 2 + 1 / dz ** 2 + 1 / (r_min * dphi) ** 2)
    if dt is None:
        dt = courant * lim
    phase = complex(np.exp(2j * math.pi * m / n_fold)) if complex_fields else 1.0 + 0j
    p = 3.0
    base = dict(
        name="test", Nr=Nr, Nphi=Nphi, Nz=Nz, dr=dr, dphi=dphi, dz=dz, r_in=r_in, dt=dt, n_fold=n_fold,
        phase=phase, complex_fields=complex_fields, has_axis=has_axis,
        npml_r_lo=npml_r[0], npml_r_hi=npml_r[1], npml_z_lo=npml_z[0], npml_z_hi=npml_z[1],
        cpml_p=p, cpml_sigma_max_r=cpml_sigma_max(p, dr), cpml_sigma_max_z=cpml_sigma_max(p, dz),
        omega=np.asarray(omega, dtype=np.float64), eps_bg_z=np.ones(Nz))
    base.update(kw)
    return ZoneInputs(**base)


def freq_from_series(x, dt):
    """omega of a (nearly) pure sinusoid from cos(w dt) = sum x[n](x[n+1]+x[n-1]) / (2 sum x[n]^2)."""
    x = np.asarray(x, dtype=np.float64)
    c = np.sum(x[1:-1] * (x[2:] + x[:-2])) / (2.0 * np.sum(x[1:-1] ** 2))
    return math.acos(c) / dt


def freq_from_complex_series(x, dt, w_guess, order=6):
    """omega of the component nearest w_guess in a sum of complex exponentials a_k exp(-i w_k t) (Prony /
    linear prediction on the series decimated to about one sample per time unit)."""
    dec = max(1, int(1.0 / dt))
    x = np.asarray(x, dtype=np.complex128)[::dec]
    h = dt * dec
    A = np.array([x[i:i + order] for i in range(len(x) - order)])
    c = np.linalg.lstsq(A, x[order:], rcond=None)[0]
    roots = np.roots(np.concatenate([[1.0], -c[::-1]]))
    w = 1j * np.log(roots) / h
    return float(w[np.argmin(np.abs(w.real - w_guess) + 10.0 * np.abs(w.imag))].real)
