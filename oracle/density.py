"""ORACLE (test infrastructure): density -> eps map and its transpose (VJP).

PAPER.md:72-76 Eq. 6: eps(p) = p (eps_h - eps_0) + eps_0; "standard
binarization and conic filters".  BASELINE.json's configs fix the variant used here
(SURVEY 8(c) A13): a separable Gaussian filter in index space (sigma cells, truncated at
+-ceil(3 sigma), weights normalised to 1, phi-periodic, r edge-clamped), then the tanh
projection  rho_bar = [tanh(beta eta) + tanh(beta (rho_f - eta))] / [tanh(beta eta) + tanh(beta (1 - eta))],
then Eq. 6, extruded over the design layer (A14).  Plain loops / NumPy float64.
"""
from __future__ import annotations

import math

import numpy as np


def gaussian_weights(sigma):
    R = int(math.ceil(3.0 * sigma))
    d = np.arange(-R, R + 1, dtype=np.float64)
    w = np.exp(-0.5 * (d / sigma) ** 2)
    return R, w / w.sum()


def filter_density(rho, sigma):
    """rho (Nr_d, Nphi) -> filtered: first along r (edge-clamped), then along phi (periodic)."""
    n_r, n_phi = rho.shape
    R, w = gaussian_weights(sigma)
    tmp = np.zeros_like(rho, dtype=np.float64)
    for i in range(n_r):
        for t, d in enumerate(range(-R, R + 1)):
            ii = min(max(i + d, 0), n_r - 1)
            tmp[i, :] += w[t] * rho[ii, :]
    out = np.zeros_like(tmp)
    for j in range(n_phi):
        for t, d in enumerate(range(-R, R + 1)):
            out[:, j] += w[t] * tmp[:, (j + d) % n_phi]
    return out


def filter_density_T(g, sigma):
    """Transpose of ``filter_density`` (scatter form)."""
    n_r, n_phi = g.shape
    R, w = gaussian_weights(sigma)
    tmp = np.zeros_like(g, dtype=np.float64)
    for j in range(n_phi):
        for t, d in enumerate(range(-R, R + 1)):
            tmp[:, (j + d) % n_phi] += w[t] * g[:, j]
    out = np.zeros_like(tmp)
    for i in range(n_r):
        for t, d in enumerate(range(-R, R + 1)):
            ii = min(max(i + d, 0), n_r - 1)
            out[ii, :] += w[t] * tmp[i, :]
    return out


def project(rho_f, beta, eta):
    den = math.tanh(beta * eta) + math.tanh(beta * (1.0 - eta))
    return (math.tanh(beta * eta) + np.tanh(beta * (rho_f - eta))) / den


def project_deriv(rho_f, beta, eta):
    den = math.tanh(beta * eta) + math.tanh(beta * (1.0 - eta))
    return beta * (1.0 - np.tanh(beta * (rho_f - eta)) ** 2) / den


def density_to_eps(dm, n_layers):
    """DensityMap -> eps on the design box, shape (Nr_d, Nphi, n_layers)."""
    rho_f = filter_density(np.asarray(dm.rho, np.float64), dm.filt_sigma)
    rho_bar = project(rho_f, dm.beta, dm.eta)
    eps2d = dm.eps0 + rho_bar * (dm.eps_h - dm.eps0)
    return np.repeat(eps2d[:, :, None], n_layers, axis=2)


def density_vjp(dm, dF_deps):
    """dF/drho (Nr_d, Nphi) from dF/deps on the design box (Nr_d, Nphi, L_d):
    sum over the layer, times (eps_h - eps_0), times the projection derivative, transposed filter."""
    g2d = dF_deps.sum(axis=2) * (dm.eps_h - dm.eps0)
    rho_f = filter_density(np.asarray(dm.rho, np.float64), dm.filt_sigma)
    g2d = g2d * project_deriv(rho_f, dm.beta, dm.eta)
    return filter_density_T(g2d, dm.filt_sigma)
