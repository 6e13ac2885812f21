"""ORACLE (test infrastructure): density -> eps map and its transpose (VJP).

PAPER.md:72-76 Eq. 6: eps(p) = p (eps_h - eps_0) + eps_0; "standard
binarization and conic filters".  BASELINE.json's configs fix the variant used here
(SURVEY 8(c) A13): a separable Gaussian filter in index space (sigma cells, truncated at
+-ceil(3 sigma), weights normalised to 1, phi-periodic, r edge-clamped), then the tanh
projection  rho_bar = [tanh(beta eta) + tanh(beta (rho_f - eta))] / [tanh(beta eta) + tanh(beta (1 - eta))],
then Eq. 6, extruded over the design layer (A14).  Plain loops / NumPy float64.

The paper's own filter ("a conic filter with a radius of 0.08 lambda" / "0.056 lambda";
DESIGN.md R22) is selected by ``conic_radius > 0``: cell (i, j) has its centre at r_i = r_first + i dr, the distance
between (i, j) and (i', j + b) is d = sqrt(((i - i') dr)^2 + (rbar b dphi)^2) with rbar = (r_i + r_i')/2 (the arc is
measured at the mean radius, which keeps the weights symmetric), w = max(0, 1 - d/R); the structure is periodic in phi
with period Nphi cells, so b runs over ALL integers with d < R and lands on cell (j + b) mod Nphi (periodic images
add); in r the sum is truncated at the design region's edges.  rho_f = sum w rho / sum w.
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


def conic_offsets(dm, n_r):
    """Largest |a| and |b| any weight can reach: a_max = floor(R/dr) capped by the region, b_max from the innermost
    arc, d >= (r_first) |b| dphi for a = 0."""
    a_max = min(int(math.floor(dm.conic_radius / dm.dr)), n_r - 1)
    b_max = int(math.floor(dm.conic_radius / (dm.r_first * dm.dphi)))
    return a_max, b_max


def conic_weight(dm, i, ii, b):
    rbar = 0.5 * ((dm.r_first + i * dm.dr) + (dm.r_first + ii * dm.dr))
    d = math.sqrt(((i - ii) * dm.dr) ** 2 + (rbar * b * dm.dphi) ** 2)
    return max(0.0, 1.0 - d / dm.conic_radius)


def conic_filter(rho, dm, normalise=True, weights_only=False):
    """out[i, j] = sum_{a, b} w(i, i + a, b) rho[i + a, (j + b) mod Nphi] (/ sum w if normalise).
    weights_only: returns sum w per cell instead."""
    n_r, n_phi = rho.shape
    a_max, b_max = conic_offsets(dm, n_r)
    out = np.zeros((n_r, n_phi))
    norm = np.zeros(n_r)
    for i in range(n_r):
        for a in range(-a_max, a_max + 1):
            ii = i + a
            if ii < 0 or ii >= n_r:
                continue
            for b in range(-b_max, b_max + 1):
                w = conic_weight(dm, i, ii, b)
                if w <= 0.0:
                    continue
                norm[i] += w
                out[i, :] += w * np.roll(rho[ii, :], -b)        # element j takes rho[ii, (j + b) mod Nphi]
    if weights_only:
        return np.repeat(norm[:, None], n_phi, axis=1)
    return out / norm[:, None] if normalise else out


def conic_filter_T(g, dm):
    """Transpose of the normalised conic filter: divide by the OUTPUT cell's weight sum, then the symmetric
    un-normalised stencil (w(i, i', b) = w(i', i, -b))."""
    norm = conic_filter(g, dm, weights_only=True)
    return conic_filter(g / norm, dm, normalise=False)


def filter_any(rho, dm):
    if dm.conic_radius > 0.0:
        return conic_filter(np.asarray(rho, np.float64), dm)
    return filter_density(np.asarray(rho, np.float64), dm.filt_sigma)


def project(rho_f, beta, eta):
    den = math.tanh(beta * eta) + math.tanh(beta * (1.0 - eta))
    return (math.tanh(beta * eta) + np.tanh(beta * (rho_f - eta))) / den


def project_deriv(rho_f, beta, eta):
    den = math.tanh(beta * eta) + math.tanh(beta * (1.0 - eta))
    return beta * (1.0 - np.tanh(beta * (rho_f - eta)) ** 2) / den


def density_to_eps(dm, n_layers):
    """DensityMap -> eps on the design box, shape (Nr_d, Nphi, n_layers)."""
    rho_f = filter_any(dm.rho, dm)
    rho_bar = project(rho_f, dm.beta, dm.eta)
    eps2d = dm.eps0 + rho_bar * (dm.eps_h - dm.eps0)
    return np.repeat(eps2d[:, :, None], n_layers, axis=2)


def density_vjp(dm, dF_deps):
    """dF/drho (Nr_d, Nphi) from dF/deps on the design box (Nr_d, Nphi, L_d):
    sum over the layer, times (eps_h - eps_0), times the projection derivative, transposed filter."""
    g2d = dF_deps.sum(axis=2) * (dm.eps_h - dm.eps0)
    rho_f = filter_any(dm.rho, dm)
    g2d = g2d * project_deriv(rho_f, dm.beta, dm.eta)
    if dm.conic_radius > 0.0:
        return conic_filter_T(g2d, dm)
    return filter_density_T(g2d, dm.filt_sigma)
