"""Pins of the oracle's density -> eps map (PAPER.md:72-76 Eq. 6; :83)."""
import numpy as np

from oracle import density as D
from workloads import DensityMap


def test_filter_preserves_constants_and_mass():
    rho = np.full((12, 9), 0.37)
    assert np.allclose(D.filter_density(rho, 3.0), 0.37, atol=1e-15)
    R, w = D.gaussian_weights(3.0)
    assert R == 9 and len(w) == 19 and abs(w.sum() - 1) < 1e-15 and np.allclose(w, w[::-1])


def test_filter_is_periodic_in_phi_and_clamped_in_r():
    rng = np.random.default_rng(0)
    rho = rng.random((10, 8))
    f = D.filter_density(rho, 1.0)
    # periodic: rolling the input in phi rolls the output
    assert np.allclose(D.filter_density(np.roll(rho, 3, axis=1), 1.0), np.roll(f, 3, axis=1), atol=1e-15)
    # brute force: out[i,j] = sum_{a,b} w_a w_b rho[clamp(i+a), (j+b) mod n]
    R, w = D.gaussian_weights(1.0)
    ref = np.zeros_like(rho)
    for i in range(10):
        for j in range(8):
            for a in range(-R, R + 1):
                for b in range(-R, R + 1):
                    ref[i, j] += w[a + R] * w[b + R] * rho[min(max(i + a, 0), 9), (j + b) % 8]
    assert np.allclose(f, ref, atol=1e-14)


def test_projection_endpoints_and_eq6():
    for beta, eta in ((8.0, 0.5), (2.0, 0.3)):
        assert abs(D.project(np.array(0.0), beta, eta)) < 1e-15
        assert abs(D.project(np.array(1.0), beta, eta) - 1.0) < 1e-15
    dm = DensityMap(rho=np.array([[0.0, 1.0]] * 2), eps0=1.0, eps_h=11.7, filt_sigma=1e-3, beta=8.0, eta=0.5)
    eps = D.density_to_eps(dm, 3)
    assert eps.shape == (2, 2, 3)
    assert np.allclose(eps[:, 0], 1.0) and np.allclose(eps[:, 1], 11.7)


def test_filter_transpose_and_vjp_vs_finite_differences():
    rng = np.random.default_rng(1)
    x, y = rng.random((16, 16)), rng.random((16, 16))
    assert abs(np.sum(D.filter_density(x, 3.0) * y) - np.sum(x * D.filter_density_T(y, 3.0))) < 1e-12
    dm = DensityMap(rho=rng.random((16, 16)), eps0=1.0, eps_h=6.25, filt_sigma=3.0, beta=8.0, eta=0.5)
    Wt = rng.standard_normal((16, 16, 4))
    f = lambda rho: float(np.sum(Wt * D.density_to_eps(DensityMap(rho, 1.0, 6.25, 3.0, 8.0, 0.5), 4)))
    g = D.density_vjp(dm, Wt)
    for (i, j) in [(0, 0), (3, 15), (8, 7), (15, 2)]:
        h = 1e-6
        rp, rm = dm.rho.copy(), dm.rho.copy()
        rp[i, j] += h
        rm[i, j] -= h
        fd = (f(rp) - f(rm)) / (2 * h)
        assert abs(g[i, j] - fd) < 1e-6 * max(1.0, abs(fd))
