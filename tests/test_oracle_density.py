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


def _conic_dm(rho, radius=4.0, r_first=2000.5, dr=1.0, dphi=None):
    dphi = (1.0 / r_first) if dphi is None else dphi
    return DensityMap(rho=rho, eps0=1.0, eps_h=6.25, beta=8.0, eta=0.5, conic_radius=radius, r_first=r_first, dr=dr,
                      dphi=dphi)


def test_conic_filter_is_the_written_out_cone_in_the_physical_metric():
    """PAPER.md:87, 133 conic filter, R22: rho_f(i, j) = sum w rho / sum w over ALL periodic images with
    w = max(0, 1 - d/R), d^2 = (a dr)^2 + (rbar b dphi)^2.  Brute force with its own loops (images enumerated over a
    generous integer range instead of the oracle's b_max), on a thin wedge whose support wraps around phi twice."""
    rng = np.random.default_rng(2)
    n_r, n_phi, Rad, r0, dr, dphi = 9, 3, 2.5, 4.5, 1.0, 0.11
    rho = rng.random((n_r, n_phi))
    f = D.conic_filter(rho, _conic_dm(rho, Rad, r0, dr, dphi))
    ref = np.zeros_like(rho)
    for i in range(n_r):
        for j in range(n_phi):
            num = den = 0.0
            for ii in range(n_r):
                for bb in range(-40, 41):
                    rbar = 0.5 * ((r0 + i * dr) + (r0 + ii * dr))
                    d = np.hypot((i - ii) * dr, rbar * bb * dphi)
                    if d < Rad:
                        num += (1.0 - d / Rad) * rho[ii, (j + bb) % n_phi]
                        den += 1.0 - d / Rad
            ref[i, j] = num / den
    assert np.allclose(f, ref, atol=1e-14)
    # the cone at r ~ 4.5 reaches b = floor(2.5 / (4.5 * 0.11)) = 5 > Nphi: images must have been added
    assert D.conic_offsets(_conic_dm(rho, Rad, r0, dr, dphi), n_r)[1] == 5


def test_conic_filter_constants_support_and_cartesian_limit():
    # constants are preserved (normalisation), also at the r edges where the cone is truncated
    dm = _conic_dm(np.full((12, 16), 0.37))
    assert np.allclose(D.conic_filter(dm.rho, dm), 0.37, atol=1e-15)
    # impulse response: support = cells with d < R in the PHYSICAL metric; halving r dphi doubles the phi reach
    imp = np.zeros((21, 32))
    imp[10, 16] = 1.0
    for scale, reach in ((1.0, 3), (0.5, 7)):
        dmi = _conic_dm(imp, radius=4.0, r_first=1e6 + 0.5, dphi=scale / 1e6)
        resp = D.conic_filter(imp, dmi, normalise=False)
        assert resp[10, 16] == 1.0 and resp[10, 16 + reach] > 0 and resp[10, 16 + reach + 1] == 0.0
        assert resp[10 + 3, 16] > 0 and resp[10 + 4, 16] == 0.0
    # r >> R with r dphi = dr: the textbook 2-D cone w = max(0, 1 - sqrt(a^2 + b^2)/R)
    dmc = _conic_dm(imp, radius=4.0, r_first=1e9 + 0.5, dphi=1.0 / 1e9)
    resp = D.conic_filter(imp, dmc, normalise=False)
    a, b = np.meshgrid(np.arange(21) - 10, np.arange(32) - 16, indexing="ij")
    assert np.allclose(resp, np.maximum(0.0, 1.0 - np.hypot(a, b) / 4.0), atol=1e-7)


def test_conic_filter_transpose_and_vjp_vs_finite_differences():
    rng = np.random.default_rng(3)
    x, y = rng.random((14, 6)), rng.random((14, 6))
    dm = _conic_dm(x, radius=3.3, r_first=5.5, dphi=2 * np.pi / (8 * 6))
    assert abs(np.sum(D.conic_filter(x, dm) * y) - np.sum(x * D.conic_filter_T(y, dm))) < 1e-12
    Wt = rng.standard_normal((14, 6, 3))
    from dataclasses import replace
    f = lambda rho: float(np.sum(Wt * D.density_to_eps(replace(dm, rho=rho), 3)))
    g = D.density_vjp(dm, Wt)
    for (i, j) in [(0, 0), (3, 5), (8, 2), (13, 4)]:
        h = 1e-6
        rp, rm = dm.rho.copy(), dm.rho.copy()
        rp[i, j] += h
        rm[i, j] -= h
        fd = (f(rp) - f(rm)) / (2 * h)
        assert abs(g[i, j] - fd) < 1e-6 * max(1.0, abs(fd))
