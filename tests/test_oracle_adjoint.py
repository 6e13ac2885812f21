"""Pins of the oracle's adjoint path (SURVEY 8(c) Steps 8-10, readings A9, A11, A12):
(i) the constructed broadband adjoint current has exactly the prescribed half-step DTFT at every design
frequency (direct summation of the time series), (ii) the adjoint gradient equals central finite
differences of the objective on a tiny zone, for real fields with two frequencies from one adjoint run and
for complex Bloch m = 1 fields."""
import math

import numpy as np
import pytest

from helpers import make_zone
from oracle import OracleZone
from workloads import focal_point_weights, gaussian_pulse_table, plane_wave_sheet


def _tiny(cplx, lambdas, n_steps, seed=0):
    Nr, Nphi, Nz = 26, 5, 40
    inp = make_zone(Nr, Nphi, Nz, r_in=20.0, n_fold=8 * 16 // Nphi, dt=0.5, complex_fields=cplx, m=1,
                    npml_r=(6, 6), npml_z=(8, 8), omega=[2 * math.pi / l for l in lambdas])
    inp.design_i0, inp.design_i1, inp.design_k0, inp.design_k1 = 8, 18, 16, 20
    inp.source_k, inp.monitor_k = 11, 28
    rng = np.random.default_rng(seed)
    inp.eps_design = 1.0 + 3.0 * rng.random(inp.design_shape)
    inp.src_A_r, inp.src_A_phi = plane_wave_sheet(Nr, Nphi, inp.dphi, cplx)
    wc = float(np.mean(inp.omega))
    # sigma_t = 20: the pulse has no DC content (exp(-(wc sigma_t)^2/2) ~ 1e-8), so no static field is left behind (A15)
    inp.src_table = gaussian_pulse_table(n_steps, inp.dt, wc, 20.0, 80.0, cplx)
    inp.n_steps = inp.n_steps_adjoint = n_steps
    inp.adj_sigma_t, inp.adj_t0 = 20.0, 80.0
    return inp


@pytest.mark.parametrize("cplx,lambdas", [(False, [20.0]), (False, [18.0, 24.0]), (True, [18.0, 24.0])])
def test_adjoint_source_has_prescribed_dtft(cplx, lambdas):
    n_steps = 600
    inp = _tiny(cplx, lambdas, n_steps)
    z = OracleZone(inp)
    z.run_forward()
    A_r, A_phi, table = z.build_adjoint_source()
    t = (np.arange(n_steps) + 0.5) * inp.dt
    mon = z.dft_fwd["monitor"]
    for (i, j) in [(7, 0), (12, 3), (19, 4)]:
        for c, A in ((0, A_r), (1, A_phi)):
            J_t = np.tensordot(table, A[:, i, j], axes=(0, 0))          # J(t_{n+1/2})
            if not cplx:
                assert np.isrealobj(J_t)
            for f, w in enumerate(inp.omega):
                Jhat = inp.dt * np.sum(J_t * np.exp(1j * w * t))
                target = np.conj(mon[f, c, i, j])
                assert abs(Jhat - target) < 1e-9 * np.abs(mon[:, c]).max()
    # zero inside the r-PML (objective mask)
    assert np.all(A_r[:, :6] == 0) and np.all(A_phi[:, -6:] == 0)


@pytest.mark.parametrize("cplx,lambdas", [(False, [18.0, 24.0]), (True, [20.0])])
def test_adjoint_gradient_matches_central_differences(cplx, lambdas):
    n_steps = 3000
    inp = _tiny(cplx, lambdas, n_steps)
    z = OracleZone(inp)
    z.run_forward()
    F0 = z.objective()
    z.build_adjoint_source()
    z.run_adjoint()
    g = z.gradient()
    voxels = [(2, 1, 0), (5, 3, 2), (8, 0, 3), (4, 4, 1)]
    h = 1e-4
    for v in voxels:
        Fs = []
        for s in (+1, -1):
            e = inp.eps_design.copy()
            e[v] += s * h
            zz = OracleZone(inp, eps_design=e)
            zz.run_forward()
            Fs.append(zz.objective())
        fd = (Fs[0] - Fs[1]) / (2 * h)
        assert abs(g[v] - fd) < 2e-4 * np.abs(g).max(), (v, g[v], fd, F0)
        assert abs(g[v] - fd) < 2e-3 * abs(fd), (v, g[v], fd)


@pytest.mark.parametrize("cplx,lambdas", [(False, [18.0, 24.0]), (True, [20.0])])
def test_focal_intensity_gradient_matches_central_differences(cplx, lambdas):
    """Pins the focal-intensity objective (Eq. 7; R20) and its adjoint source
    a = u_f conj(S_f) g / W: a missing conjugate, a missing 1/W or a wrong frequency weight fails this."""
    n_steps = 3000
    inp = _tiny(cplx, lambdas, n_steps)
    inp.focal_g = focal_point_weights(inp)
    inp.focal_u = np.array([1.0, 0.4][:len(lambdas)])
    z = OracleZone(inp)
    z.run_forward()
    z.build_adjoint_source(kind="focal_intensity")
    z.run_adjoint()
    g = z.gradient()
    h = 1e-4
    for v in [(2, 1, 0), (5, 3, 2), (8, 0, 3)]:
        Fs = []
        for s in (+1, -1):
            e = inp.eps_design.copy()
            e[v] += s * h
            zz = OracleZone(inp, eps_design=e)
            zz.run_forward()
            Fs.append(zz.objective(kind="focal_intensity"))
        fd = (Fs[0] - Fs[1]) / (2 * h)
        assert abs(g[v] - fd) < 2e-4 * np.abs(g).max(), (v, g[v], fd)
        assert abs(g[v] - fd) < 2e-3 * abs(fd), (v, g[v], fd)


def test_focal_sum_is_the_linear_functional():
    """S_f by its definition, written out with loops on a few points."""
    inp = _tiny(False, [20.0], 200)
    inp.focal_g = focal_point_weights(inp)
    z = OracleZone(inp)
    z.run_forward()
    mon = z.dft_fwd["monitor"]
    S = 0.0 + 0.0j
    for c in range(2):
        for i in range(inp.npml_r_lo, inp.Nr - inp.npml_r_hi):
            for j in range(inp.Nphi):
                S += inp.focal_g[0, c, i, j] * mon[0, c, i, j]
    assert abs(z.focal_sums()[0] - S) <= 1e-12 * abs(S)
    assert z.objective(kind="focal_intensity") == pytest.approx(abs(S) ** 2, rel=1e-12)


def test_coherent_pair_gradient_matches_central_differences():
    """The m = +1 / m = -1 members of a pair share one structure and add coherently at the focal point:
    F = u |S_+ + S_-|^2 (``lens_focal_objective``).  Each member's adjoint source carries conj(S_total), not its own
    conj(S); the structure's gradient is the sum of the members' gradients.  Central differences of F catch a missing
    cross term (own S instead of S_total moves the gradient by O(1))."""
    from dataclasses import replace
    from oracle import lens_focal_objective
    n_steps = 3000
    base = _tiny(True, [20.0], n_steps)
    members = []
    for m in (+1, -1):
        A_r, A_phi = plane_wave_sheet(base.Nr, base.Nphi, base.dphi, True, m)
        inp = replace(base, phase=complex(np.exp(2j * math.pi * m / base.n_fold)), src_A_r=A_r, src_A_phi=A_phi)
        inp.focal_g = focal_point_weights(inp, seed=7 + m)
        members.append(inp)
    u = np.array([0.7])

    def solve(eps):
        zs = [OracleZone(inp, eps_design=eps) for inp in members]
        for z in zs:
            z.run_forward()
        return zs

    zs = solve(base.eps_design)
    F0, S = lens_focal_objective(zs, u)
    # the two members must both matter, and interfere
    S_each = [z.focal_sums()[0] for z in zs]
    assert min(abs(S_each[0]), abs(S_each[1])) > 0.05 * max(abs(S_each[0]), abs(S_each[1]))
    g = np.zeros(base.design_shape)
    for z in zs:
        z.inp.focal_u = u
        z.build_adjoint_source(kind="focal_intensity", S_total=S)
        z.run_adjoint()
        g += z.gradient()
    h = 1e-4
    for v in [(2, 1, 0), (5, 3, 2), (8, 0, 3)]:
        Fs = []
        for sgn in (+1, -1):
            e = base.eps_design.copy()
            e[v] += sgn * h
            Fs.append(lens_focal_objective(solve(e), u)[0])
        fd = (Fs[0] - Fs[1]) / (2 * h)
        assert abs(g[v] - fd) < 2e-3 * abs(fd) + 2e-4 * np.abs(g).max(), (v, g[v], fd, F0)
