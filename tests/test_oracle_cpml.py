"""CPML reflection pins (BASELINE.json north_star: 'CPML reflection below 1e-4'; SURVEY 8(c) pin 4,
readings A5 and A6).  Reflection = max |E_pml - E_ref| / max |E_ref| at probe points, where E_ref is the
same run on a domain long enough that nothing comes back during the window."""
import math

import numpy as np

from helpers import make_zone
from oracle import OracleZone
from workloads import gaussian_pulse_table


def _coax_run(Nz, npml_hi, n_steps, probe_k, src_k=20):
    Nr, Nphi = 4, 1
    inp = make_zone(Nr, Nphi, Nz, r_in=10.0, n_fold=16, dt=0.5, npml_z=(12, npml_hi))
    r_half = inp.r_in + (np.arange(Nr) + 0.5)
    inp.src_A_r = (1.0 / r_half)[None, :, None] * np.ones((1, Nr, Nphi))
    inp.src_A_phi = np.zeros((1, Nr, Nphi))
    inp.src_table = gaussian_pulse_table(n_steps, inp.dt, 2 * math.pi / 20.0, 12.0, 50.0, False)
    inp.source_k = src_k
    z = OracleZone(inp)
    rec = []
    for n in range(n_steps):
        s = inp.src_table[0, n]
        z.step(J_r=np.ascontiguousarray(s * inp.src_A_r[0]), J_phi=np.ascontiguousarray(0 * inp.src_A_r[0]),
               source_k=src_k)
        rec.append(z.E[0][1, 0, probe_k])
    return np.array(rec)


def test_z_cpml_reflection_below_1e4_with_12_cells():
    """Coax TEM pulse (lambda = 20 cells) hitting a 12-cell z-CPML; PEC radial walls; single pass."""
    n_steps = 700
    with_pml = _coax_run(Nz=120, npml_hi=12, n_steps=n_steps, probe_k=80)
    ref = _coax_run(Nz=120 + 400, npml_hi=12, n_steps=n_steps, probe_k=80)
    refl = np.abs(with_pml - ref).max() / np.abs(ref).max()
    assert np.abs(ref).max() > 1e-3
    assert refl < 1e-4, refl


def _radial_run(Nr_extra, n_steps, npml=12, r_in=2000.0, Nr=160):
    """z-uniform, phi-uniform cylindrical Ez pulse (TM): Nz = 1, Nphi = 1."""
    lo = Nr_extra
    inp = make_zone(Nr + 2 * Nr_extra, 1, 1, r_in=r_in - lo, n_fold=4000, dt=0.5, npml_r=(npml, npml))
    z = OracleZone(inp)
    i = np.arange(inp.Nr) - lo
    c0, wid = Nr / 2.0, 6.0
    z.E[2][:, 0, 0] = np.exp(-((i - c0) ** 2) / (2 * wid ** 2)) * np.cos(2 * math.pi * (i - c0) / 20.0)
    rec = []
    for n in range(n_steps):
        z.step()
        rec.append(z.E[2][lo + 30:lo + Nr - 30, 0, 0].copy())
    return np.array(rec)


def test_r_cpml_reflection_at_config_radius():
    """Quasi-CPML 'full' form in r (A6/R6) at r_in = 2000 with 12 cells, TM polarisation (Ez/Hphi: pins psi_Hphi_r,
    psi_Ez_r).  Measured 2.73e-4 (SURVEY's probe, a different pulse, saw 1.3e-4): the quasi-CPML MISSES north_star's 1e-4 in r at 12 cells (R6 says so); the
    bar is the measured value + 15 %, so that any change of the r-CPML arithmetic shows."""
    n_steps = 600
    a = _radial_run(0, n_steps)
    b = _radial_run(400, n_steps)
    refl = np.abs(a - b).max() / np.abs(b).max()
    print("r-CPML TM reflection at r_in = 2000, 12 cells: %.3e" % refl)
    assert refl < 3.2e-4, refl


# ---- the E_phi / H_r / H_z polarisation: the other four psi arrays --------------------------------------------
def _te_coax_run(Nz, npml_hi, n_steps, probe_k, src_k=20, Nr=40):
    """TE01-type phi-uniform mode between PEC cylinders (E_phi(r), H_r, H_z; Nphi = 1, p = 1), driven by a J_phi sheet
    with the radial profile sin(pi i / Nr) (cut-off pi / 40 = 0.079, a quarter of the carrier 2 pi / 20)."""
    inp = make_zone(Nr, 1, Nz, r_in=1000.0, n_fold=4000, dt=0.5, npml_z=(12, npml_hi))
    A_phi = np.sin(math.pi * np.arange(Nr) / Nr)[:, None] * np.ones((Nr, 1))
    table = gaussian_pulse_table(n_steps, inp.dt, 2 * math.pi / 20.0, 12.0, 50.0, False)
    z = OracleZone(inp)
    rec = []
    for n in range(n_steps):
        z.step(J_r=np.zeros((Nr, 1)), J_phi=np.ascontiguousarray(table[0, n] * A_phi), source_k=src_k)
        rec.append(z.E[1][Nr // 2, 0, probe_k])
    assert max(np.abs(z.E[0]).max(), np.abs(z.E[2]).max(), np.abs(z.H[1]).max()) == 0.0   # the polarisation stays pure
    return np.array(rec)


def test_z_cpml_reflection_te_polarisation():
    """Pins psi_Hr_z and psi_Ephi_z (zda_oracle_core.c: the H_r and E_phi updates), which the coax TEM pulse above
    (E_r / H_phi only) never touches.  Measured 1.6e-5 with 12 cells; with the half- and integer-position CPML tables
    swapped on either of those two lines the reflection is 4.9e-2."""
    n_steps = 700
    with_pml = _te_coax_run(Nz=120, npml_hi=12, n_steps=n_steps, probe_k=80)
    ref = _te_coax_run(Nz=120 + 400, npml_hi=12, n_steps=n_steps, probe_k=80)
    assert np.abs(ref).max() > 1e-1
    refl = np.abs(with_pml - ref).max() / np.abs(ref).max()
    print("z-CPML TE reflection, 12 cells: %.3e" % refl)
    assert refl < 1e-4, refl


def _te_radial_run(Nr_extra, n_steps, npml=12, r_in=2000.0, Nr=160, Nz=24):
    """The TE twin of _radial_run: a phi-uniform cylindrical E_phi / H_z / H_r pulse between PEC plates at k = 0 and
    k = Nz, z-profile sin(pi k / Nz) (E_phi vanishes on the plates, so a z-uniform E_phi does not exist in this box)."""
    lo = Nr_extra
    inp = make_zone(Nr + 2 * Nr_extra, 1, Nz, r_in=r_in - lo, n_fold=4000, dt=0.5, npml_r=(npml, npml))
    z = OracleZone(inp)
    i = np.arange(inp.Nr) - lo
    c0, wid = Nr / 2.0, 6.0
    z.E[1][:, 0, :] = ((np.exp(-((i - c0) ** 2) / (2 * wid ** 2)) * np.cos(2 * math.pi * (i - c0) / 20.0))[:, None]
                       * np.sin(math.pi * np.arange(Nz) / Nz)[None, :])
    rec = []
    for n in range(n_steps):
        z.step()
        rec.append(z.E[1][lo + 30:lo + Nr - 30, 0, Nz // 2].copy())
    assert max(np.abs(z.E[0]).max(), np.abs(z.E[2]).max(), np.abs(z.H[1]).max()) == 0.0
    return np.array(rec)


def test_r_cpml_reflection_te_polarisation():
    """Pins psi_Hz_r and psi_Ephi_r (the H_z and E_phi updates).  Quasi-CPML at r_in = 2000, 12 cells: measured 1.59e-4
    (above north_star's 1e-4, like the TM value: R6); with the half- and integer-position tables swapped on either of
    those two lines it is 2.6e-2."""
    n_steps = 600
    a = _te_radial_run(0, n_steps)
    b = _te_radial_run(400, n_steps)
    refl = np.abs(a - b).max() / np.abs(b).max()
    print("r-CPML TE reflection at r_in = 2000, 12 cells: %.3e" % refl)
    assert refl < 1.9e-4, refl
