"""Pins of the exact cylindrical PML in r ("r' = r + i zeta_r / omega"; R25):
reflection of the outer r-slab against a long-domain reference, both polarisations, phi-uniform and Bloch m = 1, next to
the quasi-CPML's (R6) on the same pulse; the interior is untouched; long-run boundedness at the radii the library allows."""
import math

import numpy as np
import pytest

from helpers import make_zone
from oracle import OracleZone


def _outer_run(r_in, Nr, extra_hi, n_steps, exact, m=0, pol="TM", npml=12, compact=False):
    """A phi-uniform (m = 0) or one-phi-cell Bloch (m = 1) cylindrical pulse running into the OUTER r-slab; PEC inner wall."""
    Nz = 1 if pol == "TM" else 24
    inp = make_zone(Nr + extra_hi, 1, Nz, r_in=r_in, n_fold=64, dt=0.5, npml_r=(0, npml), complex_fields=(m != 0), m=m)
    inp.rpml_exact = exact
    z = OracleZone(inp)
    i = np.arange(inp.Nr)
    c0, wid = Nr * 0.55, 5.0
    prof = np.exp(-((i - c0) ** 2) / (2 * wid ** 2)) * np.cos(2 * math.pi * (i - c0) / 20.0)
    if compact:
        prof[np.abs(i - c0) > 12] = 0.0
    if pol == "TM":
        z.E[2][:, :, :] = prof[:, None, None]
    else:
        z.E[1][:, :, :] = prof[:, None, None] * np.sin(math.pi * np.arange(Nz) / Nz)[None, None, :]
    rec = []
    for _ in range(n_steps):
        z.step()
        rec.append((z.E[2] if pol == "TM" else z.E[1])[8:Nr - npml - 4, 0, Nz // 2].copy())
    return np.array(rec)


@pytest.mark.parametrize("pol", ["TM", "TE"])
@pytest.mark.parametrize("m", [0, 1])
@pytest.mark.parametrize("r_in,bar", [(1100.0, 3e-5), (100.0, 2e-4), (20.0, 5e-4)])
def test_exact_outer_r_pml_reflection(r_in, bar, m, pol):
    """12 cells.  Measured (TM / TE): r_in = 1100: 1.5e-5 / 1.3e-5 (quasi 5.1e-4 / 4.4e-4); 100: 1.1e-4 / 1.6e-5 (4e-3 / 3e-3);
    20: 2.7e-4 / 4.7e-5 (1.2e-2 / 7e-3): 30 to 40 times below the quasi-CPML, and below north_star's 1e-4 at every radius
    the library admits the exact form for (>= 1000 cells)."""
    n_steps = 400
    ref = _outer_run(r_in, 70, 300, n_steps, 0, m, pol)
    e = _outer_run(r_in, 70, 0, n_steps, 1, m, pol)
    q = _outer_run(r_in, 70, 0, n_steps, 0, m, pol)
    refl_e = np.abs(e - ref).max() / np.abs(ref).max()
    refl_q = np.abs(q - ref).max() / np.abs(ref).max()
    print("outer r-PML r_in = %5.0f m = %d %s: exact %.2e, quasi %.2e" % (r_in, m, pol, refl_e, refl_q))
    assert refl_e < bar and refl_e < refl_q / 15.0


def test_exact_mode_changes_nothing_outside_the_outer_slab():
    """Until a compactly supported pulse reaches the slab (7 cells away: 7 steps) the two modes are bit-identical: the
    interior keeps the conservative difference; afterwards they differ."""
    a = _outer_run(1100.0, 70, 0, 40, 1, compact=True)
    b = _outer_run(1100.0, 70, 0, 40, 0, compact=True)
    assert np.array_equal(a[:6], b[:6]) and not np.array_equal(a[-1], b[-1])


def test_exact_outer_pml_is_bounded_over_32000_steps_at_the_admitted_radius():
    """Random data (including static charges, the hardest case), Bloch p = exp(0.8 i), r- and z-slabs, 32 000 steps at
    r_in = 1100: max|E| stays within 20 % of its start.  (Below ~500 cells the exact form grows slowly -- x 10 over 32 000
    steps at r_in = 200 -- which is why the library admits it only for slabs beyond 1000 cells: DESIGN.md R25.)"""
    inp = make_zone(40, 5, 24, r_in=1100.0, n_fold=8, courant=0.9, npml_r=(8, 8), npml_z=(6, 6), complex_fields=True, m=0)
    inp.phase = complex(np.exp(0.8j))
    inp.rpml_exact = 1
    z = OracleZone(inp)
    rng = np.random.default_rng(0)
    for c in range(3):
        z.E[c][:] = rng.standard_normal(z.E[c].shape) + 1j * rng.standard_normal(z.E[c].shape)
    z.E[1][0] = 0
    z.E[2][0] = 0
    z.E[0][:, :, 0] = 0
    z.E[1][:, :, 0] = 0
    e0 = max(np.abs(e).max() for e in z.E)
    worst = 0.0
    for n in range(32000):
        z.step()
        if n % 2000 == 1999:
            worst = max(worst, max(np.abs(e).max() for e in z.E) / e0)
    print("exact outer r-PML, 32 000 steps at r_in = 1100: max |E| / start = %.3f" % worst)
    assert worst < 1.2
