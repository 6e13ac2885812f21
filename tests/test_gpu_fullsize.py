"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration ``bench.py`` times (fp32, fused
TMA kernel, the zone's real tiling / z-chunking / phi wrap), on sampled outputs the oracle can compute.

Method ("domain-of-dependence windows"): after n explicit leap-frog steps a field value depends only on data
within n cells of it (each step reaches one cell per axis).  So the oracle is run on a WINDOW of the big zone
(``workloads.window``: a sub-block with the same radii, dphi, z-stack, per-voxel eps, source sheet and --
where a face coincides with the zone's own boundary -- the same CPML slab), and its fields are exact copies
of the big zone's at every window point further than n + 1 cells from a cut face.  Those points are compared
element by element (relative L2 <= 1e-4, north_star); the run is long enough for the pulse to travel from
the source plane through the z-CPML and into the design layer, so the DFT accumulators are compared too."""
import numpy as np
import pytest

from oracle import OracleZone
from oracle.density import density_to_eps
from parity import rel_l2
from workloads import config2, config3, config4, config5_zones, gaussian_pulse_table, window

pytestmark = pytest.mark.gpu

TOL = 1e-4
FUSED, FUSED2 = 2, 3


def _prepare(cfg_fn, n_steps):
    from dataclasses import replace
    inp = cfg_fn(n_steps=n_steps)
    # a pulse that is already strong during the first steps (the configs' own pulse peaks hundreds of steps in)
    wc = float(np.mean(inp.omega))
    table = gaussian_pulse_table(n_steps, inp.dt, wc, 3.0, 6.0, inp.complex_fields)
    return replace(inp, src_table=table, n_steps=n_steps, n_steps_adjoint=0)


def _check_window(z, inp, eps_full, box, n, label):
    """box = (i_lo, i_hi, j_lo, j_hi, k_lo, k_hi) of the window; compares the points > n + 1 cells from cut faces."""
    from paper_2501_07979_b200 import zda
    i_lo, i_hi, j_lo, j_hi, k_lo, k_hi = box
    w = window(inp, eps_full, i_lo, i_hi, j_lo, j_hi, k_lo, k_hi, n)
    o = OracleZone(w, eps_design=w.eps_design)
    o.run_forward()
    m = n + 1
    full_phi = (j_lo == 0 and j_hi == inp.Nphi)
    si = slice(0 if i_lo == 0 else m, (i_hi - i_lo) - (0 if i_hi == inp.Nr else m))
    sj = slice(0, j_hi - j_lo) if full_phi else slice(m, (j_hi - j_lo) - m)
    sk = slice(0 if k_lo == 0 else m, (k_hi - k_lo) - (0 if k_hi == inp.Nz else m))
    errs = {}
    num = {"E": 0.0, "H": 0.0}
    den = {"E": 0.0, "H": 0.0}
    for c in range(6):
        g = z.get_field_window(c, i_lo, i_hi, j_lo, j_hi, k_lo, k_hi)[si, sj, sk].astype(np.complex128 if inp.complex_fields else np.float64)
        ref = (o.E[c] if c < 3 else o.H[c - 3])[si, sj, sk]
        tag = "E" if c < 3 else "H"
        num[tag] += float(np.linalg.norm((g - ref).ravel()) ** 2)
        den[tag] += float(np.linalg.norm(ref.ravel()) ** 2)
    for tag in ("E", "H"):
        assert den[tag] > 0.0, f"{label}: the pulse has not reached the compared region"
        errs[tag] = (num[tag] / den[tag]) ** 0.5
    # DFT accumulators on the part of the design box inside the compared region
    dk0, dk1 = w.design_k0, w.design_k1
    di0, di1 = w.design_i0, w.design_i1
    ks = slice(max(sk.start, dk0), min(sk.stop, dk1))
    isl = slice(max(si.start, di0), min(si.stop, di1))
    if ks.start < ks.stop and isl.start < isl.stop:
        ref_all = o.dft_fwd["design"]          # (F, 3, Nr_d, Nphi, L_d) on the window's design box
        for f in (0, inp.n_freq - 1):
            for c in range(3):
                gi0 = i_lo + isl.start - inp.design_i0
                gk0 = k_lo + ks.start - inp.design_k0
                g = z.get_dft_design_window(zda.ZDA_FWD, c, f, gi0, gi0 + (isl.stop - isl.start), j_lo, j_hi,
                                            gk0, gk0 + (ks.stop - ks.start))[:, sj, :]
                ref = ref_all[f, c][isl.start - di0:isl.stop - di0, sj, ks.start - dk0:ks.stop - dk0]
                if np.linalg.norm(ref.ravel()) > 0:
                    errs[f"dft_f{f}_c{c}"] = rel_l2(g, ref)
    bad = {k: v for k, v in errs.items() if not v <= TOL}
    assert not bad, f"{label}: {bad}; all {errs}"
    return errs


CASES = {
    # cfg: (builder, n_steps, k_hi of the windows)
    "config2": (config2, 26, 80),
    "config3": (config3, 42, 116),
    "config4": (config4, 50, 134),
    # one annular zone of the 24-zone lens pass (bench --workload config5): 1134 x 1387 x 200, complex Bloch, its own dt
    "config5": (lambda n_steps: config5_zones(n_zones=13, n_steps=n_steps)[12], 42, 116),
}


@pytest.mark.parametrize("cfg,kernel", [("config2", FUSED), ("config3", FUSED), ("config4", FUSED),
                                        ("config2", FUSED2), ("config3", FUSED2), ("config4", FUSED2), ("config5", 0)],
                         ids=["config2-fused", "config3-fused", "config4-fused", "config2-fused2", "config3-fused2",
                              "config4-fused2", "config5-zone12-auto"])
def test_full_size_windows(cfg, kernel):
    from paper_2501_07979_b200 import zda
    fn, n, k_hi = CASES[cfg]
    inp = _prepare(fn, n)
    eps_full = density_to_eps(inp.density, inp.design_k1 - inp.design_k0)
    z = zda.Zone(inp, precision=32, kernel=kernel)
    try:
        # AUTO = the two-step kernel wherever it applies: the plan bench.py times on config2 .. config5
        assert z.kernel_name.startswith("fused(" if kernel == FUSED else "fused2(")
        z.run_forward()
        z.check_finite()
        m = n + 1
        VECW = 128 if not inp.complex_fields else 64
        # (a) interior block around a tile corner in (r, phi): the 128-byte tile edge and a 7-row tile edge
        ic, jc = 3 * VECW, 7 * 9
        box = (ic - m - 6, ic + m + 6, jc - m - 6, jc + m + 6, 0, k_hi)
        ea = _check_window(z, inp, eps_full, box, n, cfg + " tile-corner window")
        # (b) the inner radial boundary with its r-CPML slab (window face = zone face), away from the phi wrap
        box = (0, m + 30, inp.Nphi // 2 - m - 5, inp.Nphi // 2 + m + 5, 0, k_hi)
        eb = _check_window(z, inp, eps_full, box, n, cfg + " inner r-CPML window")
        # (c) the outer radial boundary (last, partly filled tile)
        box = (inp.Nr - m - 30, inp.Nr, 100, 100 + 2 * m + 10, 0, k_hi)
        ec = _check_window(z, inp, eps_full, box, n, cfg + " outer r-CPML window")
        # (d) the phi wrap with its phase: a thin (r, z) block over ALL of phi
        box = (200, 200 + 2 * m + 8, 0, inp.Nphi, 0, k_hi)
        ed = _check_window(z, inp, eps_full, box, n, cfg + " phi-wrap window")
        print(cfg, z.kernel_name, {k: float("%.3g" % v) for d in (ea, eb, ec, ed) for k, v in d.items() if k in ("E", "H")})
    finally:
        z.close()


def _check_adjoint_window(z, inp, eps_full, box, n_fwd, n_adj, g_box, label):
    """Forward + adjoint source + adjoint run + gradient of the oracle on a window; compares the adjoint DFT accumulators
    and dF/deps at the design-box points further than n_fwd + n_adj + 2 cells from a cut face (the forward monitor DFT, hence
    the adjoint source, is exact only n_fwd + 1 cells inside the cut; the adjoint run carries that n_adj + 1 cells further)."""
    from dataclasses import replace
    from paper_2501_07979_b200 import zda
    i_lo, i_hi, j_lo, j_hi, k_lo, k_hi = box
    assert (k_lo, k_hi) == (0, inp.Nz)
    w = replace(window(inp, eps_full, i_lo, i_hi, j_lo, j_hi, k_lo, k_hi, n_fwd), n_steps_adjoint=n_adj)
    o = OracleZone(w, eps_design=w.eps_design)
    o.run_forward()
    o.build_adjoint_source()
    o.run_adjoint()
    g_ref = o.gradient()
    m = n_fwd + n_adj + 2
    full_phi = (j_lo == 0 and j_hi == inp.Nphi)
    si = slice(max(w.design_i0, 0 if i_lo == 0 else m), min(w.design_i1, (i_hi - i_lo) - (0 if i_hi == inp.Nr else m)))
    sj = slice(0, j_hi - j_lo) if full_phi else slice(m, (j_hi - j_lo) - m)
    assert si.start < si.stop and sj.start < sj.stop
    gi0 = i_lo + si.start - inp.design_i0
    Ld = inp.design_k1 - inp.design_k0
    errs = {}
    for f in range(inp.n_freq):
        num = den = 0.0
        for c in range(3):
            g = z.get_dft_design_window(zda.ZDA_ADJ, c, f, gi0, gi0 + (si.stop - si.start), j_lo, j_hi, 0, Ld)[:, sj, :]
            ref = o.dft_adj["design"][f, c][si.start - w.design_i0:si.stop - w.design_i0, sj, :]
            num += float(np.linalg.norm((g - ref).ravel()) ** 2)
            den += float(np.linalg.norm(ref.ravel()) ** 2)
        assert den > 0.0, f"{label}: the adjoint field has not reached the design box"
        errs[f"dft_adj_f{f}"] = (num / den) ** 0.5
    g = g_box[:, j_lo:j_hi, gi0:gi0 + (si.stop - si.start)].cpu().numpy().transpose(2, 1, 0)[:, sj, :]
    errs["grad"] = rel_l2(g, g_ref[si.start - w.design_i0:si.stop - w.design_i0, sj, :])
    bad = {k: v for k, v in errs.items() if not v <= (1e-3 if k == "grad" else TOL)}
    print("PARITY", label, {k: float("%.3g" % v) for k, v in errs.items()})
    assert not bad, f"{label}: {bad}; all {errs}"
    return errs


@pytest.mark.parametrize("cfg,kernel", [("config4", FUSED), ("config3", FUSED), ("config3", 0), ("config4", 0)],
                         ids=["config4-fused", "config3-fused", "config3-auto", "config4-auto"])
def test_full_size_adjoint_and_gradient_windows(cfg, kernel):
    """adjoint source, adjoint run and gradient at BENCH tiling (full grid, fp32, fused kernel, the
    zone's own z-chunks / clusters / DFT ring).  To reach the design box in a run short enough for the oracle window, the
    source and monitor planes sit inside the design layer, and the design frequencies are spread to omega = 0.25 + 0.2 f:
    with the config's own closely spaced lines a 60-step pulse basis is singular to rounding (condition number 1e14 for
    F = 6 at 70 steps; 17 with the spread ones), which would test the conditioning, not the kernels.  Grid, stack, CPML,
    density map, F and hence tiling, ring period and bytes are the bench's."""
    import torch
    from dataclasses import replace
    from paper_2501_07979_b200 import zda
    fn = {"config4": config4, "config3": config3}[cfg]
    n_fwd = n_adj = 60
    inp = fn(n_steps=n_fwd)
    F = inp.n_freq
    omega = 0.25 + 0.2 * np.arange(F)
    ks = inp.design_k0 + 10
    inp = replace(inp, omega=omega, source_k=ks, monitor_k=ks + 10, n_steps=n_fwd, n_steps_adjoint=n_adj,
                  adj_sigma_t=6.0, adj_t0=13.0,
                  src_table=gaussian_pulse_table(n_fwd, inp.dt, float(np.mean(omega)), 3.0, 6.0, inp.complex_fields))
    eps_full = density_to_eps(inp.density, inp.design_k1 - inp.design_k0)
    z = zda.Zone(inp, precision=32, kernel=kernel)
    try:
        # AUTO takes the two-step kernel: the plan bench.py times (config4 is the bench default)
        assert z.kernel_name.startswith("fused2(" if kernel == 0 else "fused(")
        z.run_forward()
        z.build_adjoint_source(want_F=False)
        z.run_adjoint()
        z.check_finite()
        nr, nphi, ld = inp.design_shape
        g_box = torch.empty((ld, nphi, nr), dtype=torch.float32, device="cuda")
        zda.zda_gradient(z.handle, g_box, None, None, 0)
        torch.cuda.synchronize()
        m = n_fwd + n_adj + 2
        VECW = 128 if not inp.complex_fields else 64
        # (a) around a tile corner in (r, phi)
        ic, jc = 3 * VECW, 7 * 40
        box = (ic - m - 6, ic + m + 6, jc - m - 6, jc + m + 6, 0, inp.Nz)
        _check_adjoint_window(z, inp, eps_full, box, n_fwd, n_adj, g_box, cfg + " adjoint tile-corner window fp32")
        # (b) the inner radial boundary: r-CPML slab and the objective mask's edge
        box = (0, m + 40, inp.Nphi // 2 - m - 4, inp.Nphi // 2 + m + 4, 0, inp.Nz)
        _check_adjoint_window(z, inp, eps_full, box, n_fwd, n_adj, g_box, cfg + " adjoint inner-r window fp32")
    finally:
        z.close()


@pytest.mark.parametrize("kernel", [FUSED, FUSED2], ids=["fused", "fused2"])
def test_full_grid_fp32_against_fp64_every_element(kernel):
    """GPU fp32 vs GPU fp64 on the FULL config-2 grid (800 x 800 x 160, the one-step kernel and the
    two-step kernel -- the plan bench.py times on config2 -- in their bench tiling), every element of all six fields and of the monitor / design accumulators after 100 steps.  The fp64
    build is the one the oracle pins element by element at small sizes, so a wrong ghost row, tile edge or chunk seam
    anywhere in the 1e8 voxels shows here: besides the relative L2 (<= 1e-4), the LARGEST single-element difference is
    held to 1e-5 of the field's maximum (fp32 rounding over 100 steps is ~1e-6)."""
    import torch
    from paper_2501_07979_b200 import zda
    n = 100
    inp = _prepare(config2, n)
    z32 = zda.Zone(inp, precision=32, kernel=kernel)
    z64 = zda.Zone(inp, precision=64, kernel=kernel)
    try:
        z32.run_forward()
        z64.run_forward()
        a = torch.empty((inp.Nz, inp.Nphi, inp.Nr), dtype=torch.float32, device="cuda")
        b = torch.empty((inp.Nz, inp.Nphi, inp.Nr), dtype=torch.float64, device="cuda")
        worst_l2 = worst_el = 0.0
        num = {"E": 0.0, "H": 0.0}; den = {"E": 0.0, "H": 0.0}; dmax = {"E": 0.0, "H": 0.0}; fmax = {"E": 0.0, "H": 0.0}
        for c in range(6):
            zda.zda_get_field(z32.handle, c, a, 0)
            zda.zda_get_field(z64.handle, c, b, 0)
            torch.cuda.synchronize()
            d = a.double() - b
            tag = "E" if c < 3 else "H"
            num[tag] += float((d * d).sum()); den[tag] += float((b * b).sum())
            dmax[tag] = max(dmax[tag], float(d.abs().max())); fmax[tag] = max(fmax[tag], float(b.abs().max()))
        for tag in ("E", "H"):
            assert den[tag] > 0
            worst_l2 = max(worst_l2, (num[tag] / den[tag]) ** 0.5)
            worst_el = max(worst_el, dmax[tag] / fmax[tag])
        nr, nphi, ld = inp.design_shape
        da = torch.empty((ld, nphi, nr), dtype=torch.complex64, device="cuda")
        db = torch.empty((ld, nphi, nr), dtype=torch.complex128, device="cuda")
        ma = torch.empty((inp.Nphi, inp.Nr), dtype=torch.complex64, device="cuda")
        mb = torch.empty((inp.Nphi, inp.Nr), dtype=torch.complex128, device="cuda")
        dft_l2 = dft_el = 0.0
        for c in range(3):
            for region, (x, y) in ((zda.ZDA_DESIGN, (da, db)), (zda.ZDA_MONITOR, (ma, mb))):
                zda.zda_get_dft(z32.handle, zda.ZDA_FWD, region, c, 0, x, 0)
                zda.zda_get_dft(z64.handle, zda.ZDA_FWD, region, c, 0, y, 0)
                torch.cuda.synchronize()
                if float(y.abs().max()) == 0.0:
                    assert float(x.abs().max()) == 0.0
                    continue
                d = x.to(torch.complex128) - y
                dft_l2 = max(dft_l2, float(d.abs().pow(2).sum().sqrt() / y.abs().pow(2).sum().sqrt()))
                dft_el = max(dft_el, float(d.abs().max() / y.abs().max()))
        print(f"PARITY config2 full grid fp32 vs fp64 kernel={kernel} | fields rel L2 %.3e, largest element %.3e of max | DFT rel L2 %.3e, "
              "largest element %.3e" % (worst_l2, worst_el, dft_l2, dft_el))
        assert worst_l2 <= TOL and dft_l2 <= TOL
        assert worst_el <= 1e-5 and dft_el <= 1e-5
    finally:
        z32.close()
        z64.close()


@pytest.mark.parametrize("cfg", ["config6", "config7"])
def test_full_size_paper_shaped_zones_whole_zone(cfg):
    """The paper-shaped zones are small enough for the oracle to run WHOLE at bench size: config6
    (1274 x 11 x 160 thin Bloch wedge, fused kernel in the tiling bench.py times) and config7 (1262 x 1 x 160 first
    zone, persistent kernel), forward + adjoint + gradient through the conic density map, every output element by element.
    Source and monitor planes are moved next to the design layer so that a short run reaches the monitor."""
    from dataclasses import replace
    from parity import compare, run_gpu, run_oracle
    from workloads import config6_thin_wedge, config7_first_zone
    n = 240 if cfg == "config6" else 600
    inp = (config6_thin_wedge if cfg == "config6" else config7_first_zone)(n_steps=n)
    wc = float(np.mean(inp.omega))
    inp = replace(inp, source_k=36, monitor_k=76, n_steps=n, n_steps_adjoint=n, adj_sigma_t=6.0, adj_t0=20.0,
                  src_table=gaussian_pulse_table(n, inp.dt, wc, 3.0, 6.0, True))
    ora = run_oracle(inp, True)
    assert ora["F"] > 0.0
    gpu = run_gpu(inp, 32, True)
    assert gpu["kernel"].startswith("fused" if cfg == "config6" else "persist")
    errs = compare(gpu, ora, TOL, 1e-3, True, cfg + " whole zone fp32")
    print(cfg, gpu["kernel"], {k: float("%.3g" % v) for k, v in errs.items()})
