"""Shared driver of the GPU-vs-oracle parity tests: runs the same ``ZoneInputs`` through the oracle
(float64 CPU, ``oracle/``) and through libzda (``paper_2501_07979_b200.zda``, C ABI) and returns both
sets of results in (r, phi, z) order.  No method arithmetic here."""
from __future__ import annotations

import numpy as np

from oracle import OracleZone
from oracle.density import density_to_eps, density_vjp


def rel_l2(a, b):
    """||a - b||_2 / ||b||_2 (b = oracle); 0 when both vanish."""
    a = np.asarray(a)
    b = np.asarray(b)
    den = float(np.linalg.norm(b.ravel()))
    num = float(np.linalg.norm((a - b).ravel()))
    if den == 0.0:
        return 0.0 if num == 0.0 else float("inf")
    return num / den


def oracle_eps_design(inp):
    if inp.density is not None:
        return density_to_eps(inp.density, inp.design_k1 - inp.design_k0)
    return inp.eps_design


def objective_kind(inp):
    """Which objective a set of inputs asks for: the focal intensity (R20) when it carries focal weights."""
    focal = getattr(inp, "focal_g", None) is not None or getattr(inp, "focal_dz", None) is not None
    return "focal_intensity" if focal else "monitor_energy"


def run_oracle(inp, adjoint=True):
    z = OracleZone(inp, eps_design=oracle_eps_design(inp))
    z.run_forward()
    kind = objective_kind(inp)
    out = dict(E=[e.copy() for e in z.E], H=[h.copy() for h in z.H],
               dft_fwd_design=z.dft_fwd["design"].copy(), dft_fwd_monitor=z.dft_fwd["monitor"].copy(),
               F=z.objective(kind=kind))
    if adjoint:
        if kind == "focal_intensity":
            out["focal_S"] = z.focal_sums()
        z.build_adjoint_source(kind=kind)
        z.run_adjoint()
        out["dft_adj_design"] = z.dft_adj["design"].copy()
        out["E_adj"] = [e.copy() for e in z.E]
        g = z.gradient()
        out["grad"] = g
        out["grad_zsum"] = g.sum(axis=2)
        if inp.density is not None:
            out["grad_rho"] = density_vjp(inp.density, g)
    return out


def run_gpu(inp, precision=32, adjoint=True, kernel=0, options=None):
    from paper_2501_07979_b200 import zda
    z = zda.Zone(inp, precision=precision, kernel=kernel, options=options)
    try:
        z.run_forward()
        out = dict(E=[z.get_field(c) for c in range(3)], H=[z.get_field(3 + c) for c in range(3)],
                   dft_fwd_design=z.dft(zda.ZDA_FWD, zda.ZDA_DESIGN), dft_fwd_monitor=z.dft(zda.ZDA_FWD, zda.ZDA_MONITOR))
        z.check_finite()
        if adjoint:
            if z.objective == zda.ZDA_OBJ_FOCAL_INTENSITY:
                out["focal_S"] = zda.zda_get_focal_sums(z.handle, inp.n_freq)
            out["F"] = z.build_adjoint_source()
            z.run_adjoint()
            out["dft_adj_design"] = z.dft(zda.ZDA_ADJ, zda.ZDA_DESIGN)
            out["E_adj"] = [z.get_field(c) for c in range(3)]
            box, zs, drho = z.gradient(True, True, inp.density is not None)
            out["grad"], out["grad_zsum"] = box, zs
            if drho is not None:
                out["grad_rho"] = drho
        out["kernel"] = z.kernel_name
        out["launches"] = z.launch_count
    finally:
        z.close()
    return out


def compare(gpu, ora, tol_field, tol_grad, adjoint=True, label=""):
    """Asserts relative-L2 parity of every result; returns the dict of errors."""
    errs = {}
    for c in range(3):
        errs[f"E{c}"] = rel_l2(gpu["E"][c], ora["E"][c])
        errs[f"H{c}"] = rel_l2(gpu["H"][c], ora["H"][c])
    # all six end-of-run components against the norm of the whole E (resp. H) field: a component that is
    # physically ~0 (rounding noise only) must not be judged against its own norm
    for tag in ("E", "H"):
        num = np.sqrt(sum(np.linalg.norm((gpu[tag][c] - ora[tag][c]).ravel()) ** 2 for c in range(3)))
        den = np.sqrt(sum(np.linalg.norm(ora[tag][c].ravel()) ** 2 for c in range(3)))
        errs[tag + "_all"] = float(num / den) if den > 0 else float(num)
    errs["dft_design"] = rel_l2(gpu["dft_fwd_design"], ora["dft_fwd_design"])
    errs["dft_monitor"] = rel_l2(gpu["dft_fwd_monitor"], ora["dft_fwd_monitor"])
    if adjoint:
        errs["F"] = abs(gpu["F"] - ora["F"]) / abs(ora["F"])
        if "focal_S" in ora:
            errs["focal_S"] = rel_l2(gpu["focal_S"], ora["focal_S"])
        errs["dft_adj"] = rel_l2(gpu["dft_adj_design"], ora["dft_adj_design"])
        errs["grad"] = rel_l2(gpu["grad"], ora["grad"])
        errs["grad_zsum"] = rel_l2(gpu["grad_zsum"], ora["grad_zsum"])
        if "grad_rho" in ora:
            errs["grad_rho"] = rel_l2(gpu["grad_rho"], ora["grad_rho"])
    field_keys = ["E_all", "H_all", "dft_design", "dft_monitor"] + (["dft_adj", "F", "focal_S"] if adjoint else [])
    bad = {k: v for k, v in errs.items() if (k in field_keys and not v <= tol_field)
           or (k.startswith("grad") and not v <= tol_grad)}
    # the achieved errors of every parity case, one line each (collected into profiles/ from the GPU run's log)
    fmax = max(v for k, v in errs.items() if k in field_keys)
    gmax = max([v for k, v in errs.items() if k.startswith("grad")] or [0.0])
    print(f"PARITY {label or '?'} | field/DFT max {fmax:.3e} (tol {tol_field:.0e}) | gradient max {gmax:.3e} (tol {tol_grad:.0e}) | "
          + " ".join(f"{k}={v:.2e}" for k, v in errs.items()))
    assert not bad, f"{label}: parity failed {bad}; all errors {errs}"
    return errs
