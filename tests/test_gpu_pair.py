"""GPU tests (``-m gpu``) of NEXT-4: the m = +1 / m = -1 pair of a zone advancing in ONE launch per time step
(zda_pair_run_forward / zda_pair_run_adjoint, fused_step_batch_kernel).  Each member against its own oracle run, fp64 at
the suite's 5e-13 and fp32 at north_star's tolerances; and the coherent lens objective with the pair batched by the
scheduler."""
import math
from dataclasses import replace

import numpy as np
import pytest

from oracle import OracleZone, lens_focal_objective
from parity import compare, rel_l2, run_oracle
from paper_2501_07979_b200 import zda
from test_gpu_parity import TOL64, TOL64_GRAD, _small
from workloads import focal_point_weights, plane_wave_sheet

pytestmark = pytest.mark.gpu


def _pair(Nr=150, Nphi=11, n_steps=300, lambdas=(18.0, 24.0)):
    """m = +1 and m = -1 members on ONE structure: a thin Bloch wedge spanning several r tiles and two phi tiles."""
    base = _small(True, list(lambdas), Nr=Nr, Nphi=Nphi, n_steps=n_steps)
    out = []
    for m in (+1, -1):
        A_r, A_phi = plane_wave_sheet(base.Nr, base.Nphi, base.dphi, True, m)
        out.append(replace(base, phase=complex(np.exp(2j * math.pi * m / base.n_fold)), src_A_r=A_r, src_A_phi=A_phi))
    return out


def _collect(z, inp):
    out = dict(E=[z.get_field(c) for c in range(3)], H=[z.get_field(3 + c) for c in range(3)])
    return out


@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("n_steps", [300, 301])
def test_pair_in_one_launch_matches_each_members_oracle(precision, n_steps):
    members = _pair(n_steps=n_steps)
    ora = [run_oracle(inp, True) for inp in members]
    zs = [zda.Zone(inp, precision=precision, kernel=zda.ZDA_KERNEL_FUSED) for inp in members]
    try:
        l0 = [z.launch_count for z in zs]
        zda.zda_pair_run_forward(zs[0].handle, zs[1].handle, n_steps)
        gpu = []
        for z, inp in zip(zs, members):
            g = dict(E=[z.get_field(c) for c in range(3)], H=[z.get_field(3 + c) for c in range(3)],
                     dft_fwd_design=z.dft(zda.ZDA_FWD, zda.ZDA_DESIGN), dft_fwd_monitor=z.dft(zda.ZDA_FWD, zda.ZDA_MONITOR))
            g["F"] = z.build_adjoint_source()
            gpu.append(g)
        zda.zda_pair_run_adjoint(zs[0].handle, zs[1].handle, n_steps)
        for z, g, inp in zip(zs, gpu, members):
            g["dft_adj_design"] = z.dft(zda.ZDA_ADJ, zda.ZDA_DESIGN)
            box, zsum, _ = z.gradient(True, True, False)
            g["grad"], g["grad_zsum"] = box, zsum
        # one launch per step for BOTH: the second member's own count holds only its accumulator visits and small kernels
        steps = 2 * n_steps
        assert zs[0].launch_count - l0[0] >= steps
        assert zs[1].launch_count - l0[1] < steps // 2
        tol = (TOL64, TOL64_GRAD) if precision == 64 else (1e-4, 1e-3)
        for b in range(2):
            compare(gpu[b], ora[b], tol[0], tol[1], True, f"batched pair member m={'+1' if b == 0 else '-1'} fp{precision} n={n_steps}")
    finally:
        for z in zs:
            z.close()


def test_pair_requirements_are_checked():
    import torch
    a, b = _pair(Nr=70, Nphi=6, n_steps=40)
    za = zda.Zone(a, precision=32, kernel=zda.ZDA_KERNEL_FUSED)
    zb_split = zda.Zone(b, precision=32, kernel=zda.ZDA_KERNEL_SPLIT)
    zb_stream = zda.Zone(b, precision=32, kernel=zda.ZDA_KERNEL_FUSED, stream=torch.cuda.Stream())
    zb_shape = zda.Zone(_small(True, [18.0, 24.0], Nr=60, Nphi=6, n_steps=40), precision=32, kernel=zda.ZDA_KERNEL_FUSED)
    zb_ok = zda.Zone(b, precision=32, kernel=zda.ZDA_KERNEL_FUSED)
    try:
        for other, word in ((zb_split, "fused"), (zb_stream, "stream"), (zb_shape, "differ"), (za, "distinct")):
            with pytest.raises(zda.ZdaError) as e:
                zda.zda_pair_run_forward(za.handle, other.handle, 40)
            assert e.value.code == zda.ZDA_E_BADARG and word in str(e.value), str(e.value)
        zda.zda_pair_run_forward(za.handle, zb_ok.handle, 40)
        with pytest.raises(zda.ZdaError) as e:          # no adjoint sources yet
            zda.zda_pair_run_adjoint(za.handle, zb_ok.handle, 40)
        assert e.value.code == zda.ZDA_E_STATE
    finally:
        for z in (za, zb_split, zb_stream, zb_shape, zb_ok):
            z.close()


@pytest.mark.parametrize("precision", [64, 32])
def test_lens_focal_gradient_batches_the_pair(precision):
    """zda_lens_focal_gradient with the two members on ONE stream: the scheduler runs them in shared launches; F, S_total and
    each member's z-summed gradient vs the oracle's coherent objective (R23), weights built by the library (R24)."""
    import torch
    members = [replace(inp, focal_dz=140.0) for inp in _pair(Nr=100, Nphi=6, n_steps=300)]
    u = np.array([1.0, 0.6])
    zs_o = [OracleZone(inp) for inp in members]
    for z in zs_o:
        z.run_forward()
    F_o, S_o = lens_focal_objective(zs_o, u)
    g_o = []
    for z in zs_o:
        z.inp.focal_u = u
        z.build_adjoint_source(kind="focal_intensity", S_total=S_o)
        z.run_adjoint()
        g_o.append(z.gradient().sum(axis=2))
    tdt = torch.float32 if precision == 32 else torch.float64
    objs = [zda.Zone(inp, precision=precision, kernel=zda.ZDA_KERNEL_FUSED) for inp in members]
    try:
        l0 = [o.launch_count for o in objs]
        g_zs = [torch.zeros((inp.Nphi, inp.design_i1 - inp.design_i0), dtype=tdt, device="cuda") for inp in members]
        F, S = zda.zda_lens_focal_gradient([o.handle for o in objs], [300, 300], [300, 300], [i.adj_t0 for i in members],
                                           [i.adj_sigma_t for i in members], u, 2, g_zs, None)
        torch.cuda.synchronize()
        assert objs[1].launch_count - l0[1] < 300          # batched: the time-step launches are counted on member 0
        tol_f, tol_g = (TOL64, TOL64_GRAD) if precision == 64 else (1e-4, 1e-3)
        assert abs(F - F_o) <= tol_f * abs(F_o), (F, F_o)
        assert rel_l2(S, S_o) <= tol_f
        for l in range(2):
            e = rel_l2(g_zs[l].cpu().numpy().T, g_o[l])
            assert e <= tol_g, (l, e)
        print("PARITY batched pair through zda_lens_focal_gradient fp%d | F %.2e S %.2e" % (precision, abs(F - F_o) / abs(F_o), rel_l2(S, S_o)))
    finally:
        for o in objs:
            o.close()
