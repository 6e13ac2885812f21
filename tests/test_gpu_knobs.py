"""GPU tests (``-m gpu``) of the paths the default plan does not reach: every remainder of the DFT
visit group, every visit period, the launch-plan options, the per-voxel eps volume, the in-run failure detector and the
scheduler's workspace check.  All through the C ABI; fp64 parity at 1e-12 means the option changes nothing."""
import math

import numpy as np
import pytest

from parity import compare, rel_l2, run_gpu, run_oracle
from paper_2501_07979_b200 import zda
from test_gpu_parity import TOL64, TOL64_GRAD, _small

pytestmark = pytest.mark.gpu

FUSED = 2


def _zone(n_steps):
    # real fields, F = 3: the plan's own visit period is 8 (fp64: (288 + 24 * 14) / 8 = 78 B against 156 B at period 2)
    return _small(False, [16.0, 20.0, 26.0], Nr=70, Nphi=17, n_steps=n_steps)      # >= 16 phi cells: both fused kernels apply


@pytest.mark.parametrize("kernel", [FUSED, 3], ids=["fused", "fused2"])
@pytest.mark.parametrize("n_steps", [401, 403, 405, 407, 400, 402])
def test_dft_ring_every_group_remainder_and_period(n_steps, kernel):
    """csrc/zda_zone_impl.cuh run_T: the last visit group holds n_steps mod period steps (1..7 with period 8); each
    remainder takes a different mix of ring slots and time buffers.  Forward DFT in fp64 against the oracle for periods
    2, 4 and 8."""
    inp = _zone(n_steps)
    ora = run_oracle(inp, adjoint=False)
    for period in (8, 4, 2):
        gpu = run_gpu(inp, 64, False, kernel, options={zda.ZDA_OPT_DFT_PERIOD: period})
        compare(gpu, ora, TOL64, TOL64_GRAD, False, f"ring kernel={kernel} n_steps={n_steps} period={period} fp64")


@pytest.mark.parametrize("opts", [{zda.ZDA_OPT_FUSED_TJ: 6}, {zda.ZDA_OPT_FUSED_TJ: 7},
                                  {zda.ZDA_OPT_FUSED_CLUSTER: 1}, {zda.ZDA_OPT_FUSED_CLUSTER: 2},
                                  {zda.ZDA_OPT_FUSED_CLUSTER: 4}, {zda.ZDA_OPT_FUSED_CHUNK: 5},
                                  {zda.ZDA_OPT_FUSED_CHUNK: 9, zda.ZDA_OPT_FUSED_CLUSTER: 3, zda.ZDA_OPT_FUSED_TJ: 6},
                                  {zda.ZDA_OPT_KERNEL: 3, zda.ZDA_OPT_FUSED_TJ: 5}, {zda.ZDA_OPT_KERNEL: 3, zda.ZDA_OPT_FUSED_TJ: 9},
                                  {zda.ZDA_OPT_KERNEL: 3, zda.ZDA_OPT_FUSED_TJ: 13, zda.ZDA_OPT_FUSED_CLUSTER: 2},
                                  {zda.ZDA_OPT_KERNEL: 3, zda.ZDA_OPT_FUSED_CHUNK: 7, zda.ZDA_OPT_FUSED_TJ: 5, zda.ZDA_OPT_FUSED_CLUSTER: 3}],
                         ids=lambda o: "-".join(f"{k}={v}" for k, v in o.items()))
@pytest.mark.parametrize("cplx", [False, True], ids=["real", "bloch"])
def test_launch_plan_options_change_nothing(opts, cplx):
    """tile height, cluster size and z-chunk length are tuning knobs; forward + adjoint + gradient in fp64
    against the oracle under each of them (300 x 21 x 70: several tiles in r and phi, several chunks)."""
    from test_gpu_parity import _multi_tile
    inp = _multi_tile(cplx)
    ora = run_oracle(inp, True)
    gpu = run_gpu(inp, 64, True, opts.get(zda.ZDA_OPT_KERNEL, FUSED), options=opts)
    compare(gpu, ora, TOL64, TOL64_GRAD, True, f"plan options {opts} {'bloch' if cplx else 'real'} fp64")


def test_option_values_are_validated():
    inp = _zone(40)
    z = zda.Zone(inp, precision=32)
    try:
        for opt, bad in ((zda.ZDA_OPT_FUSED_TJ, 4), (zda.ZDA_OPT_FUSED_CLUSTER, 9), (zda.ZDA_OPT_DFT_PERIOD, 3),
                         (zda.ZDA_OPT_CHECK_EVERY, -1), (99, 0)):
            with pytest.raises(zda.ZdaError) as e:
                zda.zda_set_option(z.handle, opt, bad)
            assert e.value.code == zda.ZDA_E_BADARG
    finally:
        z.close()
    # a zone whose workspace holds no ring (F = 1: period 2) cannot be switched to a longer period afterwards
    z = zda.Zone(_small(False, [20.0], n_steps=40), precision=32)
    try:
        with pytest.raises(zda.ZdaError) as e:
            zda.zda_set_option(z.handle, zda.ZDA_OPT_DFT_PERIOD, 8)
        assert e.value.code == zda.ZDA_E_BADARG and "ring" in str(e.value)
    finally:
        z.close()


@pytest.mark.parametrize("kernel", [1, 2, 3], ids=["split", "fused", "fused2"])
@pytest.mark.parametrize("precision", [64, 32])
def test_per_voxel_eps_volume(precision, kernel):
    """zda_set_eps_volume (north_star 'per-voxel eps'): a substrate patterned in (r, phi, z) below the design layer and a
    second patterned layer above it, which eps(z) + design box cannot express; forward + adjoint + gradient vs the oracle."""
    inp = _small(False, [18.0, 24.0], Nr=70, Nphi=17 if kernel == 3 else 9)
    rng = np.random.default_rng(7)
    vol = np.ones((inp.Nr, inp.Nphi, inp.Nz)) * np.asarray(inp.eps_bg_z)[None, None, :]
    vol[:, :, :14] = 2.13 + 0.8 * rng.random((inp.Nr, inp.Nphi, 14))          # patterned substrate (reaches into the z-PML)
    vol[10:50, :, 23:26] = 1.0 + 2.0 * rng.random((40, inp.Nphi, 3))           # second patterned layer above the design box
    vol[:, :, inp.design_k0:inp.design_k1] = 1.7                                # overwritten by eps_design inside the box
    inp.eps_volume = vol
    ora = run_oracle(inp, True)
    gpu = run_gpu(inp, precision, True, kernel)
    tol = (TOL64, TOL64_GRAD) if precision == 64 else (1e-4, 1e-3)
    compare(gpu, ora, tol[0], tol[1], True, f"eps volume fp{precision} kernel={kernel}")
    # and it matters: the same zone without the volume gives different fields
    inp.eps_volume = None
    other = run_gpu(inp, precision, False, kernel)
    assert rel_l2(other["dft_fwd_monitor"], ora["dft_fwd_monitor"]) > 1e-2


def test_eps_volume_needs_the_desc_flag():
    inp = _small(False, [20.0], n_steps=40)
    z = zda.Zone(inp, precision=32)
    try:
        with pytest.raises(zda.ZdaError) as e:
            zda.zda_set_eps_volume(z.handle, np.ones((inp.Nz, inp.Nphi, inp.Nr), np.float32), 1)
        assert e.value.code == zda.ZDA_E_STATE
    finally:
        z.close()


@pytest.mark.parametrize("kernel", [1, 2, 3], ids=["split", "fused", "fused2"])
def test_check_every_stops_a_run_that_went_non_finite(kernel):
    """ZDA_OPT_CHECK_EVERY: a NaN permittivity in one design voxel poisons E as soon as the pulse arrives; the
    run call returns ZDA_E_NAN at the first check after that instead of finishing the horizon; a clean zone passes."""
    inp = _small(False, [20.0], n_steps=200, Nphi=17 if kernel == 3 else 7)
    z = zda.Zone(inp, precision=32, kernel=kernel, options={zda.ZDA_OPT_CHECK_EVERY: 20})
    try:
        z.run_forward()                      # clean: no error
        n_clean = z.launch_count
        eps = np.array(inp.eps_design, copy=True)
        eps[3, 2, 1] = np.nan
        z.set_design_eps(eps)
        with pytest.raises(zda.ZdaError) as e:
            z.run_forward()
        assert e.value.code == zda.ZDA_E_NAN and "step" in str(e.value)
        assert z.launch_count - n_clean < n_clean      # stopped early
    finally:
        z.close()


def test_scheduler_rejects_zones_that_share_a_workspace():
    """resident zones keep their tables, materials and sheets in their workspace, so two of them cannot share
    one; zda_lens_gradient says so instead of computing with overwritten tables."""
    import torch
    inp = _small(False, [20.0], n_steps=40)
    z0 = zda.Zone(inp, precision=32)
    ws = torch.empty(z0.nbytes, dtype=torch.uint8, device="cuda")
    za = zda.Zone(inp, precision=32, workspace=ws)
    zb = zda.Zone(inp, precision=32, workspace=ws)
    try:
        with pytest.raises(zda.ZdaError) as e:
            zda.zda_lens_gradient([za.handle, zb.handle], [40, 40], [40, 40], [inp.adj_t0] * 2, [inp.adj_sigma_t] * 2)
        assert e.value.code == zda.ZDA_E_BADARG and "share" in str(e.value)
        F = zda.zda_lens_gradient([z0.handle, za.handle], [40, 40], [40, 40], [inp.adj_t0] * 2, [inp.adj_sigma_t] * 2)
        assert F[0] > 0 and F[0] == F[1]
    finally:
        for z in (z0, za, zb):
            z.close()


@pytest.mark.parametrize("kernel", [1, 2], ids=["split", "fused"])
@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("m", [+1, -1])
def test_near_to_far_weights_built_by_the_library(precision, kernel, m):
    """zda_build_focal_weights (Eq. 7-8; R24): the library builds the focal weights from the first
    Rayleigh-Sommerfeld integral itself; focal sums S_f, objective, adjoint run and gradient vs the oracle (whose own
    near-to-far transform is pinned to the closed-form aperture field in tests/test_oracle_farfield.py).  Bloch m = +-1
    wedge of n = 16: the wedge sums over the other 15 wedges are non-trivial."""
    from dataclasses import replace
    from workloads import plane_wave_sheet
    base = _small(True, [18.0, 24.0], Nr=70, Nphi=6)
    A_r, A_phi = plane_wave_sheet(base.Nr, base.Nphi, base.dphi, True, m)
    inp = replace(base, phase=complex(np.exp(2j * math.pi * m / base.n_fold)), src_A_r=A_r, src_A_phi=A_phi,
                  focal_dz=150.0, focal_u=np.array([1.0, 0.7]))
    ora = run_oracle(inp, True)
    assert abs(ora["focal_S"]).min() > 0
    gpu = run_gpu(inp, precision, True, kernel)
    tol = (TOL64, TOL64_GRAD) if precision == 64 else (1e-4, 1e-3)
    compare(gpu, ora, tol[0], tol[1], True, f"near-to-far built m={m} fp{precision} kernel={kernel}")


def test_near_to_far_selection_rule_on_the_gpu():
    """A real n-fold periodic zone (p = 1, n = 16) cannot reach an on-axis x-polarised focus: the built weights vanish."""
    inp = _small(False, [20.0], n_steps=60)
    z = zda.Zone(inp, precision=64)
    try:
        zda.zda_build_focal_weights(z.handle, 120.0, None)
        z.run_forward()
        S = zda.zda_get_focal_sums(z.handle, 1)
        mon = z.dft(zda.ZDA_FWD, zda.ZDA_MONITOR)
        assert np.abs(mon).max() > 0 and abs(S[0]) < 1e-12 * np.abs(mon).sum()
    finally:
        z.close()


def _exact_pml_zone(cplx, Nr=198, Nphi=9, n_steps=360):
    """A zone at r_in = 1100 (the exact outer r-PML is admitted from 1000 cells; R25) whose outer slab (8 cells) straddles a
    tile boundary of the fused kernel, so the halo column recomputed by the neighbouring tile lies inside the slab."""
    from helpers import make_zone
    from workloads import gaussian_pulse_table, plane_wave_sheet
    n_fold = 768
    inp = make_zone(Nr, Nphi, 40, r_in=1100.0, n_fold=n_fold, courant=0.9, complex_fields=cplx, m=1,
                    npml_r=(6, 8), npml_z=(8, 8), omega=[2 * math.pi / 18.0, 2 * math.pi / 24.0])
    inp.rpml_exact = 1
    inp.design_i0, inp.design_i1, inp.design_k0, inp.design_k1 = 7, Nr - 9, 16, 21
    inp.source_k, inp.monitor_k = 11, 29
    inp.eps_design = 1.0 + 3.0 * np.random.default_rng(2).random(inp.design_shape)
    inp.eps_bg_z = np.where(np.arange(40) < 14, 2.13, 1.0)
    inp.src_A_r, inp.src_A_phi = plane_wave_sheet(Nr, Nphi, inp.dphi, cplx)
    inp.src_table = gaussian_pulse_table(n_steps, inp.dt, float(np.mean(inp.omega)), 12.0, 50.0, cplx)
    inp.n_steps = inp.n_steps_adjoint = n_steps
    inp.adj_sigma_t, inp.adj_t0 = 14.0, 56.0
    return inp


@pytest.mark.parametrize("kernel", [1, 2], ids=["split", "fused"])
@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("cplx", [False, True], ids=["real", "bloch"])
def test_exact_outer_r_pml(precision, kernel, cplx):
    """SURVEY 8(f) NEXT-1 / DESIGN.md R25: rpml_exact = 1, forward + adjoint + gradient vs the oracle."""
    inp = _exact_pml_zone(cplx)
    ora = run_oracle(inp, True)
    gpu = run_gpu(inp, precision, True, kernel)
    tol = (TOL64, TOL64_GRAD) if precision == 64 else (1e-4, 1e-3)
    compare(gpu, ora, tol[0], tol[1], True, f"exact outer r-PML {'bloch' if cplx else 'real'} fp{precision} kernel={kernel}")
    # and it is not the quasi form: the same zone with rpml_exact = 0 differs once the pulse has reached the slab
    inp.rpml_exact = 0
    other = run_gpu(inp, precision, False, kernel)
    assert rel_l2(other["E"][2], ora["E"][2]) > 1e-6


def test_exact_outer_r_pml_is_refused_where_it_is_not_admitted():
    import ctypes
    inp = _small(False, [20.0], n_steps=40)          # r_in = 25: far below 1000 cells
    inp.rpml_exact = 1
    d, keep = zda.desc_from_inputs(inp, 32)
    assert zda.load_library().zda_zone_workspace_bytes(ctypes.byref(d), 40) == 0 and "1000" in zda.zda_last_error()
    ok = _exact_pml_zone(False, n_steps=40)
    z = zda.Zone(ok, precision=32)
    try:
        assert z.kernel_name.startswith("fused(")
        with pytest.raises(zda.ZdaError) as e:
            zda.zda_set_option(z.handle, zda.ZDA_OPT_KERNEL, zda.ZDA_KERNEL_FUSED2)
        assert e.value.code == zda.ZDA_E_BADARG
    finally:
        z.close()


@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("which", ["first-zone", "axis-m0", "annulus-bloch"])
def test_persistent_kernel(which, precision):
    """ZDA_KERNEL_PERSIST: one cooperative launch steps the whole run (grid barriers between the H and E passes).  The
    paper's one-phi-cell first zone (AUTO takes it there), an axis zone with the loop-integral phi-mean (p = 1, Nphi = 8) and
    an ordinary Bloch annulus, forward + adjoint + gradient vs the oracle."""
    from workloads import config7_first_zone, cut_down
    if which == "first-zone":
        inp, kernel = cut_down(config7_first_zone(n_steps=400), Nr=150, n_steps=400), 0
    elif which == "axis-m0":
        inp, kernel = _small(False, [20.0], Nr=40, Nphi=8, has_axis=True), 0
    else:
        inp, kernel = _small(True, [18.0, 24.0]), zda.ZDA_KERNEL_PERSIST
    ora = run_oracle(inp, True)
    gpu = run_gpu(inp, precision, True, kernel)
    assert gpu["kernel"].startswith("persist("), gpu["kernel"]
    assert gpu["launches"] < 40                       # two cooperative launches + the small kernels, not 3 per step
    tol = (TOL64, TOL64_GRAD) if precision == 64 else (1e-4, 1e-3)
    compare(gpu, ora, tol[0], tol[1], True, f"persistent kernel {which} fp{precision}")


def test_two_step_kernel_needs_the_two_ghost_row_layout():
    """Thin wedges (Nphi < 16) and axis zones keep ONE ghost row per side (their extra copies would cost 15-20 % of the
    traffic); the two-step kernel's two-row halo is then not available: ZDA_E_BADARG, AUTO never picks it."""
    z = zda.Zone(_small(True, [18.0, 24.0], Nphi=11, n_steps=40), precision=32)
    try:
        assert z.kernel_name.startswith("fused(")
        with pytest.raises(zda.ZdaError) as e:
            zda.zda_set_option(z.handle, zda.ZDA_OPT_KERNEL, zda.ZDA_KERNEL_FUSED2)
        assert e.value.code == zda.ZDA_E_BADARG and "16" in str(e.value)
    finally:
        z.close()


def test_schedule_bytes_accounting():
    """zda_schedule_bytes (bench.py's roofline.schedule_bytes): the per-step HBM bytes of the launch plan follow DESIGN.md
    7's table — fields 12 x 4 B per voxel for the one-step kernel, half of that for the two-step kernel, 18 x 4 B for the
    split pair; psi and dt/eps halve with the two-step kernel; the halo upper bound is > 0 only for the tiled kernels."""
    inp = _zone(40)
    vox = float(inp.Nr * inp.Nphi * inp.Nz)
    got = {}
    for kernel in (zda.ZDA_KERNEL_SPLIT, zda.ZDA_KERNEL_FUSED, zda.ZDA_KERNEL_FUSED2):
        z = zda.Zone(inp, precision=32, options={zda.ZDA_OPT_KERNEL: kernel})
        try:
            got[kernel] = zda.zda_schedule_bytes(z.handle, zda.ZDA_FWD)
            adj = zda.zda_schedule_bytes(z.handle, zda.ZDA_ADJ)
            assert adj["dft"] < got[kernel]["dft"]            # the adjoint run carries no monitor-plane accumulators
            assert adj["fields"] == got[kernel]["fields"]
        finally:
            z.close()
    s, f1, f2 = (got[k] for k in (zda.ZDA_KERNEL_SPLIT, zda.ZDA_KERNEL_FUSED, zda.ZDA_KERNEL_FUSED2))
    assert s["fields"] == 18 * 4 * vox and f1["fields"] == 12 * 4 * vox and f2["fields"] == 6 * 4 * vox
    assert f1["psi"] > 0 and f2["psi"] == f1["psi"] / 2 and s["psi"] == f1["psi"]
    assert f1["eps"] > 0 and f2["eps"] == f1["eps"] / 2
    assert s["halo_if_no_l2_reuse"] == 0 and f1["halo_if_no_l2_reuse"] > 0 and f2["halo_if_no_l2_reuse"] > 0
    assert all(v["dft"] > 0 for v in got.values())
