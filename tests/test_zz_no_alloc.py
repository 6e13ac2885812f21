"""GPU test (``-m gpu``) of the allocation-free entry point ``zda_density_vjp_static`` (include/zda.h): the dF_drho tail of
``zda_gradient`` with its two intermediate planes in the library's static __device__ array instead of a workspace.

Checked against the EXISTING path (``zda_gradient``'s dF_drho of a zone that ran forward + adjoint) and against the oracle's
``density_vjp``, on calls in a row that share the static array: a large map, then a small one (which finds the large one's
leftovers in the scratch), then the large one again (must reproduce the first call bit for bit).

Named ``test_zz_*`` so that pytest collects it last: the suite runs with ``pytest -x`` and a failure here must not hide
the other tests.  Needs nothing from them: it passes alone in a fresh process and after the rest of the suite."""
from dataclasses import replace

import numpy as np
import pytest

from oracle.density import density_vjp
from parity import rel_l2
from paper_2501_07979_b200 import zda
from workloads import config2, config3, cut_down

pytestmark = pytest.mark.gpu

TOL = {64: 5e-13, 32: 1e-5}     # fp64: the suite's bar (test_gpu_parity.TOL64_GRAD); fp32: same kernels, so far below 1e-3


def _existing_path(inp, precision):
    """zda_gradient of a zone after a forward and an adjoint run: (dF_deps_zsum, dF_drho), ABI layout [j][id]."""
    z = zda.Zone(inp, precision=precision)
    try:
        z.run_forward()
        z.build_adjoint_source()
        z.run_adjoint()
        _, zs, drho = z.gradient(False, True, True)
    finally:
        z.close()
    return np.ascontiguousarray(zs.T), np.ascontiguousarray(drho.T)


def _static_path(inp, precision, zs):
    """The same map through zda_density_vjp_static: device tensors in and out, nothing else."""
    import torch
    dm = inp.density
    rdt = np.float32 if precision == 32 else np.float64
    nrd, nphi = dm.rho.shape
    rho_d = torch.from_numpy(np.ascontiguousarray(np.asarray(dm.rho).T, dtype=rdt)).cuda()
    zs_d = torch.from_numpy(np.ascontiguousarray(zs, dtype=rdt)).cuda()
    out_d = torch.full((nphi, nrd), float("nan"), dtype=rho_d.dtype, device="cuda")
    before = torch.cuda.memory_allocated()
    zda.zda_density_vjp_static(precision, nrd, nphi, rho_d, zs_d, out_d, dm.eps0, dm.eps_h, dm.filt_sigma, dm.beta, dm.eta,
                               torch.cuda.current_stream())
    assert torch.cuda.memory_allocated() == before
    torch.cuda.synchronize()
    return out_d.cpu().numpy()


def _check(inp, precision, zs, drho, label):
    got = _static_path(inp, precision, zs)
    assert np.isfinite(got).all()
    err = rel_l2(got, drho)
    # the oracle's VJP of the same z-summed gradient (a box one layer deep), in (r, phi) order
    ora = density_vjp(inp.density, zs.T.astype(np.float64)[:, :, None]).T
    err_o = rel_l2(got, ora)
    print(f"PARITY {label} fp{precision}: vs zda_gradient {err:.3g}, vs oracle {err_o:.3g}")
    assert err <= TOL[precision], (label, err)
    assert err_o <= (5e-13 if precision == 64 else 1e-3), (label, err_o)
    return got


@pytest.mark.parametrize("precision", [64, 32])
def test_static_scratch_entry_point_matches_zda_gradient_on_calls_in_a_row(precision):
    big = replace(cut_down(config3(n_steps=300), Nr=170, Nphi=19, n_steps=300), n_steps_adjoint=300)
    small = replace(cut_down(config2(n_steps=300), Nr=90, Nphi=5, n_steps=300), n_steps_adjoint=300)
    assert big.density is not None and small.density is not None and big.density.conic_radius == 0.0
    ref = {name: _existing_path(inp, precision) for name, inp in (("big", big), ("small", small))}
    first = _check(big, precision, *ref["big"], "static scratch, call 1 (170 x 19 zone)")
    _check(small, precision, *ref["small"], "static scratch, call 2 (90 x 5 zone, scratch holds call 1)")
    again = _check(big, precision, *ref["big"], "static scratch, call 3 (call 1 repeated)")
    assert np.array_equal(first, again)


def test_static_scratch_entry_point_refuses_what_does_not_fit():
    """2 planes of Nr_d x Nphi elements must fit ZDA_STATIC_SCRATCH_BYTES = 16 MiB: 2 Mi cells in fp32, 1 Mi in fp64."""
    import torch
    buf = torch.zeros(8, dtype=torch.float64, device="cuda")      # never touched: the call is refused before any launch
    args = (1.0, 4.0, 2.0, 8.0, 0.5)
    for precision, nrd, nphi in ((32, 2049, 1024), (64, 1025, 1024), (64, 1 << 20, 2)):
        with pytest.raises(zda.ZdaError) as e:
            zda.zda_density_vjp_static(precision, nrd, nphi, buf, buf, buf, *args)
        assert e.value.code == zda.ZDA_E_BADARG and "static array holds 16777216 B" in str(e.value)
    for bad in ((16, 4, 2, buf, buf, buf) + args, (32, 0, 2, buf, buf, buf) + args, (32, 4, 2, None, buf, buf) + args,
                (32, 4, 2, buf, buf, buf, 1.0, 4.0, 0.0, 8.0, 0.5), (32, 4, 2, buf, buf, buf, 1.0, 4.0, 17.0, 8.0, 0.5),
                (32, 4, 2, buf, buf, buf, 1.0, 4.0, 2.0, 8.0, 1.0)):
        with pytest.raises(zda.ZdaError) as e:
            zda.zda_density_vjp_static(*bad)
        assert e.value.code == zda.ZDA_E_BADARG
    torch.cuda.synchronize()
    assert float(buf.sum()) == 0.0
    # the largest map that fits, fp32: 2 Mi cells exactly (runs; result of an all-zero gradient is all zero)
    n = 1 << 21
    rho = torch.rand(n, dtype=torch.float32, device="cuda")
    g = torch.zeros(n, dtype=torch.float32, device="cuda")
    out = torch.full((n,), float("nan"), dtype=torch.float32, device="cuda")
    zda.zda_density_vjp_static(32, 2048, 1024, rho, g, out, *args)
    torch.cuda.synchronize()
    assert float(out.abs().max()) == 0.0
