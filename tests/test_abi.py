"""CPU-side checks of the boundary: libzda.so loads and exports every symbol include/zda.h declares,
and the description checks that need no GPU (CFL, argument validation) return the documented codes."""
import ctypes
import math
import os
import re

import numpy as np

from paper_2501_07979_b200 import zda
from workloads import config1

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "zda.h")).read()
    return sorted(set(re.findall(r"^ZDA_API [\w \*]+?\b(zda_\w+)\(", text, flags=re.M)))


def test_header_symbols_are_exported():
    lib = zda.load_library()
    names = _declared_symbols()
    assert len(names) >= 18
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(zda.EXPORTS) == names


def test_desc_struct_matches_header_field_order():
    text = open(os.path.join(ROOT, "include", "zda.h")).read()
    body = text[text.index("typedef struct zda_zone_desc {"):text.index("} zda_zone_desc;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = []
    for decl in body.split(";"):
        decl = decl.strip()
        m = re.match(r"(?:typedef struct zda_zone_desc \{)?\s*(const double\*|int|double)\s+(.*)", decl, flags=re.S)
        if m:
            fields += [f.strip() for f in m.group(2).split(",")]
    assert fields == [f[0] for f in zda.zda_zone_desc._fields_]


def test_workspace_bytes_and_validation_without_gpu():
    inp = config1()
    d, keep = zda.desc_from_inputs(inp, 32)
    n32 = zda.zda_zone_workspace_bytes(d, 600)
    d64, keep64 = zda.desc_from_inputs(inp, 64)
    n64 = zda.zda_zone_workspace_bytes(d64, 600)
    vox = inp.n_voxels
    assert n32 > 12 * 4 * vox and n64 > 1.9 * n32 * 0.9
    lib = zda.load_library()
    # dt above the cylindrical CFL limit -> ZDA_E_CFL through zda_zone_create (no device touched)
    d.dt = 0.9
    out = ctypes.c_void_p()
    rc = lib.zda_zone_create(ctypes.byref(d), None, 600, 256, 1 << 30, None, ctypes.byref(out))
    assert rc == zda.ZDA_E_CFL and "CFL" in zda.zda_last_error()
    d.dt = inp.dt
    # monitor plane inside the z-PML
    d.monitor_k = 2
    assert lib.zda_zone_create(ctypes.byref(d), None, 600, 256, 1 << 30, None, ctypes.byref(out)) == zda.ZDA_E_BADARG
    d.monitor_k = inp.monitor_k
    # dphi inconsistent with n_fold
    d.dphi = 2 * math.pi / (inp.n_fold * inp.Nphi) * 1.01
    assert lib.zda_zone_create(ctypes.byref(d), None, 600, 256, 1 << 30, None, ctypes.byref(out)) == zda.ZDA_E_BADARG
    d.dphi = inp.dphi
    # complex phase with real fields
    d.phase_re, d.phase_im = math.cos(0.3), math.sin(0.3)
    assert lib.zda_zone_create(ctypes.byref(d), None, 600, 256, 1 << 30, None, ctypes.byref(out)) == zda.ZDA_E_BADARG
    d.phase_re, d.phase_im = 1.0, 0.0
    # misaligned / NULL workspace
    assert lib.zda_zone_create(ctypes.byref(d), None, 600, None, 1 << 30, None, ctypes.byref(out)) == zda.ZDA_E_BADARG
    assert lib.zda_zone_create(ctypes.byref(d), None, 600, 264, 1 << 30, None, ctypes.byref(out)) == zda.ZDA_E_BADARG
    # axis zone with an inner r-PML
    d.has_axis, d.r_in = 1, 0.0
    assert lib.zda_zone_create(ctypes.byref(d), None, 600, 256, 1 << 30, None, ctypes.byref(out)) == zda.ZDA_E_BADARG
    assert out.value is None
    del keep, keep64


def test_table_marshalling():
    t = np.array([[1 + 2j, 3 - 4j]])
    assert np.array_equal(zda.table_to_abi(t, True), np.array([[1.0, 2.0, 3.0, -4.0]]))
    assert np.array_equal(zda.table_to_abi(t.real, False), np.array([[1.0, 3.0]]))


def test_one_phi_cell_cfl_limit_in_the_library_matches_the_oracle():
    """R21: for Nphi == 1 the library's CFL check uses (K^2 + 1/2 [axis]) / (2 r_min)^2 with K = |p - 1| / dphi, like the
    oracle's cfl_limit (two independent implementations): dt just below the limit is accepted by the validator
    (zda_zone_workspace_bytes > 0), dt just above it is ZDA_E_CFL; R10's 1/(r_min dphi)^2 would reject both."""
    from oracle import cfl_limit
    from workloads import config7_first_zone
    inp = config7_first_zone(n_steps=100)
    lim = cfl_limit(inp.dr, inp.dz, inp.dphi, 0.0, True, 1, inp.phase)
    old = 1.0 / math.sqrt(1 / inp.dr ** 2 + 1 / inp.dz ** 2 + 1 / (0.5 * inp.dr * inp.dphi) ** 2)
    assert old < 0.01 < inp.dt <= lim          # the config's own dt needs R21
    d, keep = zda.desc_from_inputs(inp, 32)
    lib = zda.load_library()
    out = ctypes.c_void_p()
    d.dt = lim * (1 - 1e-9)
    assert zda.zda_zone_workspace_bytes(d, 100) > 0
    d.dt = lim * (1 + 1e-6)
    assert lib.zda_zone_create(ctypes.byref(d), None, 100, 256, 1 << 30, None, ctypes.byref(out)) == zda.ZDA_E_CFL
    # an annular one-phi-cell zone: no axis term
    d.has_axis, d.r_in, d.npml_r_lo, d.design_i0 = 0, 100.0, 12, 12
    lim_a = cfl_limit(inp.dr, inp.dz, inp.dphi, 100.0, False, 1, inp.phase)
    d.dt = lim_a * (1 - 1e-9)
    assert zda.zda_zone_workspace_bytes(d, 100) > 0
    d.dt = lim_a * (1 + 1e-6)
    assert lib.zda_zone_create(ctypes.byref(d), None, 100, 256, 1 << 30, None, ctypes.byref(out)) == zda.ZDA_E_CFL
    del keep


def test_description_limits_are_rejected_with_badarg():
    """launch-grid limits of the small kernels and the step-table bound are checked up front."""
    inp = config1()
    d, keep = zda.desc_from_inputs(inp, 32)
    lib = zda.load_library()
    assert lib.zda_zone_workspace_bytes(ctypes.byref(d), (1 << 24) + 1) == 0 and "max_steps" in zda.zda_last_error()
    d.eps_volume = 2
    assert lib.zda_zone_workspace_bytes(ctypes.byref(d), 600) == 0
    d.eps_volume = 1
    n_vol = lib.zda_zone_workspace_bytes(ctypes.byref(d), 600)
    d.eps_volume = 0
    n0 = lib.zda_zone_workspace_bytes(ctypes.byref(d), 600)
    Ld = inp.design_k1 - inp.design_k0
    assert n_vol - n0 >= 4 * (inp.Nz - Ld) * inp.Nphi * inp.Nr          # one more float per voxel outside the layer
    d.Nphi, d.n_fold = 70000, 0
    d.dphi = 1e-6
    assert lib.zda_zone_workspace_bytes(ctypes.byref(d), 600) == 0 and "Nphi" in zda.zda_last_error()
    del keep


_NOMEM_CHILD = r"""
import ctypes, resource, sys
sys.path.insert(0, %(root)r)
from paper_2501_07979_b200 import zda
from workloads import config1
inp = config1()
d, keep = zda.desc_from_inputs(inp, 64)
lib = zda.load_library(build_if_missing=False)
out = ctypes.c_void_p()
# baseline: without a memory limit the call gets as far as the first CUDA call (no device here -> ZDA_E_CUDA) or succeeds
big = 1 << 24                        # max_steps: the host twiddle table alone is 2^24 x 16 B = 268 MB
import os
vm = int(open('/proc/self/statm').read().split()[0]) * os.sysconf('SC_PAGE_SIZE')
resource.setrlimit(resource.RLIMIT_AS, (vm + (96 << 20), vm + (96 << 20)))
rc = lib.zda_zone_create(ctypes.byref(d), None, big, 256, 1 << 62, None, ctypes.byref(out))
print("RC", rc, zda.zda_last_error())
"""


def test_bad_alloc_does_not_cross_the_abi():
    """include/zda.h: 'Nothing throws or aborts across the ABI'.  A child process whose address space is capped 96 MB above
    its current size asks for a zone with 2^24 steps: the host-side twiddle table (268 MB) cannot be allocated, the
    std::bad_alloc is caught at the boundary and comes back as ZDA_E_NOMEM (an uncaught exception would abort the child)."""
    import subprocess
    import sys
    zda.load_library()            # make sure the library is built before the child loads it
    r = subprocess.run([sys.executable, "-c", _NOMEM_CHILD % {"root": ROOT}], capture_output=True, text=True, timeout=120)
    assert r.returncode == 0, r.stderr[-2000:]
    line = [l for l in r.stdout.splitlines() if l.startswith("RC")][-1]
    assert line.split()[1] == str(zda.ZDA_E_NOMEM), line
    assert "bad_alloc" in line
