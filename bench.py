#!/usr/bin/env python
"""bench.py -- throughput of the ZDA zone solve (libzda) on B200, in FDTD voxel-updates/s (fp32).

A bench *step* is one pass of the whole hot path over one synthetic zone: ``zda_run_forward`` (and, for the
forward+adjoint workloads, ``zda_build_adjoint_source`` + ``zda_run_adjoint`` + ``zda_gradient``) on the full
grid of the workload, for ``--nt`` time steps per run (default: a tenth of the config's horizon so that the
default invocation ends within minutes; ``--nt 0`` runs the full horizon -- the rate does not depend on it).
Workload at N = 1: BASELINE.json configs[1] (LWIR zone, 800 x 800 x 160, forward only).
"Measurement".

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload config2|config3|config4|config1] [--nt T]
    python bench.py --impl reference ...      # the float64 CPU oracle on a bounded sample (host cores)

Prints ONE JSON line (rank 0).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fdtd_voxel_updates_per_s"
UNIT = "voxel-updates/s"


# ------------------------------------------------------------------------------------------------
# workloads
# ------------------------------------------------------------------------------------------------
def make_workload(name: str, nt: int, rank: int = 0):
    import workloads as W
    full = {"config1": 600, "config2": 4000, "config3": 6000, "config4": 8000}[name]
    if nt <= 0:
        nt = full
    fn = {"config1": W.config1, "config2": W.config2, "config3": W.config3, "config4": W.config4}[name]
    seed = {"config1": 1, "config2": 2, "config3": 3, "config4": 4}[name] + 100 * rank
    inp = fn(seed=seed, n_steps=nt)
    return inp, nt, full


def algorithmic_bytes_per_voxel_step(inp, adjoint_run: bool = False) -> float:
    """SURVEY 8(d) / DESIGN.md "Roofline": bytes the method itself must move per voxel per time step with no
    reuse beyond one step, fp32: every field read once and written once (6 x 2 x es); CPML auxiliaries read +
    written in their slabs only (4 per slab voxel in z, 4 in r); eps (as dt/eps) read on the design box only;
    DFT accumulators (3 F complex) read + written on the design box and the monitor plane."""
    es = 8.0 if inp.complex_fields else 4.0
    Nr, Nphi, Nz = inp.Nr, inp.Nphi, inp.Nz
    vox = float(Nr) * Nphi * Nz
    fields = 12.0 * es
    cpml_z = 4.0 * 2.0 * es * (inp.npml_z_lo + inp.npml_z_hi) / Nz
    cpml_r = 4.0 * 2.0 * es * (inp.npml_r_lo + inp.npml_r_hi) / Nr
    nrd, _, ld = inp.design_shape
    design_frac = float(nrd) * Nphi * ld / vox
    eps = 4.0 * design_frac
    mon_frac = 0.0 if adjoint_run else float(Nr) * Nphi / vox
    dft = 3.0 * inp.n_freq * 8.0 * 2.0 * (design_frac + mon_frac)
    return fields + cpml_z + cpml_r + eps + dft


# ------------------------------------------------------------------------------------------------
# clocks
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.idx = gpu_index
        self.proc = None
        self.path = None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(prefix="zda_clocks_", suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.idx), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, reasons = [], [], set()
        try:
            for line in open(self.path):
                f = [x.strip() for x in line.split(",")]
                if len(f) < 9:
                    continue
                try:
                    sm.append(float(f[1])); smax.append(float(f[2]))
                except ValueError:
                    continue
                for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                    if val.lower().startswith("active"):
                        reasons.add(name)
            os.remove(self.path)
        except Exception:
            pass
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(smax)), reasons=sorted(reasons), samples=len(sm))
        return out


# ------------------------------------------------------------------------------------------------
# the oracle, timed as it stands on the host cores (cpu_baseline leg and --impl reference)
# ------------------------------------------------------------------------------------------------
def oracle_sample(inp, nphi_sample: int = 96, nt_sample: int = 24):
    """A bounded sample of the same workload for the CPU oracle: the zone's own radial extent, z stack,
    CPML, source and frequencies, with the wedge cut to ``nphi_sample`` phi-cells (dphi unchanged) and
    ``nt_sample`` time steps."""
    import workloads as W
    nphi = min(nphi_sample, inp.Nphi)
    cut = W.cut_down(inp, Nr=inp.Nr, Nphi=nphi, n_steps=min(nt_sample, inp.n_steps))
    return cut


def time_oracle(inp, adjoint: bool):
    """One oracle pass over the sample; returns (seconds, voxel_updates, threads)."""
    from oracle import OracleZone
    from oracle.density import density_to_eps
    eps = density_to_eps(inp.density, inp.design_k1 - inp.design_k0) if inp.density is not None else inp.eps_design
    z = OracleZone(inp, eps_design=eps)
    t0 = time.perf_counter()
    z.run_forward()
    runs = 1
    if adjoint:
        z.build_adjoint_source()
        z.run_adjoint()
        z.gradient()
        runs = 2
    dt = time.perf_counter() - t0
    try:
        threads = int(z.lib.zo_max_threads())
    except Exception:
        threads = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    return dt, float(inp.n_voxels) * inp.n_steps * runs, threads


def run_reference(args):
    """--impl reference: the oracle is the reference arm (no reference code exists; PAPER.md only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    inp, nt, full = make_workload(args.workload, args.nt)
    adjoint = inp.n_steps_adjoint > 0
    sample = oracle_sample(inp, nphi_sample=64, nt_sample=16)
    for _ in range(max(args.warmup, 0)):
        time_oracle(oracle_sample(inp, nt_sample=2), adjoint)
    secs, upd, threads = [], 0.0, 1
    for _ in range(args.steps):
        s, u, threads = time_oracle(sample, adjoint)
        secs.append(s); upd += u
    total = sum(secs)
    value = upd / total
    desc = (f"oracle (float64, gcc -O2 -fopenmp) on {sample.Nr}x{sample.Nphi}x{sample.Nz} cells x {sample.n_steps} "
            f"time steps{' x 2 runs (fwd+adj)' if adjoint else ''} of {args.workload} per step")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * total / max(args.steps, 1), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "grid": [inp.Nr, inp.Nphi, inp.Nz], "sample": desc},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0
