#!/usr/bin/env python
"""bench.py -- throughput of the ZDA zone solve (libzda) on B200, in FDTD voxel-updates/s (fp32).

A bench *step* is one pass of the whole hot path over one synthetic zone: ``zda_run_forward`` (and, for the
forward+adjoint workloads, ``zda_build_adjoint_source`` + ``zda_run_adjoint`` + ``zda_gradient``) on the full
grid of the workload, for ``--nt`` time steps per run (default: a tenth of the config's horizon so that the
default invocation ends within minutes; ``--nt 0`` runs the full horizon -- the rate does not depend on it).
Workload at N = 1: BASELINE.json configs[3], the ~1e9-voxel 6-wavelength zone (2000 x 2000 x 250, F = 6, forward +
adjoint + gradient) that north_star quotes its throughput target on; it fits one B200 (85 GB).  ``--workload
config2`` / ``config3`` time the LWIR and RGB zones.  See DESIGN.md "Measurement".

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
    full = {"config1": 600, "config2": 4000, "config3": 6000, "config4": 8000, "config6": 4000, "config7": 4000}[name]
    if nt <= 0:
        nt = full
    fn = {"config1": W.config1, "config2": W.config2, "config3": W.config3, "config4": W.config4,
          "config6": W.config6_thin_wedge, "config7": W.config7_first_zone}[name]
    seed = {"config1": 1, "config2": 2, "config3": 3, "config4": 4, "config6": 6, "config7": 7}[name] + 100 * rank
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


# ------------------------------------------------------------------------------------------------
# the CUDA arm (libzda through its C ABI)
# ------------------------------------------------------------------------------------------------
def _pin(torch, a: np.ndarray):
    t = torch.from_numpy(np.ascontiguousarray(a))
    try:
        return t.pin_memory()
    except Exception:
        return t


class HotPath:
    """One bench step = the whole hot path over one zone.  ``step_resident`` starts from inputs already in
    HBM (materials and source loaded before the timed region); ``step_e2e`` goes through the same C-ABI calls
    with HOST buffers: density / eps and source sheets up, objective + gradient (or monitor DFT) down."""

    def __init__(self, inp, nt, kernel=0, options=None):
        import torch
        from paper_2501_07979_b200 import zda
        self.torch, self.zda, self.inp, self.nt = torch, zda, inp, nt
        self.adjoint = inp.n_steps_adjoint > 0
        self.zone = zda.Zone(inp, precision=32, max_steps=nt, kernel=kernel, load_inputs=False, options=options)
        host = self.zone.host_inputs()
        self.table = host.pop("table")
        self.host = {k: _pin(torch, v.view(np.float32) if np.iscomplexobj(v) else v) for k, v in host.items()}
        self._load_from_host()
        nr, nphi, _ = inp.design_shape
        self.g_host = _pin(torch, np.zeros((nphi, nr), dtype=np.float32))
        self.mon_host = _pin(torch, np.zeros((inp.n_freq, 2, nphi, inp.Nr, 2), dtype=np.float32))
        self.g_dev = torch.zeros((nphi, nr), dtype=torch.float32, device="cuda")
        self.h2d = sum(int(v.numel() * v.element_size()) for v in self.host.values()) + int(self.table.nbytes)
        self.d2h = int(self.g_host.numel() * 4 + 8) if self.adjoint else int(self.mon_host.numel() * 4)
        self.runs = 2 if self.adjoint else 1
        self.updates_per_step = float(inp.n_voxels) * nt * self.runs

    def _load_from_host(self):
        zda, h, inp, z = self.zda, self.host, self.inp, self.zone.handle
        if "rho" in h:
            dm = inp.density
            if dm.conic_radius > 0:
                zda.zda_set_density_conic(z, h["rho"].data_ptr(), 1, dm.eps0, dm.eps_h, dm.conic_radius, dm.beta, dm.eta)
            else:
                zda.zda_set_density(z, h["rho"].data_ptr(), 1, dm.eps0, dm.eps_h, dm.filt_sigma, dm.beta, dm.eta)
        else:
            zda.zda_set_design_eps(z, h["eps_design"].data_ptr(), 1)
        zda.zda_set_source(z, int(np.asarray(inp.src_A_r).shape[0]), h["A_r"].data_ptr(), h["A_phi"].data_ptr(), 1,
                           self.table, self.nt)

    def step_resident(self):
        zda, z = self.zda, self.zone.handle
        zda.zda_run_forward(z, self.nt)
        if self.adjoint:
            zda.zda_build_adjoint_source(z, zda.ZDA_OBJ_MONITOR_ENERGY, self.inp.adj_t0, self.inp.adj_sigma_t, self.nt, False)
            zda.zda_run_adjoint(z, self.nt)
            zda.zda_gradient(z, None, self.g_dev.data_ptr(), None, 0)

    def step_e2e(self):
        zda, z = self.zda, self.zone.handle
        self._load_from_host()
        zda.zda_run_forward(z, self.nt)
        if self.adjoint:
            F = zda.zda_build_adjoint_source(z, zda.ZDA_OBJ_MONITOR_ENERGY, self.inp.adj_t0, self.inp.adj_sigma_t, self.nt, True)
            zda.zda_run_adjoint(z, self.nt)
            if "rho" in self.host:
                zda.zda_gradient(z, None, None, self.g_host.data_ptr(), 1)
            else:
                zda.zda_gradient(z, None, self.g_host.data_ptr(), None, 1)
            return F
        for f in range(self.inp.n_freq):
            for c in range(2):
                zda.zda_get_dft(z, zda.ZDA_FWD, zda.ZDA_MONITOR, c, f, self.mon_host[f, c].data_ptr(), 1)
        return float(self.mon_host[0, 0, 0, self.inp.Nr // 2, 0])

    def close(self):
        self.zone.close()


class LensPass:
    """BASELINE.json configs[4]: one full gradient evaluation of a 24-zone lens, zones solved back to back on the one
    GPU (a10) in ONE workspace sized for the largest zone; per zone: create, materials + source in, forward, adjoint
    source, adjoint, gradient (``zda_lens_gradient``), dF/drho out."""

    def __init__(self, nt, n_zones=24, rank=0):
        import torch
        import workloads as W
        from paper_2501_07979_b200 import zda
        self.torch, self.zda, self.nt = torch, zda, nt
        self.zones = W.config5_zones(seed=5 + 100 * rank, n_zones=n_zones, n_steps=nt)
        self.adjoint = True
        self.runs = 2
        need = 0
        for z in self.zones:
            d, _keep = zda.desc_from_inputs(z, 32)
            need = max(need, zda.zda_zone_workspace_bytes(d, nt))
        self.workspace = torch.empty(need, dtype=torch.uint8, device="cuda")
        self.host, self.dev, self.g_dev, self.g_host = [], [], [], []
        self.h2d = self.d2h = 0
        for z in self.zones:
            rho = np.ascontiguousarray(np.asarray(z.density.rho).T, dtype=np.float32)
            A_r = np.ascontiguousarray(np.asarray(z.src_A_r).transpose(0, 2, 1), dtype=np.float32)
            A_p = np.ascontiguousarray(np.asarray(z.src_A_phi).transpose(0, 2, 1), dtype=np.float32)
            h = {"rho": _pin(torch, rho), "A_r": _pin(torch, A_r), "A_phi": _pin(torch, A_p),
                 "table": zda.table_to_abi(z.src_table, False)}
            self.host.append(h)
            self.dev.append({k: (v.cuda() if k != "table" else v) for k, v in h.items()})
            self.g_dev.append(torch.zeros(rho.shape, dtype=torch.float32, device="cuda"))
            self.g_host.append(_pin(torch, np.zeros(rho.shape, dtype=np.float32)))
            self.h2d += rho.nbytes + A_r.nbytes + A_p.nbytes + h["table"].nbytes
            self.d2h += rho.nbytes + 8
        self.updates_per_step = float(sum(z.n_voxels for z in self.zones)) * nt * 2
        self.launches = 0
        self.kernel_name = ""

    def _pass(self, on_host):
        zda = self.zda
        Fs = []
        for l, z in enumerate(self.zones):
            zone = zda.Zone(z, precision=32, max_steps=self.nt, load_inputs=False, workspace=self.workspace)
            try:
                src = self.host[l] if on_host else self.dev[l]
                zone.load_inputs(src, on_host)
                F = zda.zda_lens_gradient([zone.handle], [self.nt], [self.nt], [z.adj_t0], [z.adj_sigma_t], None,
                                          [self.g_dev[l]])
                if on_host:
                    self.g_host[l].copy_(self.g_dev[l], non_blocking=True)
                Fs.append(float(F[0]))
                self.launches += zone.launch_count
                self.kernel_name = zone.kernel_name
            finally:
                zone.close()
        return Fs

    def step_resident(self):
        return self._pass(0)

    def step_e2e(self):
        return self._pass(1)


class PaperLensPass:
    """--workload config8: a lens shaped like the paper's LWIR design: the
    continuously axisymmetric first zone (config 7) and 15 thin Bloch wedges (config 6, zone numbers 2..16), 16 zones of
    ~2e6 voxels.  Every zone is RESIDENT (own workspace, 5 GB in all) and sits on one of ``n_streams`` CUDA streams;
    one ``zda_lens_gradient`` call drives them phase by phase, so zones on different streams overlap on the GPU (a zone
    is less than one wave of CTAs)."""

    def __init__(self, nt, n_streams=4, rank=0):
        import torch
        import workloads as W
        from paper_2501_07979_b200 import zda
        self.torch, self.zda, self.nt = torch, zda, nt
        self.zones = [W.config7_first_zone(seed=7 + 100 * rank, n_steps=nt)]
        self.zones += [W.config6_thin_wedge(seed=6 + ell + 100 * rank, ell=ell, n_steps=nt) for ell in range(2, 17)]
        self.adjoint, self.runs = True, 2
        self.streams = [torch.cuda.Stream() for _ in range(max(1, n_streams))]
        self.objs, self.host, self.dev, self.g_dev, self.g_host = [], [], [], [], []
        self.h2d = self.d2h = 0
        for l, z in enumerate(self.zones):
            o = zda.Zone(z, precision=32, max_steps=nt, load_inputs=False, stream=self.streams[l % len(self.streams)])
            h = {k: (_pin(torch, v) if k != "table" else v) for k, v in o.host_inputs().items()}
            self.objs.append(o)
            self.host.append(h)
            self.dev.append({k: (v.cuda() if k != "table" else v) for k, v in h.items()})
            shape = tuple(h["rho"].shape)
            self.g_dev.append(torch.zeros(shape, dtype=torch.float32, device="cuda"))
            self.g_host.append(_pin(torch, np.zeros(shape, dtype=np.float32)))
            self.h2d += sum(int(v.numel() * v.element_size()) for k, v in h.items() if k != "table") + h["table"].nbytes
            self.d2h += int(self.g_host[-1].numel()) * 4 + 8
        self.updates_per_step = float(sum(z.n_voxels for z in self.zones)) * nt * 2
        self.kernel_name = self.objs[1].kernel_name
        torch.cuda.synchronize()

    @property
    def launches(self):
        return sum(o.launch_count for o in self.objs) - self._launch_base

    @launches.setter
    def launches(self, v):
        self._launch_base = sum(o.launch_count for o in self.objs) - v

    def _pass(self, on_host):
        zda, torch = self.zda, self.torch
        for l, o in enumerate(self.objs):
            with torch.cuda.stream(o.stream):
                o.load_inputs(self.host[l] if on_host else self.dev[l], on_host)
        F = zda.zda_lens_gradient([o.handle for o in self.objs], [self.nt] * len(self.objs), [self.nt] * len(self.objs),
                                  [z.adj_t0 for z in self.zones], [z.adj_sigma_t for z in self.zones], None, self.g_dev)
        if on_host:
            for l, o in enumerate(self.objs):
                with torch.cuda.stream(o.stream):
                    self.g_host[l].copy_(self.g_dev[l], non_blocking=True)
        for st in self.streams:          # the timed region ends on the current stream: join the zone streams into it
            torch.cuda.current_stream().wait_stream(st)
        return list(F)

    def step_resident(self):
        return self._pass(0)

    def step_e2e(self):
        return self._pass(1)


def max_over_ranks(ms_local: float, dist, device) -> float:
    """Timing rule for N > 1: every rank times its own region with CUDA events; the job's time is the MAX."""
    import torch
    t = torch.tensor([ms_local], dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank_step: float, steps: int, world: int, ms: float) -> float:
    """Replicas only: every rank solves its own zone, so the whole-job rate is the units all ranks
    processed over the slowest rank's time."""
    return units_per_rank_step * steps * world / (ms * 1e-3)


def run_cuda(args):
    import torch
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: libzda has no CPU path")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # replicas only: every rank solves its own zone (seed offset), no data-path collective
    inp, nt, full = make_workload(args.workload, args.nt, rank)
    hp = HotPath(inp, nt, kernel=args.kernel, options=plan_options(args))
    zda = hp.zda
    warm = max(args.warmup, 3)

    def timed(fn, steps):
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        ev0.record()
        for _ in range(steps):
            fn()
        ev1.record()
        barrier()
        return max_over_ranks(ev0.elapsed_time(ev1), dist, "cuda")

    for _ in range(warm):
        hp.step_resident()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    l0 = hp.zone.launch_count
    ms = timed(hp.step_resident, args.steps)
    launches = hp.zone.launch_count - l0
    clocks = sampler.stop() if rank == 0 else {}
    value = whole_job_rate(hp.updates_per_step, args.steps, world, ms)

    # dominant kernel: the time-loop kernel(s).  One forward run alone, events on the zone's stream; per-launch
    # duration = run time / launches of that run (memsets excluded by timing after a throw-away reset).
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    lk0 = hp.zone.launch_count
    ev0.record()
    zda.zda_run_forward(hp.zone.handle, nt)
    ev1.record()
    torch.cuda.synchronize()
    k_ms = ev0.elapsed_time(ev1)
    k_launches = hp.zone.launch_count - lk0
    b_alg = algorithmic_bytes_per_voxel_step(inp)
    # bytes per time step of the schedule that ran (the library's own accounting of its launch plan: fields once per pass,
    # psi in slabs, dt/eps on the material planes, accumulators at their visit period incl. the ring copies of E)
    sched = zda.zda_schedule_bytes(hp.zone.handle, zda.ZDA_FWD)
    sched_bytes = sched["fields"] + sched["psi"] + sched["eps"] + sched["dft"]
    sched_gbs = sched_bytes * nt / (k_ms * 1e-3) / 1e9
    # the contract's figure: ALGORITHMIC bytes (every field read + written every step, accumulators every
    # step) over the live duration -- above the peak when temporal blocking moves fewer bytes than that
    achieved = b_alg * inp.n_voxels * nt / (k_ms * 1e-3) / 1e9
    peak, peak_src = hbm_peak()

    # end to end through the C ABI with host buffers (H2D of materials + source, D2H of the result, every step)
    hp.step_e2e()
    e2e_ms = timed(hp.step_e2e, args.steps)
    e2e_value = whole_job_rate(hp.updates_per_step, args.steps, world, e2e_ms)

    kname = hp.zone.kernel_name
    hp.close()
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        sample = oracle_sample(inp, nphi_sample=48 if hp.adjoint else 96)
        secs, upd, threads = time_oracle(sample, hp.adjoint)
        one = oracle_one_thread(args.workload, args.nt, hp.adjoint)
        cpu = {"value": upd / secs, "unit": UNIT, "cores": threads, "kind": "oracle",
               "sample": f"{sample.Nr}x{sample.Nphi}x{sample.Nz} cells x {sample.n_steps} time steps"
                         f"{' x 2 runs (fwd+adj)' if hp.adjoint else ''} of {args.workload}, float64, {secs:.1f} s",
               "one_thread": one, "cpu_model": cpu_model()}

    traffic, traffic_src = captured_traffic(args.workload, kname)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": warm,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": args.workload, "grid": [inp.Nr, inp.Nphi, inp.Nz], "complex_fields": bool(inp.complex_fields),
                   "n_freq": inp.n_freq, "time_steps_per_run": nt, "full_horizon": full, "runs_per_step": hp.runs,
                   "zone_solve_s_at_full_horizon": (ms / args.steps) * 1e-3 * full / nt,
                   "kernel": kname, "parallelism": "replicas" if world > 1 else "single",
                   "l2": "working set (fields %.1f GB) exceeds the 126 MB L2; no flush needed" % (24.0 * inp.n_voxels * (2 if inp.complex_fields else 1) / 1e9)},
        "clocks": {k: clocks.get(k) for k in ("sm_mhz", "sm_max_mhz", "reasons")},
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": hp.h2d, "d2h_bytes_per_step": hp.d2h,
                "ms_per_step": e2e_ms / args.steps},
        "gpu_launches": int(launches),
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     # dram__bytes_read.sum + dram__bytes_write.sum per time step from the committed ncu capture of THIS
                     # kernel plan (profiles/r02_traffic.json names the capture and the commit); None when the plan that
                     # ran is not the one profiled
                     "traffic": traffic, "traffic_source": traffic_src,
                     "traffic_gbs": (traffic / (k_ms / nt * 1e-3) / 1e9 if traffic else None),
                     "traffic_frac": (traffic / (k_ms / nt * 1e-3) / 1e9 / peak if traffic else None),
                     "note": "achieved = SURVEY 8(d) algorithmic bytes (alg_bytes_per_voxel_step x voxels: fields and accumulators "
                             "read + written EVERY step) / live duration per time step; it exceeds the peak where temporal blocking "
                             "(two steps per pass, accumulators visited every 8th step; bit-identical results) moves fewer bytes.  "
                             "schedule_* = the bytes the launch plan that ran must move (zda_schedule_bytes), schedule_frac <= 1 = how "
                             "close the kernels are to moving THEIR bytes at copy speed; traffic_* = DRAM bytes from the ncu capture",
                     "alg_bytes_per_voxel_step": b_alg, "algorithmic_bytes_per_launch": b_alg * inp.n_voxels,
                     "schedule_bytes": sched_bytes, "schedule_bytes_parts": sched,
                     "schedule_bytes_per_voxel_step": sched_bytes / inp.n_voxels,
                     "schedule_gbs": sched_gbs, "schedule_frac": sched_gbs / peak,
                     "peak_source": peak_src, "kernel": kname, "launches": int(k_launches),
                     "ms_per_time_step": k_ms / nt, "gvox_per_s_forward": inp.n_voxels * nt / (k_ms * 1e-3) / 1e9},
        "cpu_baseline": cpu,
    }
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()
    return 0


def captured_traffic(workload: str, kname: str):
    """DRAM bytes per time step from the committed ncu capture of this workload, ONLY if the launch plan that ran is the one
    that was profiled (profiles/r02_traffic.json: workload -> [{kernel, bytes_per_time_step, source, commit}, ...]); the file is
    written from the captures by hand, so it is keyed on the exact kernel-name string and goes silent, not stale."""
    path = os.path.join(ROOT, "profiles", "r02_traffic.json")
    try:
        with open(path) as f:
            entries = json.load(f).get(workload) or []
    except (OSError, ValueError):
        return None, None
    if isinstance(entries, dict):
        entries = [entries]
    entry = next((e for e in entries if e.get("kernel") == kname), None)    # one entry per profiled launch plan
    if entry is None:
        return None, None
    return float(entry["bytes_per_time_step"]), f"{entry['source']} @ {entry['commit']}"


def cpu_model() -> str:
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def oracle_one_thread(workload: str, nt: int, adjoint: bool):
    """The same oracle on ONE thread, on a quarter of the sample, in a child process with
    OMP_NUM_THREADS=1 (the OpenMP runtime reads it at load)."""
    import subprocess
    code = ("import sys, json; sys.path.insert(0, %r); import bench; "
            "inp, nt, full = bench.make_workload(%r, %d); "
            "s = bench.oracle_sample(inp, nphi_sample=12, nt_sample=12); "
            "secs, upd, thr = bench.time_oracle(s, %r); print(json.dumps({'value': upd / secs, 'cores': thr, 'seconds': secs}))"
            % (ROOT, workload, nt, adjoint))
    env = dict(os.environ, OMP_NUM_THREADS="1")
    try:
        out = subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, timeout=300)
        return json.loads(out.stdout.strip().splitlines()[-1])
    except Exception as e:  # the baseline is a reported extra, never a reason to lose the bench line
        return {"error": str(e)[:200]}


def run_lens(args):
    """--workload config5: the full 24-zone lens pass (a10).  Same JSON contract; `value` = aggregate voxel-updates/s
    of one gradient evaluation of the whole lens, zone creation and per-zone resets included."""
    import torch
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: libzda has no CPU path")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    nt = args.nt
    paper = args.workload == "config8"
    lp = PaperLensPass(nt, n_streams=args.streams, rank=rank) if paper else LensPass(nt, rank=rank)
    warm = max(args.warmup, 3)

    def timed(fn, steps):
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()
        ev0.record()
        for _ in range(steps):
            fn()
        ev1.record()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()
        return max_over_ranks(ev0.elapsed_time(ev1), dist, "cuda")

    for _ in range(warm):
        lp.step_resident()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    lp.launches = 0
    ms = timed(lp.step_resident, args.steps)
    launches = lp.launches
    clocks = sampler.stop() if rank == 0 else {}
    value = whole_job_rate(lp.updates_per_step, args.steps, world, ms)
    e2e_ms = timed(lp.step_e2e, args.steps)
    e2e_value = whole_job_rate(lp.updates_per_step, args.steps, world, e2e_ms)
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0
    alg = sum(0.5 * (algorithmic_bytes_per_voxel_step(z) + algorithmic_bytes_per_voxel_step(z, True)) * z.n_voxels
              for z in lp.zones) * nt * 2
    achieved = alg / (ms / args.steps * 1e-3) / 1e9
    peak, peak_src = hbm_peak()
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        sample = oracle_sample(lp.zones[8 if paper else 12], nphi_sample=48)
        secs, upd, threads = time_oracle(sample, True)
        cpu = {"value": upd / secs, "unit": UNIT, "cores": threads, "kind": "oracle",
               "sample": f"zone {8 if paper else 12} of the lens, {sample.Nr}x{sample.Nphi}x{sample.Nz} cells x {sample.n_steps} time steps "
                         f"x 2 runs, float64, {secs:.1f} s"}
    full = 4000 if paper else 5000
    cfg_extra = ({"streams": len(lp.streams), "kernel": lp.kernel_name + " (zone 0: split, one phi cell, r = 0 axis)",
                  "l2": "the 16 resident zones' fields (4 GB) exceed the 126 MB L2; no flush needed"} if paper else
                 {"kernel": lp.kernel_name + " (zone 0: split, r = 0 axis)",
                  "l2": "every zone's fields (15 GB) exceed the 126 MB L2; no flush needed"})
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": warm,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": args.workload, "zones": len(lp.zones), "voxels": int(sum(z.n_voxels for z in lp.zones)),
                   "n_freq": int(lp.zones[1].n_freq), "time_steps_per_run": nt, "full_horizon": full, "runs_per_step": 2,
                   "lens_gradient_s_at_full_horizon": (ms / args.steps) * 1e-3 * full / nt,
                   "parallelism": "replicas" if world > 1 else "single", **cfg_extra},
        "clocks": {k: clocks.get(k) for k in ("sm_mhz", "sm_max_mhz", "reasons")},
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": lp.h2d, "d2h_bytes_per_step": lp.d2h,
                "ms_per_step": e2e_ms / args.steps},
        "gpu_launches": int(launches),
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": None, "peak_source": peak_src, "kernel": "fused_step_kernel over the annular zones",
                     "note": "whole-pass figure: zone creation, resets and the once-per-run kernels are inside the time"},
        "cpu_baseline": cpu,
    }
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()
    return 0


def hbm_peak():
    """Measured copy bandwidth of this pool's B200s (driver-written MEASURED_PEAKS.json), else the
    profiling guide's fallback."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        v = float(json.load(open(p))["hbm_gbs"])
        return v, "MEASURED_PEAKS.json hbm_gbs"
    except Exception:
        return 6650.0, "B200_PROFILING.md fallback (6.65 TB/s)"


def run_pair_bench(args):
    """--workload config6p: the m = +1 / m = -1 pair of the paper-shaped thin wedge
    through zda_lens_focal_gradient with library-built near-to-far weights (R24): forward runs, coherent focal sum,
    adjoint sources, adjoint runs, gradients.  --streams 1: both members on one stream, so the scheduler batches them
    into ONE launch per time step (NEXT-4); --streams 2: one stream each (two launches per step, overlapping)."""
    import torch
    import workloads as W
    from dataclasses import replace
    from paper_2501_07979_b200 import zda
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: libzda has no CPU path")
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    nt = args.nt
    base = W.config6_thin_wedge(n_steps=nt)
    members = []
    for m in (+1, -1):
        A_r, A_phi = W.plane_wave_sheet(base.Nr, base.Nphi, base.dphi, True, m)
        members.append(replace(base, phase=complex(np.exp(2j * np.pi * m / base.n_fold)), src_A_r=A_r, src_A_phi=A_phi,
                               focal_dz=20.0 * base.Nz))
    streams = [torch.cuda.Stream() for _ in range(2)] if args.streams >= 2 else [torch.cuda.current_stream()] * 2
    zones = [zda.Zone(inp, precision=32, max_steps=nt, kernel=args.kernel, stream=st, options=plan_options(args))
             for inp, st in zip(members, streams)]
    g = [torch.zeros((inp.Nphi, inp.design_i1 - inp.design_i0), dtype=torch.float32, device="cuda") for inp in members]

    def step():
        return zda.zda_lens_focal_gradient([z.handle for z in zones], [nt, nt], [nt, nt], [i.adj_t0 for i in members],
                                           [i.adj_sigma_t for i in members], None, base.n_freq, None, g)
    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    sampler = ClockSampler(0)
    sampler.start()
    l0 = sum(z.launch_count for z in zones)
    t0 = time.perf_counter()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(args.steps):
        step()
    ev1.record()
    torch.cuda.synchronize()
    wall_ms = (time.perf_counter() - t0) * 1e3
    ms = ev0.elapsed_time(ev1) if args.streams < 2 else wall_ms     # events see only torch's current stream
    clocks = sampler.stop()
    launches = sum(z.launch_count for z in zones) - l0
    upd = 2.0 * base.n_voxels * nt * 2
    kname = zones[0].kernel_name
    for z in zones:
        z.close()
    line = {"metric": METRIC, "value": upd * args.steps / (ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": "config6p", "grid": [base.Nr, base.Nphi, base.Nz], "members": 2,
                       "batched_in_one_launch": args.streams < 2, "time_steps_per_run": nt, "kernel": kname,
                       "timing": "cuda events" if args.streams < 2 else "wall clock around synchronize (two streams)"},
            "clocks": {k: clocks.get(k) for k in ("sm_mhz", "sm_max_mhz", "reasons")},
            "gpu_launches": int(launches), "roofline": None, "cpu_baseline": None, "e2e": None}
    print(json.dumps(line), flush=True)
    return 0


def plan_options(args):
    """--opt KEY=VALUE pairs -> {ZDA_OPT_*: value} (launch-plan tuning knobs of include/zda.h, for sweeps)."""
    from paper_2501_07979_b200 import zda
    out = {}
    for kv in args.opt or []:
        k, v = kv.split("=")
        out[getattr(zda, "ZDA_OPT_" + k.upper())] = int(v)
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--workload", default="config4", choices=["config1", "config2", "config3", "config4", "config5", "config6", "config6p", "config7", "config8"])
    ap.add_argument("--streams", type=int, default=4, help="config8: CUDA streams the resident zones are spread over")
    ap.add_argument("--nt", type=int, default=-1, help="time steps per run (default full/10; 0 = full horizon)")
    ap.add_argument("--kernel", type=int, default=0, help="0 auto, 1 split, 2 fused (one step per pass), 3 fused2 (two steps per pass)")
    ap.add_argument("--opt", action="append", help="launch-plan option, e.g. --opt fused_tj=13 --opt fused_chunk=63 (ZDA_OPT_*)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.nt < 0:
        args.nt = {"config1": 600, "config2": 400, "config3": 200, "config4": 100, "config5": 40, "config6": 2000,
                   "config7": 2000, "config8": 400, "config6p": 1000}[args.workload]
    if args.impl == "reference":
        if args.workload == "config5":
            args.workload = "config3"      # the lens's zones are config-3 shaped; the oracle sample is one such zone
        if args.workload in ("config8", "config6p"):
            args.workload = "config6"      # the paper-shaped lens's zones (and the pair's members) are config-6 shaped
        return run_reference(args)
    if args.workload == "config6p":
        return run_pair_bench(args)
    if args.workload in ("config5", "config8"):
        return run_lens(args)
    return run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
