#!/usr/bin/env python
"""bench.py -- FP64 Valencia RHS cell-updates/s on one 256^3 block (WENO5 + HLLE), B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload c5-256]
                    [--recon weno5|minmod|mc] [--variant auto|tma|ldg|simple] [--no-sweep] [--sweep]

A "step" is ONE evaluation of the whole hot path (reconstruct -> HLLE -> flux divergence + sources, all three
directions) over one batch of synthetic input, i.e. one grx_valencia_rhs call = one
kernel launch.  Workload at N=1: config 5's 256^3 x 1 box (the configuration BASELINE.json's metric is quoted
on: "WENO5+HLLE, 256^3"), seeded smooth random state on a perturbed conformally flat metric with shift and
K_ij (inputs.sweep_boxes).  Inputs (4.6 GB) are far larger than the 126 MB L2, so no flush between steps.
With N>1 (torchrun) every rank evaluates its own block of the same shape (weak scaling, no data-path
collective: the path partitions over blocks); time = max over ranks.

Prints ONE JSON line (rank 0).  `value` = interior cells x boxes x ranks x steps / time, inputs resident in
HBM; `e2e` = same through grx_valencia_rhs_host with pinned HOST buffers (H2D of all inputs and D2H of the
result inside the timed region); `roofline` = algorithmic FP64 flops of the launch (the oracle's counted
operations) / kernel time against the FP64 peak, plus the HBM view; `cpu_baseline` =
the oracle, as it stands, on the host cores on a bounded sub-block of the same workload; `sweep` = every config-5
point and C3/C4 with both reconstructions (10 calls each), so that the driver-run line carries them.

--impl reference times the oracle (the only reference there is: the paper ships no code) on this host.
"""
import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2210_17509_b200 import inputs  # noqa: E402

METRIC = "FP64 Valencia RHS cell-updates/sec (WENO5+HLLE, 256^3)"
UNIT = "cell-updates/s"

# Algorithmic flops per cell-update of a cubic N^3 box = A + B/N: the operation count of the oracle's
# counting instance (add = mul = div = sqrt = 1, an FMA would be 2; every face once), fitted on
# N = 16, 32, 48 general-metric boxes (oracle/count_flops.py; tests/test_bench_model.py re-checks it).
FLOPS_MODEL = {"weno5": (4753.0, 6210.0), "minmod": (2545.0, 1794.0), "mc": (2642.0, 1460.0)}
# Nominal FP64 peak of a B200: 148 SMs x 64 FP64 lanes x 2 flop (FMA) x 1.965 GHz.
FP64_PEAK_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12
# The survey's own estimate of the straightforward formulation: quoted beside the
# official (oracle-counted) number as `frac_survey_count`.
FLOPS_SURVEY = {"weno5": 4085.0, "minmod": 2140.0}
# Numbers that only a profiler can give, from the `ncu --set full` captures summarised under profiles/ (per launch of
# the kernel of a step): DRAM bytes read + written, FP64-pipe utilisation (% of peak sustained active), executed FP64
# thread instructions per cell.  They belong to ONE state of the kernel sources: `csrc_sha` is the hash of
# paper_2210_17509_b200/csrc/ they were captured at, and bench.py reports them only while the hash still matches.
NCU_CAPTURE = {
    "csrc_sha": "d4fa1b786c4a",
    "source": "profiles/r3_ncu_tma.md",
    "c5-256/weno5/auto": {"traffic": 4.718020e9, "pipe_fp64_pct": 59.94, "fp64_inst_per_cell": 2750.0},
    "c5-256/minmod/auto": {"traffic": 4.660311e9, "pipe_fp64_pct": 47.87, "fp64_inst_per_cell": 1509.0},
}
KERNEL_OF_VARIANT = {"auto": "rhs_tma_kernel (rhs_fused_kernel for odd Nx)", "tma": "rhs_tma_kernel", "ldg": "rhs_fused_kernel",
                     "simple": "rhs_simple_kernel"}
SWEEP_POINTS = ("c5-32", "c5-64", "c5-128", "c5-256", "c3", "c4")
ORACLE_TIMED_POINTS = ("c5-64", "c5-128")     # sweep points at which the oracle is timed beside the kernel


KERNEL_SOURCES = ("grx_tma.cu", "grx_math.cuh", "grx_common.cuh")   # what the kernel of a step is compiled from


def csrc_sha():
    """Hash of the sources of the product kernel (what NCU_CAPTURE is keyed on)."""
    import hashlib
    h = hashlib.sha1()
    d = os.path.join(ROOT, "paper_2210_17509_b200", "csrc")
    for f in KERNEL_SOURCES:
        h.update(f.encode())
        h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:12]


def algorithmic_flops_per_cell(n, recon):
    a, b = FLOPS_MODEL[recon]
    return a + (b / 3.0) * (1.0 / n[0] + 1.0 / n[1] + 1.0 / n[2])


def redundant_flops_per_cell(n):
    """Operations the oracle's count holds twice: v_i and v^2 of the admissibility test (20 per face side, piece
    `admissible` of tests/test_bench_model.py) are evaluated again inside prim2con_point.  Two sides of 3 + sum 1/n_d faces
    per cell: 120 per cell of a large block.  `frac_no_redundancy` leaves them out of the numerator."""
    return 20.0 * 2.0 * (3.0 + 1.0 / n[0] + 1.0 / n[1] + 1.0 / n[2])


def algorithmic_bytes_per_cell(n, g):
    """24 input fields read once including ghosts + 8 output fields written on the interior."""
    tot = (n[0] + 2 * g) * (n[1] + 2 * g) * (n[2] + 2 * g)
    return 8.0 * (24.0 * tot / (n[0] * n[1] * n[2]) + 8.0)


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f), "measured"
    except OSError:
        return {"hbm_gbs": 6650.0}, "fallback"


# ------------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """Samples SM clock and throttle reasons of one GPU with NVML while a region runs."""

    def __init__(self, index, period=0.01):
        self.index, self.period = index, period
        self.samples, self.reasons = [], set()
        self.max_mhz = None
        self._stop = threading.Event()
        self._thread = None
        self._h = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM)
        except Exception:   # NVML not usable: clocks are reported as unknown
            self._h = None

    _NAMES = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
              0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
              0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}

    def _run(self):
        nv = self._nv
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self._h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h)
                for bit, name in self._NAMES.items():
                    if r & bit and name != "gpu_idle":
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def __enter__(self):
        if self._h is not None:
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thread:
            self._thread.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": 0}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ------------------------------------------------------------------------------------------------ oracle legs
def _sub_block(prob, nz_sub, ny_sub=None, nx_sub=None):
    """First nx_sub x ny_sub x nz_sub interior cells of box 0 with their ghost shell (a bounded sample of the
    same workload: the right-hand side of a cell only depends on cells within 3 of it)."""
    g = prob.nghost
    nx = min(nx_sub or prob.n[0], prob.n[0])
    ny = min(ny_sub or prob.n[1], prob.n[1])
    nz = min(nz_sub, prob.n[2])
    sl = (slice(0, 1), slice(None), slice(0, nz + 2 * g), slice(0, ny + 2 * g), slice(0, nx + 2 * g))
    return [np.ascontiguousarray(a[sl]) for a in (prob.prim, prob.metric, prob.K)], (nx, ny, nz)


def time_oracle(prob, recon, budget_s, reps=1):
    """Times the oracle (as it stands) on a sub-block sized for about `budget_s` seconds per repetition."""
    from oracle import oracle as orc
    orc.lib()
    (p, m, k), n0 = _sub_block(prob, 8, 64, 64)
    t0 = time.perf_counter()
    orc.valencia_rhs(p, m, k, prob.dx, prob.nghost, recon, prob.gamma)
    rate = n0[0] * n0[1] * n0[2] / max(time.perf_counter() - t0, 1e-6)    # calibration, cold
    want = max(rate * budget_s, 4096.0)
    nx, ny = prob.n[0], prob.n[1]
    nz = int(min(prob.n[2], max(1, want // (nx * ny))))
    if nz == 1 and want < nx * ny:
        ny = int(max(1, want // nx))
    (p, m, k), n1 = _sub_block(prob, nz, ny, nx)
    cells = n1[0] * n1[1] * n1[2]
    best = None
    for _ in range(reps):
        t0 = time.perf_counter()
        orc.valencia_rhs(p, m, k, prob.dx, prob.nghost, recon, prob.gamma)
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    return cells / best, best, n1, orc.num_threads()


def config_of(prob, recon, n_ranks):
    """`config` of the JSON line, the same object in both arms (what differs between the arms is in `arm` / `variant`)."""
    return {"workload": workload_string(prob, recon),
            "l2": "GPU arm: inputs 4.6 GB >> 126 MB L2, no flush; reference arm: host caches, not flushed",
            "parallelism": f"blocks x{n_ranks}, no collective (reference arm: rank 0's host cores)"}


def workload_string(prob, recon):
    """The same text in both arms, so that the driver sees one config."""
    return (f"{prob.name} per GPU, {recon}+HLLE, Gamma-law EOS, perturbed conformally flat metric + shift + K_ij, "
            f"{prob.nghost} ghosts; one right-hand-side evaluation per step")


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    prob = load_workload(args.workload, 0)
    from oracle import oracle as orc
    orc.lib()
    total_budget = 100.0
    per_step = total_budget / (args.steps + args.warmup)
    # one calibration inside time_oracle, then the same sub-block every step
    (p0, m0, k0), n0 = _sub_block(prob, 8, 64, 64)
    t0 = time.perf_counter()
    orc.valencia_rhs(p0, m0, k0, prob.dx, prob.nghost, args.recon, prob.gamma)
    rate = n0[0] * n0[1] * n0[2] / max(time.perf_counter() - t0, 1e-6)
    want = max(rate * per_step, 4096.0)
    nz = int(min(prob.n[2], max(1, want // (prob.n[0] * prob.n[1]))))
    ny = prob.n[1] if want >= prob.n[0] * prob.n[1] else int(max(1, want // prob.n[0]))
    (p, m, k), n1 = _sub_block(prob, nz, ny, prob.n[0])
    cells = n1[0] * n1[1] * n1[2]
    for _ in range(args.warmup):
        orc.valencia_rhs(p, m, k, prob.dx, prob.nghost, args.recon, prob.gamma)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        orc.valencia_rhs(p, m, k, prob.dx, prob.nghost, args.recon, prob.gamma)
    dt = time.perf_counter() - t0
    value = cells * args.steps / dt
    sample = f"first {n1[0]}x{n1[1]}x{n1[2]} interior cells (+3 ghosts) of the {prob.name} block, per step"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_of(prob, args.recon, args.gpus), "arm": "oracle on host cores, bounded sample", "variant": "n/a",
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------------------------------------ GPU arm
def max_over_ranks(seconds, world, device):
    """Time of the slowest rank (the contract's `max over ranks`); an all-reduce only when there are ranks."""
    if world == 1:
        return float(seconds)
    import torch
    import torch.distributed as dist
    t = torch.tensor([seconds], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(cells_per_rank, world, steps, t_max):
    """Weak scaling: every rank evaluates its own block(s); the job's rate counts all of them."""
    return cells_per_rank * world * steps / t_max


def load_workload(name, rank, nbox=None):
    if name.startswith("c5-"):
        N = int(name[3:])
        nbox = nbox or dict(inputs.SWEEP).get(N, 1)
        if rank == 0:
            return inputs.sweep_boxes(N, nbox)
        # other ranks: same shapes, their own seeds (boxes rank*nbox .. rank*nbox+nbox-1 of the same family)
        prims, mets, Ks = [], [], []
        for b in range(nbox):
            prim, met, K, dx, gamma = inputs._smooth_box(N, 1000 * N + rank * nbox + b, inputs.NGHOST)
            prims.append(prim), mets.append(met), Ks.append(K)
        return inputs.Problem(f"C5-{N}^3x{nbox}", (N, N, N), nbox, inputs.NGHOST, dx, gamma, np.stack(prims),
                              np.stack(mets), np.stack(Ks), ("minmod", "weno5"))
    return inputs.by_name(name)


def time_rhs(grx, torch, prob, dev, recon, steps, warmup, stream, per_call=None):
    """`steps` calls between one pair of CUDA events on the launching stream (the returned total, what `value` and
    `ms_per_step` come from); an event between consecutive calls as well, so that the median and the best single call can
    be reported beside the mean: per_call, if a list, receives the milliseconds of every call."""
    prim, met, K = dev
    out = torch.empty_like(prim)
    for _ in range(warmup):
        grx.valencia_rhs(prim, met, K, prob.dx, prob.nghost, recon, prob.gamma, out=out, stream=stream)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
    stream.synchronize()
    ev[0].record(stream)
    for i in range(steps):
        grx.valencia_rhs(prim, met, K, prob.dx, prob.nghost, recon, prob.gamma, out=out, stream=stream)
        ev[i + 1].record(stream)
    stream.synchronize()
    if per_call is not None:
        per_call.extend(ev[i].elapsed_time(ev[i + 1]) for i in range(steps))
    return ev[0].elapsed_time(ev[steps]) * 1e-3, out


def call_stats(per_call):
    """Median and best of the per-call milliseconds (the mean is ms_per_step)."""
    if not per_call:
        return {}
    a = sorted(per_call)
    n = len(a)
    return {"ms_median": a[n // 2] if n % 2 else 0.5 * (a[n // 2 - 1] + a[n // 2]), "ms_best": a[0]}


def time_zone_cycles(grx, torch, prob, dev, recon, stream, nsteps=5, ct=False):
    """zone-cycles/s = steps x cells / time of grx_step_rk: SSP-RK2, periodic ghost fill, every stage =
    RHS + update fused with con2prim + ghost fill, all on the device."""
    prim0, met, K = dev
    prim = prim0.clone()
    grx_bc = "periodic"
    cons = grx.prim2con(prim, met, prob.nghost, prob.gamma)
    ws_bytes = grx.step_workspace_bytes(prim.shape, prob.nghost, 2) + (grx.ct_workspace_bytes(prim.shape, prob.nghost) if ct else 0)
    ws = torch.empty(ws_bytes // 8, dtype=torch.float64, device="cuda")
    nfail = torch.zeros(1, dtype=torch.int64, device="cuda")
    dt = 0.2 * min(prob.dx)
    grx.step_rk(cons, prim, met, K, prob.dx, prob.nghost, recon, prob.gamma, dt, 1, rk=2, bc=grx_bc, workspace=ws, nfail=nfail,
                stream=stream, ct=ct)      # warm-up step; also makes the ghosts periodic
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    stream.synchronize()
    e0.record(stream)
    grx.step_rk(cons, prim, met, K, prob.dx, prob.nghost, recon, prob.gamma, dt, nsteps, rk=2, bc=grx_bc, workspace=ws,
                nfail=nfail, stream=stream, ct=ct)
    e1.record(stream)
    stream.synchronize()
    t = e0.elapsed_time(e1) * 1e-3
    ok = bool(torch.isfinite(cons[prob.interior]).all().item())
    return {"value": prob.cells * nsteps / t, "unit": "zone-cycles/s", "steps": nsteps, "ms_per_step": 1e3 * t / nsteps,
            "scheme": f"SSP-RK2, {recon}+HLLE{' + flux-CT' if ct else ''}, Gamma-law con2prim, periodic ghosts, static metric; {prob.name}",
            "con2prim_failures": int(nfail.item()), "finite": ok,
            "paper_context": "setupA 0.47e8 zone-cycles/s at 240^3 on one V100 (PAPER.md l.341): other hardware, context only"}


def time_ct(grx, torch, prob, dev, recon, stream, steps=10):
    """NEXT-2: grx_valencia_rhs_ct = right-hand side (face fluxes of calB written by the same launch) + face kernel for the
    lines next to the block + flux-CT kernel."""
    prim, met, K = dev
    out = torch.empty_like(prim)
    ws = torch.empty((prim.shape[0], 6) + tuple(prim.shape[2:]), dtype=torch.float64, device="cuda")
    for _ in range(3):
        grx.valencia_rhs_ct(prim, met, K, prob.dx, prob.nghost, recon, prob.gamma, out=out, workspace=ws, stream=stream)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    stream.synchronize()
    e0.record(stream)
    for _ in range(steps):
        grx.valencia_rhs_ct(prim, met, K, prob.dx, prob.nghost, recon, prob.gamma, out=out, workspace=ws, stream=stream)
    e1.record(stream)
    stream.synchronize()
    t = e0.elapsed_time(e1) * 1e-3 / steps
    return {"value": prob.cells / t, "unit": UNIT, "ms_per_call": 1e3 * t, "kernels_per_call": 3,
            "scheme": f"flux-CT of calB (reading R30), {recon}+HLLE; {prob.name}"}


def time_halo_overlap(grx, torch, prob, dev, recon, stream, world, nsteps=3):
    """NEXT-4: SSP-RK2 steps of a z-slab ring (this rank's block = one slab; periodic in x, y per rank and in z over the
    ring of ranks; a single rank is its own neighbour) with the ghost exchange overlapped with the interior planes
    (paper_2210_17509_b200/halo.py) and, for comparison, exchanged first."""
    from paper_2210_17509_b200 import halo
    prim0, met, K = dev
    g = prob.nghost
    res = {}
    for overlap in (True, False):
        prim = prim0.clone()
        grx.fill_ghosts(prim, g, "periodic", 7, stream=stream)
        cons = grx.prim2con(prim, met, g, prob.gamma)
        ex = halo.ZSlabExchange(prim, g)
        work = (torch.empty_like(cons), torch.empty_like(cons))
        dt = 0.2 * min(prob.dx)
        halo.step_rk2_zslabs(ex, cons, prim, met, K, prob.dx, g, recon, prob.gamma, dt, 1, work, overlap=overlap, stream=stream)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record(stream)
        halo.step_rk2_zslabs(ex, cons, prim, met, K, prob.dx, g, recon, prob.gamma, dt, nsteps, work, overlap=overlap,
                             stream=stream)
        e1.record(stream)
        torch.cuda.synchronize()
        t = max_over_ranks(e0.elapsed_time(e1) * 1e-3, world, "cuda")
        res["overlapped" if overlap else "exchange_first"] = {"zone_cycles_per_s": prob.cells * world * nsteps / t,
                                                              "ms_per_step": 1e3 * t / nsteps}
        res["finite"] = bool(torch.isfinite(cons[prob.interior]).all().item())
        res["bytes_per_exchange_per_rank"] = ex.bytes_per_exchange
        del ex, work, cons, prim
    res["ranks"] = world
    res["scheme"] = (f"z-slab ring of {world} rank(s), one {prob.name} block each, SSP-RK2, {recon}+HLLE, periodic; "
                     "2 exchanges of 2 x 3 ghost planes x 8 fields per step")
    return res


def time_vertex(grx, torch, prob, dev, recon, stream, steps=5):
    """NEXT-3: grx_valencia_rhs_vertex (metric / K_ij at the cell vertices; here: the block's cell-centred fields sampled
    onto the (N+1)^3 vertex grid by edge replication -- the timing does not depend on the values) and grx_tmunu_vertices."""
    prim, met, K = dev

    def to_vertices(a):
        v = torch.empty((a.shape[0], a.shape[1]) + tuple(s + 1 for s in a.shape[2:]), dtype=a.dtype, device=a.device)
        v[:, :, :-1, :-1, :-1] = a
        v[:, :, -1, :-1, :-1] = a[:, :, -1]
        v[:, :, :, -1, :-1] = v[:, :, :, -2, :-1]
        v[:, :, :, :, -1] = v[:, :, :, :, -2]
        return v

    met_v, K_v = to_vertices(met), to_vertices(K)
    out = torch.empty_like(prim)
    T = torch.empty((prim.shape[0], 10) + tuple(met_v.shape[2:]), dtype=torch.float64, device="cuda")
    res = {}
    for name, call in (("rhs_vertex", lambda: grx.valencia_rhs_vertex(prim, met_v, K_v, prob.dx, prob.nghost, recon, prob.gamma,
                                                                      out=out, stream=stream)),
                       ("tmunu_vertices", lambda: grx.tmunu_vertices(prim, met_v, prob.nghost, prob.gamma, out=T, stream=stream))):
        for _ in range(2):
            call()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        stream.synchronize()
        e0.record(stream)
        for _ in range(steps):
            call()
        e1.record(stream)
        stream.synchronize()
        t = e0.elapsed_time(e1) * 1e-3 / steps
        res[name] = {"ms_per_call": 1e3 * t, "cell_updates_per_s": prob.cells / t}
    fl = algorithmic_flops_per_cell(prob.n, recon) * prob.cells / (res["rhs_vertex"]["ms_per_call"] * 1e-3) / 1e12
    res["rhs_vertex"]["frac_of_cell_centred_count"] = fl / FP64_PEAK_NOMINAL_TFLOPS
    # T^{mu nu}: 8 prims read (cached 64-point stencils), 10 metric fields read, 10 components written per vertex
    res["tmunu_vertices"]["hbm_frac"] = 28 * 8 * prob.cells / (res["tmunu_vertices"]["ms_per_call"] * 1e-3) / 1e9 / \
        measured_peaks()[0].get("hbm_gbs", 6650.0)
    res["scheme"] = f"metric and K_ij at the cell vertices (R31), T^mu nu from 4th-order interpolated primitives (R32); {prob.name}"
    return res


class Probe:
    """libgrx_probe.so (csrc/probe/grx_probe.h): the FP64 micro-benchmarks.  Bench-side code, not the product library."""

    def __init__(self):
        import ctypes as C
        from paper_2210_17509_b200 import build
        self.C = C
        self.lib = C.CDLL(build.build_probe())
        self.lib.grx_probe_dfma_peak.argtypes = [C.c_int, C.c_void_p, C.POINTER(C.c_double), C.c_void_p]
        self.lib.grx_probe_fp64_issue.argtypes = [C.c_int, C.c_int, C.c_void_p, C.POINTER(C.c_double), C.c_void_p]

    def _call(self, fn, *args, sink, stream):
        n = self.C.c_double(0.0)
        rc = fn(*args, self.C.c_void_p(sink.data_ptr()), self.C.byref(n), self.C.c_void_p(stream.cuda_stream))
        if rc != 0:
            raise RuntimeError(f"libgrx_probe: CUDA error {rc}")
        return n.value

    def dfma_peak(self, iters, sink, stream):
        return self._call(self.lib.grx_probe_dfma_peak, iters, sink=sink, stream=stream)

    def fp64_issue(self, mode, iters, sink, stream):
        return self._call(self.lib.grx_probe_fp64_issue, mode, iters, sink=sink, stream=stream)


def measure_dfma_peak(probe, torch, stream):
    sink = torch.zeros(1, dtype=torch.float64, device="cuda")
    probe.dfma_peak(2000, sink, stream)
    best = 0.0
    for _ in range(5):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        flops = probe.dfma_peak(20000, sink, stream)
        e1.record(stream)
        stream.synchronize()
        best = max(best, flops / (e0.elapsed_time(e1) * 1e-3))
    return best / 1e12


ISSUE_PROBE_MODES = ("dfma_fixed_operands", "dfma_three_registers", "dmul", "dmul+imad", "dmul+sts64", "dmul+shfl",
                     "dfma_three_registers_mixed_parity", "dfma_accumulate_in_place", "dfma_operand_shared_by_two",
                     "dfma_two_registers+constant")


def measure_issue_probe(probe, torch, stream, sm_mhz):
    """FP64 lanes per clock per SM (64 = nominal) of the issue probe's patterns (csrc/probe/grx_probe.h): what an FP64
    instruction costs with three register operands (in several placements), and next to integer, store and shuffle
    instructions."""
    sink = torch.zeros(1, dtype=torch.float64, device="cuda")
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    hz = (sm_mhz or 1965.0) * 1e6
    res = {}
    for mode, name in enumerate(ISSUE_PROBE_MODES):
        probe.fp64_issue(mode, 500, sink, stream)
        best = 0.0
        for _ in range(3):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            n = probe.fp64_issue(mode, 4000, sink, stream)
            e1.record(stream)
            stream.synchronize()
            best = max(best, n / (e0.elapsed_time(e1) * 1e-3))
        res[name] = round(best / hz / sms, 2)
    return res


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2210_17509_b200 import build, grx

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the CUDA path has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        build.build()
        build.build_probe()
    if world > 1:
        dist.barrier()
    grx.lib()
    grx.set_variant(args.variant)
    stream = torch.cuda.current_stream()

    prob = load_workload(args.workload, rank)
    recon = args.recon
    host = [torch.from_numpy(np.ascontiguousarray(a)) for a in (prob.prim, prob.metric, prob.K)]
    dev = tuple(t.cuda() for t in host)
    if rank != 0:
        # only rank 0 runs the oracle: the other ranks keep one (pinned) host copy of their inputs, not two
        host = [t.pin_memory() for t in host]
        prob.prim = prob.metric = prob.K = None
    cells = prob.cells
    g = prob.nghost

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    # ---- device-resident timing (the headline `value`), clocks sampled during it
    time_rhs(grx, torch, prob, dev, recon, 0, max(args.warmup, 3), stream)
    barrier()
    with ClockSampler(local) as cs:
        per_call = []
        t_dev, out = time_rhs(grx, torch, prob, dev, recon, args.steps, 0, stream, per_call)
        barrier()
    clocks = cs.summary()
    if clocks["samples"] < 5:
        # timed region too short for NVML's sampling period: sample the same kernel over >= 0.5 s (untimed)
        n_extra = int(max(10, 0.6 / max(t_dev / args.steps, 1e-6)))
        with ClockSampler(local) as cs2:
            time_rhs(grx, torch, prob, dev, recon, n_extra, 0, stream)
        c2 = cs2.summary()
        c2["note"] = "sampled over an untimed repeat of the timed kernel (timed region shorter than the NVML period)"
        clocks = c2
    t_max = max_over_ranks(t_dev, world, "cuda")
    value = whole_job_rate(cells, world, args.steps, t_max)

    # ---- end to end through grx_valencia_rhs_host: pinned host buffers, H2D + kernel + D2H per step
    e2e_steps = max(1, min(args.steps, 5))
    hp, hm, hk = (t if t.is_pinned() else t.pin_memory() for t in host)
    ho = torch.empty_like(hp).pin_memory()
    ws = torch.empty(grx.host_workspace_bytes(hp.shape, g) // 8, dtype=torch.float64, device="cuda")
    grx.valencia_rhs_host(hp, hm, hk, prob.dx, g, recon, prob.gamma, ho, ws, stream=stream)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(e2e_steps):
        grx.valencia_rhs_host(hp, hm, hk, prob.dx, g, recon, prob.gamma, ho, ws, stream=stream)
    e1.record(stream)
    stream.synchronize()
    e2e_value = whole_job_rate(cells, world, e2e_steps, max_over_ranks(e0.elapsed_time(e1) * 1e-3, world, "cuda"))
    e2e_ok = bool(np.array_equal(ho.numpy()[prob.interior], out.cpu().numpy()[prob.interior]))
    h2d = int(sum(t.numel() for t in (hp, hm, hk)) * 8)
    d2h = int(ho.numel() * 8)
    del ws, hp, hm, hk, ho

    # ---- NEXT-4: z-slab ring with the ghost exchange overlapped (every rank takes part; with more than one rank only on
    # request, as the point-to-point path has been exercised on CPU ranks only)
    halo_res = None
    if (world == 1 and not args.no_sweep and prob.nbox == 1) or args.halo:
        halo_res = time_halo_overlap(grx, torch, prob, dev, recon, stream, world)

    if rank != 0:
        if world > 1:
            dist.barrier()
            dist.destroy_process_group()
        return 0

    # ---- roofline of the (single) kernel of a step; its launch duration = step time (one launch per step)
    peaks, peak_src = measured_peaks()
    t_launch = t_dev / args.steps
    fl_cell = algorithmic_flops_per_cell(prob.n, recon)
    by_cell = algorithmic_bytes_per_cell(prob.n, g)
    ach_tflops = fl_cell * cells / t_launch / 1e12
    ach_gbs = by_cell * cells / t_launch / 1e9
    probe = Probe()
    dfma = measure_dfma_peak(probe, torch, stream)
    roofline = {
        "bound": "alu", "kernel": KERNEL_OF_VARIANT[args.variant], "achieved": ach_tflops, "peak": FP64_PEAK_NOMINAL_TFLOPS,
        "unit": "TFLOP/s", "frac": ach_tflops / FP64_PEAK_NOMINAL_TFLOPS,
        "peak_source": "nominal FP64: 148 SM x 64 lanes x 2 x 1.965 GHz (MEASURED_PEAKS.json has no FP64 entry)",
        "peak_dfma_measured": dfma, "frac_of_dfma_measured": ach_tflops / dfma if dfma > 0 else None,
        "frac_no_redundancy": (fl_cell - redundant_flops_per_cell(prob.n)) * cells / t_launch / 1e12 / FP64_PEAK_NOMINAL_TFLOPS,
        "redundant_flops_per_cell": redundant_flops_per_cell(prob.n),
        "flops_per_cell": fl_cell, "flops_source": "operations of the oracle's counting instance, pinned piece by piece "
                                                   "against hand counts (tests/test_bench_model.py)",
        "frac_survey_count": (FLOPS_SURVEY[recon] * cells / t_launch / 1e12 / FP64_PEAK_NOMINAL_TFLOPS
                              if recon in FLOPS_SURVEY else None),
        "flops_per_cell_survey": FLOPS_SURVEY.get(recon),
        "bytes_per_cell": by_cell,
        "hbm": {"achieved": ach_gbs, "peak": peaks.get("hbm_gbs"), "unit": "GB/s", "peak_source": peak_src,
                "frac": ach_gbs / peaks["hbm_gbs"] if peaks.get("hbm_gbs") else None},
        "traffic": None,
        "fp64_lanes_per_clk_per_sm": measure_issue_probe(probe, torch, stream, clocks.get("sm_mhz")),
    }
    # profiler-only numbers: reported only for the state of the kernel sources they were captured at
    sha = csrc_sha()
    cap = NCU_CAPTURE.get(f"{args.workload}/{recon}/{args.variant}")
    if cap and NCU_CAPTURE["csrc_sha"] == sha:
        roofline["traffic"] = cap["traffic"]
        roofline["ncu"] = dict(cap, source=NCU_CAPTURE["source"], csrc_sha=sha)
        if cap.get("fp64_inst_per_cell"):
            # one executed FP64 instruction = one lane-slot of the pipe whatever it does (an FMA counts 2 flops)
            roofline["frac_executed_slots"] = cap["fp64_inst_per_cell"] * cells / t_launch / (148 * 64 * 1.965e9)
    elif cap is None:
        roofline["ncu"] = {"csrc_sha": sha, "note": "no ncu capture for this workload / reconstruction / variant"}
    else:
        roofline["ncu"] = {"csrc_sha": sha, "note": "no ncu capture for this state of csrc/ (captured at %s)" % NCU_CAPTURE["csrc_sha"]}

    # ---- the oracle on the host cores, bounded sample of the same workload
    cpu_rate, cpu_t, n1, cores = time_oracle(prob, recon, budget_s=args.cpu_seconds)
    cpu_baseline = {"value": cpu_rate, "unit": UNIT, "cores": cores, "kind": "oracle",
                    "sample": f"first {n1[0]}x{n1[1]}x{n1[2]} interior cells (+3 ghosts) of the same block, "
                              f"one evaluation, {cpu_t:.1f} s"}

    sweep = None
    if not args.no_sweep and args.workload == "c5-256":
        sweep = sweep_points(grx, torch, stream, SWEEP_POINTS, 10, 3, peaks, keep=("c5-256", prob, dev))

    # ---- NEXT-1: device-resident time steps on the same block (context: the paper's setupA, l.329-341: static spacetime,
    # ideal gas, RK2, WENO5, periodic boundaries, 3 ghosts -> 0.47e8 zone-cycles/s at 240^3 on one V100)
    zone_cycles = ct = vertex = None
    if not args.no_sweep:
        zone_cycles = time_zone_cycles(grx, torch, prob, dev, recon, stream)
        ct = time_ct(grx, torch, prob, dev, recon, stream)
        ct["zone_cycles"] = time_zone_cycles(grx, torch, prob, dev, recon, stream, ct=True)
        vertex = time_vertex(grx, torch, prob, dev, recon, stream)

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": 1e3 * t_max / args.steps, **call_stats(per_call), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_of(prob, recon, world), "arm": "one grx_valencia_rhs call per step", "variant": args.variant,
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "steps": e2e_steps, "matches_device_path": e2e_ok},
        "gpu_launches": args.steps,
        "roofline": roofline,
        "cpu_baseline": cpu_baseline,
    }
    if sweep is not None:
        line["sweep"] = sweep
    if zone_cycles is not None:
        line["zone_cycles"] = zone_cycles
    if ct is not None:
        line["constrained_transport"] = ct
    if vertex is not None:
        line["vertex_centred"] = vertex
    if halo_res is not None:
        line["halo_overlap"] = halo_res
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def sweep_points(grx, torch, stream, names, steps, warmup, peaks, keep=None):
    """Times every (workload, reconstruction) point: `steps` calls after `warmup`, CUDA events on the launching
    stream.  One workload is resident at a time (inputs are generated per point to bound host memory).  `keep` is an
    already loaded (name, prob, dev) that is reused instead of being generated again."""
    pts = []
    for name in names:
        if keep is not None and keep[0] == name:
            prob, dev, own = keep[1], keep[2], False
        else:
            prob = load_workload(name, 0)
            dev = tuple(torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (prob.prim, prob.metric, prob.K))
            own = True
        for recon in prob.recons:
            calls = []
            t, _ = time_rhs(grx, torch, prob, dev, recon, steps, max(warmup, 3), stream, calls)
            tl = t / steps
            fl = algorithmic_flops_per_cell(prob.n, recon) * prob.cells / tl / 1e12
            gb = algorithmic_bytes_per_cell(prob.n, prob.nghost) * prob.cells / tl / 1e9
            pt = {"workload": prob.name, "recon": recon, "cells": prob.cells, "ms_per_call": 1e3 * tl,
                  "cell_updates_per_s": prob.cells / tl, "frac": fl / FP64_PEAK_NOMINAL_TFLOPS,
                  "hbm_frac": gb / peaks["hbm_gbs"] if peaks.get("hbm_gbs") else None}
            pt.update(call_stats(calls))
            if recon in FLOPS_SURVEY:
                pt["frac_survey_count"] = FLOPS_SURVEY[recon] * prob.cells / tl / 1e12 / FP64_PEAK_NOMINAL_TFLOPS
            if name in ORACLE_TIMED_POINTS:
                # the oracle is timed at these sizes too (bounded sample of box 0, 2 s)
                rate, secs, n1, cores = time_oracle(prob, recon, budget_s=2.0)
                pt["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
                                      "sample": f"first {n1[0]}x{n1[1]}x{n1[2]} interior cells of box 0, one evaluation, {secs:.1f} s"}
            pts.append(pt)
        if own:
            del dev, prob
            torch.cuda.empty_cache()
    return pts


def run_sweep(args):
    """Config-5 sweep + the other configs: one JSON line per point (not the driver's contract line)."""
    import torch
    from paper_2210_17509_b200 import build, grx
    build.build()
    grx.lib()
    grx.set_variant(args.variant)
    stream = torch.cuda.current_stream()
    peaks, _ = measured_peaks()
    for pt in sweep_points(grx, torch, stream, SWEEP_POINTS + ("c2", "c1"), args.steps, args.warmup, peaks):
        print(json.dumps(pt), flush=True)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c5-256")
    ap.add_argument("--recon", default="weno5", choices=["weno5", "minmod", "mc"])
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="wall-clock budget of the oracle sample")
    ap.add_argument("--variant", default="auto", choices=["auto", "tma", "ldg", "simple"],
                    help="kernel selector (auto = product path)")
    ap.add_argument("--no-sweep", action="store_true", help="leave the config sweep out of the contract line")
    ap.add_argument("--sweep", action="store_true", help="time every config instead of the contract line")
    ap.add_argument("--halo", action="store_true", help="also time the z-slab ring with overlapped ghost exchange (NEXT-4) "
                                                        "when there is more than one rank")
    args = ap.parse_args()
    if args.steps < 1:
        raise SystemExit("--steps must be >= 1")
    if args.impl == "reference":
        return run_reference(args)
    if args.sweep:
        return run_sweep(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
