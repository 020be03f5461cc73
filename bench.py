"""bench.py -- 3D-RISM iteration throughput of librism3d.so on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload C4]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P \
        bench.py --gpus N --steps K --warmup W

A "step" is ONE 3D-RISM iteration = one pass of the loop rows S1-S7 of DESIGN.md (closure, forward 3D FFT,
tail subtraction + chi mat-vec, inverse 3D FFT, residual + Gram row, MDIIS solve, MDIIS update) over the whole
grid of the workload, with a FULL MDIIS history (the warm-up runs at least M iterations so that every timed
step reads all 2M history fields).  The setup kernel (S0) and the free energy (S8) are timed separately and
are part of the end-to-end solve (`e2e`).  One JSON line on stdout (rank 0); DESIGN.md "Measurement" explains
every key.  N > 1 runs N independent replicas (one solute per GPU, no data-path collective: DESIGN.md
"Multi-GPU").

`--impl reference` times the CPU oracle (oracle/, numpy fp64, as it stands) on a bounded sample of the same
workload; it is the only other place besides `cpu_baseline` where this file executes oracle code.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "3D-RISM iterations/s"
UNIT = "iterations/s"
# fp64 flops counted per atom - grid point pair by the setup rooflines: the w pair evaluation of
# SURVEY.md section 8(d) (25 + 8 n_v: distance, 1/r, exp, then per site the screened Coulomb and 12-6 terms), the phi
# pair on its common far path (distance 8, float rsqrt seed + two Newton steps 14, one FMA 2), the gradient pair
FLOPS_W_PAIR = lambda n_v: 25 + 8 * n_v
FLOPS_PHI_PAIR = 24
FLOPS_GRAD_PAIR = lambda n_v: 30 + 12 * n_v


# ---------------------------------------------------------------------------------------------------------
# algorithmic HBM words per grid-point*site and iteration of each loop kernel
# ---------------------------------------------------------------------------------------------------------
def kernel_words(n_v: int, m_hist: int) -> dict:
    """m_hist = stored MDIIS entries during the timed steps (= M once the history is full)."""
    return {
        "closure_zfwd": m_hist + 3.0,           # read M stored Z_i (pending MDIIS update) and w; write tau and c_sr(z-transformed)
        "y_fwd": 2.0,                           # in place
        "kspace_x": 2.0 + 1.0 / n_v,            # in place + phi~ (one complex per 2 points, shared by the sites)
        "y_inv": 2.0,
        "zinv_gram_solve": m_hist + 3.0,        # read work, tau, the M-1 stored residuals; write R and Z = tau + b R
    }


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ---------------------------------------------------------------------------------------------------------
# clocks: nvidia-smi sampled DURING the timed region
# ---------------------------------------------------------------------------------------------------------
class ClockSampler:
    QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")

    def __init__(self, device_index: int):
        self.path = tempfile.mktemp(prefix="rism3d_clocks_", suffix=".csv")
        self.proc = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(device_index), f"--query-gpu={self.QUERY}", "--format=csv,noheader,nounits",
                 "-lms", "20"], stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except OSError:
            self.proc = None

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        try:
            with open(self.path) as f:
                for line in f:
                    parts = [x.strip() for x in line.split(",")]
                    if len(parts) < 7:
                        continue
                    try:
                        sm.append(float(parts[0])); smax.append(float(parts[1])); power.append(float(parts[2]))
                    except ValueError:
                        continue
                    for nm, v in zip(names, parts[3:7]):
                        if v.lower().startswith("active"):
                            reasons.add(nm)
            os.unlink(self.path)
        except OSError:
            pass
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "power_w_max": float(max(power)),
                "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------------------------------------
# distributed plumbing (replicas: a barrier and a max / sum over ranks of scalars, nothing on the data path)
# ---------------------------------------------------------------------------------------------------------
def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def dist_init(backend: str):
    import torch.distributed as dist
    rank, _, world = dist_env()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, world


def reduce_scalars(values, op: str, device):
    """max / sum over ranks of a list of floats -> list of floats (identity when world size is 1)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [float(v) for v in values]
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX if op == "max" else dist.ReduceOp.SUM)
    return [float(v) for v in t.cpu()]


def aggregate_throughput(units_local: float, ms_local: float, device):
    """Whole-job throughput of a replicated run: units of ALL ranks / the slowest rank's time.
    -> (units_total / s, max ms)"""
    (ms_max,) = reduce_scalars([ms_local], "max", device)
    (units,) = reduce_scalars([units_local], "sum", device)
    return units / (ms_max * 1e-3), ms_max


# ---------------------------------------------------------------------------------------------------------
# workload
# ---------------------------------------------------------------------------------------------------------
def workload_inputs(name: str, rank: int = 0):
    """-> (cfg, solvent, solute, (k0, dk, chi)).  Replica r of a multi-GPU run gets its own seeded solute."""
    from workloads import get_config, load_chi, make_solute, solvent_by_name
    from workloads import solutes as _sol
    cfg = get_config(name)
    sv = solvent_by_name(cfg.solvent)
    if rank == 0 or name in ("C1",):
        sol = make_solute(name)
    else:
        base_seed = {"C2": 2, "C3": 3, "C4": 4, "C5": 5}[name]
        sol = getattr(_sol, "make_" + name.lower())(seed=base_seed + 100 * rank)
    return cfg, sv, sol, load_chi(sv.name)


def workload_label(cfg, sol) -> str:
    return (f"{cfg.name}: {sol.n_atoms}-atom synthetic solute ({sol.name}), {cfg.solvent}, grid {cfg.n}^3 at "
            f"{cfg.spacing} A, {cfg.closure}{'-%d' % cfg.pse_order if cfg.closure == 'PSE' else ''}, "
            f"MDIIS {cfg.mdiis_nvec} vectors, fp64")


# ---------------------------------------------------------------------------------------------------------
# the oracle on a bounded sample (cpu_baseline leg and --impl reference)
# ---------------------------------------------------------------------------------------------------------
class OracleSample:
    """The oracle (oracle/, numpy fp64, as it stands) on the workload's box, solvent, closure and MDIIS settings:
    at the workload's own grid when n_sample == cfg.n (no scaling anywhere), else on a coarser n_sample^3 grid over the
    same box, its iterations/s scaled by the grid-point*site count.  The solute is the first `atoms` atoms: one oracle
    iteration costs the same whatever the atoms are, and its (untimed) O(N N_a) numpy setup costs seconds per atom at
    256^3."""

    def __init__(self, name: str, n_sample: int, atoms: int):
        from oracle import rism3d as o3
        cfg, sv, sol, (k0, dk, chi) = workload_inputs(name)
        self.cfg, self.sv = cfg, sv
        self.n = min(n_sample, cfg.n)
        self.spacing = cfg.spacing * cfg.n / self.n
        na = min(atoms, sol.n_atoms)
        t0 = time.perf_counter()
        self.orc = o3.Rism3dOracle(self.n, self.spacing, sv.n_v, closure=cfg.closure, pse_order=cfg.pse_order,
                                   mdiis_nvec=cfg.mdiis_nvec, mdiis_b=cfg.mdiis_b, mdiis_restart=cfg.mdiis_restart)
        self.orc.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
        t1 = time.perf_counter()
        self.orc.set_solute(sol.xyz[:na], sol.q[:na], sol.sigma[:na], sol.eps[:na], rcut=cfg.rcut)
        self.setup_s_per_atom = (time.perf_counter() - t1) / max(na, 1)
        self.init_s = t1 - t0
        self.pt_sites_sample = float(self.n ** 3 * sv.n_v)
        self.pt_sites_full = float(cfg.n ** 3 * sv.n_v)
        self.full_size = self.n == cfg.n
        grid = (f"the workload's own {cfg.n}^3 grid at {cfg.spacing:g} A" if self.full_size else
                f"a {self.n}^3 grid at {self.spacing:g} A over the same {cfg.n * cfg.spacing:g} A box "
                f"(1/{int(self.pt_sites_full / self.pt_sites_sample)} of the points; rate scaled by grid-point*site count)")
        self.label = (f"{cfg.name} settings ({sv.n_v} sites, {cfg.closure}, MDIIS {cfg.mdiis_nvec}) on {grid}, "
                      f"first {na} atoms of the solute")

    def run(self, steps: int, warmup: int):
        """-> seconds per oracle iteration on the sample"""
        self.orc.iterate(max(warmup, 0), 0.0)
        t0, c0 = time.perf_counter(), time.process_time()
        self.orc.iterate(steps, 0.0)
        wall = time.perf_counter() - t0
        self.threads_used = max(1, int(round((time.process_time() - c0) / wall)))   # CPU time / wall time
        self.history_entries = min(self.cfg.mdiis_nvec, max(warmup, 0) + steps)
        return wall / steps

    def iterations_per_s_full(self, s_per_iter_sample: float) -> float:
        return (self.pt_sites_sample / s_per_iter_sample) / self.pt_sites_full


def host_info() -> dict:
    model = ""
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    model = line.split(":", 1)[1].strip()
                    break
    except OSError:
        pass
    mem_gb = 0.0
    try:
        import psutil
        mem_gb = psutil.virtual_memory().available / 1e9
    except Exception:
        pass
    return {"cpu_model": model, "nproc": os.cpu_count(), "host_mem_available_gb": round(mem_gb, 1)}


# seconds per oracle iteration, measured once on an 8-core build box (used only to pick a sample that fits the time
# budget; the reported numbers are always timed live)
ORACLE_EST_S_PER_ITER = {256: 27.0, 128: 3.2, 64: 0.3, 32: 0.04}
ORACLE_FULL_GRID_HOST_GB = 20.0


def pick_sample_grid(cfg, n_iterations: int, budget_s: float, mem_gb: float) -> int:
    """largest grid <= the workload's whose n_iterations oracle iterations fit the budget (and the host memory)"""
    n = cfg.n
    while n > 32:
        est = ORACLE_EST_S_PER_ITER.get(n, 27.0 * (n / 256.0) ** 3) * n_iterations
        mem_ok = n < 256 or mem_gb >= ORACLE_FULL_GRID_HOST_GB * (cfg.mdiis_nvec / 10.0 if n_iterations >= cfg.mdiis_nvec else 0.6)
        if est <= budget_s and mem_ok:
            return n
        n //= 2
    return n


def run_reference(args):
    """The reference arm = the CPU oracle on the box's host cores.  A step is one oracle iteration of a bounded sample
    of the workload: the workload's own grid when W + K iterations of it fit ~15 minutes, else the largest coarser grid
    over the same box that does (rate then scaled by grid-point*site count; `cpu_baseline.sample` says which)."""
    rank, _, world = dist_env()
    if rank != 0:
        return 0
    from workloads import get_config
    cfg0 = get_config(args.workload)
    hi = host_info()
    warm = max(args.warmup, 0)
    # budget: the driver allows this arm 30 minutes; W + K = 25 oracle iterations on the full 256^3 x 4 grid take ~7-11 min
    # (17-27 s each), so the workload's own grid is used (full_size: true) and ms_per_step x steps matches the run
    n_s = pick_sample_grid(cfg0, warm + args.steps, 900.0, hi["host_mem_available_gb"])
    smp = OracleSample(args.workload, n_s, 8 if n_s >= 256 else 32)
    s_per = smp.run(args.steps, warm)
    val = smp.iterations_per_s_full(s_per)
    cfg = smp.cfg
    from workloads import make_solute
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": s_per * 1e3 * smp.pt_sites_full / smp.pt_sites_sample,
        "ms_per_step_sample": s_per * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": bench_config(cfg, make_solute(cfg.name), 1),
        "cpu_baseline": dict(value=val, unit=UNIT, cores=smp.threads_used, kind="oracle", sample=smp.label,
                             full_size=smp.full_size, timing="host perf_counter (CPU program)",
                             mdiis_history_entries=smp.history_entries, **hi),
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def bench_config(cfg, sol, world: int) -> dict:
    """the `config` object of the JSON line -- the same for both arms"""
    return {"workload": workload_label(cfg, sol), "parallelism": f"replicas x{world} (no collective on the data path)",
            "l2": "inputs larger than L2 (working set of a replica: (2M + 3) field-sets of %.2f GB)" % (cfg.n ** 3 * 4 * 8 / 1e9 if cfg.solvent != "water" else cfg.n ** 3 * 2 * 8 / 1e9),
            "mdiis_history": "full (M entries) during the timed steps", "rcut_A": cfg.rcut}


# ---------------------------------------------------------------------------------------------------------
# the CUDA path
# ---------------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device for --impl ours (there is no CPU fallback)")
    import paper_2403_01039_b200 as lib
    rank, local_rank, world = dist_env()
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist_init("nccl")
    import torch.distributed as dist

    cfg, sv, sol, (k0, dk, chi) = workload_inputs(args.workload, rank)
    M, n_v = cfg.mdiis_nvec, sv.n_v
    pt_sites = float(cfg.n ** 3 * n_v)
    solver = lib.Solver(cfg.n, cfg.spacing, n_v, closure=cfg.closure, pse_order=cfg.pse_order, mdiis_nvec=M,
                        mdiis_b=cfg.mdiis_b, mdiis_restart=cfg.mdiis_restart, temperature=cfg.temperature,
                        kappa=cfg.kappa, r_min=cfg.r_min, device=local_rank)
    solver.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
    setup_ms = solver.set_solute(sol.xyz, sol.q, sol.sigma, sol.eps, rcut=cfg.rcut)
    workspace_gb = solver.workspace.numel() / 1e9
    dfma_tflops = solver.measure_dfma_peak()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    # ---- device-resident throughput: K iterations with a full history -------------------------------------
    warm = max(args.warmup, M, 3)
    solver.iterate(warm, 0.0)
    launches0 = solver.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    # clocks are sampled (every 20 ms) from here to the end of the end-to-end solve: the timed steps alone last tens of
    # milliseconds, the per-kernel pass and the whole solve that follow keep the device under the same kernels
    sampler = ClockSampler(local_rank) if rank == 0 else None
    barrier()
    ev0.record(solver.stream)
    n_done, rms_end = solver.iterate(args.steps, 0.0)
    ev1.record(solver.stream)
    barrier()
    ms_local = ev0.elapsed_time(ev1)
    launches = solver.launch_count() - launches0
    value, ms_max = aggregate_throughput(float(args.steps), ms_local, dev)

    # ---- per-kernel CUDA-event times (second pass over the same number of steps) -----------------------------
    solver.set_profiling(True)
    solver.iterate(args.steps, 0.0)
    kern_ms, prof_n = solver.timings()
    solver.set_profiling(False)
    peak, peak_src = load_peaks()
    words = kernel_words(n_v, M)
    kernels = {}
    for name, ms in kern_ms.items():
        gb = words[name] * 8.0 * pt_sites / 1e9
        kernels[name] = {"ms": ms, "algorithmic_gb": gb, "gbs": (gb / (ms * 1e-3) if ms > 0 else 0.0),
                         "frac": (gb / (ms * 1e-3) / peak if ms > 0 else 0.0)}
    dominant = max(kernels, key=lambda k: kernels[k]["ms"])
    traffic = ncu_traffic(dominant, args.workload)
    roofline = {"bound": "hbm", "kernel": dominant, "achieved": kernels[dominant]["gbs"], "peak": peak, "unit": "GB/s",
                "frac": kernels[dominant]["frac"], "traffic": traffic,
                # NOT measured by this run: the stored figure of one committed ncu --set full capture of the same kernel
                "traffic_source": "profiles/traffic.json (static: copied from a committed ncu --set full capture, not re-measured by this run)" if traffic is not None else None,
                "peak_source": peak_src,
                "algorithmic_bytes_per_launch": kernels[dominant]["algorithmic_gb"] * 1e9,
                "iteration": {"ms_sum_of_kernels": sum(k["ms"] for k in kernels.values()),
                              "algorithmic_gb": sum(k["algorithmic_gb"] for k in kernels.values()),
                              "frac": sum(k["algorithmic_gb"] for k in kernels.values()) /
                              (sum(k["ms"] for k in kernels.values()) * 1e-3) / peak},
                "kernels": kernels}

    # ---- end to end: one whole solve from HOST inputs to HOST results through the C ABI ------------------------
    e2e = None
    clocks = None
    if not args.no_e2e:
        g_host = torch.empty((n_v, cfg.n, cfg.n, cfg.n), dtype=torch.float64, pin_memory=True)
        g_np = g_host.numpy()
        barrier()
        t0 = time.perf_counter()
        setup_ms_e2e = solver.set_solute(sol.xyz, sol.q, sol.sigma, sol.eps, rcut=cfg.rcut)    # H2D atoms + S0
        it_conv, rms_conv = solver.iterate(args.max_iter, cfg.tol)                              # S1-S7 to 1e-6
        t1 = time.perf_counter()
        mu, mu_site = solver.free_energy()                                                      # S8 + D2H scalars
        t2 = time.perf_counter()
        for s in range(n_v):
            lib.rism3d_get_field(solver.ctx, lib.FIELDS["G"], s, g_np[s].ctypes.data, False)    # D2H g
        torch.cuda.synchronize(dev)
        t3 = time.perf_counter()
        (e2e_s,) = reduce_scalars([t3 - t0], "max", dev)
        (it_total,) = reduce_scalars([float(it_conv)], "sum", dev)
        clocks = sampler.stop() if sampler else None
        sampler = None
        e2e = {"value": it_total / e2e_s, "unit": UNIT,
               "h2d_bytes_per_step": int(sol.n_atoms * 6 * 8), "d2h_bytes_per_step": int(g_np.nbytes + 8 * (n_v + 1) + 64),
               "what": "one whole solve per replica: set_solute (host atom arrays -> device, S0) + iterate to rms < tol + "
                       "free_energy + g of every site copied to pinned host memory; a 'step' of this leg is the solve",
               "seconds_to_converge": e2e_s, "iterations_to_converge": int(it_conv), "converged": bool(rms_conv < cfg.tol),
               "tol": cfg.tol, "rms": rms_conv, "setup_ms": setup_ms_e2e, "loop_s": t1 - t0 - setup_ms_e2e * 1e-3,
               "free_energy_ms": (t2 - t1) * 1e3, "phi_ms": solver.phi_ms(), "get_g_ms": (t3 - t2) * 1e3,
               "dmu_kcal_mol": mu, "g_max": float(g_np.max())}
    if sampler is not None:
        clocks = sampler.stop()

    # ---- setup (S0) and gradient against the measured fp64 FMA peak (they are bound by plain fp64 arithmetic) ---------
    setup = None
    if rank == 0:
        npts, na = float(cfg.n ** 3), float(sol.n_atoms)
        if cfg.rcut > 0:
            dv = cfg.spacing ** 3
            pairs_w = na * 4.0 / 3.0 * np.pi * cfg.rcut ** 3 / dv          # pairs inside the cutoff (spheres inside the box)
        else:
            pairs_w = npts * na
        t0 = time.perf_counter()
        solver.get_field_device("PHI", 0)                                   # forces the deferred phi kernel when it has not run
        phi_ms = solver.phi_ms()
        setup = {"bound": "alu", "peak_tflops_fp64": dfma_tflops, "peak_source": "measured (rism3d_measure_dfma_peak, independent DFMA chains)",
                 "setup_ms": setup_ms, "what": ("w from the cell list + phi~ (the loop's inputs)" if cfg.rcut > 0 else "w + phi all pairs, phi~"),
                 "w_pairs": pairs_w, "w_flops_per_pair": FLOPS_W_PAIR(n_v),
                 "w_pairs_per_s_upper": pairs_w / (setup_ms * 1e-3),
                 "w_frac_of_dfma_peak_upper": pairs_w * FLOPS_W_PAIR(n_v) / (setup_ms * 1e-3) / 1e12 / dfma_tflops if dfma_tflops else None,
                 "note": "setup_ms also holds the phi~ kernels; with a cutoff most of the w kernel's time goes into distance tests of "
                         "candidate atoms outside the cutoff, which the pair count does not include"}
        if cfg.rcut > 0 and phi_ms > 0:
            setup.update({"phi_ms": phi_ms, "phi_pairs": npts * na, "phi_flops_per_pair": FLOPS_PHI_PAIR,
                          "phi_pairs_per_s": npts * na / (phi_ms * 1e-3),
                          "phi_frac_of_dfma_peak": npts * na * FLOPS_PHI_PAIR / (phi_ms * 1e-3) / 1e12 / dfma_tflops if dfma_tflops else None})
        if not args.no_e2e:
            torch.cuda.synchronize(dev)
            t0 = time.perf_counter()
            solver.gradient()
            grad_ms = (time.perf_counter() - t0) * 1e3
            setup.update({"gradient_ms": grad_ms, "gradient_pairs": npts * na, "gradient_flops_per_pair": FLOPS_GRAD_PAIR(n_v),
                          "gradient_frac_of_dfma_peak": npts * na * FLOPS_GRAD_PAIR(n_v) / (grad_ms * 1e-3) / 1e12 / dfma_tflops if dfma_tflops else None})

    # ---- context: the hand-written 3D transform pair next to cuFFT (torch.fft, never on the product path) ------------
    fft_cmp = None
    if rank == 0 and not args.no_fft_compare:
        try:
            xr = torch.randn((n_v, cfg.n, cfg.n, cfg.n), dtype=torch.float64, device=dev)

            def timed(fn, reps=5):
                fn()
                torch.cuda.synchronize(dev)
                t = []
                for _ in range(reps):
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record(); fn(); e1.record()
                    torch.cuda.synchronize(dev)
                    t.append(e0.elapsed_time(e1))
                return float(np.median(t))

            def ours():
                solver.fft_inverse(solver.fft_forward(xr))

            def cufft():
                torch.fft.irfftn(torch.fft.rfftn(xr, dim=(1, 2, 3)), s=(cfg.n,) * 3, dim=(1, 2, 3))

            fft_cmp = {"ours_pair_ms": timed(ours), "cufft_pair_ms": timed(cufft),
                       "what": "forward + inverse real 3D transform of the n_v-site field. ours: the standalone passes behind "
                               "rism3d_debug_fft_forward/inverse on the half-integer k grid (6 kernels + 2 device copies + 2 "
                               "allocations, host-synchronous calls); cuFFT: torch.fft.rfftn + irfftn (D2Z + Z2D, integer k grid: "
                               "the half-integer shift would cost it two more element-wise passes). In the loop the transforms "
                               "are fused with the closure, the k-space arithmetic and the residual, so neither number is "
                               "a share of ms_per_step."}
            del xr
        except Exception as ex:                                   # context only: never fail the bench on it
            fft_cmp = {"error": str(ex)[:200]}

    # ---- extra (context, not the headline): the same solve with the paper's own GPU accelerator, modified Anderson ----
    anderson = None
    if not args.no_e2e and not args.no_anderson:
        solver.close()
        solver = lib.Solver(cfg.n, cfg.spacing, n_v, closure=cfg.closure, pse_order=cfg.pse_order, mdiis_b=0.6,
                            temperature=cfg.temperature, kappa=cfg.kappa, r_min=cfg.r_min, device=local_rank,
                            accelerator="ANDERSON", anderson_s=(0.2, 0.0))
        solver.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
        barrier()
        t0 = time.perf_counter()
        a_setup = solver.set_solute(sol.xyz, sol.q, sol.sigma, sol.eps, rcut=cfg.rcut)
        a_it, a_rms = solver.iterate(args.max_iter, cfg.tol)
        a_mu, _ = solver.free_energy()
        for s in range(n_v):
            lib.rism3d_get_field(solver.ctx, lib.FIELDS["G"], s, g_np[s].ctypes.data, False)
        torch.cuda.synchronize(dev)
        t1 = time.perf_counter()
        (a_s,) = reduce_scalars([t1 - t0], "max", dev)
        anderson = {"what": "modified Anderson, two histories, b = 0.6, s = (0.2, 0) (PAPER.md:264-298): 3 stored pairs "
                            "instead of 10, (2*3 + 12 + 1/n_v) words per pt*site and iteration",
                    "seconds_to_converge": a_s, "iterations_to_converge": int(a_it), "converged": bool(a_rms < cfg.tol),
                    "ms_per_iteration": (a_s - a_setup * 1e-3) / max(a_it, 1) * 1e3, "dmu_kcal_mol": a_mu}

    # ---- extra (context): the same solve with the dynamic damping b = -0.2 log10(rms) of PAPER.md:308 (opt-in: the
    # update then reads X_i and R_i, M more words per pt*site and iteration), and the iteration counts on C2 ------------
    dyn = None
    if rank == 0 and world == 1 and not args.no_e2e and not args.no_anderson:
        solver.close()
        solver = lib.Solver(cfg.n, cfg.spacing, n_v, closure=cfg.closure, pse_order=cfg.pse_order, mdiis_nvec=M,
                            mdiis_b=cfg.mdiis_b, mdiis_restart=cfg.mdiis_restart, temperature=cfg.temperature,
                            kappa=cfg.kappa, r_min=cfg.r_min, device=local_rank, mdiis_dynamic_b=(0.1, 1.0))
        solver.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        d_setup = solver.set_solute(sol.xyz, sol.q, sol.sigma, sol.eps, rcut=cfg.rcut)
        d_it, d_rms = solver.iterate(args.max_iter, cfg.tol)
        d_mu, _ = solver.free_energy()
        for s_ in range(n_v):
            lib.rism3d_get_field(solver.ctx, lib.FIELDS["G"], s_, g_np[s_].ctypes.data, False)
        torch.cuda.synchronize(dev)
        d_s = time.perf_counter() - t0
        dyn = {"what": "MDIIS with b = clamp(-0.2 log10(rms), 0.1, 1) (PAPER.md:308, DESIGN.md Q18): (3M + 12 + 1/n_v) words per "
                       "pt*site and iteration instead of (2M + 12 + 1/n_v)",
               "seconds_to_converge": d_s, "iterations_to_converge": int(d_it), "converged": bool(d_rms < cfg.tol),
               "ms_per_iteration": (d_s - d_setup * 1e-3) / max(d_it, 1) * 1e3, "dmu_kcal_mol": d_mu,
               "static_b_iterations": e2e["iterations_to_converge"] if e2e else None}
        c2 = {}
        cfg2, sv2, sol2, (k02, dk2, chi2) = workload_inputs("C2")
        for label, dynb in (("static", None), ("dynamic", (0.1, 1.0))):
            s2 = lib.Solver(cfg2.n, cfg2.spacing, sv2.n_v, closure=cfg2.closure, mdiis_nvec=cfg2.mdiis_nvec, mdiis_b=cfg2.mdiis_b,
                            mdiis_restart=cfg2.mdiis_restart, device=local_rank, mdiis_dynamic_b=dynb)
            s2.set_solvent_chi(sv2.q, sv2.sigma, sv2.eps, sv2.rho, k02, dk2, chi2)
            s2.set_solute(sol2.xyz, sol2.q, sol2.sigma, sol2.eps, rcut=cfg2.rcut)
            c2[label] = int(s2.iterate(3000, cfg2.tol)[0])
            s2.close()
        dyn["C2_iterations_to_converge"] = c2

    # ---- the other large configs, briefly (device-resident iterations only): C3 and the memory-ceiling C5 --------------
    others = None
    if rank == 0 and world == 1 and not args.no_others and args.workload == "C4":
        solver.close()
        others = {}
        for name in ("C1", "C2", "C3", "C5"):
            try:
                others[name] = quick_workload(lib, name, local_rank, peak, max_iter=args.max_iter)
            except Exception as ex:                               # e.g. not enough device memory for C5
                others[name] = {"error": str(ex)[:200]}
        torch.cuda.empty_cache()
        slab = {}
        for n_ranks in (2, 8):
            try:
                slab[f"x{n_ranks}"] = slab_lockstep(lib, args.workload, local_rank, n_ranks)
            except Exception as ex:
                slab[f"x{n_ranks}"] = {"error": str(ex)[:200]}
            torch.cuda.empty_cache()
        others["slab_decomposition"] = slab
        try:
            others["rism1d"] = rism1d_block(lib, cfg.solvent, local_rank)
        except Exception as ex:
            others["rism1d"] = {"error": str(ex)[:200]}

    # ---- the oracle on the host cores (rank 0, single-GPU runs only) --------------------------------------------
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        hi = host_info()
        n_s = pick_sample_grid(cfg, 1 + args.cpu_steps, 120.0, hi["host_mem_available_gb"])
        smp = OracleSample(args.workload, n_s, 8 if n_s >= 256 else 32)
        s_per = smp.run(args.cpu_steps, 1)
        cpu = dict(value=smp.iterations_per_s_full(s_per), unit=UNIT, cores=smp.threads_used, kind="oracle",
                   sample=smp.label + f"; {args.cpu_steps} timed iterations after 1 warm-up (the MDIIS history holds "
                                      f"{smp.history_entries} of {M} entries: the oracle's accelerator cost is still growing)",
                   full_size=smp.full_size, s_per_iteration_sample=s_per, setup_s_per_atom=smp.setup_s_per_atom, **hi)

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "history_fill_iterations": warm - args.warmup,   # untimed iterations beyond --warmup that fill the MDIIS history (M entries)
            "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": bench_config(cfg, sol, world), "workspace_gb": workspace_gb,
            "pt_site_updates_per_s": value * pt_sites, "setup_ms": setup_ms, "rms_after_timed_steps": rms_end,
            "roofline": roofline, "setup": setup, "other_workloads": others, "cpu_baseline": cpu, "e2e": e2e, "e2e_modified_anderson": anderson, "e2e_dynamic_damping": dyn, "fft_compare": fft_cmp, "gpu_launches": int(launches), "clocks": clocks,
        }
        print(json.dumps(line), flush=True)
    solver.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


NVLINK_GBS_PER_DIRECTION = 900.0      # NVLink 5 per GPU and direction (nominal; no second GPU here to measure it)


def slab_lockstep(lib, name: str, device: int, n_ranks: int, steps: int = 10) -> dict:
    """The slab decomposition (include/rism3d.h "Slab decomposition") measured on ONE GPU: the n_ranks contexts of one
    solve live in this process, peer tables point at each other's arrays, and the phases run rank after rank on one
    stream.  What this times is every rank's own kernel work (CUDA events per rank and phase); what it cannot time is
    the NVLink traffic (here the 'remote' rows land in the same HBM) and the overlap between ranks."""
    import torch
    cfg, sv, sol, (k0, dk, chi) = workload_inputs(name)
    M, n_v = cfg.mdiis_nvec, sv.n_v
    stream = torch.cuda.Stream(torch.device("cuda", device))
    ranks = [lib.SlabSolver(cfg.n, cfg.spacing, n_v, n_ranks, r, closure=cfg.closure, pse_order=cfg.pse_order, mdiis_nvec=M,
                            mdiis_b=cfg.mdiis_b, mdiis_restart=cfg.mdiis_restart, temperature=cfg.temperature,
                            kappa=cfg.kappa, r_min=cfg.r_min, device=device, stream=stream) for r in range(n_ranks)]
    try:
        setup_ms = []
        for r in ranks:
            r.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
            setup_ms.append(r.set_solute(sol.xyz, sol.q, sol.sigma, sol.eps, rcut=cfg.rcut))
        loc = [r.local for r in ranks]
        for r in ranks:
            r.connect_peers([l["K"] for l in loc], [l["gram"] for l in loc], [l["flags"] for l in loc])
        lib.iterate_in_lockstep(ranks, max(M, 3), 0.0)                   # fill the history
        ms = np.zeros((n_ranks, 4))
        for r in ranks:
            r.begin(0.0)
        with torch.cuda.stream(stream):
            for _ in range(steps):
                for ph in range(4):
                    for k, r in enumerate(ranks):
                        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                        e0.record(stream)
                        r.phase(ph)
                        e1.record(stream)
                        e1.synchronize()
                        ms[k, ph] += e0.elapsed_time(e1)
        for r in ranks:
            r.end()
        ms /= steps
        per_rank = ms.sum(axis=1)
        block = loc[0]["block_bytes"]
        out_bytes = (n_ranks - 1) * block                                # leaves a rank per transposition
        nvlink_ms = 2.0 * out_bytes / (NVLINK_GBS_PER_DIRECTION * 1e9) * 1e3
        return {"workload": workload_label(cfg, sol), "n_ranks": n_ranks,
                "how": "all ranks in one process on one GPU, peer tables, phases in lockstep (sequential)",
                "phase_ms_slowest_rank": {"closure_zfwd+y_fwd": float(ms[:, 0].max()), "kspace_x": float(ms[:, 1].max()),
                                          "y_inv+zinv_gram": float(ms[:, 2].max()), "gram_solve": float(ms[:, 3].max())},
                "ms_per_iteration_slowest_rank": float(per_rank.max()), "ms_per_iteration_all_ranks": float(per_rank.sum()),
                "setup_ms_slowest_rank": float(max(setup_ms)),
                "bytes_leaving_a_rank_per_iteration": int(2 * out_bytes),
                "nvlink_ms_per_iteration_at_nominal_900_GBs": nvlink_ms,
                "note": "per-rank kernel time only: on n_ranks GPUs the ranks run side by side and the rows cross NVLink "
                        "inside the y passes' stores / loads; neither is measurable on one GPU"}
    finally:
        for r in ranks:
            r.close()


def rism1d_block(lib, solvent_name: str, device: int) -> dict:
    """The GPU 1D solvent solve (include/rism1d.h) that makes the chi table of the workload's solvent: the production
    settings of oracle/make_chi_tables.py (16 384 radial points at 0.025 A, seven-step charge ramp, MDIIS 10, b = 0.3,
    tol 1e-10), wall time with the host in the loop, and how far the result is from the stored table."""
    import torch
    from workloads import load_chi, solvent_by_name
    sv = solvent_by_name(solvent_name)
    ramp = (0.0, 0.25, 0.5, 0.75, 0.85, 0.95, 1.0)
    one = lib.Solver1d(sv.n_s, n_points=16384, dr=0.025, mdiis_nvec=10, mdiis_b=0.3, mdiis_restart=0.0, device=device)
    try:
        one.set_solvent(sv.q[sv.site_type], sv.sigma[sv.site_type], sv.eps[sv.site_type], sv.species_rho[sv.site_species],
                        sv.site_species, sv.bond)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        iters, rms = 0, 0.0
        for lam in ramp:
            n, rms = one.solve(lam, 3000, 1e-10)
            iters += n
        chi = one.chi_types(sv.site_type)
        chi_t, pressure, _ = one.thermo()
        secs = time.perf_counter() - t0
        k0, dk, table = load_chi(sv.name)
        return {"solvent": sv.name, "full_sites": int(sv.n_s), "radial_points": 16384, "charge_ramp": list(ramp),
                "iterations": int(iters), "seconds": secs, "ms_per_iteration": secs / max(iters, 1) * 1e3,
                "kernel_launches": int(one.launch_count()), "rms_last": rms, "chi_T_A3_mol_per_kcal": chi_t,
                "pressure_kcal_per_mol_A3": pressure,
                "max_rel_diff_to_stored_oracle_table": float(np.max(np.abs(chi[:table.shape[0]] - table)) / np.max(np.abs(table)))}
    finally:
        one.close()


def run_slab(args):
    """--decompose slab: ONE solve shared by all ranks (strong scaling), one process per GPU, SlabSolver.iterate with
    the process group's all-to-all between the phases.  Prints the contract line with "scaling": "strong"."""
    import torch
    import paper_2403_01039_b200 as lib
    rank, local_rank, world = dist_env()
    if world < 2:
        raise RuntimeError("--decompose slab needs at least 2 ranks (torchrun --nproc-per-node N)")
    local_rank = local_rank % torch.cuda.device_count()                   # (--backend gloo: ranks may share a GPU)
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist_init(args.backend)
    import torch.distributed as dist
    if args.backend != "nccl":
        dev = None                                                        # scalars of the timing reductions stay on the host
    cfg, sv, sol, (k0, dk, chi) = workload_inputs(args.workload, 0)      # every rank the same solute
    M, n_v = cfg.mdiis_nvec, sv.n_v
    s = lib.SlabSolver(cfg.n, cfg.spacing, n_v, world, rank, closure=cfg.closure, pse_order=cfg.pse_order, mdiis_nvec=M,
                       mdiis_b=cfg.mdiis_b, mdiis_restart=cfg.mdiis_restart, temperature=cfg.temperature, kappa=cfg.kappa,
                       r_min=cfg.r_min, device=local_rank, exportable=args.peer)
    if args.peer:
        # every rank maps the others' workspaces (CUDA IPC): the y passes store to / load from the other GPUs directly and
        # rism3d_iterate runs whole iterations with in-stream barriers.  One GPU per rank only: the barrier kernels of
        # the ranks wait for one another.
        if torch.cuda.device_count() < world:
            raise RuntimeError("--peer needs one GPU per rank")
        s.connect_peers_ipc()
    s.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
    setup_ms = s.set_solute(sol.xyz, sol.q, sol.sigma, sol.eps, rcut=cfg.rcut)
    warm = max(args.warmup, M, 3)
    s.iterate(warm, 0.0)
    launches0 = s.launch_count()
    sampler = ClockSampler(local_rank) if rank == 0 else None
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    dist.barrier(); torch.cuda.synchronize()
    ev0.record(s.stream)
    s.iterate(args.steps, 0.0)
    ev1.record(s.stream)
    dist.barrier(); torch.cuda.synchronize()
    (ms_max,) = reduce_scalars([ev0.elapsed_time(ev1)], "max", dev)
    launches = s.launch_count() - launches0
    # end to end: host atoms -> converged solve -> host g slabs
    g_host = torch.empty((n_v,) + s.shape, dtype=torch.float64, pin_memory=True)
    g_np = g_host.numpy()
    dist.barrier(); torch.cuda.synchronize()
    t0 = time.perf_counter()
    s.set_solute(sol.xyz, sol.q, sol.sigma, sol.eps, rcut=cfg.rcut)
    it_conv, rms_conv = s.iterate(args.max_iter, cfg.tol)
    mu, _ = s.free_energy()
    for g in range(n_v):
        lib.rism3d_get_field(s.ctx, lib.FIELDS["G"], g, g_np[g].ctypes.data, False)
    torch.cuda.synchronize()
    (e2e_s,) = reduce_scalars([time.perf_counter() - t0], "max", dev)
    clocks = sampler.stop() if sampler else None
    if rank == 0:
        cfgd = bench_config(cfg, sol, world)
        cfgd["parallelism"] = (f"slab x{world}: one solve, x planes in r space, y rows in k space, two all-to-all transposes "
                               f"per iteration ({'peer stores over NVLink' if args.peer else args.backend})")
        print(json.dumps({
            "metric": METRIC, "value": args.steps / (ms_max * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "history_fill_iterations": warm - args.warmup,
            "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "strong",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": cfgd, "setup_ms": setup_ms,
            "e2e": {"value": it_conv / e2e_s, "unit": UNIT, "h2d_bytes_per_step": int(sol.n_atoms * 6 * 8),
                    "d2h_bytes_per_step": int(g_np.nbytes + 64), "seconds_to_converge": e2e_s,
                    "iterations_to_converge": int(it_conv), "converged": bool(rms_conv < cfg.tol), "dmu_kcal_mol": mu},
            "gpu_launches": int(launches), "clocks": clocks}), flush=True)
    s.close()
    dist.destroy_process_group()
    return 0


def whole_solve(s, cfg, sol, n_v: int, max_iter: int) -> dict:
    """One whole solve of a config through the public calls, host clock around it: set_solute (host atoms in), iterate to
    rms < cfg.tol, free_energy (s-to-converge, iterations, pt-site updates/s for every config;
    the paper's own yardstick is iterations to 1e-6).  g stays on the device here (the C4 e2e leg of the
    main line is the one that also copies it out)."""
    import torch
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    setup_ms = s.set_solute(sol.xyz, sol.q, sol.sigma, sol.eps, rcut=cfg.rcut)
    t1 = time.perf_counter()
    try:
        it, rms = s.iterate(max_iter, cfg.tol)
        diverged = False
    except Exception as ex:                                        # RISM3D_ERR_DIVERGED
        it, rms, diverged = len(s.rms_history()), float("nan"), str(ex)[:120]
    torch.cuda.synchronize()
    t2 = time.perf_counter()
    mu = s.free_energy()[0] if not diverged else float("nan")
    torch.cuda.synchronize()
    t3 = time.perf_counter()
    loop_s = t2 - t1
    return {"seconds_to_converge": t3 - t0, "iterations_to_converge": int(it), "converged": bool(rms < cfg.tol),
            "tol": cfg.tol, "rms": rms, "mdiis_b": s.params.mdiis_b, "setup_ms": setup_ms, "loop_s": loop_s,
            "pt_site_updates_per_s": (float(cfg.n) ** 3 * n_v * it / loop_s if loop_s > 0 else 0.0),
            "ms_per_iteration_in_solve": (loop_s * 1e3 / it if it else None),
            "dmu_kcal_mol": mu, **({"diverged": diverged} if diverged else {})}


def quick_workload(lib, name: str, device: int, peak: float, steps: int = 10, max_iter: int = 1500) -> dict:
    """ms per iteration and per-kernel roofline fractions of another config (full MDIIS history, device resident), then a
    whole solve to the config's tolerance (whole_solve)"""
    import torch
    cfg, sv, sol, (k0, dk, chi) = workload_inputs(name)
    M, n_v = cfg.mdiis_nvec, sv.n_v
    pt_sites = float(cfg.n ** 3 * n_v)
    s = lib.Solver(cfg.n, cfg.spacing, n_v, closure=cfg.closure, pse_order=cfg.pse_order, mdiis_nvec=M, mdiis_b=cfg.mdiis_b,
                   mdiis_restart=cfg.mdiis_restart, temperature=cfg.temperature, kappa=cfg.kappa, r_min=cfg.r_min, device=device)
    try:
        s.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
        setup_ms = s.set_solute(sol.xyz, sol.q, sol.sigma, sol.eps, rcut=cfg.rcut)
        s.iterate(max(M, 3), 0.0)
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record(s.stream)
        s.iterate(steps, 0.0)
        ev1.record(s.stream)
        torch.cuda.synchronize()
        ms = ev0.elapsed_time(ev1) / steps
        s.set_profiling(True)
        s.iterate(steps, 0.0)
        kern_ms, _ = s.timings()
        s.set_profiling(False)
        words = kernel_words(n_v, M)
        out = {"workload": workload_label(cfg, sol), "ms_per_iteration": ms, "setup_ms": setup_ms,
               "workspace_gb": s.workspace.numel() / 1e9,
               "iteration_frac_of_hbm_peak": sum(words.values()) * 8.0 * pt_sites / 1e9 / (ms * 1e-3) / peak,
               "kernels": {k: {"ms": v, "frac": (words[k] * 8.0 * pt_sites / 1e9 / (v * 1e-3) / peak if v > 0 else 0.0)}
                           for k, v in kern_ms.items()}}
        if cfg.n <= 128:
            out["note"] = "field-set of 67 MB: largely L2 resident, the HBM roofline does not bind"
        out["solve"] = whole_solve(s, cfg, sol, n_v, max_iter)
        # a config that does not reach the tolerance with the default damping is re-run with
        # a smaller b, and the b that worked is recorded
        for b_try in (0.3, 0.15):
            if out["solve"]["converged"]:
                break
            s.close()
            s = lib.Solver(cfg.n, cfg.spacing, n_v, closure=cfg.closure, pse_order=cfg.pse_order, mdiis_nvec=M, mdiis_b=b_try,
                           mdiis_restart=cfg.mdiis_restart, temperature=cfg.temperature, kappa=cfg.kappa, r_min=cfg.r_min,
                           device=device)
            s.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
            first = out["solve"]
            out["solve"] = whole_solve(s, cfg, sol, n_v, max_iter)
            out["solve"]["earlier_attempts"] = first.get("earlier_attempts", []) + [
                {k: first[k] for k in ("mdiis_b", "iterations_to_converge", "rms", "converged")}]
        return out
    finally:
        s.close()
        del s


def ncu_traffic(kernel: str, workload: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel`, from the committed ncu --set full summary
    (profiles/traffic.json, written by hand from the capture named there); None when no capture covers it."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    if not os.path.exists(p):
        return None
    with open(p) as f:
        t = json.load(f)
    return t.get(workload, {}).get(kernel)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C4", choices=["C1", "C2", "C3", "C4", "C5"])
    ap.add_argument("--max-iter", type=int, default=1500, help="iteration cap of the end-to-end solve")
    ap.add_argument("--cpu-steps", type=int, default=3, help="timed oracle iterations of the cpu_baseline leg")
    ap.add_argument("--no-others", action="store_true", help="skip the C1 / C2 / C3 / C5 runs of other_workloads")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-anderson", action="store_true", help="skip the extra modified-Anderson solve")
    ap.add_argument("--no-fft-compare", action="store_true", help="skip the cuFFT comparison")
    ap.add_argument("--backend", default="nccl", choices=["nccl", "gloo"],
                    help="process group of --decompose slab (gloo: the blocks travel through host memory; lets several "
                         "ranks share one GPU, for testing)")
    ap.add_argument("--peer", action="store_true",
                    help="--decompose slab in peer mode: CUDA IPC mappings, transposes inside the y passes' stores and loads")
    ap.add_argument("--decompose", default="replicas", choices=["replicas", "slab"],
                    help="N > 1: N independent solves (default, weak scaling) or ONE solve in x / y slabs (strong scaling)")
    args = ap.parse_args()
    if args.steps < 1:
        ap.error("--steps must be >= 1")
    if args.impl == "reference":
        return run_reference(args)
    return run_slab(args) if args.decompose == "slab" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
