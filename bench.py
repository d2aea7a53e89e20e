"""Benchmark of the lattice Boltzmann hot path (BASELINE.json metric: MLUPS and achieved HBM GB/s as a
fraction of the B200 peak, per lattice/model, one GPU).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg4] [--precision 64|32]
                    [--impl ours|reference] [--no-extras]

A "step" is ONE time step of the whole hot path (moments, psi, Shan-Chen force, velocity, BGK + Guo
collision, scalar lattice, in-place streaming, boundaries: DESIGN.md rows a1-a8) over the whole grid.
The headline workload is BASELINE.json configs[3]: D3Q19 BGK + Guo force, 256^3, halfway bounce-back
walls in z, fp64 ("throughput timed over 1000 steps"); the other configs are reported in "per_model"
with the same kernels and timing method.  Inputs are seeded and synthetic (workloads.py), resident in
HBM before the timed region; the population array (2.55 GB) is far larger than the 126 MB L2, so no
explicit L2 flush is needed between steps (config.l2 says so).

Prints ONE JSON line (rank 0).  Multi-GPU: the path does not shard (north_star: one GPU, one domain),
so --gpus N runs N independent replicas ("replicas only", weak scaling, no data-path collective).

--impl reference times the CPU oracle (oracle/, test infrastructure) on a bounded sample of the same
workload on the host cores; it is the only other place this file executes oracle/.
"""
import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads  # noqa: E402

HBM_NOMINAL_GBS = 8000.0      # north_star: "the B200's ~8 TB/s"
HBM_FALLBACK_GBS = 6650.0     # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent


def measured_peak():
    """(GB/s, 'measured'|'fallback')"""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured"
    except Exception:
        return HBM_FALLBACK_GBS, "fallback"


def ncu_traffic(workload, kernel):
    """(bytes, provenance) of dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the
    newest `ncu --set full` capture listed in profiles/r*_traffic.csv -- a number copied from a capture, NOT measured in
    this run -- or (None, why).  A row counts only if it names this workload AND the kernel that ran now."""
    import csv
    import glob
    best = None
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", "r*_traffic.csv"))):
        try:
            with open(path) as fh:
                for row in csv.DictReader(fh):
                    if row["workload"] == workload and row["kernel"] == kernel:
                        best = (float(row["traffic_bytes_per_launch"]),
                                "%s: %s (%s)" % (os.path.basename(path), row["source"], row.get("commit", "commit n/a")))
        except Exception:
            pass
    return best if best is not None else (None, "no ncu capture of %s for this workload under profiles/" % kernel)


def shape_of(cfg):
    S = 2 if cfg["model"] in ("SC2", "SC2_ADE") else 1
    Q = 19 if cfg["lattice"] == "D3Q19" else 9
    Qs = (7 if cfg["lattice"] == "D3Q19" else 5) if cfg["model"] == "SC2_ADE" else (Q if cfg["model"] == "BGK_T" else 0)
    B = 8 if cfg["params"]["precision"] == 64 else 4
    N = cfg["grid"][0] * cfg["grid"][1] * cfg["grid"][2]
    sc = cfg["model"] != "BGK"
    return dict(S=S, Q=Q, Qs=Qs, B=B, N=N, sc=sc)


def algorithmic_bytes(cfg):
    """Algorithmic bytes per lattice update:
    step kernel: every population read once and written once (+ one compulsory psi read per component);
    psi pass: psi written once per component (its re-read of the flow populations is NOT algorithmic:
    it is this design's overhead and shows up as a lower fraction)."""
    s = shape_of(cfg)
    step = (2 * (s["S"] * s["Q"] + s["Qs"]) + (s["S"] if s["sc"] else 0)) * s["B"]
    psi = (s["S"] if s["sc"] else 0) * s["B"]
    return step, psi


def max_over_ranks(ms, dist=None, device="cpu"):
    """max over ranks of a per-rank elapsed time (the contract's multi-GPU timing rule)"""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(ms)
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_mlups(world, cells_per_replica, steps, ms):
    """whole-job MLUPS of `world` independent replicas that all finished within `ms` (replicas only)"""
    return world * cells_per_replica * steps / (ms * 1e-3) / 1e6


def replica_seed(rank):
    return 1 + rank


class ClockSampler:
    """Samples SM clock and throttle reasons during the timed region (NVML; B200_PROFILING.md clocks line)."""

    def __init__(self, index=0, period=0.05):
        self.index, self.period = index, period
        self.samples, self.reasons = [], set()
        self.max_mhz = None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _loop(self):
        nv = self.nv
        names = {
            "hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
            "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
            "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
            "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4),
            "hw_power_brake": getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80),
        }
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop.wait(self.period)

    def __enter__(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self):
        s = sorted(self.samples)
        return {"sm_mhz": (s[len(s) // 2] if s else None), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s)}


# --------------------------------------------------------------------------------------------
# GPU arm
# --------------------------------------------------------------------------------------------
def time_device(cfg, steps, warmup, device, seed, sampler=None, barrier=None, path=None, mask_frac=0.0):
    """Times `steps` time steps with populations resident in HBM.  Returns a dict with the elapsed
    ms (CUDA events on the context's stream), the per-kernel device times measured with event pairs
    around every launch in a second pass of the same length, and the launch count."""
    import torch
    import paper_2502_12955_b200 as lbm
    sim = lbm.LBM(*cfg["grid"], cfg["lattice"], cfg["model"], device=device, **cfg["params"])
    if path is not None:
        sim.set_path(*path)
    sim.init_from_seed(seed)
    if mask_frac:                                             # seeded random solid nodes (benchmark lines with a mask)
        g = torch.Generator(device="cpu").manual_seed(1234)
        sim.set_mask((torch.rand(sim.N, generator=g) < mask_frac).to(torch.uint8))
    sim.step(warmup)
    sim.synchronize()
    if barrier is not None:
        barrier()
    l0 = sim.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ctx = sampler if sampler is not None else _Null()
    with ctx:
        e0.record(sim.stream)
        sim.step(steps)
        e1.record(sim.stream)
        e1.synchronize()
    ms = e0.elapsed_time(e1)
    launches = sim.launch_count() - l0
    if barrier is not None:
        barrier()
    # second pass: the dominant kernel's own average duration (event pair around every launch)
    nk = min(steps, 200)
    sim.kernel_timing(True)
    sim.step(nk)
    step_ms, step_n = sim.kernel_time_ms(0)
    psi_ms, psi_n = sim.kernel_time_ms(1)
    sim.kernel_timing(False)
    # sanity: the state is finite (a NaN-producing run is not a benchmark)
    m = sim.get_macros(u=False, phi=False, C_=False)
    finite = bool(torch.isfinite(m["rho"]).all().item())
    del m
    used_path = sim.get_path()
    try:
        sim.check()                                           # deferred device-side errors (bounded waits of the tile path)
    except Exception:
        finite = False
    s = shape_of(cfg)
    if used_path == "pipeline":
        kernel = "k_tile"
    elif cfg["model"] == "BGK" and s["B"] == 4 and cfg["grid"][0] % 2 == 0 and not cfg["params"].get("bc", (0, 0, 0))[0]:
        kernel = "k_step_v2"
    else:
        kernel = "k_step"
    sim.close()
    torch.cuda.empty_cache()
    return dict(ms=ms, launches=launches, step_ms=step_ms, step_n=step_n, psi_ms=psi_ms, psi_n=psi_n, finite=finite,
                path=used_path, kernel=kernel)


class _Null:
    def __enter__(self):
        return self

    def __exit__(self, *a):
        pass


def time_e2e(cfg, steps, device, seed):
    """The same metric through lbm_run_host: pinned HOST buffers in and out, the host->device copy of
    the canonical populations and the device->host copy of rho and u inside the timed region."""
    import torch
    import paper_2502_12955_b200 as lbm
    s = shape_of(cfg)
    sim = lbm.LBM(*cfg["grid"], cfg["lattice"], cfg["model"], device=device, **cfg["params"])
    sim.init_from_seed(seed)
    f_dev = sim.get_populations()
    f_host = torch.empty(f_dev.numel(), dtype=f_dev.dtype, pin_memory=True)
    f_host.copy_(f_dev)
    del f_dev
    d = 3 if cfg["lattice"] == "D3Q19" else 2
    rho = torch.empty(s["S"] * s["N"], dtype=f_host.dtype, pin_memory=True)
    u = torch.empty(d * s["N"], dtype=f_host.dtype, pin_memory=True)
    sim.run_host(f_host, min(steps, 3), rho=rho, u=u)       # warm-up call (same path)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(sim.stream)
    sim.run_host(f_host, steps, rho=rho, u=u)
    e1.record(sim.stream)
    e1.synchronize()
    ms = e0.elapsed_time(e1)
    ok = bool(torch.isfinite(rho).all().item())
    h2d = f_host.numel() * f_host.element_size()
    d2h = (rho.numel() + u.numel()) * rho.element_size()
    sim.close()
    del f_host, rho, u
    torch.cuda.empty_cache()
    return dict(ms=ms, h2d=h2d, d2h=d2h, finite=ok)


def model_line(name, cfg, r, steps, peak):
    """per-model entry: MLUPS, achieved algorithmic GB/s of the whole step and of each kernel"""
    s = shape_of(cfg)
    step_b, psi_b = algorithmic_bytes(cfg)
    mlups = s["N"] * steps / (r["ms"] * 1e-3) / 1e6
    gbs = (step_b + psi_b) * s["N"] * steps / (r["ms"] * 1e-3) / 1e9
    out = {"workload": name, "lattice": cfg["lattice"], "model": cfg["model"], "grid": list(cfg["grid"]),
           "dtype": "f64" if s["B"] == 8 else "f32", "steps": steps, "ms_per_step": r["ms"] / steps,
           "mlups": round(mlups, 1), "algorithmic_bytes_per_update": step_b + psi_b,
           "hbm_gbs": round(gbs, 1), "frac_of_measured": round(gbs / peak, 4),
           "frac_of_nominal_8TBs": round(gbs / HBM_NOMINAL_GBS, 4),
           "population_mb": round((s["S"] * s["Q"] + s["Qs"]) * s["N"] * s["B"] / 1e6, 1),
           "finite": r["finite"]}
    out["path"], out["kernel"] = r.get("path"), r.get("kernel")
    if r["step_n"]:
        t = r["step_ms"] / r["step_n"]
        out["step_kernel_ms"] = round(t, 5)
        out["step_kernel_gbs"] = round(step_b * s["N"] / (t * 1e-3) / 1e9, 1)
    if r["psi_n"]:
        t = r["psi_ms"] / r["psi_n"]
        out["psi_kernel_ms"] = round(t, 5)
    return out


# --------------------------------------------------------------------------------------------
# CPU arm: the oracle as it stands (single-threaded), on a bounded sample of the workload
# --------------------------------------------------------------------------------------------
def oracle_sample_grid(cfg, budget_cells):
    """A sub-grid of the workload with about budget_cells cells: the wall axis (z for cfg4) keeps its
    full extent, the periodic axes shrink by powers of two."""
    g = list(cfg["grid"])
    bc = cfg["params"].get("bc", (0, 0, 0))
    axes = [a for a in range(3) if not bc[a] and g[a] > 1]
    while g[0] * g[1] * g[2] > budget_cells and axes:
        a = max(axes, key=lambda k: g[k])
        if g[a] <= 8:
            break
        g[a] //= 2
    return tuple(g)


def time_oracle(cfg, steps, warmup, seconds):
    """(MLUPS, sample description, seconds spent).  The sample grid is chosen from a one-step probe so
    that warmup + steps oracle steps take about `seconds`."""
    from oracle.ref_lbm import RefLBM
    over = {}
    if cfg["params"].get("init_kind") == "RANDOM_DROPLETS":
        over = dict(rmin=4.0, rmax=8.0, vol_frac=0.05)       # droplets that fit the sample grid
    probe_grid = oracle_sample_grid(cfg, 1 << 18)           # larger than the host L2: an honest rate
    pc = dict(cfg, grid=probe_grid, params=dict(cfg["params"], **over))
    ref = RefLBM(*pc["grid"], pc["lattice"], pc["model"], **pc["params"])
    ref.init_from_seed(1)
    ref.step(1)
    t0 = time.perf_counter()
    ref.step(2)
    rate = 2 * ref.N / (time.perf_counter() - t0)            # cell updates / s
    ref.close()
    budget = int(0.7 * rate * seconds / max(1, steps + warmup))
    grid = oracle_sample_grid(cfg, max(budget, 1 << 12))
    sc = dict(cfg, grid=grid, params=dict(cfg["params"], **over))
    ref = RefLBM(*sc["grid"], sc["lattice"], sc["model"], **sc["params"])
    ref.init_from_seed(1)
    ref.step(warmup)
    t0 = time.perf_counter()
    ref.step(steps)
    dt = time.perf_counter() - t0
    n = ref.N
    ref.close()
    desc = "%s %s %s grid %dx%dx%d (sub-grid of %dx%dx%d), %d steps, single thread" % (
        cfg["lattice"], cfg["model"], "f64" if cfg["params"]["precision"] == 64 else "f32",
        grid[0], grid[1], grid[2], cfg["grid"][0], cfg["grid"][1], cfg["grid"][2], steps)
    return n * steps / dt / 1e6, desc, dt


_ORACLE_WORKER = """
import json, sys, time
sys.path.insert(0, sys.argv[1])
from oracle.ref_lbm import RefLBM
a = json.loads(sys.argv[2])
ref = RefLBM(*a["grid"], a["lattice"], a["model"], **a["params"])
ref.init_from_seed(1)
ref.step(1)
t0 = time.perf_counter()
ref.step(a["steps"])
print(ref.N * a["steps"], time.perf_counter() - t0)
"""


def time_oracle_all_cores(cfg, steps, budget_cells, timeout=150.0):
    """The oracle is single-threaded and stays so; this is the optional second figure of SURVEY 8(d): one independent
    oracle instance per host core (separate processes, the same sample grid each, bounded by `timeout`), aggregate
    MLUPS = all updates / the slowest instance's time.  Labelled as such; not a tuned program."""
    import subprocess
    cores = min(os.cpu_count() or 1, 32)                   # bounded: every instance holds two copies of its populations
    over = dict(rmin=4.0, rmax=8.0, vol_frac=0.05) if cfg["params"].get("init_kind") == "RANDOM_DROPLETS" else {}
    grid = oracle_sample_grid(cfg, budget_cells)
    params = dict(cfg["params"], **over)
    params = {k: (list(v) if isinstance(v, tuple) else v) for k, v in params.items() if k != "wall_u"}
    arg = json.dumps(dict(grid=list(grid), lattice=cfg["lattice"], model=cfg["model"], params=params, steps=steps))
    procs = [subprocess.Popen([sys.executable, "-c", _ORACLE_WORKER, ROOT, arg], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL,
                              text=True) for _ in range(cores)]
    updates, dt = 0, 0.0
    t_end = time.time() + timeout
    try:
        for pr in procs:
            out, _ = pr.communicate(timeout=max(1.0, t_end - time.time()))
            u, d = out.split()
            updates += int(u)
            dt = max(dt, float(d))
    finally:
        for pr in procs:
            if pr.poll() is None:
                pr.kill()
    desc = "%d independent single-thread oracle processes, each %s %s grid %dx%dx%d, %d steps" % (
        cores, cfg["lattice"], cfg["model"], grid[0], grid[1], grid[2], steps)
    return updates / dt / 1e6, cores, desc


def workload_name(key, cfg):
    s = shape_of(cfg)
    return "%s: %s %s %s %dx%dx%d" % (key, cfg["lattice"], cfg["model"], "fp64" if s["B"] == 8 else "fp32",
                                      cfg["grid"][0], cfg["grid"][1], cfg["grid"][2])


def run_reference(args, cfg, key):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    mlups, desc, dt = time_oracle(cfg, args.steps, args.warmup, seconds=90.0)
    line = {"impl": "reference", "metric": "MLUPS", "value": round(mlups, 3), "unit": "MLUPS", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64" if cfg["params"]["precision"] == 64 else "f32", "data": "synthetic",
            "config": {"workload": workload_name(key, cfg), "sample": desc},
            "cpu_baseline": {"value": round(mlups, 3), "unit": "MLUPS", "cores": 1, "kind": "oracle", "sample": desc},
            "e2e": {"value": round(mlups, 3), "unit": "MLUPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# per-model lines of the default run: (key, config overrides, steps, warmup).  BASELINE.json configs
# 1-3 at paper size are L2-resident (0.3 / 4.7 / 38 MB): their rate is launch/L2-bound and their "HBM
# fraction" is flagged l2_resident; the 8192^2 rows run the same D2Q9 kernels HBM-bound.
# (key, overrides, grid, steps, warmup[, path[, note[, mask fraction]]])
EXTRAS = [
    ("cfg4", dict(precision=32), None, 1000, 50),
    ("cfg5", dict(), None, 100, 10),
    ("cfg5", dict(), None, 40, 5, ("register", 0), "two launches per step: psi pass + fused step (DESIGN.md 6.3)"),
    ("cfg1", dict(), None, 2000, 100),
    ("cfg2", dict(), None, 2000, 100),
    ("cfg3", dict(), None, 1000, 50),
    ("cfg1", dict(), (8192, 8192, 1), 100, 10),
    ("cfg2", dict(radius=2000.0), (8192, 8192, 1), 100, 10),
    ("cfg3", dict(), (8192, 8192, 1), 50, 5),
    ("cfg3", dict(), (8192, 8192, 1), 30, 5, ("pipeline", 0), "resident-tile path (opt-in for D2Q9: slower there, DESIGN.md 6.3)"),
    ("cfg4", dict(bc=(0, 0, 0), force=(0.0, 0.0, 0.0), init_kind="TAYLOR_GREEN", u0=0.05, tau=(0.5019, 0.5019)),
     (128, 128, 128), 1000, 50, None, "the paper's 3D Taylor-Green size, 2,097,152 cells (PAPER.md:854: 1056 MLUPS on a V100)"),
    # the paper's 3D Couette benchmark (1,000,000 cells, 1202 MLUPS on a V100): moving-wall kernel variant
    ("cfg4", dict(bc=(0, 0, 1), force=(0.0, 0.0, 0.0), wall_u={(2, 1): (0.02, 0.0, 0.0)}), (100, 100, 100), 1000, 50, None,
     "the paper's 3D Couette size, 1,000,000 cells, top wall moving (PAPER.md:848: 1202 MLUPS on a V100); L2-resident"),
    ("cfg4", dict(bc=(0, 0, 1), force=(0.0, 0.0, 0.0), wall_u={(2, 1): (0.02, 0.0, 0.0)}), (256, 256, 256), 500, 20, None,
     "Couette, moving-wall kernel variant at an HBM-bound size"),
    # paper-shaped Rayleigh-Taylor setup: two components between walls in y, gravity, 1200 x 400
    ("cfg3", dict(bc=(0, 1, 0), force=(0.0, -1e-5, 0.0), G_ads=(0.0, 0.0)), (1200, 400, 1), 500, 50, None,
     "Rayleigh-Taylor-shaped: walls in y + body force"),
    ("cfg3", dict(forcing=1), (8192, 8192, 1), 50, 5, None, "velocity-shift forcing scheme (Eq. 16-19)"),
    ("cfgT", dict(), (256, 256, 256), 200, 20, None, "BGK + internal-energy lattice (IEDDF, Eq. 27-30)"),
    ("cfgT", dict(tau_s=0.9, rho_solid=2.0), (256, 256, 256), 200, 20, None,
     "the same with 20 % random solid nodes carrying the solid-phase energy lattice (Eq. 31-33)", 0.2),
]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=50)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg4", choices=sorted(workloads.CONFIGS))
    ap.add_argument("--precision", type=int, default=None, choices=[32, 64])
    ap.add_argument("--grid", type=int, nargs=3, default=None, help="override the grid (profiling runs)")
    ap.add_argument("--path", default=None, help="register | pipeline[:rows_per_pencil] (default: the library's choice)")
    ap.add_argument("--no-extras", action="store_true", help="skip per_model, e2e and cpu_baseline (profiling runs)")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3                                       # timing rule: W >= 3
    over = {} if args.precision is None else {"precision": args.precision}
    cfg = workloads.config(args.workload, grid=args.grid, **over)
    if args.impl == "reference":
        run_reference(args, cfg, args.workload)
        return

    import torch
    import paper_2502_12955_b200 as lbm
    from paper_2502_12955_b200 import build as _build
    if int(os.environ.get("LOCAL_RANK", "0")) == 0:
        _build.build()                                        # no-op when liblbm.so is up to date (needs nvcc otherwise)
    else:
        t_wait = time.time()
        while not _build.up_to_date() and time.time() - t_wait < 900:
            time.sleep(1.0)                                   # rank 0 is building
    lbm.lib()                                                 # fails loudly when liblbm.so is missing
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the hot path has no CPU fallback")
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    device = "cuda:%d" % local
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(device))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    peak, peak_kind = measured_peak()
    sampler = ClockSampler(index=local) if rank == 0 else None
    # replicas only: rank r runs its own seeded copy of the workload (no data-path collective)
    path = None
    if args.path:
        pp = args.path.split(":")
        path = (pp[0], int(pp[1]) if len(pp) > 1 else 0)
    r = time_device(cfg, args.steps, args.warmup, device, seed=replica_seed(rank), sampler=sampler, barrier=barrier,
                    path=path)
    ms = max_over_ranks(r["ms"], dist, device)
    s = shape_of(cfg)
    step_b, psi_b = algorithmic_bytes(cfg)
    value = aggregate_mlups(world, s["N"], args.steps, ms)
    e2e = None
    if not args.no_extras:
        e = time_e2e(cfg, args.steps, device, seed=replica_seed(rank))
        ems = max_over_ranks(e["ms"], dist, device)
        e2e = {"value": round(aggregate_mlups(world, s["N"], args.steps, ems), 1), "unit": "MLUPS",
               "h2d_bytes_per_step": e["h2d"] / args.steps, "d2h_bytes_per_step": e["d2h"] / args.steps,
               "call": "lbm_run_host(f_host, n=%d, rho_host, u_host): one upload of the populations, %d steps, "
                       "one download of rho and u, pinned host memory" % (args.steps, args.steps),
               "ms": round(ems, 3), "finite": e["finite"]}
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # roofline of the dominant kernel (the fused step kernel): algorithmic bytes per launch / its
    # average launch duration, measured live with CUDA event pairs on the launching stream
    k_ms = r["step_ms"] / max(1, r["step_n"])
    achieved = step_b * s["N"] / (k_ms * 1e-3) / 1e9
    traffic, traffic_source = ncu_traffic(workload_name(args.workload, cfg), r["kernel"])
    line = {
        "metric": "MLUPS", "value": round(value, 1), "unit": "MLUPS", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64" if s["B"] == 8 else "f32", "data": "synthetic",
        "config": {"workload": workload_name(args.workload, cfg), "parallelism": "replicas only" if world > 1 else "1 gpu",
                   "l2": "inputs larger than L2 (%.0f MB populations vs 126 MB), no flush" %
                         ((s["S"] * s["Q"] + s["Qs"]) * s["N"] * s["B"] / 1e6),
                   "streaming": "in-place AA pattern, one population copy", "path": r["path"]},
        "hbm_gbs": round((step_b + psi_b) * s["N"] * args.steps / (ms * 1e-3) / 1e9 , 1),
        "roofline": {"bound": "hbm", "kernel": "%s (fused collide+stream)" % r["kernel"], "achieved": round(achieved, 1),
                     "peak": peak, "peak_kind": "%s: torch copy_ bandwidth (a fraction a little above 1.0 means the kernel "
                                                "beats a plain copy, not that it beats the hardware)" % peak_kind,
                     "unit": "GB/s", "frac": round(achieved / peak, 4),
                     "frac_of_nominal_8TBs": round(achieved / HBM_NOMINAL_GBS, 4),
                     "algorithmic_bytes_per_update": step_b, "kernel_ms": round(k_ms, 5),
                     "kernel_ms_how": "second pass of the same length with a CUDA event pair around every launch "
                                      "(adds event overhead: may slightly exceed ms_per_step)",
                     "traffic": traffic, "traffic_source": traffic_source},
        "gpu_launches": r["launches"],
        "clocks": sampler.summary() if sampler is not None else None,
        "finite": r["finite"],
    }
    if e2e is not None:
        line["e2e"] = e2e
    if not args.no_extras and world == 1:
        per = [model_line(workload_name(args.workload, cfg), cfg, r, args.steps, peak)]
        for key, ov, grid, k, w, *rest in EXTRAS:
            c = workloads.config(key, grid=grid, **ov)
            epath = rest[0] if rest else None
            rr = time_device(c, k, w, device, seed=1, path=epath, mask_frac=rest[2] if len(rest) > 2 else 0.0)
            ml = model_line(workload_name(key, c), c, rr, k, peak)
            if len(rest) > 1 and rest[1]:
                ml["note"] = rest[1]
            if ml["population_mb"] < 126.0:
                ml["l2_resident"] = True
            per.append(ml)
        line["per_model"] = per
        # north_star's "D3Q19 fused kernels >= 75 % of HBM bandwidth": the three D3Q19 kernels, inside roofline so that
        # they survive a truncated output tail
        fused = []
        for ml in per:
            if ml["lattice"] == "D3Q19" and ml["workload"].startswith(("cfg4: D3Q19 BGK fp64 256", "cfg4: D3Q19 BGK fp32 256", "cfg5:")) \
                    and "Couette" not in ml.get("note", ""):
                fused.append({k2: ml[k2] for k2 in ("workload", "path", "kernel", "mlups", "ms_per_step", "hbm_gbs",
                                                     "frac_of_measured", "frac_of_nominal_8TBs", "step_kernel_ms") if k2 in ml})
        line["roofline"]["d3q19_fused"] = fused
        mlups, desc, _ = time_oracle(cfg, 6, 1, seconds=20.0)
        line["cpu_baseline"] = {"value": round(mlups, 3), "unit": "MLUPS", "cores": 1, "kind": "oracle", "sample": desc}
        try:
            am, cores, adesc = time_oracle_all_cores(cfg, 6, 1 << 19)
            line["cpu_baseline"]["all_cores"] = {"value": round(am, 3), "unit": "MLUPS", "cores": cores, "sample": adesc}
        except Exception as exc:                               # the single-thread figure above is the baseline
            line["cpu_baseline"]["all_cores"] = {"unavailable": repr(exc)[:200]}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
