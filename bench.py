#!/usr/bin/env python
"""bench.py -- throughput of the full RK2 Kurganov-Tadmor step (both stages + inversion + regularisation + ghost cells).

  python bench.py --gpus N --steps K --warmup W            (this implementation, CUDA C-ABI library)
  python bench.py --impl reference --steps K --warmup W    (the CPU oracle on a bounded sample, host cores)

Workload at N=1: BASELINE.json configs[2] -- 128^3 cells, 3+1d viscous non-conformal, 15 FP64 fields per cell, seeded
Gaussian hotspots (stand-in for the paper's MC-Glauber event).  One "step" = one full RK2 step of
the whole grid.  metric = cell-updates/s.  The path does not shard (BASELINE.json north_star: one GPU, no collectives):
with N > 1 every rank runs an independent replica (event seed + rank), no data-path collective, "weak" scaling.
Prints ONE JSON line (rank 0)."""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_1608_06577_b200 import inputs  # noqa: E402

METRIC = "cell-updates/s (full RK2 KT step, FP64) at 128^3 viscous"
METRIC_F32 = "cell-updates/s (full RK2 KT step, single-precision build) at 128^3 viscous"
UNIT = "cell-updates/s"
ALG_BYTES_PER_CELL_UPDATE = 856.0      # 107 doubles per cell-update, each state array read/written once per stage
ALG_BYTES_STAGE = {"stage1": (25 + 21) * 8.0, "stage2": (40 + 21) * 8.0}
# Raw `ncu --csv` metric page of one RK2 step of THIS workload (four launches, in launch order), committed with the build it was taken
# from; the command is in profiles/r02_metrics.md.  bench.py reads DRAM traffic, executed DFMA/DADD/DMUL and FP64-pipe utilisation per
# launch from it (they are properties of the build, not of a run: ncu replays kernels and cannot be on while timing).
NCU_METRICS_CSV = os.path.join(ROOT, "profiles", "r03_metrics.csv")


def metrics_page(workload="config3", physics="config3", precision="f64", storage=0, variant=0):
    """The committed raw ncu page of the configuration a line is printed for (profiles/r03_metrics.md names the command of each), or None:
    FP64 default pipeline only - the pages hold FP64 op counts and the launch order velocity / stage / velocity / stage."""
    if precision != "f64" or storage or variant:
        return None
    tag = workload if workload != "config3" else ("paper" if physics == "paper" else "config3")
    if workload != "config3" and physics == "paper":
        return None
    return NCU_METRICS_CSV if tag == "config3" else os.path.join(ROOT, "profiles", "r03_metrics_%s.csv" % tag)
LAUNCH_KEYS = ("velocity1", "stage1", "velocity2", "stage2")


def ncu_metrics(path=NCU_METRICS_CSV):
    """{launch key: {metric: value}} from the committed raw ncu CSV (rows: one per launch and metric), or {} if it is absent or does
    not hold exactly one step of the default pipeline (velocity, stage, velocity, stage)."""
    import csv
    if not os.path.exists(path):
        return {}
    rows = list(csv.reader(l for l in open(path) if l.startswith('"')))
    if not rows:
        return {}
    h = rows[0]
    try:
        ki, mi, vi, ii = h.index("Kernel Name"), h.index("Metric Name"), h.index("Metric Value"), h.index("ID")
    except ValueError:
        return {}
    per, order = {}, []
    for r in rows[1:]:
        if r[ii] not in per:
            per[r[ii]] = {"kernel": r[ki]}
            order.append(r[ii])
        try:
            per[r[ii]][r[mi]] = float(r[vi].replace(",", ""))
        except ValueError:
            pass
    if len(order) != 4:
        return {}
    out = {}
    for key, lid in zip(LAUNCH_KEYS, order):
        if ("velocity" in key) != ("velocity" in per[lid]["kernel"]):
            return {}
        out[key] = per[lid]
    return out


def host_cpu():
    model = "unknown"
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                model = line.split(":", 1)[1].strip()
                break
    except OSError:
        pass
    return model, os.cpu_count()


def workload(rank=0, physics="config3", which="config3"):
    """configs[2] of BASELINE.json (default); physics="paper": the same grid and hotspots with the paper's own equation of state
    (lattice, Eqs. 19-20) and zeta/s(T) (Eq. 17, T_c = 200 MeV) - SURVEY 8(f) NEXT-1 - for a second, labelled bench line.
    which = "config4" / "config5": the batched 2+1d and the large 3+1d configurations of BASELINE.json (labelled extra lines)."""
    over = dict(eos=2, zeta_model=3, zeta_amp=1.0, zeta_T0=0.2 / inputs.HBARC) if physics == "paper" else {}
    if which == "config4":
        prm, init, _ = inputs.config_batched2d(seed=inputs.BASE_SEED + 1000 * rank, **over)
    elif which == "config5":
        prm, init, _ = inputs.config_3d(512, 512, 128, 0.05, 0.05, 0.1, n_hot=200, n_steps=50, seed=inputs.BASE_SEED + rank, **over)
    else:
        prm, init, _ = inputs.config_3d(seed=inputs.BASE_SEED + rank, **over)
    return prm, init


def max_over_ranks(x, dist, device):
    """Timing of a multi-rank run = the slowest rank (the only collective of the replica mode; none on the data path)."""
    if dist is None:
        return float(x)
    import torch

    t = torch.tensor([x], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(ncell_per_rank, steps, world, seconds):
    """Whole-job throughput of `world` independent replicas: all ranks' cell-updates / max-over-ranks time."""
    return ncell_per_rank * steps * world / seconds


class ClockSampler:
    """SM clock, power and throttle reasons sampled WHILE the timed region runs: NVML polled every ~2 ms from a thread (the timed
    region of a short run is far shorter than nvidia-smi's polling period); falls back to `nvidia-smi -lms 20` without pynvml."""
    REASONS = (("hw_slowdown", "HwSlowdown"), ("hw_thermal_slowdown", "HwThermalSlowdown"), ("sw_thermal_slowdown", "SwThermalSlowdown"),
               ("sw_power_cap", "SwPowerCap"))
    Q = "index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown," \
        "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, gpu_index):
        self.gpu = gpu_index
        self.sm, self.power, self.reasons = [], [], set()
        self.sm_max = None
        self.stop_flag = threading.Event()
        self.thread = None
        self.proc = None
        self.file = None
        self.nvml = None
        try:
            import pynvml

            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = gpu_index
            if vis:
                ids = [x.strip() for x in vis.split(",") if x.strip()]
                if gpu_index < len(ids) and ids[gpu_index].isdigit():
                    phys = int(ids[gpu_index])
            self.handle = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.sm_max = float(pynvml.nvmlDeviceGetMaxClockInfo(self.handle, pynvml.NVML_CLOCK_SM))
            self.nvml = pynvml
        except Exception:
            self.nvml = None

    def _poll(self):
        nv = self.nvml
        while not self.stop_flag.is_set():
            try:
                self.sm.append(float(nv.nvmlDeviceGetClockInfo(self.handle, nv.NVML_CLOCK_SM)))
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.handle) / 1000.0)
                mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self.handle)
                for name, suffix in self.REASONS:
                    if mask & getattr(nv, "nvmlClocksEventReason" + suffix):
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.002)

    def start(self):
        if self.nvml is not None:
            self.thread = threading.Thread(target=self._poll, daemon=True)
            self.thread.start()
            return
        try:
            self.file = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=self.file, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": self.sm_max, "reasons": [], "samples": 0, "power_w_max": None, "source": "nvml" if self.nvml else "nvidia-smi"}
        if self.thread is not None:
            self.stop_flag.set()
            self.thread.join(timeout=2)
        elif self.proc is not None:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except Exception:
                self.proc.kill()
            self.file.flush()
            self.file.seek(0)
            mx = []
            for line in self.file.read().splitlines():
                c = [x.strip() for x in line.split(",")]
                if len(c) < 9:
                    continue
                try:
                    self.sm.append(float(c[1])); mx.append(float(c[2])); self.power.append(float(c[3]))
                except ValueError:
                    continue
                for (name, _), v in zip(self.REASONS, c[5:9]):
                    if v.lower().startswith("active"):
                        self.reasons.add(name)
            try:
                os.unlink(self.file.name)
            except OSError:
                pass
            if mx:
                self.sm_max = float(max(mx))
        if self.sm:
            out.update(sm_mhz=float(np.median(self.sm)), sm_max_mhz=self.sm_max, reasons=sorted(self.reasons), samples=len(self.sm),
                       power_w_max=float(max(self.power)) if self.power else None)
        return out


def oracle_sample(prm, init, nx, ny, nz):
    """Central cut-out of the workload for the CPU oracle (bounded sample of the same initial data)."""
    nz = min(nz, prm["nz"])
    z0, y0, x0 = (prm["nz"] - nz) // 2, (prm["ny"] - ny) // 2, (prm["nx"] - nx) // 2
    cut = lambda a: np.ascontiguousarray(a[..., 0:1, z0:z0 + nz, y0:y0 + ny, x0:x0 + nx])
    sub = dict(prm, nx=nx, ny=ny, nz=nz, n_batch=1)
    return sub, cut(init["e"]), cut(init["u"])


def time_oracle(prm, init, dims, steps, warmup=0):
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import vh_oracle

    sub, e, u = oracle_sample(prm, init, *dims)
    o = vh_oracle.Oracle(sub)
    o.set_initial(e, u)
    if warmup:
        o.step(warmup)
    dt = o.time_steps(steps)
    ncell = dims[0] * dims[1] * dims[2]
    what = "the full %dx%dx%d workload" % dims if dims == (prm["nx"], prm["ny"], prm["nz"]) else "central %dx%dx%d cut-out of the 128^3 initial data" % dims
    return ncell * steps / dt, dt, "%s, %d RK2 step(s), serial C++ oracle -O2, 1 core" % (what, steps)


def algorithmic_flops(prm, init):
    """MINIMAL algorithmic flop count per cell-update: the oracle with an operation-counting scalar on a 16^3 cut-out; every interface
    charged once, every limited slope once, compares excluded, exact 0 / +-1 constants not counted; weights of SURVEY.md 8(d).
    Returns (flops, per-class op counts, flops per oracle section).  Test infrastructure used for the report only."""
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import vh_oracle

    sub, e, u = oracle_sample(prm, init, 16, 16, 16)
    return vh_oracle.algorithmic_flops_per_cell_update(sub, e, u)


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    prm, init = workload(0, args.physics)
    dims = (64, 64, 32)
    warm = args.warmup
    value, dt, sample = time_oracle(prm, init, dims, args.steps, warmup=warm)
    model, ncores = host_cpu()
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": warm,
        "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": "configs[2]: 128^3 3+1d viscous non-conformal, seeded hotspots; bounded sample " + sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample, "host_cpu": model, "host_cores_total": ncores},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def run_small(args, vh, torch, dev, rank):
    """configs[0] (1d shock tube, 200 cells, 100 steps) and configs[1] (2+1d viscous Gubser, 201^2, 400 steps) of BASELINE.json: wall time
    of the WHOLE run, CUDA events around vh_step(n_steps) after one untimed run, best of five; the serial oracle's
    full run beside it.  Labelled extra lines: these grids are launch-bound (a step is four launches of a few microseconds of work), so no
    roofline fraction is printed."""
    if rank != 0:
        return 0
    if args.workload == "config1":
        prm, init, n_steps, _ = inputs.config_shocktube()
        what = "configs[0] (labelled extra line): 1d ideal shock tube, 200 cells, 100 steps"
    else:
        prm, init, n_steps, _ = inputs.config_gubser()
        what = "configs[1] (labelled extra line): 2+1d conformal viscous Gubser flow, 201x201, 400 steps"
    t = lambda a: None if a is None else torch.as_tensor(a, device=dev)
    s = vh.Solver(prm, device=dev)
    arrays = (t(init["e"]), t(init["u"]), t(init.get("pi")), t(init.get("Pi")))
    best, launches = None, 0
    for rep in range(6):                      # rep 0 is the warm-up run
        s.set_initial(*arrays)
        torch.cuda.synchronize()
        n0 = s.launch_count()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record(); s.step(n_steps); ev1.record()
        torch.cuda.synchronize()
        launches = s.launch_count() - n0
        if rep > 0:
            best = ev0.elapsed_time(ev1) if best is None else min(best, ev0.elapsed_time(ev1))
    st = s.status()
    s.close()
    ncell = prm["nx"] * prm["ny"] * prm["nz"]
    line = {"metric": METRIC.replace("at 128^3 viscous", "whole run of " + args.workload), "value": ncell * n_steps / (best * 1e-3), "unit": UNIT, "n_gpus": 1,
            "steps": n_steps, "warmup": n_steps, "ms_per_step": best / n_steps, "run_ms": best, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": {"workload": what}, "gpu_launches": int(launches), "roofline": None,
            "status": {"n_inversion_failures": st["n_inversion_failures"], "n_nonfinite": st["n_nonfinite"]}}
    if not args.no_cpu_baseline:
        sys.path.insert(0, os.path.join(ROOT, "oracle"))
        import vh_oracle
        o = vh_oracle.Oracle(prm)
        o.set_initial(init["e"], init["u"], init.get("pi"), init.get("Pi"))
        t0 = time.perf_counter(); o.step(n_steps); dt = time.perf_counter() - t0
        line["cpu_baseline"] = {"value": ncell * n_steps / dt, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": "the full run, serial C++ oracle -O2, 1 core", "seconds": dt}
    print(json.dumps(line))
    return 0


def run_slab(args, vh, torch, dist, dev, rank, world, local):
    """ONE grid split into eta-slabs, one per rank, neighbour exchange of boundary planes after every kernel (vh.SlabSolver):
    strong scaling.  A labelled extra line - the default N > 1 mode stays independent replicas (north_star: no sharding).  The same event on
    every rank (seed of rank 0); time = max over ranks of the CUDA-event time of K steps including the exchanges."""
    if dist is None:
        import torch.distributed as dist      # a 1-rank group: SlabSolver then owns the whole grid and exchanges nothing
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1"); os.environ.setdefault("MASTER_PORT", "29533")
        dist.init_process_group("nccl", rank=0, world_size=1, device_id=dev)
    prm, init = workload(0, args.physics, args.workload)
    if args.precision == "f32":
        prm["newton_rtol"] = 2e-6
    W, K = max(args.warmup, 3), args.steps
    s = vh.SlabSolver(prm, device=dev, precision=args.precision)
    s.set_initial(torch.as_tensor(init["e"], device=dev), torch.as_tensor(init["u"], device=dev))
    s.step(W)
    torch.cuda.synchronize(); dist.barrier(); torch.cuda.synchronize()
    sampler = ClockSampler(local)
    sampler.start()
    n0 = s.s.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    s.step(K)
    ev1.record()
    torch.cuda.synchronize(); dist.barrier(); torch.cuda.synchronize()
    launches = s.s.launch_count() - n0
    clocks = sampler.stop()
    ms = max_over_ranks(ev0.elapsed_time(ev1), dist, dev)
    st = s.status()
    fails = torch.tensor([float(st["n_inversion_failures"])], device=dev, dtype=torch.float64)
    dist.all_reduce(fails)
    halo = (s.s.halo_size(0) + s.s.halo_size(1)) * 8 * 2          # bytes a rank sends per face per step (two exchanges of each kind)
    s.close()
    ncell = prm["nx"] * prm["ny"] * prm["nz"]
    if rank == 0:
        print(json.dumps({
            "metric": METRIC.replace("at 128^3 viscous", "at %dx%dx%d viscous, ONE grid in %d eta-slabs" % (prm["nx"], prm["ny"], prm["nz"], world)),
            "value": ncell * K / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": ms / K, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": args.precision, "data": "synthetic",
            "config": {"workload": "labelled extra line (the default N > 1 mode is independent replicas): %s split along eta, %d planes per rank, neighbour "
                                   "send/recv of 2 planes x 21 arrays + 1 plane of state velocities per face after every kernel (%s backend)"
                                   % (args.workload, prm["nz"] // world, dist.get_backend()), "halo_bytes_per_face_per_step": halo},
            "gpu_launches": int(launches), "clocks": clocks, "status": {"n_inversion_failures": int(fails.item())}}))
    dist.barrier()
    dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--variant", type=int, default=0, help="stage-kernel variant (vh_set_kernel_variant), 0 = default")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-paper-physics", action="store_true", help="skip the second, labelled measurement with the lattice EOS and Eq. 17 zeta/s")
    ap.add_argument("--precision", default="f64", choices=["f64", "f32"], help="f32: the single-precision build (libvh_f32.so; SURVEY 8(f) NEXT-3), a labelled extra line")
    ap.add_argument("--workload", default="config3", choices=["config3", "config4", "config5", "config1", "config2"],
                    help="config4 (256 batched 2+1d events) / config5 (512x512x128): labelled extra lines; the default is the BASELINE.json metric")
    ap.add_argument("--decomposition", default="replicas", choices=["replicas", "slab"],
                    help="N > 1: independent replicas (the default: BASELINE.json north_star fixes one GPU, no sharding) or ONE grid split into eta-slabs "
                         "with neighbour exchange over NCCL (vh.SlabSolver; SURVEY 8(e), strong scaling; a labelled extra line)")
    ap.add_argument("--storage", type=int, default=0, choices=[0, 1], help="1: reduced-storage mode (5 pi + 3 u components, PAPER.md:476; SURVEY 8(f) NEXT-3), a labelled extra line")
    ap.add_argument("--physics", default="config3", choices=["config3", "paper"], help="paper: lattice EOS + Eq. 17 zeta/s on the config-3 grid")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch

    from paper_1608_06577_b200 import vh

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)
    W = max(args.warmup, 3)
    K = args.steps

    if args.decomposition == "slab":
        return run_slab(args, vh, torch, dist, dev, rank, world, local)
    if args.workload in ("config1", "config2"):
        return run_small(args, vh, torch, dev, rank)
    prm, init = workload(rank, args.physics, args.workload)
    other = (args.workload != "config3")
    f32 = (args.precision == "f32")
    prm["storage"] = args.storage
    if f32:
        prm["newton_rtol"] = 2e-6          # the stopping rule of Eq. 72 at single precision (the f32 library refuses anything below 1e-6)
    ncell = prm["nx"] * prm["ny"] * prm["nz"] * prm["n_batch"]
    s = vh.Solver(prm, device=dev, precision=args.precision)
    if args.variant:
        s.set_kernel_variant(args.variant)
    e_d = torch.as_tensor(init["e"], device=dev)
    u_d = torch.as_tensor(init["u"], device=dev)
    s.set_initial(e_d, u_d)
    xoff = 4 if f32 else 2
    s_bytes = (43 if args.storage else 67) * ((prm["nx"] + xoff + 2 + 15) // 16 * 16) * (prm["ny"] + 4) * (prm["nz"] + 4 if prm["nz"] > 1 else 1) * prm["n_batch"] * (4 if f32 else 8)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    # ---------------- device-resident throughput: W warm-up steps, then exactly K timed steps
    s.step(W)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    n0 = s.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    s.step(K)
    ev1.record()
    barrier()
    launches = s.launch_count() - n0
    clocks = sampler.stop()
    ms = ev0.elapsed_time(ev1)
    ms = max_over_ranks(ms, dist, dev)
    value = aggregate_value(ncell, K, world, ms * 1e-3)
    st = s.status()

    # ---------------- per-kernel durations (CUDA events around each launch on the launching stream)
    prof = s.step_profile(min(K, 10))       # keyed by kernel: velocity1, stage1, velocity2, stage2 (variant 1: stage1, ghost1, stage2, ghost2)

    # ---------------- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region (default workload only)
    pin = lambda a: torch.as_tensor(np.ascontiguousarray(a)).pin_memory()
    f_dev = s.get_fields()
    h_e, h_u = pin(f_dev["e"].cpu().numpy()), pin(f_dev["u"].cpu().numpy())
    h_pi, h_Pi = pin(f_dev["q"][4:14].cpu().numpy()), pin(f_dev["q"][14].cpu().numpy())
    shape = s.shape
    kw = dict(dtype=torch.float64, pin_memory=True)
    out = dict(q=torch.empty((15,) + shape, **kw), e=torch.empty(shape, **kw), p=torch.empty(shape, **kw), u=torch.empty((4,) + shape, **kw))
    del f_dev
    h2d = (h_e.numel() + h_u.numel() + h_pi.numel() + h_Pi.numel()) * 8
    d2h = sum(v.numel() for v in out.values()) * 8
    E = 1 if other else max(1, args.e2e_steps)
    s.set_initial(h_e, h_u, h_pi, h_Pi); s.step(1); s.get_fields(out=out)      # warm-up (allocates staging buffers)
    barrier()
    t0 = time.perf_counter()
    for _ in range(E):
        s.set_initial(h_e, h_u, h_pi, h_Pi)
        s.step(1)
        s.get_fields(out=out)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    e2e_s = max_over_ranks(e2e_s, dist, dev)
    e2e_value = aggregate_value(ncell, E, world, e2e_s)

    # ---------------- peaks measured in the same run by the library's own microbenchmarks
    copy_gbs, fp64_gflops = vh.measure_peaks(n_bytes=1 << 30, repeats=10)
    fp32_gflops = vh.measure_fp32_peak(repeats=10) if f32 else None
    alu_gflops = fp32_gflops if f32 else fp64_gflops      # the ALU peak of the precision the library computes in
    bscale = 0.5 if f32 else 1.0                          # bytes per stored value relative to FP64
    s.close()

    # ---------------- second, labelled workload: the paper's own physics (lattice EOS, Eq. 17 zeta/s) on the same grid
    paper_line = None
    if world == 1 and args.physics == "config3" and not args.variant and not args.no_paper_physics and not f32 and not args.storage and not other:
        prm2, init2 = workload(rank, "paper")
        s2 = vh.Solver(prm2, device=dev)
        s2.set_initial(torch.as_tensor(init2["e"], device=dev), torch.as_tensor(init2["u"], device=dev))
        s2.step(W)
        torch.cuda.synchronize()
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a0.record(); s2.step(K); a1.record()
        torch.cuda.synchronize()
        ms2 = a0.elapsed_time(a1)
        st2 = s2.status()
        prof2 = s2.step_profile(min(K, 10))
        s2.close()
        paper_line = {"workload": "configs[2] grid and hotspots with the paper's own physics: lattice EOS (Eqs. 19-20), zeta/s of Eq. 17 (T_c = 200 MeV)",
                      "ms_per_step": ms2 / K, "value": ncell * K / (ms2 * 1e-3), "unit": UNIT, "per_kernel_ms": prof2,
                      "n_inversion_failures": st2["n_inversion_failures"], "n_nonfinite": st2["n_nonfinite"]}

    if rank == 0:
        peaks_file = os.path.join(ROOT, "MEASURED_PEAKS.json")
        hbm_peak, hbm_src = 6650.0, "fallback (B200_PROFILING.md)"
        if os.path.exists(peaks_file):
            try:
                hbm_peak, hbm_src = float(json.load(open(peaks_file))["hbm_gbs"]), "MEASURED_PEAKS.json"
            except Exception:
                pass
        flops_cu, mix, by_section = algorithmic_flops(prm, init)
        flops_inv_cu = by_section["invert"]
        variant1 = (args.variant == 1) or args.storage == 1
        default_pipeline = (args.variant == 0) and args.storage == 0
        # Kernel shares of the algorithmic work: the velocity kernel does the interface-state inversions
        # (Eq. 72 at every reconstructed state), the stage kernel everything else; one stage = half of a cell-update.
        alg_kernel = {k: 0.5 * (flops_inv_cu if "velocity" in k else flops_cu - flops_inv_cu) for k in LAUNCH_KEYS}
        if variant1:
            alg_kernel = {"stage1": 0.5 * flops_cu, "stage2": 0.5 * flops_cu}
        bytes_kernel = {k: v * bscale for k, v in {"stage1": ALG_BYTES_STAGE["stage1"], "stage2": ALG_BYTES_STAGE["stage2"], "velocity1": 10 * 8.0, "velocity2": 10 * 8.0}.items()}
        page = metrics_page(args.workload, args.physics, args.precision, args.storage, args.variant)
        ncu = ncu_metrics(page) if page else {}
        ex_kernel, pipe_kernel, traffic_kernel = {}, {}, {}
        for k, m in ncu.items():
            try:
                ex_kernel[k] = (2.0 * m["smsp__sass_thread_inst_executed_op_dfma_pred_on.sum"] + m["smsp__sass_thread_inst_executed_op_dadd_pred_on.sum"]
                                + m["smsp__sass_thread_inst_executed_op_dmul_pred_on.sum"]) / ncell
                pipe_kernel[k] = m["sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active"] / 100.0
                traffic_kernel[k] = m["dram__bytes_read.sum"] + m["dram__bytes_write.sum"]
            except KeyError:
                pass
        # dominant kernel: the longest of the step's launches, velocity kernels included
        cand = [k for k in prof if k in alg_kernel]
        dom = max(cand, key=lambda k: prof[k])
        dur = prof[dom] * 1e-3
        # Useful flops of a launch: the minimal algorithmic count, but never more than the kernel executes (2 DFMA + DADD + DMUL, ncu):
        # where the kernel gets by with fewer flops than the count, the count still holds work the method does not need.
        useful = {k: min(alg_kernel[k], ex_kernel.get(k, alg_kernel[k])) for k in cand}
        flops_launch = useful[dom] * ncell
        bytes_launch = bytes_kernel[dom] * ncell
        t_alu = flops_launch / (alu_gflops * 1e9)
        t_hbm = bytes_launch / (hbm_peak * 1e9)
        if t_alu >= t_hbm:
            roof = {"bound": "alu", "achieved": flops_launch / dur / 1e12, "peak": alu_gflops / 1e3, "unit": "TFLOP/s"}
        else:
            roof = {"bound": "hbm", "achieved": bytes_launch / dur / 1e9, "peak": hbm_peak, "unit": "GB/s"}
        # a fraction is printed only where the executed flops of THIS configuration's kernels are on file (min(alg, executed) numerator);
        # without a page the minimal count alone would be the numerator, which is known to be too kind (frac_on_minimal_count keeps it, labelled)
        roof["frac"] = roof["achieved"] / roof["peak"] if dom in ex_kernel else None
        useful_step = sum(useful.values())
        step_roof_s = max(useful_step * ncell / (alu_gflops * 1e9), ALG_BYTES_PER_CELL_UPDATE * bscale * ncell / (hbm_peak * 1e9))
        kname = ("velocity_tile_kernel" if "velocity" in dom else "stage_tile_kernel") if default_pipeline else ("stage_reduced_kernel" if args.storage else ("stage_cell_kernel" if variant1 else "stage_kernel"))
        roof.update({
            "traffic": traffic_kernel.get(dom), "traffic_source": os.path.relpath(page, ROOT) if dom in traffic_kernel else None,
            "kernel": "%s (%s)" % (kname, dom), "launch_ms": prof[dom],
            "peak_source": ("FP32 FMA microbenchmark, same run (vh_measure_fp32_peak)" if f32 else "FP64 FMA microbenchmark, same run (vh_measure_peaks)") if roof["bound"] == "alu" else hbm_src,
            "numerator": "min(minimal algorithmic flops, executed flops) of this kernel per cell x cells per launch" if dom in ex_kernel else
                         "minimal algorithmic flops (NO ncu capture of this configuration is committed: on config 3 the kernels execute 1.4x fewer flops than this count, so frac here is that much too kind)",
            "alg_flops_this_kernel_per_cell": alg_kernel[dom], "executed_flops_per_cell": ex_kernel.get(dom),
            "alg_over_executed": (alg_kernel[dom] / ex_kernel[dom]) if dom in ex_kernel else None,
            "fp64_pipe_util": pipe_kernel.get(dom),
            "frac_on_minimal_count": alg_kernel[dom] * ncell / dur / (alu_gflops * 1e9),
            "alg_flops_per_cell_update": flops_cu, "alg_flops_by_section_per_cell_update": {k: round(v, 1) for k, v in by_section.items()},
            "executed_flops_per_cell_update": sum(ex_kernel.values()) if len(ex_kernel) == 4 else None,
            "alg_bytes_per_cell_update": ALG_BYTES_PER_CELL_UPDATE * bscale, "alg_bytes_this_kernel_per_cell": bytes_kernel[dom],
            "flop_weights": "add/mul 1, div 10, sqrt 15, exp 25, pow 30, tanh 40 (SURVEY 8(d)); compares carry no weight; counted on the oracle with "
                            "each interface once, each limited slope once, exact 0/+-1 constants not counted",
            "op_mix_per_cell_update": {k: round(v, 1) for k, v in mix.items()},
            "hbm_view": {"achieved_gbs": bytes_launch / dur / 1e9, "peak_gbs": hbm_peak, "peak_source": hbm_src, "frac": bytes_launch / dur / 1e9 / hbm_peak,
                         "copy_gbs_same_run": copy_gbs},
            "step_roofline_ms": step_roof_s * 1e3, "step_frac": step_roof_s / (ms / K * 1e-3) if len(ex_kernel) == len(cand) else None,
            "per_kernel_ms": prof,
            "per_kernel": {k: {"ms": prof[k], "alg_flops_per_cell": alg_kernel[k], "executed_flops_per_cell": ex_kernel.get(k),
                               "frac": useful[k] * ncell / (prof[k] * 1e-3) / (alu_gflops * 1e9) if k in ex_kernel else None, "fp64_pipe_util": pipe_kernel.get(k),
                               "traffic": traffic_kernel.get(k), "alg_bytes": bytes_kernel[k] * ncell} for k in cand},
        })
        line = {
            "metric": (METRIC_F32 if f32 else METRIC).replace("at 128^3 viscous", {"config4": "on 256 x 201^2 batched 2+1d viscous events", "config5": "at 512x512x128 viscous"}.get(args.workload, "at 128^3 viscous")), "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": ms / K,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": args.precision, "data": "synthetic",
            "config": {"workload": ("SINGLE-PRECISION BUILD (labelled extra line, not the BASELINE.json metric, which is FP64): " if f32 else "") + ("REDUCED-STORAGE MODE (5 pi + 3 u components stored, 43 instead of 67 arrays; labelled extra line): " if args.storage else "") + ({"config4": "configs[3] (labelled extra line): 256 independent 2+1d events of 201x201 in one launch; physics of ", "config5": "configs[4] (labelled extra line): 512x512x128, 200 hotspots; physics of "}.get(args.workload, "")) + ("configs[2]: 128x128x128 3+1d viscous non-conformal (EOS 1, eta/s=0.2, Gaussian zeta/s), 40 seeded hotspots, "
                                    "dtau=0.025, one independent replica per GPU (no sharding, no collective)") if args.physics == "config3" else
                                   ("configs[2] grid and hotspots with the paper's own physics: lattice EOS (Eqs. 19-20), zeta/s of Eq. 17 (T_c = 200 MeV), "
                                    "eta/s=0.2; one independent replica per GPU"),
                       "l2": "state (%d padded arrays, %.2f GB) exceeds the 126 MB L2; no flush needed" % (43 if args.storage else 67, s_bytes / 1e9), "kernel_variant": args.variant,
                       "paper_context": "GTX 980 Ti, FP32, lattice EOS: 244.45 ms/step = 8.58e6 cell-updates/s (PAPER.md Table 3; another machine, not a target)"},
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": E,
                    "what": "per step: vh_set_initial(host e,u,pi,Pi) + vh_step(1) + vh_get_fields(host q,e,p,u), pinned buffers"},
            "gpu_launches": int(launches),
            "clocks": clocks,
            "roofline": roof,
            "status": {"n_inversion_failures": st["n_inversion_failures"], "n_nonfinite": st["n_nonfinite"], "min_reg_factor": st["min_reg_factor"]},
            "measured_peaks_same_run": {"copy_gbs": copy_gbs, "fp64_fma_gflops": fp64_gflops, "fp32_fma_gflops": fp32_gflops},
        }
        if paper_line is not None:
            line["paper_physics"] = paper_line
        if world == 1 and not args.no_cpu_baseline and not other:
            # SURVEY 8(d) "Oracle timing": the serial oracle on the FULL workload for 3 steps (about 40 s), 1 core, CPU model and core count stated
            v, dt, sample = time_oracle(prm, init, (prm["nx"], prm["ny"], prm["nz"]), 3)
            model, ncores = host_cpu()
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample, "seconds": dt, "host_cpu": model,
                                    "host_cores_total": ncores}
        print(json.dumps(line))
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
