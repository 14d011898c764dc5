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
UNIT = "cell-updates/s"
ALG_BYTES_PER_CELL_UPDATE = 856.0      # 107 doubles per cell-update, each state array read/written once per stage
ALG_BYTES_STAGE = {"stage1": (25 + 21) * 8.0, "stage2": (40 + 21) * 8.0}
# dram__bytes_read.sum + dram__bytes_write.sum of one launch of the stage kernel at 128^3 from the committed ncu --set full
# capture (profiles/r01c_ncu_summary.md); valid for the default workload (128^3) only
NCU_TRAFFIC_BYTES = {"stage1": 629327104 + 353338112, "stage2": 932169216 + 358881024}      # profiles/r01c_ncu_summary.md


def workload(rank=0, physics="config3"):
    """configs[2] of BASELINE.json (default); physics="paper": the same grid and hotspots with the paper's own equation of state
    (lattice, Eqs. 19-20) and zeta/s(T) (Eq. 17, T_c = 200 MeV) - SURVEY 8(f) NEXT-1 - for a second, labelled bench line."""
    over = dict(eos=2, zeta_model=3, zeta_amp=1.0, zeta_T0=0.2 / inputs.HBARC) if physics == "paper" else {}
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
    z0, y0, x0 = (prm["nz"] - nz) // 2, (prm["ny"] - ny) // 2, (prm["nx"] - nx) // 2
    cut = lambda a: np.ascontiguousarray(a[..., z0:z0 + nz, y0:y0 + ny, x0:x0 + nx])
    sub = dict(prm, nx=nx, ny=ny, nz=nz)
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
    return ncell * steps / dt, dt, "central %dx%dx%d cut-out of the 128^3 initial data, %d RK2 step(s), serial C++ oracle -O2" % (dims[0], dims[1], dims[2], steps)


def algorithmic_flops(prm, init):
    """Measured algorithmic flop count per cell-update (oracle with an operation-counting scalar on a 16^3 cut-out, every
    interface charged once; weights of SURVEY.md 8(d)).  Test infrastructure used for the report only."""
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import vh_oracle

    sub, e, u = oracle_sample(prm, init, 16, 16, 16)
    flops, plain, per = vh_oracle.algorithmic_flops_per_cell_update(sub, e, u)
    return flops, plain, per


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    prm, init = workload(0, args.physics)
    dims = (64, 64, 32)
    warm = min(args.warmup, 1)
    value, dt, sample = time_oracle(prm, init, dims, args.steps, warmup=warm)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": warm,
        "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": "configs[2]: 128^3 3+1d viscous non-conformal, seeded hotspots; bounded sample " + sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
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

    prm, init = workload(rank, args.physics)
    ncell = prm["nx"] * prm["ny"] * prm["nz"] * prm["n_batch"]
    s = vh.Solver(prm, device=dev)
    if args.variant:
        s.set_kernel_variant(args.variant)
    e_d = torch.as_tensor(init["e"], device=dev)
    u_d = torch.as_tensor(init["u"], device=dev)
    s.set_initial(e_d, u_d)

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

    # ---------------- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
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
    E = max(1, args.e2e_steps)
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
    s.close()

    if rank == 0:
        peaks_file = os.path.join(ROOT, "MEASURED_PEAKS.json")
        hbm_peak, hbm_src = 6650.0, "fallback (B200_PROFILING.md)"
        if os.path.exists(peaks_file):
            try:
                hbm_peak, hbm_src = float(json.load(open(peaks_file))["hbm_gbs"]), "MEASURED_PEAKS.json"
            except Exception:
                pass
        flops_cu, plain_cu, mix = algorithmic_flops(prm, init)
        flops_inv_cu = mix.pop("flops_interface_inversions")
        # Kernel shares of the algorithmic work: the velocity kernel does the interface-state inversions
        # (Eq. 72 at every reconstructed state), the stage kernel everything else; one stage = half of a cell-update.
        variant1 = (args.variant == 1)
        stage_keys = ("stage1", "stage2")
        dom = max(stage_keys, key=lambda k: prof[k])            # dominant kernel: the longer of the two stage-kernel launches
        dur = prof[dom] * 1e-3
        flops_stage = 0.5 * (flops_cu if variant1 else flops_cu - flops_inv_cu)
        flops_launch = flops_stage * ncell
        # algorithmic bytes of the stage kernel: the state arrays of SURVEY 8(d) (each read / written once per stage) plus,
        # in the split pipeline, the six state velocities it reads back (they are a by-product, not state: not counted)
        bytes_launch = ALG_BYTES_STAGE[dom] * ncell
        t_alu = flops_launch / (fp64_gflops * 1e9)
        t_hbm = bytes_launch / (hbm_peak * 1e9)
        if t_alu >= t_hbm:
            roof = {"bound": "alu", "achieved": flops_launch / dur / 1e12, "peak": fp64_gflops / 1e3, "unit": "TFLOP/s"}
        else:
            roof = {"bound": "hbm", "achieved": bytes_launch / dur / 1e9, "peak": hbm_peak, "unit": "GB/s"}
        roof["frac"] = roof["achieved"] / roof["peak"]
        step_roof_s = max(flops_cu * ncell / (fp64_gflops * 1e9), ALG_BYTES_PER_CELL_UPDATE * ncell / (hbm_peak * 1e9))
        roof.update({
            "traffic": NCU_TRAFFIC_BYTES.get(dom) if (ncell == 128 ** 3 and not args.variant and args.physics == "config3") else None, "kernel": "stage_tile_kernel (%s)" % dom if not variant1 else "stage_cell_kernel (%s)" % dom,
            "launch_ms": prof[dom],
            "peak_source": "FP64 FMA microbenchmark, same run (vh_measure_peaks)" if roof["bound"] == "alu" else hbm_src,
            "alg_flops_per_cell_update": flops_cu, "alg_flops_interface_inversions_per_cell_update": flops_inv_cu,
            "alg_flops_this_kernel_per_cell": flops_stage, "alg_bytes_per_cell_update": ALG_BYTES_PER_CELL_UPDATE,
            "alg_bytes_this_kernel_per_cell": ALG_BYTES_STAGE[dom],
            "flop_weights": "add/mul/cmp 1, div 10, sqrt 15, exp 25, pow 30, tanh 40 (SURVEY 8(d)); counted on the oracle, each interface once",
            "op_mix_per_cell_update": {k: round(v, 1) for k, v in mix.items()},
            "hbm_view": {"achieved_gbs": bytes_launch / dur / 1e9, "peak_gbs": hbm_peak, "peak_source": hbm_src, "frac": bytes_launch / dur / 1e9 / hbm_peak,
                         "copy_gbs_same_run": copy_gbs},
            "step_roofline_ms": step_roof_s * 1e3, "step_frac": step_roof_s / (ms / K * 1e-3),
            "per_kernel_ms": prof,
        })
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": ms / K,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": ("configs[2]: 128x128x128 3+1d viscous non-conformal (EOS 1, eta/s=0.2, Gaussian zeta/s), 40 seeded hotspots, "
                                    "dtau=0.025, one independent replica per GPU (no sharding, no collective)") if args.physics == "config3" else
                                   ("configs[2] grid and hotspots with the paper's own physics: lattice EOS (Eqs. 19-20), zeta/s of Eq. 17 (T_c = 200 MeV), "
                                    "eta/s=0.2; one independent replica per GPU"),
                       "l2": "state (61 arrays, 1.34 GB) exceeds the 126 MB L2; no flush needed", "kernel_variant": args.variant,
                       "paper_context": "GTX 980 Ti, FP32, lattice EOS: 244.45 ms/step = 8.58e6 cell-updates/s (PAPER.md Table 3; another machine, not a target)"},
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": E,
                    "what": "per step: vh_set_initial(host e,u,pi,Pi) + vh_step(1) + vh_get_fields(host q,e,p,u), pinned buffers"},
            "gpu_launches": int(launches),
            "clocks": clocks,
            "roofline": roof,
            "status": {"n_inversion_failures": st["n_inversion_failures"], "n_nonfinite": st["n_nonfinite"], "min_reg_factor": st["min_reg_factor"]},
            "measured_peaks_same_run": {"copy_gbs": copy_gbs, "fp64_fma_gflops": fp64_gflops},
        }
        if world == 1 and not args.no_cpu_baseline:
            v, dt, sample = time_oracle(prm, init, (96, 96, 64), 2)
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample, "seconds": dt}
        print(json.dumps(line))
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
