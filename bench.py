#!/usr/bin/env python
"""bench.py -- ensemble member-steps/s of the CN/RK3 ensemble DNS step (arXiv 2306.12739) on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--impl reference]

One "step" = one dns_step(1): the whole hot path (3 RK stages x {z-FFT, fused x-line kernel, z-FFT, per-pair DMMA
kernel; the mean-flow kernel runs beside the last two on a side stream}: 15 launches) over the whole ensemble.  At N = 1 the workload is BASELINE.json configs[1]
(plane Couette, Re = 1000, 32 x 49 x 32, E = 64, fp64).  For N > 1 (torchrun, one rank per GPU) every rank advances
its own 64 members (weak scaling; members are independent, no data-path collective -- SURVEY.md 8(e)).
Prints ONE JSON line on rank 0 (contract in the task statement): value = whole-job member-steps/s with the state
resident in HBM; e2e = the same through the C ABI with HOST buffers (H2D + step + D2H every step);
roofline = the dominant kernel against the measured HBM / fp64 peaks; cpu_baseline = the oracle on the host cores.
`--impl reference` times the oracle (oracle/dns_oracle.py) alone, as it stands, on a bounded sample.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2306_12739_b200 import inputs  # noqa: E402

METRIC = "ensemble member-steps/s (fp64, device-timed)"
UNIT = "member-steps/s"
FP64_PEAK_TFLOPS = 37.0   # measured on this pool's B200: DMMA.8x8x4 and DFMA both 37.0 TFLOP/s


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons with NVML while the timed region runs."""

    def __init__(self, index=0, period=0.05):
        super().__init__(daemon=True)
        self.period, self.index = period, index
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._halt = threading.Event()
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
        }
        while not self._halt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self):
        self._halt.set()
        self.join(timeout=2)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def workload_counts(cfg, E):
    """Algorithmic bytes / flops per kernel class per STAGE for E members."""
    Ni, P = cfg.Ny - 2, (cfg.Nx // 2) * (cfg.Nz - 1)
    Mx, Mz, nkx, nkz = 3 * cfg.Nx // 2, 3 * cfg.Nz // 2, cfg.Nx // 2, cfg.Nz - 1
    S = Ni * P * 16.0 * E                       # one spectral field, interior rows (bytes)
    I = Ni * Mz * nkx * 16.0 * E                # one mixed (kx, z) field
    lg = np.log2
    fz = 5.0 * Mz * lg(Mz)                      # flops of one complex length-Mz FFT
    fx = 5.0 * Mx * lg(Mx)
    nmat = nkx * (cfg.Nz // 2) - 1
    Kh, Kho = (Ni + 1) // 2, Ni // 2
    return {
        "fft_z_inv": {"bytes": 5 * S + 8 * I, "flops": 8 * Ni * nkx * E * fz},
        "line_fft_x_products": {"bytes": 11 * I + Ni * Mz * E * 16.0, "flops": Ni * Mz * E * (8 * fx + 15.0 * Mx)},
        "fft_z_fwd": {"bytes": 3 * I + 3 * S, "flops": 3 * Ni * nkx * E * fz},
        # reads Nu,Nv,Nw,v_t,eta_t (+ F,G history), writes v', u, w, du, dw (+ history / eta): ~13 fields, plus the
        # parity-folded matrices (3 per pair, half size); flops of the 7 products in the reflection-parity basis.
        # The mean flow (row a10) runs on a side stream under this class's events: its bytes are added here.
        "ypair_dmma": {"bytes": 13 * S + 3 * (Kh * Kh + Kho * Kho) * 8.0 * nmat + Ni * Mz * E * 16.0 + 12 * cfg.Ny * E * 8.0,
                       "flops": 7 * 2.0 * (Kh * Kh + Kho * Kho) * 2 * E * (P - 1)},
    }


def run_reference(args):
    """--impl reference: the oracle alone, as it stands, on the host cores (bounded sample per step)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from oracle.dns_oracle import Oracle
    cfg = inputs.CONFIGS[args.config]
    total = args.steps + args.warmup
    Es = 8 if total <= 30 else (2 if total <= 120 else 1)
    Es = min(Es, cfg.E)
    o = Oracle(*inputs.plan_args(cfg, E=Es))
    st = inputs.make_state(cfg, range(Es))
    o.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
    o.step(args.warmup)
    t0 = time.perf_counter()
    o.step(args.steps)
    dt = time.perf_counter() - t0
    val = Es * args.steps / dt
    cores = _blas_threads()
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(args.steps, 1), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "sample": f"{Es} of {cfg.E} members per step", "device": "host CPU"},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"{Es} members x {args.steps} steps of {cfg.name}"},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def _blas_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [i.get("num_threads", 1) for i in threadpool_info()]
        return int(max(n)) if n else os.cpu_count()
    except Exception:
        return os.cpu_count()


def cpu_baseline(cfg):
    """The oracle as it stands on the host cores: a bounded sample (about 10-30 s) of the bench workload."""
    from oracle.dns_oracle import Oracle
    Es, nst = min(16, cfg.E), 8
    o = Oracle(*inputs.plan_args(cfg, E=Es))
    st = inputs.make_state(cfg, range(Es))
    o.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
    t0 = time.perf_counter()
    o.step(nst)
    dt = time.perf_counter() - t0
    return {"value": Es * nst / dt, "unit": UNIT, "cores": _blas_threads(), "kind": "oracle",
            "sample": f"{Es} members x {nst} steps of {cfg.name} ({dt:.1f} s)"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config number (1-based); 2 = configs[1]")
    ap.add_argument("--members", type=int, default=0, help="override E per GPU (config 5 sweep)")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sweep", action="store_true",
                    help="BASELINE config 5: one JSON line per ensemble size E in inputs.SWEEP_E (per-kernel times and "
                         "roofline fractions versus E); not the default bench line")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "b200":
        args.warmup = 3
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    from paper_2306_12739_b200 import binding, shard

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the library has no CPU path")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    base = inputs.CONFIGS[5 if args.sweep else args.config]
    sizes = list(inputs.SWEEP_E) if args.sweep else [args.members or base.E]
    for E_gpu in sizes:
        if args.sweep:
            args.steps, args.warmup = 50, 5                  # BASELINE config 5: 50 steps per ensemble size
        cfg_all = base.with_E(E_gpu * world)                 # weak scaling: E_gpu members on every rank
        mine = shard.member_range(cfg_all.E, rank, world)
        cfg = base.with_E(len(mine))
        plan = binding.Plan(*inputs.plan_args(cfg), device=f"cuda:{local}")
        st = inputs.make_state(cfg_all, mine)
        plan.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
        stream = torch.cuda.current_stream()

        def barrier():
            if world > 1:
                dist.barrier()
            torch.cuda.synchronize()

        # ---- device-resident timing: W warm-up steps, then exactly K steps between two events
        plan.step(args.warmup)
        barrier()
        sampler = ClockSampler(local)
        sampler.start()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record(stream)
        plan.step(args.steps)
        ev1.record(stream)
        barrier()
        ms = ev0.elapsed_time(ev1)
        clocks = sampler.stop()
        ms_max = shard.max_over_ranks(ms) if world > 1 else ms
        value = cfg_all.E * args.steps / (ms_max * 1e-3)

        # ---- per-kernel-class durations with CUDA events on the same stream (live, same state)
        nprof = min(max(args.steps // 10, 3), 20)
        prof = plan.step_profile(nprof)
        counts = workload_counts(cfg, cfg.E)
        hbm_peak, peak_src = measured_peaks()
        kernels = {}
        for name, msum in prof.items():
            per_launch_s = msum * 1e-3 / (3 * nprof)
            c = counts[name]
            t_hbm, t_alu = c["bytes"] / (hbm_peak * 1e9), c["flops"] / (FP64_PEAK_TFLOPS * 1e12)
            kernels[name] = {"us_per_launch": per_launch_s * 1e6, "share": msum / max(sum(prof.values()), 1e-30),
                             "GBps": c["bytes"] / per_launch_s * 1e-9, "TFLOPs": c["flops"] / per_launch_s * 1e-12,
                             "bound": "hbm" if t_hbm >= t_alu else "fp64",
                             "frac": max(t_hbm, t_alu) / per_launch_s}
        dom = max(kernels, key=lambda k: kernels[k]["share"])
        kd = kernels[dom]
        traffic = None
        tpath = os.path.join(ROOT, "profiles", "dominant_kernel_traffic.json")
        if os.path.exists(tpath):
            try:
                tj = json.load(open(tpath))
                if tj.get("kernel") == dom and tj.get("workload") == cfg.name:
                    traffic = tj.get("dram_bytes_per_launch")
            except Exception:
                traffic = None
        if kd["bound"] == "hbm":
            roofline = {"bound": "hbm", "achieved": kd["GBps"], "peak": hbm_peak, "unit": "GB/s",
                        "frac": kd["GBps"] / hbm_peak, "traffic": traffic}
        else:
            roofline = {"bound": "tensor" if dom == "ypair_dmma" else "alu", "achieved": kd["TFLOPs"],
                        "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": kd["TFLOPs"] / FP64_PEAK_TFLOPS,
                        "traffic": traffic}
        roofline.update({"kernel": dom, "peak_source": peak_src + "; fp64 37.0 TFLOP/s measured DMMA/DFMA microbenchmark",
                         "us_per_launch": kd["us_per_launch"], "share_of_step": kd["share"]})

        # ---- end to end through the C ABI with HOST (pinned) buffers: H2D + step + D2H every step
        pin = [torch.from_numpy(np.ascontiguousarray(st[k])).pin_memory() for k in ("vhat", "etahat", "U00", "W00")]
        outs = [torch.empty_like(t).pin_memory() for t in pin]
        h2d = sum(t.numel() * t.element_size() for t in pin)
        d2h = sum(t.numel() * t.element_size() for t in outs)
        ne2e = min(args.steps, 20)
        for _ in range(2):
            plan.set_state(*pin)
            plan.step(1)
            plan.get_state(outs)
        barrier()
        t0 = time.perf_counter()
        for _ in range(ne2e):
            plan.set_state(*pin)
            plan.step(1)
            plan.get_state(outs)
        barrier()
        e2e_s = time.perf_counter() - t0
        e2e_s = shard.max_over_ranks(e2e_s) if world > 1 else e2e_s
        e2e = {"value": cfg_all.E * ne2e / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "steps": ne2e, "note": "dns_set_state(host pinned) + dns_step(1) + dns_get_state(host pinned) per step"}

        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg.name, "members_per_gpu": cfg.E, "members_total": cfg_all.E,
                       "parallelism": f"member-shards x{world} (no collective in dns_step)",
                       "l2_policy": "working set %.0f MB per GPU > 126 MB L2 (no flush needed)" % (plan.workspace_bytes / 1e6)
                       if plan.workspace_bytes > 2 * 126e6 else "working set fits L2; not flushed between steps (stated)",
                       "input_sha256": st["sha256"][:16]},
            "clocks": clocks, "e2e": e2e, "gpu_launches": args.steps * plan.launches_per_step(),
            "roofline": roofline, "kernels": kernels,
        }
        if rank == 0 and world == 1 and not args.no_cpu_baseline and not args.sweep:
            line["cpu_baseline"] = cpu_baseline(base)
        plan.close()
        if rank == 0:
            print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
