#!/usr/bin/env python
"""bench.py -- ensemble member-steps/s of the CN/RK3 ensemble DNS step (arXiv 2306.12739) on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--form convective] [--impl reference]

One "step" = one dns_step(1): the whole hot path (3 RK stages x {z-FFT, fused x-line kernel, z-FFT, per-pair DMMA
kernel; the mean-flow kernel runs beside the last two on a side stream}: 15 launches) over the whole ensemble.  At N = 1
the workload is BASELINE.json configs[3] (Poiseuille at constant mass flux, 48 x 65 x 48, E = 256, fp64): BASELINE.json's
metric names no configuration, and this is the largest single-GPU workload of the five (the paper's C1/P1 x-z
resolution) -- `--config 2` gives configs[1].  For N > 1 (torchrun, one rank per GPU) every rank advances
its own E members (weak scaling; members are independent, no data-path collective -- SURVEY.md 8(e)).
Prints ONE JSON line on rank 0 (contract in the task statement): value = whole-job member-steps/s with the state
resident in HBM, in the paper's convective form of the nonlinear term; "rotational" = the same
measurement in the rotational form; e2e = through the C ABI with HOST buffers (H2D + step + D2H
every step); roofline = the dominant kernel against the measured HBM / fp64 peaks (the fp64 peak is measured live by
dns_debug_fp64_peak); cpu_baseline = the oracle on the host cores.
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
FP64_PEAK_FALLBACK = 37.0   # used only if the live microbenchmark fails (148 SMs x 64 FMA/clk x 2 x 1.965 GHz = 37.2)


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


def workload_counts(cfg, E, rot=False):
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
    if rot:   # 6 fields in and out of the z inverse, 6 in + 3 out of the line kernel (3 + 2 transforms), eta' as a 14th field
        return {
            "fft_z_inv": {"bytes": 6 * S + 6 * I, "flops": 6 * Ni * nkx * E * fz},
            "line_fft_x_products": {"bytes": 9 * I + Ni * Mz * E * 16.0, "flops": Ni * Mz * E * (5 * fx + 9.0 * Mx)},
            "fft_z_fwd": {"bytes": 3 * I + 3 * S, "flops": 3 * Ni * nkx * E * fz},
            "ypair_dmma": {"bytes": 14 * S + 3 * (Kh * Kh + Kho * Kho) * 8.0 * nmat + Ni * Mz * E * 16.0 + 12 * cfg.Ny * E * 8.0,
                           "flops": 7 * 2.0 * (Kh * Kh + Kho * Kho) * 2 * E * (P - 1)},
        }
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
    Es, nst = (min(16, cfg.E), 8) if cfg.Nx * cfg.Ny * cfg.Nz < 60000 else (min(8, cfg.E), 4)
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
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--config", type=int, default=4,
                    help="BASELINE.json config number (1-based); 4 = configs[3], the largest single-GPU workload")
    ap.add_argument("--form", default="both", choices=["both", "convective", "rotational"],
                    help="nonlinear term: the headline is the paper's convective form; 'both' adds the rotational "
                         "form (row f1) as a second measurement in the same line")
    ap.add_argument("--members", type=int, default=0, help="override E per GPU (config 5 sweep)")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true",
                    help="skip the threaded end-to-end measurement (for runs under ncu only: `e2e` is then null)")
    ap.add_argument("--opt", action="append", default=[], metavar="NAME=VALUE",
                    help="dns_debug_set_option before the plans are created (experiments, e.g. --opt line_96=1); "
                         "the options used are recorded in config.options")
    ap.add_argument("--no-extras", action="store_true",
                    help="skip the `other_configs` (configs 1-3 and the config-5 sweep, 20 steps each) and `rows` (linearised "
                         "ensemble, optimal-disturbance loop, coupled step, statistics) blocks of the default line")
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
    for o in args.opt:
        name, val = o.split("=", 1)
        if binding.dns_debug_set_option(name, int(val)) != binding.DNS_OK:
            raise SystemExit(f"unknown option {name}")
    base = inputs.CONFIGS[5 if args.sweep else args.config]
    sizes = list(inputs.SWEEP_E) if args.sweep else [args.members or base.E]
    hbm_peak, peak_src = measured_peaks()
    fp64 = {"dfma_tflops": None, "dmma_tflops": None, "mixed_dfma_dmma_tflops": None}
    for kind, key in ((0, "dfma_tflops"), (1, "dmma_tflops"), (2, "mixed_dfma_dmma_tflops")):
        st_, tf = binding.dns_debug_fp64_peak(kind, 0.4)
        if st_ == binding.DNS_OK:
            fp64[key] = tf
    fp64_peak = max([v for k, v in fp64.items() if v and k != "mixed_dfma_dmma_tflops"] or [FP64_PEAK_FALLBACK])
    fp64_src = ("fp64 %.1f TFLOP/s measured live (dns_debug_fp64_peak: DFMA %.1f, DMMA.8x8x4 %.1f; 0.4 s each)"
                % (fp64_peak, fp64["dfma_tflops"] or 0.0, fp64["dmma_tflops"] or 0.0)) if fp64["dfma_tflops"] \
        else "fp64 %.1f TFLOP/s fallback (units x clock)" % FP64_PEAK_FALLBACK

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def measure(cfg, cfg_all, st, rot, steps=None, warmup=None, coupling=None):
        """Device-resident timing of `steps` (default args.steps) steps + per-kernel-class durations, one form of the
        nonlinear term; coupling: dns_plan_set_coupling mode (row f2) or None."""
        steps = args.steps if steps is None else steps
        warmup = args.warmup if warmup is None else warmup
        plan = binding.Plan(*inputs.plan_args(cfg), device=f"cuda:{local}",
                            form=binding.DNS_FORM_ROTATIONAL if rot else binding.DNS_FORM_CONVECTIVE,
                            coupling=binding.DNS_COUPLING_NONE if coupling is None else coupling)
        plan.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
        stream = torch.cuda.current_stream()
        plan.step(warmup)
        barrier()
        sampler = ClockSampler(local)
        sampler.start()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record(stream)
        plan.step(steps)
        ev1.record(stream)
        barrier()
        ms = ev0.elapsed_time(ev1)
        clocks = sampler.stop()
        ms_max = shard.max_over_ranks(ms) if world > 1 else ms
        value = cfg_all.E * steps / (ms_max * 1e-3)
        # per-kernel-class durations with CUDA events on the same stream (live, same state)
        nprof = min(max(steps // 10, 3), 20)
        prof = plan.step_profile(nprof)
        counts = workload_counts(cfg, cfg.E, rot)
        kernels = {}
        for name, msum in prof.items():
            per_launch_s = msum * 1e-3 / (3 * nprof)
            c = counts[name]
            t_hbm, t_alu = c["bytes"] / (hbm_peak * 1e9), c["flops"] / (fp64_peak * 1e12)
            kernels[name] = {"us_per_launch": per_launch_s * 1e6, "share": msum / max(sum(prof.values()), 1e-30),
                             "GBps": c["bytes"] / per_launch_s * 1e-9, "TFLOPs": c["flops"] / per_launch_s * 1e-12,
                             "alg_bytes_per_launch": c["bytes"], "alg_flops_per_launch": c["flops"],
                             "bound": "hbm" if t_hbm >= t_alu else "fp64",
                             "frac": max(t_hbm, t_alu) / per_launch_s,
                             "traffic": traffic_lookup(name, cfg, rot)[0]}
        return plan, value, ms_max, clocks, kernels

    ncu_extra = {}

    def traffic_lookup(kernel, cfg, rot):
        """DRAM bytes per launch of one kernel class from the committed ncu capture of the same workload and form
        (profiles/dominant_kernel_traffic.csv, copied from `ncu --set full` reports; see profiles/r2k_kernels.md)."""
        tpath = os.path.join(ROOT, "profiles", "dominant_kernel_traffic.csv")
        try:
            import csv
            for rec in csv.DictReader(open(tpath)):
                if rec.get("kernel") == kernel and rec.get("workload") == cfg.name and \
                        rec.get("form", "convective") == ("rotational" if rot else "convective"):
                    ncu_extra[(kernel, rot)] = float(rec.get("fp64_pipe_active_pct") or 0.0)
                    return float(rec["dram_bytes_per_launch"]), rec.get("source")
        except Exception:
            pass
        return None, None

    def roofline_of(kernels, cfg, rot):
        dom = max(kernels, key=lambda k: kernels[k]["share"])
        kd = kernels[dom]
        traffic, tsrc = traffic_lookup(dom, cfg, rot)
        if kd["bound"] == "hbm":
            r = {"bound": "hbm", "achieved": kd["GBps"], "peak": hbm_peak, "unit": "GB/s", "frac": kd["GBps"] / hbm_peak}
        else:
            r = {"bound": "tensor" if dom == "ypair_dmma" else "alu", "achieved": kd["TFLOPs"], "peak": fp64_peak,
                 "unit": "TFLOP/s", "frac": kd["TFLOPs"] / fp64_peak}
        # context from the same ncu capture: how busy the fp64 pipe was (the line kernel is bound by fp64 instruction issue,
        # DESIGN.md sections 5 and 7; DFMA and DMMA share that pipe)
        r["fp64_pipe_active_pct_ncu"] = ncu_extra.get((dom, rot))
        r.update({"traffic": traffic, "traffic_source": tsrc, "kernel": dom, "peak_source": peak_src + "; " + fp64_src,
                  "alg_bytes_per_launch": kd["alg_bytes_per_launch"], "us_per_launch": kd["us_per_launch"],
                  "share_of_step": kd["share"]})
        return r

    def measure_e2e(cfg, cfg_all, st, nchunk):
        """End to end through the C ABI with HOST (pinned) buffers, every step: dns_set_state(host) + dns_step(1) +
        dns_get_state(host).  Members are independent, so the ensemble is cut into `nchunk` plans on
        their own streams, each driven by its own host thread: the copies of one chunk overlap the step of another."""
        import concurrent.futures as cf
        bounds = [shard.member_range(cfg.E, c, nchunk) for c in range(nchunk)]
        bounds = [b for b in bounds if len(b)]
        work = []
        for b in bounds:
            sl = slice(b.start, b.stop)
            strm = torch.cuda.Stream(device=local)
            with torch.cuda.stream(strm):
                pl = binding.Plan(*inputs.plan_args(cfg.with_E(len(b))), device=f"cuda:{local}")
            pin = [torch.from_numpy(np.ascontiguousarray(st[k][sl])).pin_memory() for k in ("vhat", "etahat", "U00", "W00")]
            outs = [torch.empty_like(t).pin_memory() for t in pin]
            work.append((pl, pin, outs))
        h2d = sum(t.numel() * t.element_size() for _, pin, _ in work for t in pin)
        d2h = sum(t.numel() * t.element_size() for _, _, outs in work for t in outs)
        ne2e = max(3, min(args.steps, 10))

        def drive(w, n):
            torch.cuda.set_device(local)
            pl, pin, outs = w
            for _ in range(n):
                pl.set_state(*pin)
                pl.step(1)
                pl.get_state(outs)

        with cf.ThreadPoolExecutor(len(work)) as ex:
            list(ex.map(lambda w: drive(w, 2), work))
            barrier()
            t0 = time.perf_counter()
            list(ex.map(lambda w: drive(w, ne2e), work))
            barrier()
            e2e_s = time.perf_counter() - t0
        for pl, _, _ in work:
            pl.close()
        e2e_s = shard.max_over_ranks(e2e_s) if world > 1 else e2e_s
        return {"value": cfg_all.E * ne2e / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "steps": ne2e, "chunks": len(work),
                "note": "dns_set_state(host pinned) + dns_step(1) + dns_get_state(host pinned) per step and member chunk; "
                        "%d chunks of members on their own plans, streams and host threads" % len(work)}

    def other_configs():
        """The other BASELINE configs and the config-5 sweep in short form (north_star: "all five configs"): 20 timed steps
        each after 5 warm-up steps, convective form, same timing and per-class fractions as the headline."""
        out = []
        todo = [(f"config{c}", inputs.CONFIGS[c]) for c in (1, 2, 3) if c != args.config]
        todo += [(f"config5_E{E}", inputs.CONFIGS[5].with_E(E)) for E in inputs.SWEEP_E]
        for tag, c in todo:
            st_ = inputs.make_state(c)
            plan, value, ms_max, _, kernels = measure(c, c, st_, False, steps=20, warmup=5)
            out.append({"tag": tag, "workload": c.name, "value": value, "unit": UNIT, "ms_per_step": ms_max / 20,
                        "steps": 20, "launches_per_step": plan.launches_per_step(), "workspace_MB": plan.workspace_bytes / 1e6,
                        "frac": {k: round(v["frac"], 4) for k, v in kernels.items()},
                        "us_per_launch": {k: round(v["us_per_launch"], 2) for k, v in kernels.items()}})
            plan.close()
        return out

    def timed(fn, stream):
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        ev0.record(stream)
        fn()
        ev1.record(stream)
        torch.cuda.synchronize()
        return ev0.elapsed_time(ev1)

    def rows_block(cfg4, st4, base_value):
        """One device-timed measurement for each SURVEY.md 8(f) row that is not the headline: the linearised forward /
        adjoint ensemble at the paper's size (48 x 65 x 48, 45 disturbances, t_f = 5), one
        optimal-disturbance loop, the coupled ensemble's cost over the uncoupled step, and dns_stats_accumulate."""
        stream = torch.cuda.current_stream()
        rows = {}
        c2 = cfg4.with_E(2)
        s2 = inputs.make_state(c2)
        dns = binding.Plan(*inputs.plan_args(c2), device=f"cuda:{local}")
        dns.set_state(s2["vhat"], s2["etahat"], s2["U00"], s2["W00"])
        n_list, Eg = [1, 2, 3], 15
        lin = binding.LinPlan(c2.Nx, c2.Ny, c2.Nz, n_list, Eg, c2.Re, c2.Lx, c2.Lz, 5 * c2.dt, device=f"cuda:{local}")
        lin.set_base(dns, 1)
        pert = inputs.make_broadband_state(c2.with_E(lin.E), range(20, 20 + lin.E))
        lin.set_state(np.stack([pert["vhat"][e, n_list[e // Eg]] for e in range(lin.E)]),
                      np.stack([pert["etahat"][e, n_list[e // Eg]] for e in range(lin.E)]))
        lin.orthonormalise()
        # algorithmic bytes of one linear stage: z inverse 5 S + 8 I, pointwise vector 8 I + 3 I, z forward 3 I + 3 S,
        # per-pair kernel 13 S + the matrices of the 3 kx rows; S, I = one spectral / mixed field with ONE kx row
        Ni, nkz, Mz = c2.Ny - 2, c2.Nz - 1, 3 * c2.Nz // 2
        S, I = Ni * nkz * 16.0 * lin.E, Ni * Mz * 16.0 * lin.E
        Kh, Kho = (Ni + 1) // 2, Ni // 2
        mats = 3 * (Kh * Kh + Kho * Kho) * 8.0 * len(n_list) * (c2.Nz // 2)
        stage_bytes = 21 * S + 22 * I + mats
        nlin = 50
        for adj, tag in ((False, "lin_step_forward"), (True, "lin_step_adjoint")):
            lin.step(5, adj)
            ms = timed(lambda: lin.step(nlin, adj), stream)
            rows[tag] = {"value": lin.E * nlin / (ms * 1e-3), "unit": UNIT, "ms_per_step": ms / nlin, "members": lin.E,
                         "launches_per_step": binding.dns_lin_launches_per_step(lin.h),
                         "alg_bytes_per_step": 3 * stage_bytes, "GBps": 3 * stage_bytes * nlin / (ms * 1e-3) * 1e-9,
                         "frac_hbm": 3 * stage_bytes * nlin / (ms * 1e-3) * 1e-9 / hbm_peak,
                         "workload": f"{c2.Nx}x{c2.Ny}x{c2.Nz}, kx modes {n_list} x {Eg} disturbances, dt_lin = 5 dt"}
            lin.orthonormalise()
        nopt, niter = 20, 2
        lin.optimals(2, 1)
        t0 = time.perf_counter()
        gains = lin.optimals(nopt, niter)                     # synchronises at its end
        wall = time.perf_counter() - t0
        rows["lin_optimals"] = {"ms": wall * 1e3, "nsteps": nopt, "niter": niter,
                                "lin_steps_total": 2 * nopt * niter, "ms_per_lin_step": wall * 1e3 / (2 * nopt * niter),
                                "max_gain": float(np.max(gains)),
                                "note": "orthonormalise + niter x (nsteps forward, energies, nsteps adjoint, orthonormalise)"}
        ms = timed(lambda: [lin.orthonormalise() for _ in range(10)], stream)
        rows["lin_orthonormalise"] = {"ms": ms / 10, "members": lin.E, "groups": len(n_list)}
        lin.close()
        dns.close()
        # coupled ensemble (row f2) on the headline workload: the same 20 steps with dns_plan_set_coupling
        plan, value, ms_max, _, _ = measure(cfg4, cfg4, st4, False, steps=20, warmup=5,
                                            coupling=binding.DNS_COUPLING_STREAMWISE_MEAN)
        rows["coupled_step"] = {"value": value, "unit": UNIT, "ms_per_step": ms_max / 20,
                                "launches_per_step": plan.launches_per_step(),
                                "cost_over_uncoupled": base_value / value - 1.0, "workload": cfg4.name}
        # one-point statistics (row f4) of the same plan's state: reads u, v, w of every member once
        plan.stats_reset()
        plan.stats_accumulate()
        ms = timed(lambda: [plan.stats_accumulate() for _ in range(20)], stream)
        P = (cfg4.Nx // 2) * (cfg4.Nz - 1)
        sb = 3 * cfg4.Ny * P * 16.0 * cfg4.E
        rows["stats_accumulate"] = {"us_per_call": ms * 1e3 / 20, "alg_bytes_per_call": sb,
                                    "GBps": sb / (ms * 1e-3 / 20) * 1e-9, "frac_hbm": sb / (ms * 1e-3 / 20) * 1e-9 / hbm_peak}
        plan.close()
        return rows

    for E_gpu in sizes:
        if args.sweep:
            args.steps, args.warmup = 50, 5                  # BASELINE config 5: 50 steps per ensemble size
        cfg_all = base.with_E(E_gpu * world)                 # weak scaling: E_gpu members on every rank
        mine = shard.member_range(cfg_all.E, rank, world)
        cfg = base.with_E(len(mine))
        st = inputs.make_state(cfg_all, mine)
        forms = {"both": (False, True), "convective": (False,), "rotational": (True,)}[args.form]
        if args.sweep:
            forms = forms[:1]
        res = {}
        for rot in forms:
            plan, value, ms_max, clocks, kernels = measure(cfg, cfg_all, st, rot)
            res[rot] = dict(value=value, ms_max=ms_max, clocks=clocks, kernels=kernels, launches=plan.launches_per_step(),
                            ws=plan.workspace_bytes, roofline=roofline_of(kernels, cfg, rot))
            plan.close()
        head = res[forms[0]]
        e2e = None if args.no_e2e else measure_e2e(cfg, cfg_all, st, 1 if (args.sweep or cfg.E < 8) else 4)

        line = {
            "metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": head["ms_max"] / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg.name, "members_per_gpu": cfg.E, "members_total": cfg_all.E,
                       "nonlinear_form": "rotational" if forms[0] else "convective (PAPER.md:147)",
                       "parallelism": f"member-shards x{world} (no collective in dns_step)",
                       "l2_policy": "working set %.0f MB per GPU > 126 MB L2 (no flush needed)" % (head["ws"] / 1e6)
                       if head["ws"] > 2 * 126e6 else "working set fits L2; not flushed between steps (stated)",
                       "input_sha256": st["sha256"][:16], **({"options": args.opt} if args.opt else {})},
            "clocks": head["clocks"], "e2e": e2e, "gpu_launches": args.steps * head["launches"],
            "roofline": head["roofline"], "kernels": head["kernels"], "fp64_peak": fp64,
        }
        if len(forms) > 1:
            r = res[True]
            line["rotational"] = {"value": r["value"], "unit": UNIT, "ms_per_step": r["ms_max"] / args.steps,
                                  "clocks": r["clocks"], "roofline": r["roofline"], "kernels": r["kernels"],
                                  "note": "same workload, steps and timing with dns_plan_set_form(DNS_FORM_ROTATIONAL), "
                                          "SURVEY.md 8(f) row f1"}
        if world == 1 and not args.sweep and not args.no_extras and args.config == 4 and not args.members and not args.opt:
            try:
                line["other_configs"] = other_configs()
                line["rows"] = rows_block(cfg, st, head["value"])
            except Exception as exc:                              # the headline line must still be printed
                line["extras_error"] = repr(exc)
        if rank == 0 and world == 1 and not args.no_cpu_baseline and not args.sweep:
            line["cpu_baseline"] = cpu_baseline(base)
        if rank == 0:
            print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
