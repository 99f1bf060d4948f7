#!/usr/bin/env python
"""bench.py -- throughput of the EMRI_MC hot path on B200 (contract: see DESIGN.md section 8).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config i] [--impl reference]

A "step" is one pass of the whole hot path -- emri_loglike: orbit RK4 (a), synthesis (b), cuFFT Z2Z
(c: one complex transform per walker carries both channels), likelihood reduction (d) -- over one ensemble of K walkers of BASELINE.json:configs[i]
(default i = 1: K=64, N=2^20, n_max=10).  Inputs are synthetic and seeded (workloads.py).  Prints ONE
JSON line.  `value` = walker*samples/s with inputs resident in HBM; `e2e` = the same through
emri_loglike_host with pinned HOST buffers (copies inside the timed region).  With N > 1 (torchrun)
every rank runs its own K walkers (the path shards by walker, no data-path collective): weak scaling.

`--impl reference` times the CPU oracle (oracle/, test infrastructure) on the host cores instead.
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

from paper_2311_17174_b200 import workloads as W  # noqa: E402

METRIC = "AK waveform+logL evaluations/sec (walkers x samples/s)"
UNIT = "walker*samples/s"
ORBIT_KERNELS = 10          # orbit_init, 3 x (orbit_sweep, orbit_correct), orbit_tail, orbit_fixup, orbit_aux
CHUNK = 128                 # walkers per synth / cuFFT / loglike launch (emri_plan_set_chunk default)

# Algorithmic work of synth_kernel per (walker, sample): FP64 flops EXECUTED by the kernel as it stands, counted
# by ncu (2 dfma + dmul + dadd, smsp__sass_thread_inst_executed_op_*_pred_on.sum) on the configs' own inputs:
# profiles/counts_r1.md.  SURVEY 8(d)-2 asks for counted instructions in place of its estimate 600 + 170 n_max
# (2300 at n_max = 10), which the re-summed harmonic series undercuts by 3.7x.
COUNTED_FLOPS = {5: 546.0, 10: 619.0, 20: 921.0, 30: 1213.0}
# DRAM bytes of one synth_kernel launch (dram__bytes_read.sum + dram__bytes_write.sum, same ncu pass)
SYNTH_TRAFFIC = {0: 415488.0, 1: 1073785088.0, 2: 4438271488.0, 3: 4444701696.0}


def counted_flops_per_walker_sample(n_max):
    ks = sorted(COUNTED_FLOPS)
    return float(np.interp(n_max, ks, [COUNTED_FLOPS[k] for k in ks]))


def load_measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f), "measured"
    except Exception:
        return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """samples SM clock and throttle reasons through NVML while the timed region runs"""

    def __init__(self, index):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._nv = None

    def _run(self):
        nv = self._nv
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40,
                 "hw_power_brake_slowdown": 0x80, "sync_boost": 0x10}
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self._h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop.wait(0.02)

    def start(self):
        if self._nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()

    def stop(self):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def host_cores():
    try:
        return len(os.sched_getaffinity(0))
    except Exception:
        return os.cpu_count() or 1


def oracle_sample(cfg, P, walkers, stride, with_likelihood):
    """Time the oracle, as it stands, on `walkers` walkers (one per thread), every `stride`-th sample.
    Returns (seconds, walker*samples processed)."""
    from concurrent.futures import ThreadPoolExecutor
    from oracle.oracle import Oracle
    orc = Oracle()
    orc.set_anchor(cfg.index == 5)
    idx = None if stride == 1 else np.arange(0, cfg.N, stride, dtype=np.int64)
    n = cfg.N if idx is None else idx.size
    psd = W.lisa_psd_barack_cutler(cfg.N, cfg.dt) if with_likelihood else None

    def one(k):
        hI, hII, st = orc.waveform(P[k], cfg.N, cfg.dt, cfg.n_max, idx=idx)
        if with_likelihood and idx is None:
            H = np.stack([orc.rfft(hI), orc.rfft(hII)])
            return orc.loglike(H, np.zeros_like(H), psd, cfg.N, cfg.dt)
        return float(hI[0])

    t0 = time.perf_counter()
    with ThreadPoolExecutor(max_workers=walkers) as ex:      # ctypes releases the GIL during the call
        list(ex.map(one, range(walkers)))
    return time.perf_counter() - t0, walkers * n


def run_reference(args, cfg):
    """--impl reference: the CPU oracle on the host cores; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    cores = host_cores()
    walkers = min(cores, cfg.K)
    P = W.draw_params(cfg, K=walkers)
    # one step = the oracle waveform of `walkers` walkers at every `stride`-th sample of the N-sample series
    stride = 32
    for _ in range(args.warmup):
        oracle_sample(cfg, P, walkers, stride * 8, False)
    t, units = 0.0, 0
    for _ in range(args.steps):
        dt_, u = oracle_sample(cfg, P, walkers, stride, False)
        t += dt_
        units += u
    value = units / t
    sample = f"oracle waveform (orbit + every {stride}th of N={cfg.N} samples) of {walkers} walkers, one per thread, per step"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"configs[{cfg.index}]: K={cfg.K} N={cfg.N} dt={cfg.dt} n_max={cfg.n_max}"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": walkers, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def run_gpu(args, cfg):
    import torch
    import torch.distributed as dist
    from paper_2311_17174_b200 import emri

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(x):
        if world == 1:
            return x
        t = torch.tensor([x], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    emri.load()
    K, N = cfg.K, cfg.N
    # every rank draws its own ensemble (weak scaling: K walkers per GPU)
    from paper_2311_17174_b200 import sharding
    P = W.draw_params(sharding.rank_config(cfg, rank))
    psd = W.lisa_psd_barack_cutler(N, cfg.dt)
    plan = emri.Plan(N, cfg.dt, cfg.n_max, K, psd)
    if cfg.index == 5:
        plan.set_anchor(True)            # the paper's convention: initial conditions at the LSO, integrated backwards
    p_d = torch.from_numpy(P).to(dev)
    # data = the library's own injection of walker 0 (+ seeded coloured noise when the config says so)
    spec = plan.waveform_fft(p_d[:1].contiguous())
    D = spec[0].clone()
    if cfg.noise_seed:
        D += torch.from_numpy(W.noise_fft(N, cfg.dt, psd, cfg.noise_seed)).to(dev)
    logL = torch.empty(K, dtype=torch.float64, device=dev)
    status = torch.zeros(K, dtype=torch.int32, device=dev)

    mcmc = cfg.index in (4, 5)
    if mcmc:
        # configs[4]: a step is one full stretch-move update (both half-ensembles), proposals / accept on the device
        lo_d, hi_d = (torch.from_numpy(v).to(dev) for v in W.prior_box(cfg))
        acc = torch.zeros(K, dtype=torch.int32, device=dev)
        plan.loglike(p_d, D, logL, status)
        X = p_d.clone()
        counter = [0]

        def one_step():
            for half in (0, 1):
                plan.stretch_step(X, logL, D, lo_d, hi_d, 2.0, 20231117, counter[0], half, accepted=acc)
            counter[0] += 1
    else:
        def one_step():
            plan.loglike(p_d, D, logL, status)

    for _ in range(max(args.warmup, 3)):
        one_step()
    barrier()
    sampler = ClockSampler(torch.cuda.current_device() if "CUDA_VISIBLE_DEVICES" not in os.environ else local)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(args.steps):
        one_step()
    e1.record()
    barrier()
    ms = max_over_ranks(e0.elapsed_time(e1))
    n_bad = int((status != 0).sum().item())
    if mcmc:        # the chain has moved X and logL; the e2e check below is against the initial ensemble
        logL = plan.loglike(p_d, D, status=status)
    logL_host = logL.cpu().numpy()

    # ---- end to end: pinned host buffers in, logL out, through emri_loglike_host
    P_pin = torch.from_numpy(P).pin_memory()
    D_pin = D.cpu().pin_memory()
    L_pin = torch.empty(K, dtype=torch.float64).pin_memory()
    S_pin = torch.zeros(K, dtype=torch.int32).pin_memory()
    for _ in range(2):
        plan.loglike_host_ptr(P_pin.data_ptr(), K, D_pin.data_ptr(), L_pin.data_ptr(), S_pin.data_ptr())
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        plan.loglike_host_ptr(P_pin.data_ptr(), K, D_pin.data_ptr(), L_pin.data_ptr(), S_pin.data_ptr())
    torch.cuda.synchronize()
    e2e_ms = max_over_ranks((time.perf_counter() - t0) * 1e3)
    clocks = sampler.stop()
    assert np.array_equal(L_pin.numpy(), logL_host), "host and device entry points disagree"

    # ---- per-stage device times (CUDA events inside the plan, on the launching stream), same steps again
    plan.enable_timings(True)
    stage = {"orbit": 0.0, "synth": 0.0, "fft": 0.0, "like": 0.0}
    for _ in range(args.steps):
        plan.loglike(p_d, D, logL, status)
        for k_, v in plan.timings().items():
            stage[k_] += v / args.steps
    plan.enable_timings(False)

    if rank == 0:
        peaks, peaks_src = load_measured_peaks()
        fp64_probe = emri.probe_fp64_peak()
        fp64_probe3 = emri.probe_fp64_peak3()
        sm_max = clocks["sm_max_mhz"] or peaks.get("sm_max_mhz", 1965.0)
        sms = torch.cuda.get_device_properties(dev).multi_processor_count
        fp64_nominal = sms * 64 * 2 * sm_max * 1e6 * 1e-12        # 64 FP64 lanes / SM / clk
        n_chunks = (K + CHUNK - 1) // CHUNK
        fpws = counted_flops_per_walker_sample(cfg.n_max)
        flops = fpws * K * N
        achieved = flops / (stage["synth"] * 1e-3) * 1e-12
        roofline = {"bound": "alu", "kernel": "synth_kernel", "achieved": achieved, "peak": fp64_nominal,
                    "unit": "TFLOP/s", "frac": achieved / fp64_nominal, "traffic": SYNTH_TRAFFIC.get(cfg.index),
                    "peak_source": f"derived: {sms} SMs x 64 FP64 lanes x 2 x {sm_max:.0f} MHz (DESIGN.md section 7)",
                    "peak_dfma_probe": fp64_probe, "frac_of_probe": achieved / fp64_probe,
                    "peak_dfma_probe_3_register_operands": fp64_probe3,
                    "launches_per_step": n_chunks, "ms_per_launch": stage["synth"] / n_chunks,
                    "flops_per_walker_sample": fpws, "flops_source": "counted by ncu (profiles/counts_r1.md)" + (", figure of configs[2] at the same n_max" if mcmc else ""),
                    "algorithmic_bytes_per_launch": 16.0 * min(K, CHUNK) * N}
        # the reduction reads the packed spectrum Z[K][N] complex128 once (D and 1/S_n stay in L2)
        like_gbs = (16.0 * K * N) / (stage["like"] * 1e-3) * 1e-9 if stage["like"] > 0 else None
        cores = host_cores()
        walkers = min(cores, K)
        # the oracle leg runs at N = 1 only (a scaling run does not repeat it on every N)
        cpu_t, cpu_units = oracle_sample(cfg, P, walkers, 1 if N <= (1 << 20) else 4, True) if world == 1 else (None, 0)
        out = {
            "metric": METRIC, "value": world * K * N * args.steps / (ms * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"configs[{cfg.index}]: K={K} walkers/GPU N={N} dt={cfg.dt} n_max={cfg.n_max}, "
                                   f"data = injection{' + coloured noise' if cfg.noise_seed else ''}",
                       "l2": f"per-step working set {2 * K * (N + 2) * 8 / 1e6:.0f} MB > 126 MB L2 (no flush needed)",
                       "parallelism": f"walker-sharded x{world}, no collective"},
            "likelihoods_per_s": world * K * args.steps / (ms * 1e-3),
            "clocks": clocks,
            "e2e": {"value": world * K * N * args.steps / (e2e_ms * 1e-3), "unit": UNIT,
                    "h2d_bytes_per_step": int(P_pin.numel() * 8 + D_pin.numel() * 16),
                    "d2h_bytes_per_step": int(L_pin.numel() * 8 + S_pin.numel() * 4), "ms_per_step": e2e_ms / args.steps},
            "gpu_launches": (ORBIT_KERNELS + 2 * n_chunks + 1) * args.steps,
            "stage_ms": stage,
            "roofline": roofline,
            "like_kernel": {"bound": "hbm", "kernel": "loglike_kernel", "achieved_gbs": like_gbs,
                            "peak_gbs": peaks.get("hbm_gbs"), "frac": (like_gbs / peaks["hbm_gbs"]) if like_gbs else None,
                            "peak_source": f"MEASURED_PEAKS.json copy bandwidth ({peaks_src})"},
            "fft": {"bound": "hbm", "kernel": "cuFFT Z2Z (vendor)", "achieved_gbs": (32.0 * K * N) / (stage["fft"] * 1e-3) * 1e-9
                    if stage["fft"] > 0 else None, "note": "one read + one write of Z per transform counted"},
            "cpu_baseline": ({"value": cpu_units / cpu_t, "unit": UNIT, "cores": walkers, "kind": "oracle",
                              "sample": f"oracle waveform+rfft+logL of {walkers} walkers (one per thread), "
                                        f"{cpu_units // walkers} of N={N} samples each, {cpu_t:.1f} s"}
                             if cpu_t else {"value": None, "unit": UNIT, "cores": 0, "kind": "oracle",
                                            "sample": "timed at N = 1 only"}),
            "walkers_with_status": n_bad,
        }
        print(json.dumps(out))
    plan.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=1,
                    help="index into BASELINE.json:configs (0-4; 4 = stretch-move steps); 5 = the paper's own run shape")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    args = ap.parse_args()
    cfg = W.CONFIGS[args.config]
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_gpu(args, cfg)


if __name__ == "__main__":
    main()
