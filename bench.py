#!/usr/bin/env python
"""bench.py -- throughput of the EMRI_MC hot path on B200 (contract: see DESIGN.md section 8).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config i] [--psd bc|robson] [--impl reference]

A "step" is one pass of the whole hot path -- emri_loglike: orbit RK4 (a), synthesis (b), transform (c), likelihood
reduction (d) -- over one ensemble of K walkers of BASELINE.json:configs[i].  Default i = 3, the largest single-GPU
configuration (K=1024, N=2^21, n_max=30); the other configs are parity-test cases, reachable with --config.
Inputs are synthetic and seeded (workloads.py).  Prints ONE JSON line.  `value` = walker*samples/s with inputs resident
in HBM; `e2e` = the same through emri_loglike_host with pinned HOST buffers (copies inside the timed region).  With N > 1
(torchrun) every rank runs its own K walkers (the path shards by walker, no data-path collective): weak scaling.

`--impl reference` times the CPU oracle (oracle/, test infrastructure) on the host cores instead: the SAME work in kind
as the `cpu_baseline` leg of the GPU arm (orbit + waveform at every sample + rfft + logL), on a bounded sample.
"""
import argparse
import hashlib
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2311_17174_b200 import sharding, workloads as W  # noqa: E402

METRIC = "AK waveform+logL evaluations/sec (walkers x samples/s)"
UNIT = "walker*samples/s"
CHUNK = 128                 # walkers per synth / transform / loglike launch (emri_plan_set_chunk default)
COUNTS_FILE = os.path.join(ROOT, "profiles", "counts_r3.json")
COUNTED_SOURCES = ("paper_2311_17174_b200/csrc/synth.cuh", "paper_2311_17174_b200/csrc/emri.cu")   # kernel + its launch heuristics
# The oracle leg covers the first N / ORACLE_DECIMATE[i] samples of the window (same dt, n_max, parameters): a bounded
# sample of the workload sized to a few seconds of host time per step.
ORACLE_DECIMATE = {0: 1, 1: 1, 2: 4, 3: 4, 4: 4, 5: 4}


def git_blob_sha(path):
    """`git hash-object` of a file, computed here (the GPU box has no .git)"""
    data = open(path, "rb").read()
    return hashlib.sha1(b"blob %d\0" % len(data) + data).hexdigest()


def counted_work(cfg_index, n_max):
    """Algorithmic work of synth_kernel per (walker, sample): FP64 flops EXECUTED by the kernel as built, 2 dfma + dmul +
    dadd, formed HERE from the raw ncu thread-instruction counters of one launch that profiles/counts_r3.json records
    (the same rows are in profiles/counts_r3.md with the command), and the launch's DRAM bytes.  The file also records the
    git blob hash of the kernel source it was counted on: a different source gives (None, None, 'stale')."""
    try:
        with open(COUNTS_FILE) as f:
            c = json.load(f)
    except Exception as e:
        return None, None, f"missing ({e.__class__.__name__})"
    for rel in COUNTED_SOURCES:
        if c.get("sources", {}).get(rel) != git_blob_sha(os.path.join(ROOT, rel)):
            return None, None, "stale"
    e = c.get("configs", {}).get(str(cfg_index))
    if not e or e.get("n_max") != n_max:
        return None, None, "not counted for this config"
    flops = (2.0 * e["dfma"] + e["dmul"] + e["dadd"]) / (float(e["walkers_per_launch"]) * float(e["samples"]))
    return flops, float(e["dram_bytes_read"]) + float(e["dram_bytes_write"]), \
        f"2 dfma + dmul + dadd of one launch, ncu counters on the configs' own inputs ({os.path.relpath(COUNTS_FILE, ROOT)}, source hash verified)"


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


def psd_of(args, N, dt):
    return W.lisa_psd_robson(N, dt) if args.psd == "robson" else W.lisa_psd_barack_cutler(N, dt)


def workload_config(cfg, args):
    """the `config` object: identical in the GPU arm and the reference arm"""
    return {"workload": f"configs[{cfg.index}]: K={cfg.K} walkers per GPU, N={cfg.N}, dt={cfg.dt} s, n_max={cfg.n_max}, "
                        f"data = injection{' + coloured noise' if cfg.noise_seed else ''}, "
                        f"PSD = {'Robson-Cornish-Liu' if args.psd == 'robson' else 'Barack-Cutler'}"
                        + (", a step = one stretch-move update of the ensemble" if cfg.index in (4, 5) else "")
                        + (f", orbit by adaptive DP5(4) at rtol {args.adaptive:g}" if getattr(args, "adaptive", 0) else ""),
            "l2": f"per-step working set {16 * cfg.K * cfg.N / 1e6:.0f} MB > 126 MB L2: no flush needed"
                  if 16 * cfg.K * cfg.N > 126e6 else "per-step working set fits L2 (launch-bound case, reported as is)"}


class OracleLeg:
    """The oracle as it stands, one walker per host thread: orbit + waveform at EVERY sample + rfft of both channels +
    logL against a zero data spectrum, over the first N' = N / ORACLE_DECIMATE samples of the window (same dt, n_max and
    parameter rows).  Used by the `cpu_baseline` leg of the GPU arm (one step) and by --impl reference (every step)."""

    def __init__(self, cfg, args):
        from oracle.oracle import Oracle
        self.cfg = cfg
        self.orc = Oracle(anchor=(cfg.index == 5))
        self.walkers = min(host_cores(), cfg.K)
        self.P = W.draw_params(cfg, K=self.walkers)
        self.Np = 1 << ((cfg.N // ORACLE_DECIMATE.get(cfg.index, 4)).bit_length() - 1)      # a power of two (the oracle's FFT)
        self.psd = psd_of(args, self.Np, cfg.dt)

    def describe(self, seconds=None):
        s = (f"oracle orbit + waveform at every sample + rfft + logL of {self.walkers} walkers (one per thread) over the "
             f"first {self.Np} of N={self.cfg.N} samples")
        return s + (f", {seconds:.1f} s" if seconds is not None else " per step")

    def step(self, n=None):
        """returns (seconds, walker*samples processed)"""
        from concurrent.futures import ThreadPoolExecutor
        n = self.Np if n is None else n
        psd = self.psd if n == self.Np else W.lisa_psd_barack_cutler(n, self.cfg.dt)
        orc, cfg = self.orc, self.cfg

        def one(k):
            hI, hII, st = orc.waveform(self.P[k], n, cfg.dt, cfg.n_max)
            H = np.stack([orc.rfft(hI), orc.rfft(hII)])
            return orc.loglike(H, np.zeros_like(H), psd, n, cfg.dt)

        t0 = time.perf_counter()
        with ThreadPoolExecutor(max_workers=self.walkers) as ex:      # ctypes releases the GIL during the call
            list(ex.map(one, range(self.walkers)))
        return time.perf_counter() - t0, self.walkers * n


def run_reference(args, cfg):
    """--impl reference: the CPU oracle on the host cores; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    leg = OracleLeg(cfg, args)
    for _ in range(args.warmup):
        leg.step(n=1 << 12)                      # loads the library and the thread pool; a CPU has nothing else to warm
    t, units = 0.0, 0
    for _ in range(args.steps):
        dt_, u = leg.step()
        t += dt_
        units += u
    value = units / t
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": workload_config(cfg, args),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": leg.walkers, "kind": "oracle", "sample": leg.describe()},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def run_gpu(args, cfg):
    import torch
    import torch.distributed as dist
    from paper_2311_17174_b200 import emri, probe

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

    emri.load()
    K, N = cfg.K, cfg.N
    # every rank draws its own ensemble (weak scaling: K walkers per GPU)
    P = W.draw_params(sharding.rank_config(cfg, rank))
    psd = psd_of(args, N, cfg.dt)
    plan = emri.Plan(N, cfg.dt, cfg.n_max, K, psd)
    if cfg.index == 5:
        plan.set_anchor(True)            # the paper's convention: initial conditions at the LSO, integrated backwards
    if args.adaptive:
        # the paper's own kind of integrator: embedded pair, step control, dense output
        plan.set_integrator((args.adaptive, args.adaptive * np.array([1.0, 1e-9, 1.0, 1e-5, 1.0])))
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

    warmup = max(args.warmup, 3)
    for _ in range(warmup):
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
    ms = sharding.max_over_ranks(e0.elapsed_time(e1), world, dev)
    launches = plan.launch_count()                # kernels of this library enqueued by the LAST call (cuFFT's excluded)
    if mcmc:
        launches = 2 * launches
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
    e2e_ms = sharding.max_over_ranks((time.perf_counter() - t0) * 1e3, world, dev)
    clocks = sampler.stop()
    assert np.array_equal(L_pin.numpy(), logL_host), "host and device entry points disagree"

    # ---- per-stage device times (CUDA events inside the plan, on the launching stream), same steps again
    plan.enable_timings(True)
    stage = {"orbit": 0.0, "synth": 0.0, "fft": 0.0, "like": 0.0}
    for _ in range(args.steps):
        plan.loglike(p_d, D, logL, status)
        for k_, v in plan.timings().items():
            stage[k_] += v / args.steps
    paths = plan.synth_report()
    # the plain path (full cuFFT transform + streaming reduction kernel) for comparison: a few steps, stage times only
    fused = plan.transform_is_fused()
    plain = None
    if fused:
        plan.set_transform(False)
        plain = {"orbit": 0.0, "synth": 0.0, "fft": 0.0, "like": 0.0}
        n_plain = min(args.steps, 3)
        plan.loglike(p_d, D, logL, status)
        for _ in range(n_plain):
            plan.loglike(p_d, D, logL, status)
            for k_, v in plan.timings().items():
                plain[k_] += v / n_plain
        plan.set_transform(True)
    plan.enable_timings(False)

    if rank == 0:
        peaks, peaks_src = load_measured_peaks()
        fp64_probe = probe.fp64_peak()
        fp64_probe3 = probe.fp64_peak3()
        sm_max = clocks["sm_max_mhz"] or peaks.get("sm_max_mhz", 1965.0)
        sms = torch.cuda.get_device_properties(dev).multi_processor_count
        fp64_nominal = sms * 64 * 2 * sm_max * 1e6 * 1e-12        # 64 FP64 lanes / SM / clk
        n_chunks = (K + CHUNK - 1) // CHUNK
        # configs[4] runs the kernel of configs[2] on a ball of walkers around one injection: counted on its own inputs
        fpws, traffic, src = counted_work(cfg.index, cfg.n_max)
        achieved = fpws * K * N / (stage["synth"] * 1e-3) * 1e-12 if fpws else None
        # peak = the dependent-free DFMA probe of THIS run (probe.cu: 2 register operands reused, all SMs), the derived
        # figure beside it (they agree to ~2 % at 1965 MHz; MEASURED_PEAKS.json has no FP64 entry)
        roofline = {"bound": "alu", "kernel": "synth_kernel", "achieved": achieved, "peak": fp64_probe,
                    "unit": "TFLOP/s", "frac": (achieved / fp64_probe) if achieved else None, "traffic": traffic,
                    "peak_source": "measured in this run: DFMA probe on all SMs (paper_2311_17174_b200/csrc/probe.cu)",
                    "peak_derived": fp64_nominal,
                    "peak_derived_from": f"{sms} SMs x 64 FP64 lanes x 2 x {sm_max:.0f} MHz (DESIGN.md section 7)",
                    "frac_of_derived": (achieved / fp64_nominal) if achieved else None,
                    "peak_dfma_probe_3_register_operands": fp64_probe3,
                    "launches_per_step": n_chunks, "ms_per_launch": stage["synth"] / n_chunks,
                    "flops_per_walker_sample": fpws, "flops_source": src,
                    "algorithmic_bytes_per_launch": 16.0 * min(K, CHUNK) * N,
                    "paths": paths}
        # Stages (c)+(d).  Fused (fft2_like_kernel): z is read once, the intermediate of the two-pass transform is written
        # and read once: 48 B per walker*sample through HBM, ~85 FP64 instructions per element beside it.  Plain path: the
        # reduction kernel alone reads the spectrum once, 16 B per walker*sample.
        bytes_ws = 48.0 if fused else 16.0
        like_gbs = (bytes_ws * K * N) / (stage["like"] * 1e-3) * 1e-9 if stage["like"] > 0 else None
        cd_gbs = (16.0 * K * N) / ((stage["fft"] + stage["like"]) * 1e-3) * 1e-9
        red_gbs = (16.0 * K * N) / (plain["like"] * 1e-3) * 1e-9 if plain and plain["like"] > 0 else None
        if world == 1:        # the oracle leg runs at N = 1 only (a scaling run does not repeat it on every N)
            leg = OracleLeg(cfg, args)
            cpu_t, cpu_units = leg.step()
            cpu = {"value": cpu_units / cpu_t, "unit": UNIT, "cores": leg.walkers, "kind": "oracle",
                   "sample": leg.describe(cpu_t)}
        else:
            cpu = {"value": None, "unit": UNIT, "cores": 0, "kind": "oracle", "sample": "timed at N = 1 only"}
        out = {
            "metric": METRIC, "value": sharding.whole_job_value(K * N, args.steps, ms, world), "unit": UNIT,
            "n_gpus": world, "steps": args.steps, "warmup": warmup, "ms_per_step": ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(cfg, args),
            "parallelism": f"walker-sharded x{world}, no collective",
            "likelihoods_per_s": world * K * args.steps / (ms * 1e-3),
            "clocks": clocks,
            "e2e": {"value": sharding.whole_job_value(K * N, args.steps, e2e_ms, world), "unit": UNIT,
                    "h2d_bytes_per_step": int(P_pin.numel() * 8 + D_pin.numel() * 16),
                    "d2h_bytes_per_step": int(L_pin.numel() * 8 + S_pin.numel() * 4), "ms_per_step": e2e_ms / args.steps},
            "gpu_launches": launches * args.steps,
            "stage_ms": stage,
            "roofline": roofline,
            "like_kernel": {"bound": "hbm", "kernel": plan.like_kernel_name(), "achieved_gbs": like_gbs,
                            "bytes_per_walker_sample": bytes_ws,
                            "peak_gbs": peaks.get("hbm_gbs"), "frac": (like_gbs / peaks["hbm_gbs"]) if like_gbs else None,
                            "peak_source": f"MEASURED_PEAKS.json copy bandwidth ({peaks_src})"},
            "plain_path": None if not plain else {
                "note": "emri_plan_set_transform(0): full cuFFT transform + loglike_kernel, stage times of a few steps",
                "stage_ms": plain,
                "reduction_kernel": {"bound": "hbm", "kernel": "loglike_kernel", "achieved_gbs": red_gbs,
                                     "bytes_per_walker_sample": 16.0, "peak_gbs": peaks.get("hbm_gbs"),
                                     "frac": (red_gbs / peaks["hbm_gbs"]) if red_gbs else None}},
            "transform_and_likelihood": {"bound": "hbm", "achieved_gbs": cd_gbs, "frac": cd_gbs / peaks["hbm_gbs"],
                                         "note": "stages (c)+(d) together against one read of z (16 B per walker*sample)"},
            "cpu_baseline": cpu,
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
    ap.add_argument("--config", type=int, default=3,
                    help="index into BASELINE.json:configs (0-4; 4 = stretch-move steps); 5 = the paper's own run shape")
    ap.add_argument("--psd", default="bc", choices=["bc", "robson"],
                    help="noise curve: Barack-Cutler (the paper's example) or Robson-Cornish-Liu (its second model)")
    ap.add_argument("--adaptive", type=float, default=0.0, metavar="RTOL",
                    help="stage (a) by the adaptive Dormand-Prince 5(4) pair with this relative tolerance instead of fixed-step RK4")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    args = ap.parse_args()
    cfg = W.CONFIGS[args.config]
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_gpu(args, cfg)


if __name__ == "__main__":
    main()
