#!/usr/bin/env python
"""bench.py -- Wilson Dslash throughput on B200 (BASELINE.json metric), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W]            # the CUDA library (default config 3)
    python bench.py --impl reference [--steps K] [--warmup W]       # the CPU oracle, same metric/config
    python bench.py --sweep [--sweep-csv PATH]                      # config 5: 120 variants, top-10
    python bench.py --advisor [--advisor-csv PATH]                  # the paper's own 84 variants on 32x32x32x16
    python bench.py --costmodel                                     # the Advisor's cost model fitted on measured variant runtimes
    python bench.py --probe                                         # read/write/copy/4:1-mix bandwidth, FP64 FMA rate of this board
    python bench.py --cg | --eo | --decomposition slab              # solver, even-odd operator, multi-GPU slab form
    python bench.py --kernel direct|wpipe|march ...                        # force a kernel instead of letting dslash_tune pick

A "step" is one application of D (one dslash_apply = one kernel launch covering SURVEY.md section 8(a)
steps a1-a7) to one seeded synthetic lattice that is already resident in HBM in the native layout.  Before the timed
region the library picks its kernel by measurement (dslash_tune), then the device idles 1 s.
`value` = 1320 flop/site * sites of all ranks / max-over-ranks device time (CUDA events on the
launching stream) of the K timed steps; `repeats` = the same region four more times (median, min); `sustained` = the same
after ~0.6 s of continuous load, when the board runs against its power cap (what a solver sees); `parity` = the buffer the
timed region wrote, compared with the oracle on the whole lattice (outside the timed region).
For lattices whose working set fits L2 (configs[0], [1]: an application takes 3-11 us) the K applications of a timed region
are captured once in a CUDA graph and replayed (--graph auto): the eager loop measured the host's launch rate there.
`e2e` = the same metric through dslash_apply_host with pinned HOST buffers (H2D copy of gauge and spinor, pack, apply, unpack,
D2H copy of the result inside the timed region).
Multi-GPU: default = replicas (every rank its own lattice, weak scaling, no collective: north_star keeps the path on one
GPU); --decomposition slab = one lattice cut along t with a halo exchange per application (strong scaling).
"""
import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "Dslash GFLOP/s (1320 flop/site) & HBM GB/s vs peak, 32^3x64 FP64, 1 B200"
FLOP_PER_SITE = 1320
SEED = 230103636
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md fallback, used only if MEASURED_PEAKS.json is absent

# BASELINE.json configs (index = position in `configs`); bytes/site = compulsory traffic:
# spinor in once + 4 links once + spinor out once.
CONFIGS = {
    "1": dict(dims=(4, 4, 4, 4), precision="f64", recon12=False, name="configs[0]: 4^4 FP64"),
    "2": dict(dims=(16, 16, 16, 16), precision="f64", recon12=False, name="configs[1]: 16^4 FP64 (L2-resident)"),
    "3": dict(dims=(32, 32, 32, 64), precision="f64", recon12=False, name="configs[2]: 32^3x64 FP64, 18-real links"),
    "3r": dict(dims=(32, 32, 32, 64), precision="f64", recon12=True, name="configs[2]: 32^3x64 FP64, 12-real links"),
    "4": dict(dims=(48, 48, 48, 96), precision="f32", recon12=False, name="configs[3]: 48^3x96 FP32"),
    "5": dict(dims=(24, 24, 24, 24), precision="f64", recon12=False, name="configs[4]: 24^4 FP64 (sweep lattice)"),
}

# dram__bytes_read.sum + dram__bytes_write.sum per launch and the FP64-pipe utilisation of the dominant kernel, copied from
# the committed `ncu --set full` captures (profiles/); None until captured for that workload and kernel.
NCU_FIGURES = {
    "32x32x32x64_f64_soa_r18_direct": dict(traffic=2032698000, fp64_pipe_pct=31.0, source="profiles/r01_ncu_tuned_kernel.txt"),
    "32x32x32x64_f64_soa_r18_wpipe": dict(traffic=2051962000, fp64_pipe_pct=None, source="profiles/r01f_wpipe.md"),
    "32x32x32x64_f64_soa_r18_march": dict(traffic=2000138688, fp64_pipe_pct=30.3, source="profiles/r03_ncu_march_raw.csv"),
    "32x32x32x64_f64_soa_r12_march": dict(traffic=1593540816, fp64_pipe_pct=37.9, source="profiles/r02b_skeleton.md"),
    "48x48x48x96_f32_soa_r18_direct": dict(traffic=5294248000, fp64_pipe_pct=None, source="profiles/r03_ncu_direct_cfg4_raw.csv"),
}
KERNEL_NAMES = {"direct": "dslash_tuned_kernel", "wpipe": "dslash_wpipe_kernel", "march": "dslash_march_kernel"}


KERNEL_IDS = {1: "direct", 5: "wpipe", 6: "march"}  # DSLASH_KERNEL_*


def bytes_per_site(precision, recon12):
    real = 8 if precision == "f64" else 4
    return (24 + 4 * (12 if recon12 else 18) + 24) * real


def hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ------------------------------------------------------------------ clocks during the timed region (NVML)
class ClockSampler:
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown"}

    def __init__(self, index):
        self.samples, self.power, self.reasons, self.max_mhz, self.ok = [], [], set(), None, False
        self._stop = threading.Event()
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.ok = False

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
                try:
                    r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for bit, name in self.REASONS.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.002)

    def __enter__(self):
        if self.ok:
            self.t = threading.Thread(target=self._run, daemon=True)
            self.t.start()
        return self

    def __exit__(self, *exc):
        if self.ok:
            self._stop.set()
            self.t.join()

    def summary(self):
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": 0}
        return {"sm_mhz": float(np.median(self.samples)), "sm_min_mhz": int(min(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples),
                "power_w": float(np.median(self.power)) if self.power else None}


# ------------------------------------------------------------------ CPU oracle legs
def oracle_timing(dims, g64, p64, nsites, steps, warmup, nthreads=0):
    """Time the oracle as it stands on `nsites` seeded sample sites per step (the whole lattice if nsites >= V);
    returns (GFLOP/s, s/step, threads, sites, last output)."""
    import oracle
    from paper_2301_03636_b200 import inputs
    v = inputs.volume(dims)
    cores = oracle.max_threads() if nthreads <= 0 else nthreads
    if nsites >= v:
        fn = lambda: oracle.dslash(p64, g64, dims, nthreads)
        n = v
    else:
        sites = np.sort(np.random.default_rng([SEED, 77]).choice(v, size=nsites, replace=False)).astype(np.int64)
        fn = lambda: oracle.dslash_sites(p64, g64, dims, sites, nthreads)
        n = nsites
    out = None
    for _ in range(warmup):
        out = fn()
    t0 = time.perf_counter()
    for _ in range(steps):
        out = fn()
    dt = (time.perf_counter() - t0) / max(steps, 1)
    return FLOP_PER_SITE * n / dt / 1e9, dt, cores, n, out


def run_reference(args, cfg):
    """--impl reference: the oracle (oracle/dslash_oracle.c, unmodified) on the host cores."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from paper_2301_03636_b200 import inputs
    dims = cfg["dims"]
    g, p = inputs.fields(dims, SEED + 3, cfg["precision"], check=False)
    g64, p64 = inputs.promote(g), inputs.promote(p)
    v = inputs.volume(dims)
    nsites = v if args.ref_sites <= 0 else min(v, args.ref_sites)
    gflops, dt, cores, n, _ = oracle_timing(dims, g64, p64, nsites, args.steps, args.warmup)
    sample = ("the whole %s lattice per step (oracle_dslash)" % "x".join(map(str, dims)) if n == v else
              "%d seeded sample sites of the %s lattice per step (oracle_dslash_sites)" % (n, "x".join(map(str, dims))))
    line = {
        "impl": "reference", "metric": METRIC, "value": gflops, "unit": "GFLOP/s", "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg["name"], "dims": list(dims), "sample": sample, "sites_per_step": int(n)},
        "cpu_baseline": {"value": gflops, "unit": "GFLOP/s", "cores": cores, "nproc": os.cpu_count(), "kind": "oracle", "sample": sample},
        "e2e": {"value": gflops, "unit": "GFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------ the CUDA arm
USE_GRAPH = False  # set by run_cuda: the K applications of a timed region are captured in one CUDA graph and replayed


def time_applies(torch, lat, out, inp, gauge, steps, warmup, group, sampler_index):
    graph = None
    if USE_GRAPH:
        # A lattice whose application takes ~10 us is bound by the HOST's launch rate when every step is a ctypes call
        # (measured: 12.4 us per step on 16^4 whatever the tile).  The same K launches captured once and replayed by the
        # device measure the kernels.  Still K launches of the library's kernel per timed region, each through dslash_apply.
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            for _ in range(warmup):
                lat.apply(out, inp, gauge)
            side.synchronize()
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=side):
                for _ in range(steps):
                    lat.apply(out, inp, gauge)
        torch.cuda.current_stream().wait_stream(side)
        graph.replay()  # one untimed replay (uploads the graph)
    else:
        for _ in range(warmup):
            lat.apply(out, inp, gauge)
    torch.cuda.synchronize()
    group.barrier()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(sampler_index) as cs:
        e0.record()
        if graph is not None:
            graph.replay()
        else:
            for _ in range(steps):
                lat.apply(out, inp, gauge)
        e1.record()
        torch.cuda.synchronize()
    group.barrier()
    ms = group.max_over_ranks(e0.elapsed_time(e1))
    return ms, cs.summary()


def lattice_options(B, lat, args):
    if args.tile:
        lat.set_tile(args.tile)
    if args.occupancy is not None:
        B.dslash_set_option(lat.ctx, B.DSLASH_OPT_OCCUPANCY, args.occupancy)
    if args.kernel:
        lat.set_kernel(args.kernel)
    if args.x_shuffle is not None:
        B.dslash_set_option(lat.ctx, B.DSLASH_OPT_X_SHUFFLE, args.x_shuffle)
    if args.l2_policy is not None:
        B.dslash_set_option(lat.ctx, B.DSLASH_OPT_L2_POLICY, args.l2_policy)
    if args.march_policy is not None:
        B.dslash_set_option(lat.ctx, B.DSLASH_OPT_MARCH_POLICY, args.march_policy)
    if args.march_lead is not None:
        B.dslash_set_option(lat.ctx, B.DSLASH_OPT_MARCH_LEAD, args.march_lead)
    if args.pipe_slots is not None:
        B.dslash_set_option(lat.ctx, B.DSLASH_OPT_PIPE_SLOTS, args.pipe_slots)
    if args.pipe_warps is not None:
        B.dslash_set_option(lat.ctx, B.DSLASH_OPT_PIPE_WARPS, args.pipe_warps)


def run_cuda(args, cfg):
    import torch
    from paper_2301_03636_b200 import binding as B
    from paper_2301_03636_b200 import checks, device, inputs, replicas

    rank, world, local = replicas.env_ranks()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA library has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    group = replicas.Group("nccl", torch.device("cuda", local))
    dims, prec = cfg["dims"], cfg["precision"]
    v = inputs.volume(dims)
    global USE_GRAPH
    USE_GRAPH = args.graph == "on" or (args.graph == "auto" and bytes_per_site(prec, cfg["recon12"]) * v < 126e6)
    g, p = inputs.fields(dims, SEED + 3 + 1000 * rank, prec, check=False)  # every rank its own replica

    results = {}
    clocks = None
    launches = 0
    timed_out = None  # the buffer the main timed region wrote, canonical layout, host
    for tag, recon12 in (("main", cfg["recon12"]), ("other_recon", not cfg["recon12"])):
        if tag == "other_recon" and not args.both_recon:
            continue
        with device.Lattice(dims, prec, args.layout, recon12, device="cuda:%d" % local) as lat:
            lattice_options(B, lat, args)
            gd, pd, od = lat.upload_gauge(g), lat.upload_spinor(p), lat.new_spinor()
            tuned = None
            if not args.kernel and not args.no_tune:
                # outside the timed region: the library picks its kernel by measurement, for the regime the timed region will
                # mostly run in (a board leaves its boost window after ~100 back-to-back applications of this lattice)
                long_run = (args.steps + args.warmup) * v > 250 * (1 << 21)
                B.dslash_set_option(lat.ctx, B.DSLASH_OPT_TUNE_MODE, B.DSLASH_TUNE_SUSTAINED if long_run else B.DSLASH_TUNE_BURST)
                tuned = lat.tune(od, pd, gd)
                time.sleep(1.0)               # back to idle: the timed region starts from the same state with or without tuning
            od.fill_(0x7f)                    # whatever the timed region leaves behind is what `parity` looks at
            n0 = B.dslash_launch_count(lat.ctx)
            ms, ck = time_applies(torch, lat, od, pd, gd, args.steps, args.warmup, group, local)
            n1 = B.dslash_launch_count(lat.ctx)
            bps = bytes_per_site(prec, recon12)
            results[tag] = dict(ms=ms, ms_per_step=ms / args.steps,
                                gflops=replicas.whole_job_rate(FLOP_PER_SITE * v, world, ms / args.steps) / 1e9,
                                gbs=bps * v / (ms / args.steps) / 1e6, bps=bps, recon12=recon12,
                                tile=list(B.dslash_get_tile(lat.ctx)),
                                kernel=KERNEL_IDS[B.dslash_get_kernel(lat.ctx)],
                                occupancy=B.dslash_get_option(lat.ctx, B.DSLASH_OPT_OCCUPANCY),
                                x_shuffle=B.dslash_get_option(lat.ctx, B.DSLASH_OPT_X_SHUFFLE),
                                l2_policy=B.dslash_get_option(lat.ctx, B.DSLASH_OPT_L2_POLICY),
                                pipe_slots=B.dslash_get_option(lat.ctx, B.DSLASH_OPT_PIPE_SLOTS),
                                pipe_warps=B.dslash_get_option(lat.ctx, B.DSLASH_OPT_PIPE_WARPS),
                                tuned_ms=None if tuned is None else tuned[1])
            if tag == "main":
                clocks, launches = ck, n1 - n0 - args.warmup
                if not args.no_parity and rank == 0:
                    timed_out = lat.download_spinor(od)
                # "x5 repeats, median and min" -- four more regions of the same K steps, each from idle
                reps = [ms / args.steps]
                for _ in range(max(0, args.repeats - 1)):
                    time.sleep(0.5)
                    ms_r, _ = time_applies(torch, lat, od, pd, gd, args.steps, args.warmup, group, local)
                    reps.append(ms_r / args.steps)
                results["repeats"] = reps
                if args.sustained_steps > 0:
                    # ~0.6 s of continuous load, when the board runs against its power cap; the library re-picks its kernel for
                    # that regime (DSLASH_TUNE_SUSTAINED), again outside the timed region
                    kernel_s = results[tag]["kernel"]
                    if tuned is not None:
                        B.dslash_set_option(lat.ctx, B.DSLASH_OPT_TUNE_MODE, B.DSLASH_TUNE_SUSTAINED)
                        ks, _ = lat.tune(od, pd, gd)
                        kernel_s = KERNEL_IDS.get(ks, str(ks))
                    ms_s, ck_s = time_applies(torch, lat, od, pd, gd, args.sustained_steps, args.heat_steps, group, local)
                    results["sustained"] = dict(ms_per_step=ms_s / args.sustained_steps, clocks=ck_s, kernel=kernel_s,
                                                gbs=bps * v / (ms_s / args.sustained_steps) / 1e6,
                                                gflops=replicas.whole_job_rate(FLOP_PER_SITE * v, world, ms_s / args.sustained_steps) / 1e9)
            del gd, pd, od

    main = results["main"]
    peak, peak_src = hbm_peak()
    key = "%s_%s_%s_r%d_%s" % ("x".join(map(str, dims)), prec, args.layout, 12 if main["recon12"] else 18, main["kernel"])
    ncu = NCU_FIGURES.get(key, {})
    working_set = main["bps"] * v
    l2_resident = working_set < 126e6  # the whole working set of an application fits the 126 MB L2: repeated applies never reach HBM
    if l2_resident:
        # report it, but never as an HBM fraction
        roofline = {"bound": "l2", "achieved": main["gbs"], "peak": None, "unit": "GB/s", "frac": None, "traffic": None,
                    "note": "working set %.1f MB fits the 126 MB L2: algorithmic GB/s served from L2, no HBM roofline applies"
                            % (working_set / 1e6),
                    "kernel": KERNEL_NAMES.get(main["kernel"], main["kernel"]),
                    "algorithmic_bytes_per_site": main["bps"], "algorithmic_bytes_per_launch": working_set}
    else:
        roofline = {"bound": "hbm", "achieved": main["gbs"], "peak": peak, "unit": "GB/s", "frac": main["gbs"] / peak,
                    "traffic": ncu.get("traffic"), "traffic_source": ncu.get("source"),
                    "fp64_pipe_pct": ncu.get("fp64_pipe_pct"), "fp64_pipe_source": ncu.get("source"),
                    "peak_source": peak_src, "kernel": KERNEL_NAMES.get(main["kernel"], main["kernel"]),
                    "algorithmic_bytes_per_site": main["bps"], "algorithmic_bytes_per_launch": working_set,
                    "frac_of_nominal_8TBs": main["gbs"] / 8000.0,
                    "regime": "burst: K steps from idle (board at its boost clock); see `sustained` for the power-capped regime"}
        if "sustained" in results:
            roofline["sustained_frac"] = results["sustained"]["gbs"] / peak

    # end to end through the C ABI with pinned HOST buffers (H2D + pack + apply + unpack + D2H per step)
    e2e = None
    if not args.no_e2e:
        with device.Lattice(dims, prec, args.layout, cfg["recon12"], device="cuda:%d" % local) as lat:
            lattice_options(B, lat, args)
            gh = torch.from_numpy(np.ascontiguousarray(g)).pin_memory()
            ph = torch.from_numpy(np.ascontiguousarray(p)).pin_memory()
            oh = torch.empty(ph.shape, dtype=ph.dtype).pin_memory()
            stream = lat.stream()
            n_e2e = max(1, min(args.steps, args.e2e_steps))
            for _ in range(2):
                h2d, d2h = B.dslash_apply_host(lat.ctx, oh.data_ptr(), ph.data_ptr(), gh.data_ptr(), B.DSLASH_MAP_MINIMAL, stream)
            torch.cuda.synchronize()
            group.barrier()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(n_e2e):
                B.dslash_apply_host(lat.ctx, oh.data_ptr(), ph.data_ptr(), gh.data_ptr(), B.DSLASH_MAP_MINIMAL, stream)
            e1.record()
            torch.cuda.synchronize()
            group.barrier()
            ms_e = group.max_over_ranks(e0.elapsed_time(e1))
            e2e = {"value": replicas.whole_job_rate(FLOP_PER_SITE * v, world, ms_e / n_e2e) / 1e9, "unit": "GFLOP/s", "h2d_bytes_per_step": int(h2d),
                   "d2h_bytes_per_step": int(d2h), "ms_per_step": ms_e / n_e2e, "steps": n_e2e,
                   "gb_per_s_h2d": h2d / (ms_e / n_e2e) / 1e6,
                   "path": "dslash_apply_host(DSLASH_MAP_MINIMAL), pinned host buffers, canonical layout; t-slabs pipelined over three streams"}
            if timed_out is not None:  # the end-to-end path must give the same field as the device-resident one
                e2e["max_abs_diff_vs_timed_buffer"] = float(np.abs(oh.numpy().reshape(timed_out.shape) - timed_out).max())
            del gh, ph, oh

    cpu_baseline = None
    parity = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        g64, p64 = inputs.promote(g), inputs.promote(p)
        nsite = v if args.cpu_sites <= 0 else min(v, args.cpu_sites)
        gf, dt, cores, n, ref = oracle_timing(dims, g64, p64, nsite, 3, 1)
        # the same oracle on ONE thread, on a sample an eighth as large (SURVEY.md section 8(d) asks for both)
        gf1, dt1, _, n1s, _ = oracle_timing(dims, g64, p64, max(1, min(v, 1 << 21) // 8), 1, 0, nthreads=1)
        cpu_baseline = {"value": gf, "unit": "GFLOP/s", "cores": cores, "nproc": os.cpu_count(), "kind": "oracle",
                        "seconds_per_application": dt,
                        "single_thread": {"value": gf1, "unit": "GFLOP/s", "seconds": dt1, "sites": int(n1s)},
                        "sample": "mean of 3 applications (after 1 warm-up) to %d of %d sites (%s)"
                                  % (n, v, "whole lattice" if n == v else "seeded sample")}
        if timed_out is not None and n == v:
            # parity of the buffer the timed region wrote, against the oracle's whole-lattice result (DESIGN.md Reading R10)
            e = float(checks.parity_error(timed_out, ref))
            parity = {"e": e, "sites": int(v), "kernel": main["kernel"], "tolerance": 1e-12 if prec == "f64" else 1e-5,
                      "ok": bool(e <= (1e-12 if prec == "f64" else 1e-5)),
                      "metric": "max_k |g_k - r_k| / max(|r_k|, rms(r)) over complex components, whole lattice, oracle = oracle_dslash"}

    if rank == 0:
        reps = results["repeats"]
        line = {
            "metric": METRIC, "value": main["gflops"], "unit": "GFLOP/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": main["ms_per_step"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": prec, "data": "synthetic",
            "config": {"workload": cfg["name"], "dims": list(dims), "layout": args.layout, "recon": 12 if main["recon12"] else 18,
                       "tile": main["tile"], "kernel": main["kernel"],
                       "kernel_chosen_by": "dslash_tune (measured before the timed region)" if main["tuned_ms"] is not None else "option", "occupancy_option": main["occupancy"],
                       "x_shuffle_option": main["x_shuffle"], "l2_policy_option": main["l2_policy"], "pipe_slots": main["pipe_slots"], "pipe_warps": main["pipe_warps"], "sites": v, "parallelism": "replicas x%d" % world,
                       "launch": "the K applications of a timed region are one CUDA graph replay (K dslash_apply launches captured once)" if USE_GRAPH
                                 else "K dslash_apply calls from the host",
                       "l2": ("working set %.1f MB fits L2: L2-resident by design of this config" % (working_set / 1e6)) if l2_resident else
                             ("inputs larger than L2: %.2f GB working set per apply vs 126 MB L2, no flush needed" % (working_set / 1e9))},
            "hbm_gbs": None if l2_resident else main["gbs"], "roofline": roofline, "parity": parity,
            "repeats": {"n": len(reps), "ms_per_step": reps, "median": float(np.median(reps)), "min": float(np.min(reps)),
                        "note": "the K-step region repeated, each after 0.5 s idle; the first entry is `ms_per_step`"},
            "cpu_baseline": cpu_baseline, "e2e": e2e, "clocks": clocks,
            "gpu_launches": int(launches),
        }
        if "sustained" in results:
            su = results["sustained"]
            line["sustained"] = {"value": su["gflops"], "ms_per_step": su["ms_per_step"], "hbm_gbs": su["gbs"],
                                 "roofline_frac": None if l2_resident else su["gbs"] / peak, "steps": args.sustained_steps, "heat_steps": args.heat_steps,
                                 "clocks": su["clocks"], "kernel": su["kernel"],
                                 "note": "after heat_steps back-to-back applies (SM clock under the power cap); kernel re-picked by "
                                         "dslash_tune in DSLASH_TUNE_SUSTAINED mode unless --kernel / --no-tune"}
        if "other_recon" in results:
            o = results["other_recon"]
            line["also"] = {"recon": 12 if o["recon12"] else 18, "value": o["gflops"], "ms_per_step": o["ms_per_step"],
                            "hbm_gbs": o["gbs"], "roofline_frac": None if l2_resident else o["gbs"] / peak, "kernel": o["kernel"]}
        if args.all_configs and not l2_resident and "sustained" in results:
            # the honest ceiling of the sustained leg: the board's own 4:1 read/write rate after the same kind of heat
            sp = probe_sustained(local)
            roofline["sustained_peak"] = {"value": sp["read4_write1"]["GB/s"], "unit": "GB/s", "kind": "dslash_probe READ4_WRITE1 after 0.5 s of "
                                          "back-to-back launches (csrc/dslash_probe.cu)", "sm_mhz": sp["read4_write1"]["sm_mhz"],
                                          "reasons": sp["read4_write1"]["reasons"], "copy_gbs": sp["copy"]["GB/s"],
                                          "copy_sm_mhz": sp["copy"]["sm_mhz"]}
            roofline["sustained_frac_of_sustained_peak"] = results["sustained"]["gbs"] / sp["read4_write1"]["GB/s"]
        if args.all_configs:
            # north_star: "throughput on the synthetic lattices below ... with the variant sweep's top-10 ranking reported":
            # BASELINE.json configs[0], [1], [3], [4] after the headline (configs[2]), then the 120-variant sweep on configs[4]
            line["configs"] = [measure_other_config(k, args, group, local, peak) for k in ("1", "2", "4", "5")]
            sw = sweep_line(args)
            line["sweep"] = {"workload": sw["sweep"], "variants": sw["variants"], "all_parity_ok": sw["all_parity_ok"],
                             "worst_parity": sw["worst_parity"], "ymax_minus_ymin_ms": sw["spread_ms"],
                             "top10": [{k: r[k] for k in ("rank", "index", "layout", "collapse", "tpb", "spt", "median_ms", "gflops")}
                                       for r in sw["top10"]],
                             "slowest_ms": sw["slowest"]["median_ms"], "tuned_kernel": sw["tuned_kernel"]}
        if B.SKELETON:
            line["skeleton"] = True
            line["metric"] = "NOT A BENCH VALUE: data-movement skeleton (arithmetic compiled out, --skeleton); " + line["metric"]
        print(json.dumps(line))
    group.close()
    return 0


def measure_other_config(key, args, group, local, peak):
    """One compact entry of the default line's `configs` array: BASELINE.json's other lattices through the same protocol as
    the headline (kernel picked by dslash_tune outside the timed region, K steps from idle, parity of the buffer the timed
    region wrote against the oracle's whole-lattice result, a sustained leg for lattices that reach HBM)."""
    import torch
    import oracle
    from paper_2301_03636_b200 import binding as B
    from paper_2301_03636_b200 import checks, device, inputs
    global USE_GRAPH
    cfg = CONFIGS[key]
    dims, prec = cfg["dims"], cfg["precision"]
    v = inputs.volume(dims)
    bps = bytes_per_site(prec, cfg["recon12"])
    working_set = bps * v
    l2_resident = working_set < 126e6
    USE_GRAPH = l2_resident  # the same rule as --graph auto
    steps = max(args.steps, 100) if l2_resident else args.steps
    g, p = inputs.fields(dims, SEED + 3, prec, check=False)
    entry = {"workload": cfg["name"], "dims": list(dims), "dtype": prec, "sites": v, "steps": steps,
             "launch": "CUDA graph replay of the K applies" if l2_resident else "K dslash_apply calls from the host"}
    with device.Lattice(dims, prec, args.layout, cfg["recon12"], device="cuda:%d" % local) as lat:
        gd, pd, od = lat.upload_gauge(g), lat.upload_spinor(p), lat.new_spinor()
        B.dslash_set_option(lat.ctx, B.DSLASH_OPT_TUNE_MODE, B.DSLASH_TUNE_BURST)
        lat.tune(od, pd, gd)
        time.sleep(1.0)
        od.fill_(0x7f)
        ms, ck = time_applies(torch, lat, od, pd, gd, steps, args.warmup, group, local)
        got = lat.download_spinor(od)
        kernel = KERNEL_IDS[B.dslash_get_kernel(lat.ctx)]
        gbs = bps * v / (ms / steps) / 1e6
        entry.update(kernel=kernel, tile=list(B.dslash_get_tile(lat.ctx)), ms_per_step=ms / steps,
                     gflops=FLOP_PER_SITE * v / (ms / steps) / 1e6, clocks=ck)
        if l2_resident:
            entry.update(bound="l2", hbm_gbs=None, roofline_frac=None, sustained_frac=None, l2_gbs=gbs,
                         note="working set %.1f MB fits the 126 MB L2: no HBM roofline applies" % (working_set / 1e6))
        else:
            entry.update(bound="hbm", hbm_gbs=gbs, roofline_frac=gbs / peak)
            sustained_frac = None
            if args.sustained_steps > 0:  # the same amount of traffic as the headline's heat + timed region
                scale = (960.0 * (1 << 21)) / working_set
                heat, n = max(3, int(args.heat_steps * scale)), max(3, int(args.sustained_steps * scale))
                B.dslash_set_option(lat.ctx, B.DSLASH_OPT_TUNE_MODE, B.DSLASH_TUNE_SUSTAINED)
                ks, _ = lat.tune(od, pd, gd)
                ms_s, ck_s = time_applies(torch, lat, od, pd, gd, n, heat, group, local)
                sustained_frac = bps * v / (ms_s / n) / 1e6 / peak
                entry["sustained"] = {"ms_per_step": ms_s / n, "kernel": KERNEL_IDS.get(ks, str(ks)), "steps": n, "heat_steps": heat,
                                      "sm_mhz": ck_s.get("sm_mhz"), "reasons": ck_s.get("reasons")}
            entry["sustained_frac"] = sustained_frac
        del gd, pd, od
    tol = 1e-12 if prec == "f64" else 1e-5
    ref = oracle.dslash(inputs.promote(p), inputs.promote(g), dims)  # whole lattice (DESIGN.md Reading R10)
    e = float(checks.parity_error(got, ref))
    entry["parity"] = {"e": e, "sites": int(v), "tolerance": tol, "ok": bool(e <= tol)}
    return entry


# ------------------------------------------------------------------ multi-GPU: one global lattice cut into T-slabs
def run_slab(args, cfg):
    """--decomposition slab: the --config lattice is cut along t across the ranks (paper_2301_03636_b200/slab.py);
    every apply exchanges one face of spin-projected half-spinors with each t-neighbour over torch.distributed (NCCL)
    and overlaps the exchange with the interior slices (dslash_slab_* calls of the C ABI).  Strong scaling: value = 1320 * V_global / max-over-ranks time."""
    import torch
    from paper_2301_03636_b200 import binding as B
    from paper_2301_03636_b200 import inputs, replicas, slab
    rank, world, local = replicas.env_ranks()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA library has no CPU fallback")
    torch.cuda.set_device(local)
    group = replicas.Group("nccl", torch.device("cuda", local))
    dims, prec = cfg["dims"], cfg["precision"]
    v = inputs.volume(dims)
    g, p = inputs.fields(dims, SEED + 3, prec, check=False)  # every rank generates the same global fields from the seed
    rk = slab.SlabDslash(dims, prec, args.layout, cfg["recon12"], group=group, device="cuda:%d" % local)
    gd, pd, od = rk.upload_gauge(g), rk.upload_spinor(p), rk.lat.new_spinor()
    del g, p
    for _ in range(args.warmup):
        rk.apply(od, pd, gd)
    torch.cuda.synchronize()
    group.barrier()
    torch.cuda.synchronize()
    n0 = B.dslash_launch_count(rk.lat.ctx)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local) as cs:
        e0.record()
        for _ in range(args.steps):
            rk.apply(od, pd, gd)
        e1.record()
        torch.cuda.synchronize()
    group.barrier()
    ms = group.max_over_ranks(e0.elapsed_time(e1)) / args.steps
    launches = B.dslash_launch_count(rk.lat.ctx) - n0
    bps = bytes_per_site(prec, cfg["recon12"])
    peak, peak_src = hbm_peak()
    if rank == 0:
        gbs = bps * v / ms / 1e6
        line = {"metric": METRIC, "value": FLOP_PER_SITE * v / ms / 1e6, "unit": "GFLOP/s", "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
                "dtype": prec, "data": "synthetic",
                "config": {"workload": cfg["name"], "dims": list(dims), "layout": args.layout, "recon": 12 if cfg["recon12"] else 18,
                           "parallelism": "t-slabs x%d, %d slices per rank, half-spinor faces" % (world, rk.geom.lt),
                           "halo_bytes_per_rank_per_step": rk.halo_bytes_per_application,
                           "face_bytes": rk.face_bytes,
                           "l2": "inputs larger than L2 per rank" if bps * v / world > 2 * 126e6 else "per-rank working set near L2 size"},
                "hbm_gbs": gbs, "roofline": {"bound": "hbm", "achieved": gbs / world, "peak": peak, "unit": "GB/s",
                                             "frac": gbs / world / peak, "traffic": None, "peak_source": peak_src,
                                             "kernel": "slab_pack_faces_kernel + dslash_tuned_kernel (interior) + slab_boundary_kernel: 3 launches per apply"},
                "cpu_baseline": None, "e2e": None, "clocks": cs.summary(), "gpu_launches": int(launches)}
        print(json.dumps(line))
    rk.close()
    group.close()
    return 0


# ------------------------------------------------------------------ config 5: the Advisor-style sweep
def run_sweep(args):
    print(json.dumps(sweep_line(args)))
    return 0


def sweep_line(args):
    import torch
    import oracle
    from paper_2301_03636_b200 import binding as B
    from paper_2301_03636_b200 import checks, device, inputs
    cfg = CONFIGS["5"]
    dims = cfg["dims"]
    v = inputs.volume(dims)
    g, p = inputs.fields(dims, SEED + 5, "f64", check=False)
    ref = oracle.dslash(p, g, dims)
    ref_t = torch.from_numpy(np.ascontiguousarray(ref)).cuda()
    ref_c = torch.view_as_complex(ref_t)
    den = torch.maximum(ref_c.abs(), torch.sqrt(torch.mean(ref_c.abs() ** 2)))
    lats = {}
    for lay in ("aos", "soa"):
        lat = device.Lattice(dims, "f64", lay, False)
        lats[lay] = (lat, lat.upload_gauge(g), lat.upload_spinor(p), lat.new_spinor(),
                     lat._bytes(B.dslash_canonical_spinor_bytes(lat.ctx)))
    rows = []
    for i in range(B.dslash_variant_count()):
        depth, tpb, spt, layout = B.dslash_variant_at(i)
        lay = "aos" if layout == B.DSLASH_AOS else "soa"
        lat, gd, pd, od, can = lats[lay]
        lat.set_variant(depth, tpb, spt)
        od.zero_()
        lat.apply(od, pd, gd)
        B.dslash_unpack_spinor(lat.ctx, can.data_ptr(), od.data_ptr(), lat.stream())
        got_c = torch.view_as_complex(can.view(torch.float64).view(ref_t.shape))
        err = float(((got_c - ref_c).abs() / den).max())
        # 3 warm-ups, then min(100, as many as fit in 0.5 s, >= 3) timed applies, each with its own event pair
        times = []
        for _ in range(3):
            lat.apply(od, pd, gd)
        torch.cuda.synchronize()
        budget, n = 0.5, 0
        while n < 100 and (n < 3 or budget > 0):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            lat.apply(od, pd, gd)
            e1.record()
            e1.synchronize()
            ms = e0.elapsed_time(e1)
            times.append(ms)
            budget -= ms / 1e3
            n += 1
        med = float(np.median(times))
        rows.append(dict(index=i, layout=lay, collapse=depth, tpb=tpb, spt=spt, median_ms=med, min_ms=float(min(times)),
                         n=n, gflops=FLOP_PER_SITE * v / med / 1e6, parity=err, ok=bool(err <= 1e-12)))
    # the tuned kernel, same protocol, for reference
    lat, gd, pd, od, can = lats["soa"]
    lat.set_variant(B.DSLASH_VARIANT_TUNED)
    for _ in range(3):
        lat.apply(od, pd, gd)
    torch.cuda.synchronize()
    tt = []
    for _ in range(100):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        lat.apply(od, pd, gd)
        e1.record()
        e1.synchronize()
        tt.append(e0.elapsed_time(e1))
    tuned_ms = float(np.median(tt))
    for lat, *_ in lats.values():
        lat.close()
    rows.sort(key=lambda r: r["median_ms"])
    for k, r in enumerate(rows):
        r["rank"] = k + 1
    if args.sweep_csv:
        os.makedirs(os.path.dirname(os.path.abspath(args.sweep_csv)), exist_ok=True)
        with open(args.sweep_csv, "w") as f:
            cols = ["rank", "index", "layout", "collapse", "tpb", "spt", "median_ms", "min_ms", "n", "gflops", "parity", "ok"]
            f.write(",".join(cols) + "\n")
            for r in rows:
                f.write(",".join(str(r[c]) for c in cols) + "\n")
    line = {"sweep": cfg["name"], "variants": len(rows), "all_parity_ok": all(r["ok"] for r in rows),
            "worst_parity": max(r["parity"] for r in rows), "top10": rows[:10], "slowest": rows[-1],
            "spread_ms": rows[-1]["median_ms"] - rows[0]["median_ms"],
            "tuned_kernel": {"median_ms": tuned_ms, "gflops": FLOP_PER_SITE * v / tuned_ms / 1e6}}
    return line


# ------------------------------------------------------------------ the paper's own 84-variant space, training-mode style
def run_advisor(args):
    """Training mode of the paper: generate every variant of the Dslash kernel (84 for 4 loops,
    Table 1), execute each on the device, collect kernel runtime and data-transfer time, rank.  Lattice 32x32x32x16 is
    the one the paper reports Dslash predictions on.  Every kernel variant is parity-checked first."""
    import torch
    import oracle
    from paper_2301_03636_b200 import binding as B
    from paper_2301_03636_b200 import checks, device, inputs
    dims = tuple(args.advisor_dims)
    v = inputs.volume(dims)
    g, p = inputs.fields(dims, SEED + 6, "f64", check=False)
    ref = oracle.dslash(p, g, dims)
    names = {B.DSLASH_SCHED_STATIC: "static", B.DSLASH_SCHED_DYNAMIC: "dynamic", B.DSLASH_SCHED_GUIDED: "guided"}
    gh = torch.from_numpy(np.ascontiguousarray(g)).pin_memory()
    ph = torch.from_numpy(np.ascontiguousarray(p)).pin_memory()
    oh = torch.zeros(ph.shape, dtype=ph.dtype).pin_memory()
    rows = []
    kernel_cache = {}
    with device.Lattice(dims, "f64", "soa", False) as lat:
        gd, pd, od = lat.upload_gauge(g), lat.upload_spinor(p), lat.new_spinor()
        stream = lat.stream()
        for i in range(B.dslash_omp_variant_count(4)):
            x, a, b, sched, mode = B.dslash_omp_variant_at(4, i)
            B.dslash_set_omp_variant(lat.ctx, x, a, b, sched, 0, args.team_size)
            key = (x, a, b, sched)
            if key not in kernel_cache:
                od.zero_()
                lat.apply(od, pd, gd)
                err = checks.parity_error(lat.download_spinor(od), ref)
                times = []
                for _ in range(2):
                    lat.apply(od, pd, gd)
                torch.cuda.synchronize()
                budget, n = 0.3, 0
                while n < 50 and (n < 3 or budget > 0):
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record()
                    lat.apply(od, pd, gd)
                    e1.record()
                    e1.synchronize()
                    times.append(e0.elapsed_time(e1))
                    budget -= times[-1] / 1e3
                    n += 1
                kernel_cache[key] = (float(np.median(times)), err)
            k_ms, err = kernel_cache[key]
            # the offloaded region end to end: map to the device, run this variant, map back
            t_e2e = []
            for _ in range(3):
                oh.zero_()
                t0 = time.perf_counter()
                h2d, d2h = B.dslash_apply_host(lat.ctx, oh.data_ptr(), ph.data_ptr(), gh.data_ptr(), mode, stream)
                t_e2e.append((time.perf_counter() - t0) * 1e3)
            e2e_ms = float(np.median(t_e2e))
            e2e_err = checks.parity_error(oh.numpy(), ref)
            rows.append(dict(index=i, parallel_position=x, distribute_collapse=a, parallel_collapse=b, schedule=names[sched],
                             map="tofrom" if mode == B.DSLASH_MAP_TOFROM else "minimal", kernel_ms=k_ms, e2e_ms=e2e_ms,
                             transfer_gb=(h2d + d2h) / 1e9, parity=max(err, e2e_err), ok=bool(max(err, e2e_err) <= 1e-12)))
        # the library's tuned kernel, same protocol
        lat.set_variant(B.DSLASH_VARIANT_TUNED)
        for _ in range(3):
            lat.apply(od, pd, gd)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(50):
            lat.apply(od, pd, gd)
        e1.record()
        torch.cuda.synchronize()
        tuned_ms = e0.elapsed_time(e1) / 50
    rows.sort(key=lambda r: r["e2e_ms"])
    for k, r in enumerate(rows):
        r["rank"] = k + 1
    if args.advisor_csv:
        os.makedirs(os.path.dirname(os.path.abspath(args.advisor_csv)), exist_ok=True)
        cols = ["rank", "index", "parallel_position", "distribute_collapse", "parallel_collapse", "schedule", "map", "kernel_ms",
                "e2e_ms", "transfer_gb", "parity", "ok"]
        with open(args.advisor_csv, "w") as f:
            f.write(",".join(cols) + "\n")
            for r in rows:
                f.write(",".join(str(r[c]) for c in cols) + "\n")
    by_kernel = sorted({(r["parallel_position"], r["distribute_collapse"], r["parallel_collapse"], r["schedule"]): r["kernel_ms"]
                        for r in rows}.items(), key=lambda kv: kv[1])
    gb = {m: next(r["transfer_gb"] for r in rows if r["map"] == m) for m in ("tofrom", "minimal")}
    line = {"advisor": "training-mode run over the paper's variant space (PAPER.md:150-173)", "dims": list(dims),
            "variants": len(rows), "kernel_variants": len(by_kernel), "all_parity_ok": all(r["ok"] for r in rows),
            "worst_parity": max(r["parity"] for r in rows), "top10": rows[:10], "slowest": rows[-1],
            "spread_ms": rows[-1]["e2e_ms"] - rows[0]["e2e_ms"],
            "kernel_only": {"fastest": by_kernel[0], "slowest": by_kernel[-1], "tuned_kernel_ms": tuned_ms},
            "transfer_gb": gb, "transfer_ratio_tofrom_over_minimal": gb["tofrom"] / gb["minimal"]}
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------ the Advisor's cost model
COSTMODEL_LATTICES = [(8, 8, 8, 8), (8, 8, 8, 16), (12, 12, 12, 12), (16, 16, 16, 8), (16, 16, 16, 16), (12, 12, 12, 24),
                      (24, 24, 24, 12), (16, 16, 16, 32), (24, 24, 24, 24), (32, 32, 32, 16)]
COSTMODEL_FEATURES = ["parallel_position", "distribute_collapse", "parallel_collapse", "sched_static", "sched_dynamic",
                      "sched_guided", "log2_league_iterations", "log2_team_iterations", "log2_serial_iterations", "log2_volume",
                      "log2_L_T", "log2_L_X"]


def costmodel_features(dims, x, a, b, sched):
    """The 12 inputs of this build's cost model for one kernel variant on one lattice.  The paper's 33 features are not
    published (PAPER.md:305 gives only their number), so these are this build's choice (parity unpinned): the
    variant parameters of PAPER.md:156-160 and the iteration counts they imply.  Loops outer -> inner = t, z, y, x."""
    ext = [dims[3], dims[2], dims[1], dims[0]]  # Loop 0..3
    league = float(np.prod(ext[:a])) if x > 0 else 1.0              # distribute collapse(a) over Loops 0..a-1
    team = float(np.prod(ext[x:x + b]))                               # parallel for collapse(b) over Loops x..x+b-1
    serial = float(np.prod(ext)) / (league * team)                    # what one thread runs serially per parallel iteration
    return [x, a, b, float(sched == 0), float(sched == 1), float(sched == 2), np.log2(league), np.log2(team), np.log2(serial),
            np.log2(float(np.prod(ext))), np.log2(ext[0]), np.log2(ext[3])]


def collect_variant_timings(args, lattices):
    """Training mode: run every kernel structure x schedule of the paper's space on each lattice, parity-check
    it against the oracle, time it on the device.  Returns rows (features, runtime in ms, lattice, variant)."""
    import torch
    import oracle
    from paper_2301_03636_b200 import binding as B
    from paper_2301_03636_b200 import checks, device, inputs
    rows = []
    for dims in lattices:
        g, p = inputs.fields(dims, SEED + 7, "f64", check=False)
        ref = oracle.dslash(p, g, dims)
        with device.Lattice(dims, "f64", "soa", False) as lat:
            gd, pd, od = lat.upload_gauge(g), lat.upload_spinor(p), lat.new_spinor()
            seen = set()
            for i in range(B.dslash_omp_variant_count(4)):
                x, a, b, sched, _mode = B.dslash_omp_variant_at(4, i)
                if (x, a, b, sched) in seen:
                    continue
                seen.add((x, a, b, sched))
                B.dslash_set_omp_variant(lat.ctx, x, a, b, sched, 0, args.team_size)
                od.zero_()
                lat.apply(od, pd, gd)
                err = checks.parity_error(lat.download_spinor(od), ref)
                lat.apply(od, pd, gd)
                torch.cuda.synchronize()
                times, budget = [], 0.05
                while len(times) < 20 and (len(times) < 3 or budget > 0):
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record()
                    lat.apply(od, pd, gd)
                    e1.record()
                    e1.synchronize()
                    times.append(e0.elapsed_time(e1))
                    budget -= times[-1] / 1e3
                rows.append(dict(dims=dims, variant=(x, a, b, sched), ms=float(np.median(times)), parity=err,
                                 features=costmodel_features(dims, x, a, b, sched)))
    return rows


def run_costmodel_profile_one(args):
    """--costmodel --profile-one: ONE costmodel_train launch of the paper's network size on seeded random data (F = 33,
    n = 400 rows, 4 epochs of batch 16 = 100 updates, one model, cluster of 8) -- the command the ncu figures of
    profiles/r01e_costmodel.md are taken from.  Prints the launch's time per update."""
    import torch
    from paper_2301_03636_b200 import costmodel as C
    from paper_2301_03636_b200 import inputs
    dev = torch.device("cuda:0")
    f, n, epochs, batch = args.costmodel_f, 400, 4, 16
    cluster = args.costmodel_cluster
    if args.costmodel_threads:
        C.costmodel_set_option(C.COSTMODEL_OPT_THREADS, args.costmodel_threads)
    rng = np.random.default_rng([SEED, 33])
    xs = torch.from_numpy(rng.standard_normal((n, f))).to(dev)
    ys = torch.from_numpy(rng.standard_normal(n)).to(dev)
    uni = torch.from_numpy(inputs.uniforms(SEED + 100, C.costmodel_weight_count(f))[None]).to(dev)
    perms = torch.from_numpy(inputs.permutations(SEED + 100, epochs, n)[None]).to(dev)
    model = C.CostModel(f)
    updates = epochs * ((n + batch - 1) // batch)
    ms = []
    for _ in range(3):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        model.train(xs, ys, uni, perms, epochs=epochs, batch=batch, cluster_size=cluster)
        e1.record()
        torch.cuda.synchronize()
        ms.append(e0.elapsed_time(e1))
    print(json.dumps({"costmodel_profile_one": True, "f": f, "rows": n, "epochs": epochs, "batch": batch,
                      "cluster": cluster if cluster else "library default", "threads": args.costmodel_threads or "library default",
                      "updates": updates, "ms_per_launch": ms, "us_per_update": min(ms) * 1e3 / updates}))
    return 0


def run_costmodel(args):
    """The cost-model half of the Advisor on this build's own measurements: 42 kernel variants x 10 lattices -> runtime;
    80 % / 20 % split, Z-score, the paper's MLP and optimiser settings, everything on the device through
    include/advisor_costmodel.h; the NumPy oracle runs the same protocol beside it (parity of the result, CPU baseline)."""
    import torch
    from oracle import costmodel as ocm
    from paper_2301_03636_b200 import costmodel as C
    from paper_2301_03636_b200 import inputs
    dev = torch.device("cuda:0")
    t0 = time.perf_counter()
    rows = collect_variant_timings(args, COSTMODEL_LATTICES[:args.costmodel_lattices])
    collect_s = time.perf_counter() - t0
    f = len(COSTMODEL_FEATURES)
    n = len(rows)
    x = np.array([r["features"] for r in rows], dtype=np.float64)
    y_ms = np.array([r["ms"] for r in rows], dtype=np.float64)
    order = inputs.permutations(SEED + 8, 1, n)[0]
    ntr = int(round(0.8 * n))  # "80% for training and 20% for validation"
    tr, va = np.sort(order[:ntr]), np.sort(order[ntr:])
    epochs, batch, m = args.costmodel_epochs, 16, args.costmodel_models
    nw = C.costmodel_weight_count(f)
    uni = np.stack([inputs.uniforms(SEED + 100 + k, nw) for k in range(m)])
    perms = np.stack([inputs.permutations(SEED + 100 + k, epochs, ntr) for k in range(m)])
    out = {"costmodel": "MLP F-2F-4F-2F-F-1, RMSprop 0.01 x0.1/30 epochs, wd 1e-4, batch 16 (PAPER.md:305-307)",
           "features": COSTMODEL_FEATURES, "rows": n, "train_rows": ntr, "validation_rows": n - ntr, "epochs": epochs,
           "lattices": [list(d) for d in COSTMODEL_LATTICES[:args.costmodel_lattices]],
           "all_variants_parity_ok": bool(max(r["parity"] for r in rows) <= 1e-12), "collect_seconds": collect_s,
           "runtime_ms_range": [float(y_ms.min()), float(y_ms.max())], "targets": {}}
    model = C.CostModel(f)
    xd = torch.from_numpy(x).to(dev)
    ud, pd = torch.from_numpy(uni).to(dev), torch.from_numpy(perms).to(dev)
    idx_tr, idx_va = torch.from_numpy(tr).to(dev), torch.from_numpy(va).to(dev)
    for target, y in (("runtime_ms", y_ms), ("log10_runtime_ms", np.log10(y_ms))):
        yd = torch.from_numpy(y).to(dev)
        xtr, ytr, xva, yva = xd[idx_tr].contiguous(), yd[idx_tr].contiguous(), xd[idx_va].contiguous(), yd[idx_va].contiguous()
        launches0 = C.costmodel_launch_count()
        model.fit_scaler(xtr, ytr)
        xs_tr, ys_tr, xs_va, xs_all = model.scale_x(xtr), model.scale_y(ytr), model.scale_x(xva), model.scale_x(xd)
        model.train(xs_tr, ys_tr, ud, pd, epochs=epochs, batch=batch)  # warm-up launch (module load, clocks)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        params, loss = model.train(xs_tr, ys_tr, ud, pd, epochs=epochs, batch=batch)
        e1.record()
        torch.cuda.synchronize()
        train_ms = e0.elapsed_time(e1)
        e0.record()
        model.train(xs_tr, ys_tr, ud[:1], pd[:1], epochs=epochs, batch=batch)
        e1.record()
        torch.cuda.synchronize()
        train1_ms = e0.elapsed_time(e1)
        fill_ms = None
        if target == "runtime_ms":
            # the axis along which the GPU is filled: one model (seed) per SM in the same launch
            sms = torch.cuda.get_device_properties(dev).multi_processor_count
            uf = torch.from_numpy(np.stack([inputs.uniforms(SEED + 1000 + k, nw) for k in range(sms)])).to(dev)
            pf = torch.from_numpy(np.stack([inputs.permutations(SEED + 1000 + k, epochs, ntr) for k in range(sms)])).to(dev)
            model.train(xs_tr, ys_tr, uf, pf, epochs=epochs, batch=batch)
            torch.cuda.synchronize()
            e0.record()
            model.train(xs_tr, ys_tr, uf, pf, epochs=epochs, batch=batch)
            e1.record()
            torch.cuda.synchronize()
            fill_ms = e0.elapsed_time(e1)
            out["one_model_per_sm"] = {"models": sms, "train_ms": fill_ms,
                                       "model_updates_per_s": sms * epochs * ((ntr + batch - 1) // batch) / (fill_ms / 1e3)}
            del uf, pf
        pred_va = model.predict(xs_va, params)
        nrmse = []
        for k in range(m):
            pk = model.scale_y(pred_va[k].contiguous(), inverse=True)
            nrmse.append(float(model.error(pk, yva).cpu().numpy()[1]))
        pred_all = model.scale_y(model.predict(xs_all, params[:1])[0].contiguous(), inverse=True).cpu().numpy()
        launches = C.costmodel_launch_count() - launches0
        # ranking on the largest lattice: measured top-10 vs predicted top-10 of its 42 variants (model 0)
        big = [i for i, r in enumerate(rows) if r["dims"] == COSTMODEL_LATTICES[args.costmodel_lattices - 1]]
        top_meas = set(sorted(big, key=lambda i: y[i])[:10])
        top_pred = set(sorted(big, key=lambda i: pred_all[i])[:10])
        # the oracle, same protocol, model 0 (CPU baseline and parity of the outcome)
        t0 = time.perf_counter()
        mx, sx = ocm.zscore_fit(x[tr])
        my, sy = ocm.zscore_fit(y[tr])
        oxs, oys = ocm.zscore_apply(x, mx, sx), ocm.zscore_apply(y, my, sy)
        oparams, oloss = ocm.train(f, oxs[tr], oys[tr], uni[0], perms[0], epochs=epochs, batch=batch)
        opred = ocm.predict(oparams, oxs[va]) * sy[0] + my[0]
        oracle_s = time.perf_counter() - t0
        onrmse = ocm.nrmse(opred, y[va])
        steps = epochs * ((ntr + batch - 1) // batch)
        if target == "runtime_ms":
            # Sensitivity of the protocol itself: the same training stopped after k updates, CUDA path vs oracle, next to the
            # oracle vs the oracle with ONE training target moved by one ulp.  Both differences grow at the same exponential
            # rate until they saturate, which is why whole-run parameters are compared statistically (NRMSE), not digit by digit.
            oys_p = oys[tr].copy()
            oys_p[0] = np.nextafter(oys_p[0], np.inf)
            ks = [k for k in (10, 50, 100, 200, 400, 800, 1600, steps) if k <= steps]
            grow = {"updates": ks, "cuda_vs_oracle": [], "oracle_vs_oracle_one_ulp": []}
            for k in ks:
                pk, _ = model.train(xs_tr, ys_tr, ud[:1], pd[:1], epochs=epochs, batch=batch, max_steps=k)
                ok = ocm.pack(ocm.train(f, oxs[tr], oys[tr], uni[0], perms[0], epochs=epochs, batch=batch, max_steps=k)[0])
                op = ocm.pack(ocm.train(f, oxs[tr], oys_p, uni[0], perms[0], epochs=epochs, batch=batch, max_steps=k)[0])
                grow["cuda_vs_oracle"].append(float(np.abs(pk[0].cpu().numpy() - ok).max()))
                grow["oracle_vs_oracle_one_ulp"].append(float(np.abs(op - ok).max()))
            out["trajectory_sensitivity_max_abs_param_diff"] = grow
        out["targets"][target] = {
            "nrmse_validation": nrmse[0], "success_nrmse_below_0.1": bool(nrmse[0] < 0.1),
            "nrmse_models": {"n": m, "mean": float(np.mean(nrmse)), "min": float(np.min(nrmse)), "max": float(np.max(nrmse))},
            "oracle_nrmse_validation": float(onrmse), "nrmse_rel_diff_vs_oracle": float(abs(nrmse[0] - onrmse) / onrmse),
            "params_max_abs_diff_vs_oracle": float(np.abs(params[0].cpu().numpy() - ocm.pack(oparams)).max()),
            "final_epoch_loss": float(loss[0, -1].item()), "oracle_final_epoch_loss": float(oloss[-1]),
            "top10_overlap_largest_lattice": len(top_meas & top_pred),
            "train_ms_one_model": train1_ms, "us_per_update_one_model": 1e3 * train1_ms / steps,
            "train_ms_all_models": train_ms, "model_updates_per_s": m * steps / (train_ms / 1e3),
            "oracle_seconds_one_model": oracle_s, "oracle_updates_per_s": steps / oracle_s, "gpu_launches": int(launches)}
    print(json.dumps(out))
    return 0


# ------------------------------------------------------------------ ceilings of the board at hand
def probe_sustained(index, heat_s=0.5, timed_s=0.12):
    """What the board's memory system holds under CONTINUOUS load: the library's 4:1 read/write probe (the Dslash's own mix)
    and its copy probe, each launched back to back for heat_s seconds (about the duration of the headline's 1500-apply heat),
    then timed over timed_s seconds with the SM clock and throttle reasons sampled.  MEASURED_PEAKS.json's hbm_gbs is a burst
    figure (best of a few copies from idle); the sustained Dslash number has this one as its honest ceiling."""
    import torch
    from paper_2301_03636_b200 import binding as B
    dev = torch.device("cuda", index)
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    n = 1 << 26  # 16-byte units: 1 GiB per stream, far beyond L2
    src = torch.empty(4 * n * 2, dtype=torch.float64, device=dev).normal_()
    dst = torch.empty(n * 2, dtype=torch.float64, device=dev)
    st = torch.cuda.current_stream().cuda_stream
    out = {}
    for name, kind, nbytes in (("read4_write1", B.DSLASH_PROBE_READ4_WRITE1, 80 * n), ("copy", B.DSLASH_PROBE_COPY, 32 * n)):
        def launch(k):
            for _ in range(k):
                B.dslash_probe_launch(kind, dst.data_ptr(), src.data_ptr(), n, sms * 8, st)
        launch(3)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        launch(5)
        e1.record()
        torch.cuda.synchronize()
        per = e0.elapsed_time(e1) / 5 / 1e3  # seconds per launch, to size the two regions
        heat, timed = max(10, int(heat_s / per)), max(10, int(timed_s / per))
        time.sleep(1.0)
        launch(heat)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with ClockSampler(index) as cs:
            e0.record()
            launch(timed)
            e1.record()
            torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / timed
        ck = cs.summary()
        out[name] = {"GB/s": nbytes / ms / 1e6, "ms_per_launch": ms, "bytes_per_launch": nbytes, "heat_launches": heat,
                     "timed_launches": timed, "sm_mhz": ck.get("sm_mhz"), "reasons": ck.get("reasons"), "power_w": ck.get("power_w")}
    del src, dst
    return out


def run_probe(args):
    """Read / write / copy / 4:1-mix bandwidth over 4 GiB working sets and the FP64 FMA rate, each the best of 5 launches after
    1 s idle (boost window), with the library's own probe kernels (csrc/dslash_probe.cu)."""
    import torch
    from paper_2301_03636_b200 import binding as B
    dev = torch.device("cuda:0")
    torch.cuda.set_device(dev)
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    n = 1 << 26  # 16-byte units: 1 GiB per stream
    src = torch.empty(4 * n * 2, dtype=torch.float64, device=dev).normal_()
    dst = torch.empty(n * 2, dtype=torch.float64, device=dev)
    st = torch.cuda.current_stream().cuda_stream

    def best(kind, units, blocks, bytes_moved=None, flops=None):
        B.dslash_probe_launch(kind, dst.data_ptr(), src.data_ptr(), units, blocks, st)
        torch.cuda.synchronize()
        time.sleep(1.0)
        ts = []
        for _ in range(5):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            B.dslash_probe_launch(kind, dst.data_ptr(), src.data_ptr(), units, blocks, st)
            e1.record()
            e1.synchronize()
            ts.append(e0.elapsed_time(e1))
        ms = min(ts)
        return {"ms": ms, "GB/s": None if bytes_moved is None else bytes_moved / ms / 1e6,
                "TFLOP/s": None if flops is None else flops / ms / 1e9}
    blocks = sms * 8
    iters = 1 << 14
    peak, peak_src = hbm_peak()
    out = {"probe": "csrc/dslash_probe.cu, best of 5 launches after 1 s idle", "sms": sms, "blocks": blocks,
           "read": best(B.DSLASH_PROBE_READ, 4 * n, blocks, bytes_moved=64 * n),
           "write": best(B.DSLASH_PROBE_WRITE, n, blocks, bytes_moved=16 * n),
           "copy": best(B.DSLASH_PROBE_COPY, n, blocks, bytes_moved=32 * n),
           "read4_write1": best(B.DSLASH_PROBE_READ4_WRITE1, n, blocks, bytes_moved=80 * n),
           "dfma": best(B.DSLASH_PROBE_DFMA, iters, blocks, flops=2.0 * 8 * iters * blocks * 256),
           "measured_peaks_hbm_gbs": peak, "peak_source": peak_src}
    del src, dst
    out["sustained"] = probe_sustained(0)
    print(json.dumps(out))
    return 0


# ------------------------------------------------------------------ the solver around Dslash
def run_cg(args):
    """CG on M^dagger M (dslash_cg_solve) on a BASELINE lattice: what "called several times throughout the LQCD
    application" looks like.  Reports iterations, time per iteration and the operator throughput."""
    import torch
    from paper_2301_03636_b200 import binding as B
    from paper_2301_03636_b200 import device, inputs
    cfg = CONFIGS[args.config]
    dims, prec = cfg["dims"], cfg["precision"]
    v = inputs.volume(dims)
    g, b = inputs.fields(dims, SEED + 7, prec, check=False)
    with device.Lattice(dims, prec, args.layout, cfg["recon12"]) as lat:
        gd, bd, xd = lat.upload_gauge(g), lat.upload_spinor(b), lat.new_spinor()
        lat.cg_solve(xd, bd, gd, args.cg_mass, 1e-2, 5)  # warm-up (allocates the work spinors)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n0 = B.dslash_launch_count(lat.ctx)
        e0.record()
        iters, rel = lat.cg_solve(xd, bd, gd, args.cg_mass, args.cg_tol, args.cg_max_iter)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        launches = B.dslash_launch_count(lat.ctx) - n0
        # per iteration: M and M^dagger (1320 + 72 flop/site each: the epilogue a*psi + b*acc is 24 mul + 24 fma), |t|^2 (48),
        # the fused update x += alpha p, r -= alpha q, |r|^2 (4*24 + 48), p = r + beta p (48)
        flop_it = v * (2 * (1320 + 72) + 48 + 144 + 48)
        rb = 8 if prec == "f64" else 4
        # bytes: two operator applies (+ centre spinor), |t|^2 reads t, the fused update reads 4 and writes 2, p-update reads 2 writes 1
        bytes_it = v * (2 * (bytes_per_site(prec, cfg["recon12"]) + 24 * rb) + (1 + 6 + 3) * 24 * rb)
        line = {"cg": "dslash_cg_solve, M^dagger M x = b", "workload": cfg["name"], "dims": list(dims), "mass": args.cg_mass,
                "tol": args.cg_tol, "iterations": iters, "rel_residual": rel, "ms_total": ms, "ms_per_iteration": ms / max(iters, 1),
                "gflops": flop_it * iters / ms / 1e6, "algorithmic_gbs": bytes_it * iters / ms / 1e6, "gpu_launches": int(launches),
                "dtype": prec, "data": "synthetic"}
        print(json.dumps(line))
    return 0


def run_eo(args):
    """Even-odd (checkerboarded) form on a BASELINE lattice: time of one D_{eo} application and of the Schur complement Mhat,
    then dslash_eo_solve (M x = b through Mhat) beside dslash_cg_solve on the same right-hand side."""
    import torch
    from paper_2301_03636_b200 import binding as B
    from paper_2301_03636_b200 import device, inputs
    cfg = CONFIGS[args.config]
    dims, prec = cfg["dims"], cfg["precision"]
    v = inputs.volume(dims)
    rb = 8 if prec == "f64" else 4
    g, b = inputs.fields(dims, SEED + 7, prec, check=False)
    with device.Lattice(dims, prec, args.layout, cfg["recon12"]) as lat:
        ge = lat.upload_eo_gauge(g)
        be, bo = lat.upload_eo_spinor(b, 0), lat.upload_eo_spinor(b, 1)
        xe, xo, tmp = lat.new_eo_spinor(), lat.new_eo_spinor(), lat.new_eo_spinor()

        def timed(fn, steps, warmup):
            for _ in range(warmup):
                fn()
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(steps):
                fn()
            e1.record()
            torch.cuda.synchronize()
            return e0.elapsed_time(e1) / steps

        ms_d = timed(lambda: lat.eo_apply(0, 0, xe, bo, ge), args.steps, args.warmup)
        ms_m = timed(lambda: lat.eo_apply_schur(0, args.cg_mass, xe, be, tmp, ge), args.steps, args.warmup)
        # one D_{p,1-p}: V/2 output sites x 1320 flop; bytes: in half + all links (forward links of the output parity, backward
        # links of the input parity) + out half
        link_b = (12 if cfg["recon12"] else 18) * 4 * rb
        bytes_d = v * (24 * rb // 2 + link_b + 24 * rb // 2)
        lat.eo_solve(xe, xo, be, bo, ge, args.cg_mass, 1e-2, 5)  # warm-up (allocates the work fields)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n0 = B.dslash_launch_count(lat.ctx)
        e0.record()
        iters, rel = lat.eo_solve(xe, xo, be, bo, ge, args.cg_mass, args.cg_tol, args.cg_max_iter)
        e1.record()
        torch.cuda.synchronize()
        ms_solve, launches = e0.elapsed_time(e1), B.dslash_launch_count(lat.ctx) - n0
        del ge
        gd, bd, xd = lat.upload_gauge(g), lat.upload_spinor(b), lat.new_spinor()
        lat.cg_solve(xd, bd, gd, args.cg_mass, 1e-2, 5)
        torch.cuda.synchronize()
        e0.record()
        iters_plain, rel_plain = lat.cg_solve(xd, bd, gd, args.cg_mass, args.cg_tol, args.cg_max_iter)
        e1.record()
        torch.cuda.synchronize()
        ms_plain = e0.elapsed_time(e1)
        line = {"eo": "checkerboarded Dslash, Schur complement, dslash_eo_solve", "workload": cfg["name"], "dims": list(dims),
                "mass": args.cg_mass, "tol": args.cg_tol,
                "d_eo": {"ms": ms_d, "gflops": 1320 * (v // 2) / ms_d / 1e6, "algorithmic_gbs": bytes_d / ms_d / 1e6,
                         "algorithmic_bytes": bytes_d},
                "mhat": {"ms": ms_m, "gflops": (2 * 1320 + 72) * (v // 2) / ms_m / 1e6,
                         "algorithmic_gbs": (2 * bytes_d + v // 2 * 24 * rb) / ms_m / 1e6},
                "eo_solve": {"iterations": iters, "rel_residual": rel, "ms_total": ms_solve, "ms_per_iteration": ms_solve / max(iters, 1),
                             "gpu_launches": int(launches)},
                "plain_cg": {"iterations": iters_plain, "rel_residual": rel_plain, "ms_total": ms_plain,
                             "ms_per_iteration": ms_plain / max(iters_plain, 1)},
                "speedup_vs_plain_cg": ms_plain / ms_solve, "dtype": prec, "data": "synthetic"}
        print(json.dumps(line))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)  # 10 warm-up + 100 applies
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--sustained-steps", type=int, default=300, help="0: skip the power-capped (sustained) measurement")
    ap.add_argument("--heat-steps", type=int, default=1500)
    ap.add_argument("--impl", choices=["cuda", "reference"], default="cuda")
    ap.add_argument("--config", choices=sorted(CONFIGS), default="3")
    ap.add_argument("--dims", type=int, nargs=4, default=None, help="override the lattice of --config (x y z t): an off-contract "
                                                                    "workload for kernel comparisons, named as such in the line")
    ap.add_argument("--precision", choices=["f64", "f32"], default=None, help="override the precision of --config (same remark)")
    ap.add_argument("--layout", choices=["soa", "aos"], default="soa")
    ap.add_argument("--tile", type=int, nargs=4, default=None, help="tile of the tuned kernel (x y z t)")
    ap.add_argument("--occupancy", type=int, default=None, help="DSLASH_OPT_OCCUPANCY override")
    ap.add_argument("--kernel", choices=["auto", "direct", "wpipe", "march"], default=None)
    ap.add_argument("--l2-policy", type=int, default=None, help="DSLASH_OPT_L2_POLICY bits (direct kernel)")
    ap.add_argument("--march-policy", type=int, default=None, help="DSLASH_OPT_MARCH_POLICY bits (marching kernels)")
    ap.add_argument("--march-lead", type=int, default=None, help="DSLASH_OPT_MARCH_LEAD")
    ap.add_argument("--no-tune", action="store_true", help="skip dslash_tune (keep the library's static default kernel)")
    ap.add_argument("--pipe-slots", type=int, default=None, help="DSLASH_OPT_PIPE_SLOTS override (wpipe kernel)")
    ap.add_argument("--pipe-warps", type=int, default=None, help="DSLASH_OPT_PIPE_WARPS override (wpipe kernel)")
    ap.add_argument("--x-shuffle", type=int, choices=[0, 1], default=None, help="DSLASH_OPT_X_SHUFFLE override")
    ap.add_argument("--both-recon", action="store_true", default=True, help="also time the other link compression")
    ap.add_argument("--one-recon", dest="both_recon", action="store_false")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=10)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-parity", action="store_true", help="skip the whole-lattice parity check of the timed buffer")
    ap.add_argument("--graph", choices=["auto", "on", "off"], default="auto",
                    help="time the K applications of a region as one CUDA graph replay (auto: when the working set is L2-resident, "
                         "i.e. an application is too short for the host's launch rate)")
    ap.add_argument("--no-configs", action="store_true",
                    help="default run only: leave out the `configs` array (BASELINE configs[0], [1], [3], [4]) and the `sweep` summary")
    ap.add_argument("--skeleton", action="store_true",
                    help="measurement aid: time libdslash_b200_skeleton.so (python -m paper_2301_03636_b200.build --skeleton), the same "
                         "kernels with their arithmetic compiled out -- same loads, copies, hand-offs and stores.  The output is not "
                         "D psi: no parity, no cpu_baseline, no e2e; the line says \"skeleton\": true and is not a bench value")
    ap.add_argument("--repeats", type=int, default=5, help="K-step regions timed in all (median and min reported)")
    ap.add_argument("--cpu-sites", type=int, default=0, help="sites the cpu_baseline oracle run covers (0: the whole lattice, which "
                                                             "is also what the parity object needs)")
    ap.add_argument("--ref-sites", type=int, default=0, help="sites per step of --impl reference (0: the whole lattice)")
    ap.add_argument("--decomposition", choices=["replicas", "slab"], default="replicas",
                    help="multi-GPU mode: independent lattices per rank (default) or one lattice cut into T-slabs")
    ap.add_argument("--sweep", action="store_true")
    ap.add_argument("--sweep-csv", default=os.path.join(ROOT, "gpurun_out", "sweep_24x24x24x24.csv"))
    ap.add_argument("--advisor", action="store_true", help="run the paper's 84 offload variants (training-mode style)")
    ap.add_argument("--advisor-dims", type=int, nargs=4, default=[32, 32, 32, 16])
    ap.add_argument("--advisor-csv", default=os.path.join(ROOT, "gpurun_out", "advisor_variants.csv"))
    ap.add_argument("--team-size", type=int, default=128)
    ap.add_argument("--cg", action="store_true", help="time dslash_cg_solve on the --config lattice")
    ap.add_argument("--eo", action="store_true", help="time the even-odd operator, Mhat and dslash_eo_solve on the --config lattice")
    ap.add_argument("--cg-mass", type=float, default=0.2)
    ap.add_argument("--cg-tol", type=float, default=1e-8)
    ap.add_argument("--cg-max-iter", type=int, default=2000)
    ap.add_argument("--probe", action="store_true", help="read/write/copy/4:1-mix bandwidth and FP64 FMA rate of this board")
    ap.add_argument("--costmodel", action="store_true", help="fit the Advisor's cost model on the variants' measured runtimes")
    ap.add_argument("--profile-one", action="store_true", help="with --costmodel: one training launch of the paper's network size")
    ap.add_argument("--costmodel-f", type=int, default=33, help="--profile-one: number of features (33 = the paper's network)")
    ap.add_argument("--costmodel-cluster", type=int, default=8, help="--profile-one: thread blocks per model (0: library default)")
    ap.add_argument("--costmodel-threads", type=int, default=0, help="--profile-one: COSTMODEL_OPT_THREADS (0: library default)")
    ap.add_argument("--costmodel-lattices", type=int, default=len(COSTMODEL_LATTICES))
    ap.add_argument("--costmodel-epochs", type=int, default=150)
    ap.add_argument("--costmodel-models", type=int, default=16, help="independent seeds trained in the same launch")
    args = ap.parse_args()
    # the other BASELINE configs and the sweep ride on the plain default run only (the one the driver makes), not on experiments
    args.all_configs = (not args.no_configs and args.config == "3" and args.impl == "cuda" and not args.skeleton and not args.kernel
                        and not args.dims and not args.precision and not args.tile and args.decomposition != "slab"
                        and int(os.environ.get("WORLD_SIZE", "1")) == 1 and not args.no_parity)
    if args.skeleton:
        from paper_2301_03636_b200 import binding
        binding.load_skeleton()  # explicit switch: every later use of the binding in this process calls the skeleton library
        args.no_e2e = args.no_cpu_baseline = args.no_parity = True
    if args.warmup < 3 and args.impl == "cuda" and not args.sweep:
        args.warmup = 3  # timing rule: at least 3 warm-up steps
    if args.sweep:
        return run_sweep(args)
    if args.advisor:
        return run_advisor(args)
    if args.probe:
        return run_probe(args)
    if args.costmodel:
        return run_costmodel_profile_one(args) if args.profile_one else run_costmodel(args)
    if args.cg:
        return run_cg(args)
    if args.eo:
        return run_eo(args)
    cfg = dict(CONFIGS[args.config])
    if args.dims or args.precision:
        cfg["dims"] = tuple(args.dims) if args.dims else cfg["dims"]
        cfg["precision"] = args.precision or cfg["precision"]
        cfg["name"] = "off-contract: %s %s (--dims / --precision override of config %s)" % ("x".join(map(str, cfg["dims"])), cfg["precision"], args.config)
    if args.impl == "reference":
        return run_reference(args, cfg)
    if args.decomposition == "slab":
        return run_slab(args, cfg)
    return run_cuda(args, cfg)


if __name__ == "__main__":
    sys.exit(main())
