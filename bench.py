#!/usr/bin/env python
"""bench.py -- tLISI + detect throughput of the B200-native FITrig hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload stream50k] [--impl reference]

A "step" is one pass of the whole hot path (fitrig_tlisi + fitrig_detect: steps a1-a8 of DESIGN.md)
over one synthetic snapshot stack.  BASELINE.json's metric names no config, so the default workload is the largest
single-GPU one: configs[3] (4 snapshots of 50000 x 50000 fp32, 40 GB, N_T = 32, tau = 6) -- `value` with the stack
resident in HBM (fused kernel against the HBM roofline), `e2e` through fitrig_stream from 40 GB of pinned host memory
(against the PCIe rate measured in the same run: north_star's second target).  At N = 1 the default run then measures the
other BASELINE configs (meerkat, ska_aa2, imgfreq) the same way, each in a process of its own, and embeds them in the
one JSON line under "configs" (--no-configs leaves them out; an explicit --workload never adds them).

Prints ONE JSON line (rank 0).  Keys follow the driver's contract:
  value      whole-job Mpix/s (L*H*W pixels per step, summed over ranks), inputs resident in HBM,
             K steps timed with CUDA events between barrier+synchronize, max over ranks
  e2e        the same metric through fitrig_stream + fitrig_detect with HOST (pinned) snapshots:
             H2D copy of every snapshot and D2H of the tLISI map and candidate list inside the timed region
  roofline   fused kernel: algorithmic bytes / CUDA-event duration of its launches inside the timed region,
             against the measured HBM copy bandwidth of MEASURED_PEAKS.json
  cpu_baseline  the fp64 oracle (oracle/, as it stands) timed on this box's host cores (all cores, and one thread)
  ms_per_step_median / _min / _max   a second pass of the same K steps with a CUDA event after every step (PAPER.md:441
             quotes a median); the event records break the launch chain between steps, so `value` comes from the first pass
With --impl reference the oracle itself is the timed arm (host cores, no GPU work).
N > 1 (under torchrun, or started by this script when it is not): --scaling weak (default) gives every rank its own
independent stack (no data-path collective: tiles and fields are independent); --scaling strong
cuts ONE stack into row shards (one all-gather of the method's global scalars over NCCL).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "tLISI+detect snapshot Mpix/s"
UNIT = "Mpix/s"
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent
NOMINAL_HBM_GBS = 8000.0   # the "~8 TB/s" north_star quotes (HBM3e nominal); reported beside the measured copy peak
DEFAULT_WORKLOAD = "stream50k"  # BASELINE.json configs[3]: the largest single-GPU configuration
OTHER_CONFIGS = ("meerkat", "ska_aa2", "imgfreq")  # measured by the default run too, each in its own process
CPU_SAMPLE_MAX_ROWS = 16384  # the oracle legs look at no more than this many image rows of every snapshot
# dram__bytes_read.sum + dram__bytes_write.sum of ONE fused-kernel launch on the default workload, from the
# `ncu --set full` capture summarised in profiles/ (None until a capture has been taken for this build)
# (keyed to the build: `srchash` is paper_2509_21754_b200.build.source_hash() of the build the capture was taken on;
# any other build prints "traffic": null)
NCU_TRAFFIC = {"srchash": "212816b41d21bdc36f28b11a590cf5e9c50cafc2580eec2b89eefbbb4186267c", "stream50k": 40110947848, "meerkat": 1090717752}  # profiles/r03_b_ncu.md


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="fitrig", choices=["fitrig", "reference"])
    ap.add_argument("--workload", default=None, choices=["tiny", "meerkat", "ska_aa2", "stream50k", "imgfreq", "psr_like"])
    ap.add_argument("--tau", type=float, default=None)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=None)
    ap.add_argument("--channels", type=int, default=0, help="imgfreq only: use the first N of the 16 channels")
    ap.add_argument("--tile", type=int, default=32, help="N_T (the paper's default and BASELINE.json's is 32)")
    ap.add_argument("--harmonics", type=int, default=1, help="frequency branch: harmonic summing over 1,2,4..H harmonics")
    ap.add_argument("--width", type=int, default=0, help="override the image width W (e.g. 2050: W % 4 != 0 takes the generic path)")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = an independent stack per rank; strong = ONE stack cut into row shards (ShardedContext)")
    ap.add_argument("--no-pipeline", action="store_true", help="end every step with a synchronous fitrig_detect")
    ap.add_argument("--accumulate", type=int, default=1, help="snapshot accumulation g (PAPER.md:497): units = L / g - 2")
    ap.add_argument("--no-configs", action="store_true", help="default run: do not measure the other BASELINE configs")
    return ap.parse_args()


TILE = 32  # N_T of this run (--tile)
REC_BYTES = 16  # bytes of the per-tile, per-unit record the tLISI kernel writes (8 for tiles of one pixel)
ACCUMULATE = 1  # --accumulate
HARMONICS = 1  # --harmonics


def workload_desc(cfg, tau, branch, n_ch=1):
    return (f"{cfg.name}: {f'{n_ch} channels x ' if n_ch > 1 else ''}{cfg.L} snapshots x {cfg.H}x{cfg.W} fp32 "
            + (f"(BASELINE.json configs[{cfg.cfg_index - 1}]), " if cfg.cfg_index <= 5 else
               "(shape of the paper's real-data run, PAPER.md:371-395; not a BASELINE.json config), ")
            +
            f"N_T={TILE}, tau={tau:g}, branch={'image-frequency' if branch else 'image'}"
            + (f", accumulate={ACCUMULATE}" if ACCUMULATE > 1 else ""))


# ---------------------------------------------------------------------------------------------
# clocks: NVML sampled by a thread during the timed regions
# ---------------------------------------------------------------------------------------------
class ClockSampler:
    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
               0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x10: "sync_boost"}

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _loop(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in self.REASONS.items():
                    if mask & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.002)

    def start(self):
        if self.nv is not None:
            self._stop.clear()
            self._thread = threading.Thread(target=self._loop, daemon=True)
            self._thread.start()

    def stop(self):
        if self._thread is not None:
            self._stop.set()
            self._thread.join()
            self._thread = None

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": 0}
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2], "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(s)}


def measured_peak_gbs():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy bandwidth)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md, MEASURED_PEAKS.json absent)"


# ---------------------------------------------------------------------------------------------
# reference arm / cpu baseline: the oracle on the host cores
# ---------------------------------------------------------------------------------------------
def oracle_sample_rate(snaps, rows, tau, branch, repeats=1):
    """One oracle pass (O1..O7, or O8) over the first `rows` image rows of every snapshot -> seconds."""
    import numpy as np
    import oracle
    sub = [s[:rows] for s in snaps]
    best = None
    for _ in range(repeats):
        t0 = time.perf_counter()
        oracle.run(sub, tile=TILE, tau=tau, branch=branch, harmonics=HARMONICS, accumulate_g=ACCUMULATE)
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    return best


def choose_sample_rows(snaps, tau, branch, budget_s, passes):
    """Rows (multiple of 32) such that `passes` oracle passes take about budget_s."""
    H = snaps[0].shape[0]  # (the rows the caller holds: at most CPU_SAMPLE_MAX_ROWS of the image)
    probe = min(H, 256)
    t = oracle_sample_rate(snaps, probe, tau, branch)
    per_row = t / probe
    rows = int(budget_s / max(passes, 1) / max(per_row, 1e-9))
    rows = max(32, min(H, rows // 32 * 32))
    return H if rows >= H - 31 else rows


def host_stack(cfg, channel=0, max_rows=None):
    """Synthetic stack on the host as a list of [rows, W] numpy arrays, rows = min(H, max_rows): the first rows of
    every snapshot of the workload (generated on the GPU when there is one)."""
    import torch
    import synth
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    truth = synth.draw_truth(cfg, channel)
    steady = synth.steady_image(cfg, truth, dev)
    out = []
    for s in range(cfg.L):
        img = synth.snapshot(cfg, truth, steady, s)
        out.append((img if max_rows is None else img[:max_rows]).contiguous().cpu().numpy())
        del img
    return out


def cpu_model():
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.lower().startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def run_reference(args, cfg, tau, branch):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return  # rank 0 alone runs the oracle arm
    import oracle
    snaps = host_stack(cfg, max_rows=CPU_SAMPLE_MAX_ROWS)
    rows = choose_sample_rows(snaps, tau, branch, budget_s=150.0, passes=args.steps + args.warmup)
    for _ in range(args.warmup):
        oracle_sample_rate(snaps, rows, tau, branch)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_sample_rate(snaps, rows, tau, branch)
    dt = time.perf_counter() - t0
    pix = cfg.L * rows * cfg.W
    value = pix * args.steps / dt / 1e6
    sample = (f"first {rows} of {cfg.H} rows of all {cfg.L} snapshots per step "
              f"({100.0 * rows / cfg.H:.0f}% of the workload), {args.steps} steps")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_desc(cfg, tau, branch), "what": "CPU fp64 oracle (oracle/fitrig_oracle.c, "
                   "gcc -O2 -fopenmp) on the host cores; no GPU work"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", "sample": sample,
                         "cpu_model": cpu_model()},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# ---------------------------------------------------------------------------------------------
# the B200 arm
# ---------------------------------------------------------------------------------------------
def measure_h2d_gbs(torch, nbytes=1 << 30, reps=10):
    h = torch.empty(nbytes // 4, dtype=torch.float32).pin_memory()
    d = torch.empty(nbytes // 4, dtype=torch.float32, device="cuda")
    best = 0.0
    for _ in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        d.copy_(h, non_blocking=True)
        e1.record()
        torch.cuda.synchronize()
        best = max(best, nbytes / (e0.elapsed_time(e1) * 1e-3) / 1e9)
    del h, d
    return best


def timed(torch, stream, fn, barrier):
    """CUDA-event time (ms) of fn() on `stream`, bracketed by barrier + synchronize on both sides."""
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    fn()
    e1.record(stream)
    barrier()
    return e0.elapsed_time(e1)


def ncu_traffic(workload):
    """dram bytes of one fused-kernel launch from the committed ncu capture -- only if it was taken on THIS build."""
    from paper_2509_21754_b200 import build as lib_build
    if NCU_TRAFFIC.get("srchash") != lib_build.source_hash() or TILE != 32:
        return None
    return NCU_TRAFFIC.get(workload)


def run_fitrig(args, cfg, tau, branch):
    import numpy as np
    import torch
    import paper_2509_21754_b200 as fitrig
    import synth
    from paper_2509_21754_b200 import shard

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        raise RuntimeError(f"--gpus {args.gpus} but WORLD_SIZE={world}: launch through bench.py itself or torchrun with matching counts")
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the library has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    backend = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        backend = f"{dist.get_backend()} (NCCL {'.'.join(map(str, torch.cuda.nccl.version()))})"

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    dev = f"cuda:{local}"
    strong = args.scaling == "strong" and world > 1
    n_ch = cfg.n_channels if not args.channels else min(args.channels, cfg.n_channels)
    sampler = ClockSampler(local)
    stream = torch.cuda.current_stream()
    cap = 1 << 16
    outs = [np.zeros(cap, dtype=fitrig.binding.CANDIDATE_DTYPE) for _ in range(2)]
    num_sms = torch.cuda.get_device_properties(local).multi_processor_count

    if strong:
        # ---- ONE image stack cut into row shards: every rank reads only its rows of every snapshot;
        # one all-gather of 2 + 2U doubles (and 3 more in the frequency branch), then local detection and a gather
        # of the candidate lists.  Every rank draws the same stack (same seed) and keeps its own rows.
        full = synth.make_stack(cfg, device=dev, channel=0)[0]
        L, H, W = full.shape
        sc = shard.ShardedContext(H, W, L, rank, world, device=local, branch=branch, tile=TILE, harmonics=HARMONICS)
        rows = full[:, sc.r0:sc.r1].contiguous()
        del full
        torch.cuda.empty_cache()
        pix = L * H * W  # the whole job
        ctx = sc.ctx
        U, Ty, Tx = ctx.map_dims()

        def step():
            sc.tlisi(rows, None, stream)
            c_, n_ = sc.detect(tau, cap, stream)
            return sc.gather(c_, dev)

        for _ in range(max(args.warmup, 3)):
            merged = step()
        l0 = ctx.launch_count()
        sampler.start()
        ms = timed(torch, stream, lambda: [step() for _ in range(args.steps)], barrier)
        sampler.stop()
        launches = ctx.launch_count() - l0
        ms_max = shard.max_over_ranks(ms, dev)
        n_found = len(merged)

        def per_step_pass(k):
            evs = [torch.cuda.Event(enable_timing=True) for _ in range(k + 1)]
            barrier()
            evs[0].record(stream)
            for i in range(k):
                step()
                evs[i + 1].record(stream)
            barrier()
            return [evs[i].elapsed_time(evs[i + 1]) for i in range(k)]

        step_times = per_step_pass(args.steps)
        ctx.profile(True)
        timed(torch, stream, lambda: [step() for _ in range(args.steps)], barrier)
        main_tot, main_n, fin_tot, fin_n = ctx.last_timing()
        ctx.profile(False)
        my_pix = L * (sc.r1 - sc.r0) * W
        alg_bytes = 4 * my_pix + REC_BYTES * U * Ty * Tx
        ms_sync = ms_max
        e2e = None
        cpu = None
        stacks = None
    else:
        # ---- every rank owns independent stacks (different noise and field per rank): weak scaling, no data-path
        # collective.  config 5 (R19): the 16 frequency channels are a batch of independent stacks, all resident (34 GB)
        rcfg = cfg if world == 1 else cfg.replace(cfg_index=cfg.cfg_index + 100 * rank)
        stacks = [synth.make_stack(rcfg, device=dev, channel=ch)[0] for ch in range(n_ch)]
        L, H, W = stacks[0].shape
        pix = L * H * W * n_ch * world
        my_pix = L * H * W
        ctx = fitrig.Context(H, W, L, device=local, branch=branch, tile=TILE, harmonics=HARMONICS, batch=n_ch, accumulate=ACCUMULATE)
        U, Ty, Tx = ctx.map_dims()
        d_tl = torch.empty((n_ch, U, Ty, Tx), dtype=torch.float32, device=dev)

        def step_sync():
            ctx.tlisi_batch(stacks, d_tl, stream)
            return ctx.detect_batch(tau, cap, stream, out=outs[0])

        def pipelined(k):
            """K steps; the candidate list of step i is fetched after step i + 1 has been queued (two result slots),
            so the device never waits for the host.  Every step's map and list is produced and delivered."""
            res = None
            for i in range(k):
                ctx.tlisi_batch(stacks, d_tl, stream)
                ctx.detect_launch(tau, cap, stream)
                if i > 0:
                    res = ctx.detect_fetch(outs[(i - 1) & 1])
            return ctx.detect_fetch(outs[(k - 1) & 1])

        for _ in range(max(args.warmup, 3)):
            cands, n_found, per_stack = step_sync()
        pipelined(2)
        l0 = ctx.launch_count()
        sampler.start()
        if args.no_pipeline:
            ms = timed(torch, stream, lambda: [step_sync() for _ in range(args.steps)], barrier)
        else:
            ms = timed(torch, stream, lambda: pipelined(args.steps), barrier)
        sampler.stop()
        launches = ctx.launch_count() - l0
        ms_max = shard.max_over_ranks(ms, dev)

        def per_step_pass(k):
            """The same K steps once more with a CUDA event behind every step's launches (the per-step distribution)."""
            evs = [torch.cuda.Event(enable_timing=True) for _ in range(k + 1)]
            barrier()
            evs[0].record(stream)
            for i in range(k):
                if args.no_pipeline:
                    step_sync()
                else:
                    ctx.tlisi_batch(stacks, d_tl, stream)
                    ctx.detect_launch(tau, cap, stream)
                evs[i + 1].record(stream)
                if not args.no_pipeline and i > 0:
                    ctx.detect_fetch(outs[(i - 1) & 1])
            if not args.no_pipeline:
                ctx.detect_fetch(outs[(k - 1) & 1])
            barrier()
            return [evs[i].elapsed_time(evs[i + 1]) for i in range(k)]

        step_times = per_step_pass(args.steps)
        # the same steps, each ended by its own synchronous fitrig_detect (host round trip inside every step)
        ms_sync = shard.max_over_ranks(timed(torch, stream, lambda: [step_sync() for _ in range(args.steps)], barrier), dev)
        # the same steps once more with the library's CUDA events around its own launches (on the launching stream)
        ctx.profile(True)
        timed(torch, stream, lambda: [step_sync() for _ in range(args.steps)], barrier)
        main_tot, main_n, fin_tot, fin_n = ctx.last_timing()
        ctx.profile(False)
        alg_bytes = 4 * my_pix + REC_BYTES * U * Ty * Tx  # one launch = one stack: every pixel once + one record per tile and unit

    value = pix * args.steps / (ms_max * 1e-3) / 1e6

    # ---- roofline of the dominant (fused) kernel, and of the whole step ----
    plan = fitrig.plan_query(H if not strong else sc.r1 - sc.r0, W, L, num_sms=num_sms, tile=TILE, accumulate=ACCUMULATE)
    k_ms = main_tot / max(main_n, 1)
    peak, peak_src = measured_peak_gbs()
    achieved = alg_bytes / (k_ms * 1e-3) / 1e9
    read_peak = ctx.probe_read_bandwidth(stacks[0] if stacks else rows) if rank == 0 else None
    launches_per_step = n_ch if not strong else 1
    step_bytes = alg_bytes * launches_per_step + 8 * n_ch * U * Ty * Tx  # + q and tLISI written by the finalise
    step_ms = ms_max / args.steps
    # which tLISI kernel the library takes (the plan is host-only and assumes a 16-byte aligned base): rows off 16-byte
    # boundaries (W % 4 != 0) ride the fused kernel's super-row variant where the plan says fused
    path_name = ("fused-tma (super rows)" if W % 4 else "fused-tma") if plan.path == 0 else "generic"  # (fitrig_plan_query decides)
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": ncu_traffic(cfg.name), "kernel": "tlisi_fused_kernel" if path_name != "generic" else
                "tlisi_march_kernel", "kernel_ms": k_ms, "algorithmic_bytes": alg_bytes, "peak_source": peak_src,
                "read_only_peak": read_peak, "frac_of_read_only_peak": (achieved / read_peak) if read_peak else None,
                "read_only_peak_source": "fitrig_probe_read_bandwidth: plain float4 grid-stride read of the same stack, best of 5, this run",
                "finalize_ms": fin_tot / max(fin_n, 1), "kernel_launches_timed": main_n,
                "kernel_share_of_step": k_ms * launches_per_step / step_ms,
                "step_achieved": step_bytes / (step_ms * 1e-3) / 1e9, "step_frac": step_bytes / (step_ms * 1e-3) / 1e9 / peak,
                "step_bytes": step_bytes,
                "step_frac_sync": step_bytes / (ms_sync / args.steps * 1e-3) / 1e9 / peak,
                "nominal_peak": NOMINAL_HBM_GBS, "frac_of_nominal": achieved / NOMINAL_HBM_GBS,
                "nominal_peak_source": "the ~8 TB/s HBM3e figure north_star quotes; `frac` is against the measured copy bandwidth",
                "kernel_timing": "a separate pass of the same K steps, each ended by a blocking fitrig_detect, under fitrig_profile(1): "
                                 "the library's CUDA events around every tLISI kernel launch on the launching stream.  Profiling turns "
                                 "the programmatic-dependent-launch chain off, so these are the same kernels on the same data but "
                                 "not the very launches `value` was timed on"}

    # ---- end to end: host (pinned) snapshots -> fitrig_stream -> fitrig_detect -> host results ----
    if not strong:
        e2e = None
    if not strong and not args.no_e2e:
        h2d_gbs = measure_h2d_gbs(torch) if rank == 0 else None
        ectx = ctx if n_ch == 1 else fitrig.Context(H, W, L, device=local, branch=branch, tile=TILE, harmonics=HARMONICS, accumulate=ACCUMULATE)
        hosts = []
        for st_c in stacks:
            host = torch.empty((L, H, W), dtype=torch.float32, pin_memory=True)  # (page-locked at once: no pageable twin)
            host.copy_(st_c)
            hosts.append([host[s] for s in range(L)])
        h_tl = torch.empty((U, Ty, Tx), dtype=torch.float32).pin_memory()
        ksteps = args.e2e_steps or max(3, min(args.steps, int(20e9 // (4 * pix // world)) or 1))

        def e2e_step():
            n_tot = 0
            for snaps in hosts:
                ectx.stream(snaps, h_tl, stream)
                c_, n_ = ectx.detect(tau, cap, stream, out=outs[0])
                n_tot += n_
            return c_, n_tot

        for _ in range(2):
            c2, n2 = e2e_step()
        sampler.start()
        e_ms = timed(torch, stream, lambda: [e2e_step() for _ in range(ksteps)], barrier)
        sampler.stop()
        c2, n2 = e2e_step()
        e_ms = shard.max_over_ranks(e_ms, dev) / ksteps
        assert n2 == n_found, "streamed and resident paths disagree on the candidate count"
        e2e = {"value": pix / (e_ms * 1e-3) / 1e6, "unit": UNIT, "h2d_bytes_per_step": 4 * pix // world,
               "d2h_bytes_per_step": n_ch * (4 * U * Ty * Tx + 16) + 16 * int(min(n_found, 4096 * n_ch)), "ms_per_step": e_ms,
               "steps": ksteps, "api": "fitrig_stream + fitrig_detect (pinned host snapshots, row strips)",
               "roofline": {"bound": "pcie", "achieved": 4 * pix / world / (e_ms * 1e-3) / 1e9, "peak": h2d_gbs,
                            "unit": "GB/s", "frac": (4 * pix / world / (e_ms * 1e-3) / 1e9 / h2d_gbs) if h2d_gbs else None,
                            "peak_source": "pinned 1 GiB cudaMemcpyAsync H2D, best of 10, this run"}}
        # ---- real-time leg: fitrig_push, one snapshot per call from pinned host memory (Fig. 14 timeline) ----
        # ---- the copy / kernel timeline of one more streamed pass (library CUDA events, fitrig_stream_timeline) ----
        ectx.profile(True)
        ectx.stream(hosts[0], h_tl, stream)
        torch.cuda.synchronize()
        tl = ectx.stream_timeline()
        ectx.profile(False)
        if len(tl):
            copy_ms = float((tl[:, 1] - tl[:, 0]).sum())
            kern_ms = float((tl[:, 3] - tl[:, 2]).sum())
            # time a kernel spends while the copy stream is busy with a LATER strip's copy
            hidden = 0.0
            for i in range(len(tl)):
                for j in range(i + 1, len(tl)):
                    hidden += max(0.0, float(min(tl[i, 3], tl[j, 1]) - max(tl[i, 2], tl[j, 0])))
            e2e["timeline"] = {"strips": int(len(tl)), "span_ms": float(tl[:, 3].max() - tl[:, 0].min()), "copy_ms_sum": copy_ms,
                               "kernel_ms_sum": kern_ms, "kernel_ms_hidden_under_later_copies": hidden,
                               "first_strips_ms": [[round(float(v), 4) for v in row] for row in tl[:4]],
                               "columns": "copy start, copy end, kernel start, kernel end (ms from the first copy's start)",
                               "source": "fitrig_stream_timeline: CUDA events of one streamed pass of stack 0 under fitrig_profile(1), outside the timed region"}
        if ACCUMULATE == 1:  # (fitrig_push does not accumulate)
            window = 3 if branch == 0 else min(L, 18)
            pctx = fitrig.Context(H, W, window, device=local, tile=TILE, branch=branch, harmonics=HARMONICS)
            snaps0 = hosts[0]

            def push_pass():
                tot = 0
                for s_ in snaps0 + [None]:
                    u_, c_, n_ = pctx.push(s_, tau, None, cap, stream, out=outs[0])
                    tot += n_
                pctx.push_reset()
                return tot

            push_pass()
            barrier()
            t_wall = time.perf_counter()
            n_rt = push_pass()
            barrier()
            p_ms = shard.max_over_ranks((time.perf_counter() - t_wall) * 1e3, dev)
            e2e["realtime"] = {"value": world * L * H * W / (p_ms * 1e-3) / 1e6, "unit": UNIT, "ms_per_snapshot": p_ms / L,
                               "api": "fitrig_push (one pinned host snapshot per call, running M, candidates per unit"
                                      + (f"; frequency branch: Eq. 10-12 over the cube of the last {window - 2} units" if branch else "") + ")",
                               "candidates": int(n_rt), "h2d_gbs": 4 * L * H * W / (p_ms * 1e-3) / 1e9,
                               "timer": "host wall clock around the pass (every push synchronises)"}
            pctx.close()
        if ectx is not ctx:
            ectx.close()
        del hosts

    # ---- the oracle beside it (rank 0, N = 1 only) ----
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle
        snaps_np = [stacks[0][s][:CPU_SAMPLE_MAX_ROWS].contiguous().cpu().numpy() for s in range(L)]
        rows_s = choose_sample_rows(snaps_np, tau, branch, budget_s=12.0, passes=1)
        npass, t_cpu = 0, 0.0
        while t_cpu < 12.0 and npass < 1000:  # about 12 s of CPU work: repeat the pass when one is shorter
            t_cpu += oracle_sample_rate(snaps_np, rows_s, tau, branch)
            npass += 1
        cores = oracle.num_threads()
        cpu = {"value": npass * L * rows_s * W / t_cpu / 1e6, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"{npass} passes over the first {rows_s} of {H} rows of all {L} snapshots"
                         f"{' of channel 0' if n_ch > 1 else ''} ({t_cpu:.1f} s in total)",
               "cpu_model": cpu_model()}
        # the same oracle on ONE thread (single thread and all cores), a smaller sample of the same rows
        oracle.set_threads(1)
        try:
            rows_1 = choose_sample_rows(snaps_np, tau, branch, budget_s=6.0, passes=1)
            npass1, t1 = 0, 0.0
            while t1 < 6.0 and npass1 < 1000:
                t1 += oracle_sample_rate(snaps_np, rows_1, tau, branch)
                npass1 += 1
            cpu["single_thread"] = {"value": npass1 * L * rows_1 * W / t1 / 1e6, "unit": UNIT, "cores": 1,
                                    "sample": f"{npass1} passes over the first {rows_1} of {H} rows of all {L} snapshots ({t1:.1f} s in total)"}
        finally:
            oracle.set_threads(cores)
        del snaps_np

    if rank == 0:
        from paper_2509_21754_b200 import build as lib_build
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": step_ms, "ms_per_step_median": float(np.median(step_times)),
            "ms_per_step_min": float(min(step_times)), "ms_per_step_max": float(max(step_times)),
            "ms_per_step_distribution": "a second pass of the same K steps with a CUDA event recorded behind every step's launches "
                                        "(PAPER.md:441 quotes a median; rank 0); an event record between two steps breaks the "
                                        "programmatic-dependent-launch chain, so `value` and `ms_per_step` come from the first, unbroken pass",
            "higher_is_better": True,
            "scaling": "strong" if strong else "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_desc(cfg, tau, branch, n_ch), "tile": TILE, "tau": tau, "harmonics": HARMONICS,
                       "candidates_per_step": int(n_found),
                       "step": ("one image cut into row shards: fitrig_tlisi on the shard + all-gather of 2+2U doubles + "
                                "fitrig_shard_import + fitrig_detect + candidate gather, every step synchronous") if strong else
                               ("fitrig_tlisi_batch + fitrig_detect (synchronous, one host round trip per step)" if args.no_pipeline else
                                "fitrig_tlisi_batch + fitrig_detect_launch; fitrig_detect_fetch of step i after step i+1 was queued "
                                "(two result slots; every step's map and candidate list is produced and delivered inside the timed region)"),
                       "ms_per_step_sync": ms_sync / args.steps,
                       "l2": f"input {4 * pix // world / 1e6:.0f} MB per step vs 126 MB L2: "
                             + ("larger than L2, no flush" if 4 * pix // world > 2 * 126e6 else "fits L2 (launch-latency-bound config)"),
                       "plan": {"path": path_name, "units_per_cta": plan.units_per_cta, "box_tiles": plan.box_tiles,
                                "warps_per_cta": plan.warps_per_cta, "stages": plan.stages, "grid": plan.grid},
                       "build": lib_build.source_hash()[:16], "dist_backend": backend},
            "clocks": sampler.summary(), "e2e": e2e, "gpu_launches": int(launches) * world,
            "roofline": roofline, "cpu_baseline": cpu,
        }
    ctx.close()
    if rank == 0:
        if world == 1 and args.default_run and not args.no_configs:
            # the other BASELINE configs, each measured by this same script in a process of its own (the 40 GB of this run
            # are released first), summarised under one key of the one line
            del stacks, d_tl
            torch.cuda.empty_cache()
            line["configs"] = {name: sub_record(args, name) for name in OTHER_CONFIGS}
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def sub_record(args, name):
    """`bench.py --workload name` in a child process -> the keys that summarise it (never raises: a failure is recorded)."""
    import subprocess
    cmd = [sys.executable, os.path.abspath(__file__), "--workload", name, "--steps", str(args.steps), "--warmup", str(args.warmup),
           "--no-cpu-baseline"] + (["--no-e2e"] if name == "imgfreq" else [])
    t0 = time.perf_counter()
    try:
        r = subprocess.run(cmd, capture_output=True, text=True, timeout=300)
        rec = json.loads(r.stdout.strip().splitlines()[-1])
    except Exception as e:  # noqa: BLE001
        return {"error": f"{type(e).__name__}: {e}"[:300], "command": " ".join(cmd[1:])}
    rf, e2e = rec["roofline"], rec.get("e2e")
    out = {"workload": rec["config"]["workload"], "value": rec["value"], "unit": rec["unit"], "steps": rec["steps"],
           "ms_per_step": rec["ms_per_step"], "ms_per_step_median": rec["ms_per_step_median"], "ms_per_step_min": rec["ms_per_step_min"],
           "ms_per_step_max": rec["ms_per_step_max"], "ms_per_step_sync": rec["config"]["ms_per_step_sync"],
           "candidates_per_step": rec["config"]["candidates_per_step"], "clocks": rec["clocks"], "gpu_launches": rec["gpu_launches"],
           "roofline": {k: rf[k] for k in ("bound", "kernel", "kernel_ms", "achieved", "peak", "unit", "frac", "frac_of_nominal", "algorithmic_bytes",
                                           "read_only_peak", "kernel_share_of_step", "finalize_ms", "step_frac", "step_frac_sync", "traffic")},
           "e2e": None if not e2e else {"value": e2e["value"], "unit": e2e["unit"], "ms_per_step": e2e["ms_per_step"], "steps": e2e["steps"],
                                        "h2d_bytes_per_step": e2e["h2d_bytes_per_step"], "d2h_bytes_per_step": e2e["d2h_bytes_per_step"],
                                        "roofline": e2e["roofline"]},
           "command": "python bench.py " + " ".join(cmd[2:]), "wall_s": round(time.perf_counter() - t0, 1)}
    return out


def relaunch_under_torchrun(args):
    """`python bench.py --gpus N` with N > 1 and no torchrun around it: start the N ranks ourselves."""
    import socket
    import subprocess
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    sys.exit(subprocess.call(cmd))


def main():
    global TILE, HARMONICS, REC_BYTES, ACCUMULATE
    args = parse_args()
    TILE, HARMONICS, ACCUMULATE = args.tile, args.harmonics, args.accumulate
    REC_BYTES = 8 if TILE == 1 else 16
    import synth
    args.default_run = args.workload is None
    if args.default_run:
        args.workload = DEFAULT_WORKLOAD
    cfg = synth.CONFIGS[args.workload]
    if args.workload == "stream50k":  # (both arms, so that they name the same workload)
        # SURVEY.md 8(d), cfg 4: "if the host cannot lock 40 GB, fall back to 4 x 36000^2 (20.7 GB)" -- decided from the
        # memory the box reports as available (the pinned copy of the stack + the oracle's sample + slack)
        try:
            import psutil
            avail = psutil.virtual_memory().available
        except Exception:  # noqa: BLE001
            avail = None
        if avail is not None and avail < 64e9:
            cfg = synth.scaled(cfg, 36000, 36000, name="stream50k_fallback36000")
    if args.width:
        cfg = cfg.replace(W=args.width, name=f"{cfg.name}_w{args.width}")
    tau = args.tau if args.tau is not None else cfg.tau
    branch = 1 if args.workload in ("imgfreq", "psr_like") else 0
    if args.impl == "reference":
        run_reference(args, cfg, tau, branch)
    elif args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        relaunch_under_torchrun(args)
    else:
        run_fitrig(args, cfg, tau, branch)


if __name__ == "__main__":
    main()
