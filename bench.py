#!/usr/bin/env python
"""bench.py -- tLISI + detect throughput of the B200-native FITrig hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload meerkat] [--impl reference]

A "step" is one pass of the whole hot path (fitrig_tlisi + fitrig_detect: steps a1-a8 of DESIGN.md)
over one synthetic snapshot stack.  Default workload = BASELINE.json configs[1] (MeerKAT-like,
64 x 2048 x 2048 fp32, N_T = 32, tau = 5), the configuration the metric is quoted on.

Prints ONE JSON line (rank 0).  Keys follow the driver's contract:
  value      whole-job Mpix/s (L*H*W pixels per step, summed over ranks), inputs resident in HBM,
             K steps timed with CUDA events between barrier+synchronize, max over ranks
  e2e        the same metric through fitrig_stream + fitrig_detect with HOST (pinned) snapshots:
             H2D copy of every snapshot and D2H of the tLISI map and candidate list inside the timed region
  roofline   fused kernel: algorithmic bytes / CUDA-event duration of its launches inside the timed region,
             against the measured HBM copy bandwidth of MEASURED_PEAKS.json
  cpu_baseline  the fp64 oracle (oracle/, as it stands) timed on this box's host cores
With --impl reference the oracle itself is the timed arm (host cores, no GPU work).
Under torchrun (N > 1) every rank processes its own independent stack (weak scaling, no data-path
collective: tiles and fields are independent).
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
# dram__bytes_read.sum + dram__bytes_write.sum of ONE fused-kernel launch on the default workload, from the
# `ncu --set full` capture summarised in profiles/ (None until a capture has been taken for this build)
NCU_TRAFFIC_BYTES = {"meerkat": 1091050016}  # profiles/r01_e_final.md: 1 083 252 000 read + 7 798 016 written


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="fitrig", choices=["fitrig", "reference"])
    ap.add_argument("--workload", default="meerkat", choices=["tiny", "meerkat", "ska_aa2", "stream50k", "imgfreq", "psr_like"])
    ap.add_argument("--tau", type=float, default=None)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=None)
    ap.add_argument("--channels", type=int, default=0, help="imgfreq only: use the first N of the 16 channels")
    ap.add_argument("--tile", type=int, default=32, help="N_T (the paper's default and BASELINE.json's is 32)")
    ap.add_argument("--harmonics", type=int, default=1, help="frequency branch: harmonic summing over 1,2,4..H harmonics")
    return ap.parse_args()


TILE = 32  # N_T of this run (--tile)
HARMONICS = 1  # --harmonics


def workload_desc(cfg, tau, branch, n_ch=1):
    return (f"{cfg.name}: {f'{n_ch} channels x ' if n_ch > 1 else ''}{cfg.L} snapshots x {cfg.H}x{cfg.W} fp32 "
            + (f"(BASELINE.json configs[{cfg.cfg_index - 1}]), " if cfg.cfg_index <= 5 else
               "(shape of the paper's real-data run, PAPER.md:371-395; not a BASELINE.json config), ")
            +
            f"N_T={TILE}, tau={tau:g}, branch={'image-frequency' if branch else 'image'}")


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
        oracle.run(sub, tile=TILE, tau=tau, branch=branch, harmonics=HARMONICS)
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    return best


def choose_sample_rows(snaps, tau, branch, budget_s, passes):
    """Rows (multiple of 32) such that `passes` oracle passes take about budget_s."""
    H = snaps[0].shape[0]
    probe = min(H, 256)
    t = oracle_sample_rate(snaps, probe, tau, branch)
    per_row = t / probe
    rows = int(budget_s / max(passes, 1) / max(per_row, 1e-9))
    rows = max(32, min(H, rows // 32 * 32))
    return H if rows >= H - 31 else rows


def host_stack(cfg, channel=0):
    """Synthetic stack on the host as a list of [H, W] numpy arrays (generated on the GPU when there is one)."""
    import torch
    import synth
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    truth = synth.draw_truth(cfg, channel)
    steady = synth.steady_image(cfg, truth, dev)
    out = []
    for s in range(cfg.L):
        out.append(synth.snapshot(cfg, truth, steady, s).cpu().numpy())
    return out


def run_reference(args, cfg, tau, branch):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return  # rank 0 alone runs the oracle arm
    import oracle
    snaps = host_stack(cfg)
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
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
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


def run_fitrig(args, cfg, tau, branch):
    import numpy as np
    import torch
    import paper_2509_21754_b200 as fitrig
    import synth
    from paper_2509_21754_b200 import shard

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the library has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    dev = f"cuda:{local}"
    # every rank owns an independent stack (different noise and field per rank): weak scaling
    # config 5 (R19): the 16 frequency channels are a batch of independent stacks, all resident (34 GB)
    n_ch = cfg.n_channels if not args.channels else min(args.channels, cfg.n_channels)
    rcfg = cfg if world == 1 else cfg.replace(cfg_index=cfg.cfg_index + 100 * rank)
    stacks = [synth.make_stack(rcfg, device=dev, channel=ch)[0] for ch in range(n_ch)]
    stack = stacks[0]
    L, H, W = stack.shape
    pix = L * H * W * n_ch
    ctx = fitrig.Context(H, W, L, device=local, branch=branch, tile=TILE, harmonics=HARMONICS)
    U, Ty, Tx = ctx.map_dims()
    d_tl = torch.empty((U, Ty, Tx), dtype=torch.float32, device=dev)
    cap = 1 << 16
    out = np.zeros(cap, dtype=fitrig.binding.CANDIDATE_DTYPE)
    stream = torch.cuda.current_stream()

    def step():
        n_tot = 0
        for st_c in stacks:
            ctx.tlisi(st_c, d_tl, stream)
            c_, n_ = ctx.detect(tau, cap, stream, out=out)
            n_tot += n_
        return c_, n_tot

    sampler = ClockSampler(local)
    for _ in range(max(args.warmup, 3)):
        cands, n_found = step()
    ctx.profile(True)
    barrier()
    l0 = ctx.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler.start()
    e0.record(stream)
    for _ in range(args.steps):
        step()
    e1.record(stream)
    barrier()
    sampler.stop()
    launches = ctx.launch_count() - l0
    ms = e0.elapsed_time(e1)
    # CUDA events the library recorded around its own launches, on the launching stream, during the timed region
    main_tot, main_n, fin_tot, fin_n = ctx.last_timing()
    ctx.profile(False)
    ms_max = shard.max_over_ranks(ms, dev)  # device time of the slowest rank
    value = world * pix * args.steps / (ms_max * 1e-3) / 1e6

    # ---- roofline of the dominant (fused) kernel ----
    plan = fitrig.plan_query(H, W, L, num_sms=torch.cuda.get_device_properties(local).multi_processor_count, tile=TILE)
    # one launch = one channel's stack: every snapshot pixel read once + one 16-byte record per tile and unit
    alg_bytes = 4 * (pix // n_ch) + 16 * U * Ty * Tx
    traffic = NCU_TRAFFIC_BYTES.get(cfg.name) if TILE == 32 else None
    k_ms = main_tot / max(main_n, 1)
    peak, peak_src = measured_peak_gbs()
    achieved = alg_bytes / (k_ms * 1e-3) / 1e9
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": traffic, "kernel": "tlisi_fused_kernel" if plan.path == 0 else
                "tlisi_generic_kernel", "kernel_ms": k_ms, "algorithmic_bytes": alg_bytes, "peak_source": peak_src,
                "finalize_ms": fin_tot / max(fin_n, 1), "kernel_launches_timed": main_n, "kernel_share_of_step": k_ms * n_ch * args.steps / ms}

    # ---- end to end: host (pinned) snapshots -> fitrig_stream -> fitrig_detect -> host results ----
    e2e = None
    if not args.no_e2e:
        h2d_gbs = measure_h2d_gbs(torch) if rank == 0 else None
        hosts = []
        for st_c in stacks:
            host = torch.empty((L, H, W), dtype=torch.float32).pin_memory()
            host.copy_(st_c)
            hosts.append([host[s] for s in range(L)])
        h_tl = torch.empty((U, Ty, Tx), dtype=torch.float32).pin_memory()
        ksteps = args.e2e_steps or max(3, min(args.steps, int(20e9 // (4 * pix)) or 1))

        def e2e_step():
            n_tot = 0
            for snaps in hosts:
                ctx.stream(snaps, h_tl, stream)
                c_, n_ = ctx.detect(tau, cap, stream, out=out)
                n_tot += n_
            return c_, n_tot

        for _ in range(2):
            c2, n2 = e2e_step()
        barrier()
        sampler.start()
        f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        f0.record(stream)
        for _ in range(ksteps):
            c2, n2 = e2e_step()
        f1.record(stream)
        barrier()
        sampler.stop()
        e_ms = shard.max_over_ranks(f0.elapsed_time(f1), dev) / ksteps
        assert n2 == n_found, "streamed and resident paths disagree on the candidate count"
        e2e = {"value": world * pix / (e_ms * 1e-3) / 1e6, "unit": UNIT, "h2d_bytes_per_step": 4 * pix,
               "d2h_bytes_per_step": n_ch * (4 * U * Ty * Tx + 16) + 16 * int(min(n_found, 4096 * n_ch)), "ms_per_step": e_ms,
               "steps": ksteps, "api": "fitrig_stream + fitrig_detect (pinned host snapshots, row strips)",
               "roofline": {"bound": "pcie", "achieved": 4 * pix / (e_ms * 1e-3) / 1e9, "peak": h2d_gbs,
                            "unit": "GB/s", "frac": (4 * pix / (e_ms * 1e-3) / 1e9 / h2d_gbs) if h2d_gbs else None,
                            "peak_source": "pinned 1 GiB cudaMemcpyAsync H2D, best of 10, this run"}}
        # ---- real-time leg: fitrig_push, one snapshot per call from pinned host memory (Fig. 14 timeline) ----
        if branch == 0:
            pctx = fitrig.Context(H, W, 3, device=local, tile=TILE)
            snaps0 = hosts[0]

            def push_pass():
                tot = 0
                for s_ in snaps0 + [None]:
                    u_, c_, n_ = pctx.push(s_, tau, None, cap, stream, out=out)
                    tot += n_
                pctx.push_reset()
                return tot

            push_pass()
            barrier()
            g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            g0.record(stream)
            t_wall = time.perf_counter()
            n_rt = push_pass()
            g1.record(stream)
            barrier()
            p_ms = shard.max_over_ranks((time.perf_counter() - t_wall) * 1e3, dev)
            e2e["realtime"] = {"value": world * L * H * W / (p_ms * 1e-3) / 1e6, "unit": UNIT, "ms_per_snapshot": p_ms / L,
                               "api": "fitrig_push (one pinned host snapshot per call, running M, candidates per unit)",
                               "candidates": int(n_rt), "h2d_gbs": 4 * L * H * W / (p_ms * 1e-3) / 1e9,
                               "timer": "host wall clock around the pass (every push synchronises)"}
            pctx.close()
        del hosts

    # ---- the oracle beside it (rank 0, N = 1 only) ----
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle
        snaps_np = [stack[s].cpu().numpy() for s in range(L)]
        rows = choose_sample_rows(snaps_np, tau, branch, budget_s=12.0, passes=1)
        npass, t_cpu = 0, 0.0
        while t_cpu < 12.0 and npass < 1000:  # about 12 s of CPU work: repeat the pass when one is shorter
            t_cpu += oracle_sample_rate(snaps_np, rows, tau, branch)
            npass += 1
        cpu = {"value": npass * L * rows * W / t_cpu / 1e6, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
               "sample": f"{npass} passes over the first {rows} of {H} rows of all {L} snapshots"
                         f"{' of channel 0' if n_ch > 1 else ''} ({t_cpu:.1f} s in total)"}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_max / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_desc(cfg, tau, branch, n_ch), "tile": TILE, "tau": tau, "harmonics": HARMONICS,
                       "candidates_per_step": int(n_found),
                       "l2": f"input {4 * pix / 1e6:.0f} MB per step vs 126 MB L2: "
                             + ("larger than L2, no flush" if 4 * pix > 2 * 126e6 else "fits L2 (launch-latency-bound config)"),
                       "plan": {"path": "fused-tma" if plan.path == 0 else "generic", "units_per_cta": plan.units_per_cta, "box_tiles": plan.box_tiles,
                                "warps_per_cta": plan.warps_per_cta, "stages": plan.stages, "grid": plan.grid}},
            "clocks": sampler.summary(), "e2e": e2e, "gpu_launches": int(launches) * world,
            "roofline": roofline, "cpu_baseline": cpu,
        }
        print(json.dumps(line))
    ctx.close()
    if dist is not None:
        dist.destroy_process_group()


def main():
    global TILE, HARMONICS
    args = parse_args()
    TILE, HARMONICS = args.tile, args.harmonics
    import synth
    cfg = synth.CONFIGS[args.workload]
    tau = args.tau if args.tau is not None else cfg.tau
    branch = 1 if args.workload in ("imgfreq", "psr_like") else 0
    if args.impl == "reference":
        run_reference(args, cfg, tau, branch)
    else:
        run_fitrig(args, cfg, tau, branch)


if __name__ == "__main__":
    main()
