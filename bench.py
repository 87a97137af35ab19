#!/usr/bin/env python
"""bench.py — throughput of the GH right-hand-side hot path (arXiv 1804.09101) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload c4|c3|c2|c1|c5]

Metric (BASELINE.json): GH RHS grid-point evaluations per second, FP64.  One "step" is one pass of the whole
hot path (rows A2-A8) over the workload: one `gh_rk_step_norms` = 3 x [Chebyshev + angular derivatives,
fused Jacobian + pointwise RHS + face mask + RK3 stage update as its epilogue], with the constraint norms of the step's
input state as an epilogue of the first stage (A8 fused into A5).  value = 3 * P * K / T.
Protocol (the paper's): W >= 3 warm-up steps, then K timed steps with the library's
per-launch events OFF; `ms_per_step` = T / K over the whole region, `ms_per_step_median` = median of the K per-step CUDA-event
times; the per-kernel split comes from a SECOND pass with the per-launch events on; the FP64 peak the derivative kernels
are quoted against is measured in the same run (gh_fp64_peak).
`--workload c5` is the size sweep of BASELINE.json configs[4]: one JSON line per member (single shells N_r = L+1 = n and
single cubes N^3, 1e3 ... 3.3e7 points): gh_rhs points/s, derivative-kernel FP64 rate, k_rhs GB/s.

Default workload: C4 (BASELINE.json configs[3], the production-like isolated-BH domain: 40 shells + 24 cube
blocks, spin 0.9, replicated to >= 4M points, reading S13) - the configuration the HBM-roofline part of the
metric is meaningful on (C1/C2 are L2-resident latency cases).  All inputs are seeded and synthetic
(analytic Kerr-Schild data + smooth seeded perturbations).

N > 1 (torchrun): the path does not shard inside one call ("replicas only"): every rank runs its own
replica of the workload on its own GPU, no data-path collective; value = N * 3 * P * K / max-over-ranks(T).

`--impl reference` times the CPU oracle (oracle/, test infrastructure, as it stands) on a bounded sample of the
same workload on the host cores; rank 0 only.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "gh_rhs_grid_point_evals_per_s"
UNIT = "points/s"

# algorithmic traffic per grid point and launch, DESIGN.md §5
BYTES_RHS_PT = (50 + 150 + 4 + 12 + 50) * 8      # k_rhs as gh_rhs: 216 reads (+ table lookups, cached) + 50 writes = 2 128 B
# inside gh_rk_step the stage update (A7) is the epilogue of k_rhs: stage 1 moves the same 2 128 B (writes u1 instead of
# d_t u), stages 2 and 3 also read u0: 2 528 B.  Average over the three launches of a step:
BYTES_RHS_RK_PT = (BYTES_RHS_PT + 2 * (BYTES_RHS_PT + 50 * 8)) / 3.0
FLOP_RHS_PT = 4391                                # SURVEY.md §8(a) A4+A5 instrumented count


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


# FP64 peak for the derivative kernels (bound "alu"): measured IN THIS RUN by the library's probe (gh_fp64_peak: register-
# resident DMMA m8n8k4 and DFMA kernels; the two share one datapath).  Round 1 measured 37.1 / 33.9 TFLOP/s
# (profiles/r01_fp64_peak.md); nominal 148 SM x 64 FMA x 2 x 1.965 GHz = 37.2.


# ------------------------------------------------------------------------------------------------------------------
# workload construction (host, numpy; seeded)
# ------------------------------------------------------------------------------------------------------------------
def make_config(name: str, min_points: int):
    from paper_1804_09101_b200 import configs

    if name == "c4":
        cfg = configs.c4(min_points=min_points)
        base = configs.c4(replicate=False)
        label = (f"C4 production-like isolated-BH domain: {cfg['replicas']} x (40 shells N_r 12..24, L 12..32 + 24 cube "
                 f"blocks N 16..32), Kerr-Schild a=0.9, perturbation 1e-5, one RK3 step + constraint norms")
        return cfg, base, label
    if name == "c3":
        cfg = configs.c3()
        return cfg, cfg, "C3 isolated Kerr BH a=0.7: 8 shells N_r=16 L=16, perturbation 1e-5, RK3 step + constraint norms"
    if name == "c2":
        cfg = configs.c2()
        cfg["dt"] = 0.25 * configs.min_spacing(cfg["descs"])
        return cfg, cfg, "C2 one 24^3 block, a=0.5 (L2-resident latency case)"
    if name == "c1":
        cfg = configs.c1()
        cfg["dt"] = 0.25 * configs.min_spacing(cfg["descs"])
        return cfg, cfg, "C1 one shell N_r=8 L=8, a=0 (L2-resident latency case)"
    raise SystemExit(f"unknown workload {name}")


def base_inputs(base_cfg, coords):
    from paper_1804_09101_b200 import inputs

    return inputs.initial_data(base_cfg["descs"], coords, base_cfg["spin"], base_cfg["amplitude"], base_cfg["id"])


# ------------------------------------------------------------------------------------------------------------------
# clocks during the timed region (B200_PROFILING.md "clocks line")
# ------------------------------------------------------------------------------------------------------------------
class ClockSampler:
    QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu = gpu_index
        self.proc = None
        self.lines = []
        self.thread = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.gpu), f"--query-gpu={self.QUERY}", "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._pump, daemon=True)
        self.thread.start()

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        if self.thread is not None:
            self.thread.join(timeout=2)
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax.append(float(f[1])); power.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "power_w_max": float(max(power)),
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------------------------
# the CPU oracle, timed on a bounded sample (cpu_baseline leg and --impl reference)
# ------------------------------------------------------------------------------------------------------------------
def oracle_sample(base_cfg, budget_points: int = 60_000):
    """Pick subdomains of the workload (alternating shells / blocks, in order) until ~budget_points points."""
    from paper_1804_09101_b200 import configs

    descs = base_cfg["descs"]
    shells = [s for s, d in enumerate(descs) if d["kind"] == "shell"]
    blocks = [s for s, d in enumerate(descs) if d["kind"] == "block"]
    order = []
    for i in range(max(len(shells), len(blocks))):
        if i < len(shells):
            order.append(shells[i])
        if i < len(blocks):
            order.append(blocks[i])
    pick, pts = [], 0
    for s in order:
        pick.append(s)
        pts += configs.num_points(descs[s])
        if pts >= budget_points:
            break
    return pick, pts


def time_oracle(base_cfg, pick, steps: int, warmup: int, threads=None):
    """One 'step' = one oracle RHS evaluation (Real=double build, OpenMP) of every picked subdomain."""
    from oracle.gh_oracle import Oracle
    from paper_1804_09101_b200 import inputs

    ora = Oracle("double", threads=threads)
    descs = [base_cfg["descs"][s] for s in pick]
    coords = [ora.coords(d) for d in descs]
    us, Hs = [], []
    for s, d, xyz in zip(pick, descs, coords):
        u, H = inputs.initial_data([d], [xyz], base_cfg["spin"], base_cfg["amplitude"], base_cfg["id"])
        us.append(u[0]); Hs.append(H[0])
    pts = sum(u.shape[1] for u in us)
    for _ in range(warmup):
        ora.rhs(descs[0], us[0], Hs[0])
    t0 = time.perf_counter()
    for _ in range(steps):
        for d, u, H in zip(descs, us, Hs):
            ora.rhs(d, u, H)
    dt = time.perf_counter() - t0
    try:
        cores = len(os.sched_getaffinity(0))
    except AttributeError:
        cores = os.cpu_count() or 1
    omp = os.environ.get("OMP_NUM_THREADS")
    if omp:
        cores = min(cores, int(omp))
    if threads is not None:
        cores = min(cores, int(threads))
    return pts * steps / dt, dt / steps, cores, pts


# ------------------------------------------------------------------------------------------------------------------
# algorithmic work per launch of each kernel, from the descriptors
# ------------------------------------------------------------------------------------------------------------------
def kernel_work(descs):
    from paper_1804_09101_b200 import configs

    P = sum(configs.num_points(d) for d in descs)
    Ps = sum(configs.num_points(d) for d in descs if d["kind"] == "shell")
    Pb = P - Ps
    cheb_flop = ang_flop = ang_exec = 0.0
    from paper_1804_09101_b200 import opcount

    for d in descs:
        p = configs.num_points(d)
        if d["kind"] == "shell":
            cheb_flop += 50.0 * p * (2 * d["n"][0] - 1)
            ang_flop += 50.0 * p * 8 * (2 * d["n"][1] + 1)     # S1 + S2 + S3 of K_ang: 8 (2L+1) flop / point / component
            ang_exec += opcount.shell_executed_dmma_flop(50, d["n"][0], d["n"][1])   # what the folded, tile-padded kernel issues
        else:
            cheb_flop += 50.0 * p * sum(2 * n - 1 for n in d["n"])
    return {
        "P": P,
        "k_rhs": {"bytes": float(BYTES_RHS_RK_PT) * P, "flop": float(FLOP_RHS_PT + 200) * P, "bound": "hbm"},
        "k_con": {"bytes": (50 + 120 + 4) * 8.0 * P, "flop": 1200.0 * P, "bound": "hbm"},
        "k_cheb": {"bytes": 8.0 * (50 * Ps + 50 * Ps + 50 * Pb + 150 * Pb), "flop": cheb_flop, "bound": "alu"},
        "k_ang": {"bytes": 8.0 * (50 + 100) * Ps, "flop": ang_flop, "flop_executed": ang_exec, "bound": "alu"},
    }


def read_traffic(kernel: str, P: int):
    """dram bytes per launch of `kernel` from the committed ncu summary profiles/ncu_traffic.csv
    (columns: kernel,P,dram_bytes_per_launch; see profiles/README.md), if taken on this workload size; else None."""
    p = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    if not os.path.exists(p):
        return None
    with open(p) as f:
        for ln in f:
            c = [x.strip() for x in ln.split(",")]
            if len(c) >= 3 and c[0] == kernel:
                try:
                    if int(c[1]) == int(P):
                        return float(c[2])
                except ValueError:
                    continue
    return None


# ------------------------------------------------------------------------------------------------------------------
# multi-rank bookkeeping ("replicas only"): no data-path collective, only the timing reduction
# ------------------------------------------------------------------------------------------------------------------
def max_over_ranks(values, dist, device):
    """MAX over ranks of each entry of `values` (device times); identity when dist is None."""
    if dist is None:
        return [float(v) for v in values]
    import torch

    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def whole_job_value(world: int, points_per_rank: int, steps: int, ms_max: float) -> float:
    """Replicas: every rank evaluates 3 RHS per step on its own copy; the job's rate divides by the slowest rank's time."""
    return world * 3.0 * points_per_rank * steps / (ms_max * 1e-3)


# ------------------------------------------------------------------------------------------------------------------
# our arm
# ------------------------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch

    from paper_1804_09101_b200 import build as _build
    from paper_1804_09101_b200 import gh

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the library has no CPU fallback (use --impl reference for the oracle)")
    if rank == 0:
        _build.build()
    dist = None
    if world > 1:
        import torch.distributed as dist_

        dist = dist_
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local_rank}"))
        dist.barrier()
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    if args.workload == "c5":
        if rank == 0:
            run_sweep(args, dev)
        if dist is not None:
            dist.barrier(); dist.destroy_process_group()
        return

    cfg, base, label = make_config(args.workload, args.min_points)
    descs = cfg["descs"]
    nbase = len(base["descs"])
    reps = len(descs) // nbase
    dom = gh.Domain(descs, device=dev)
    if args.no_graph:
        dom.set_option(gh.GH_OPT_NO_GRAPH, 1)
    P, S = dom.P, dom.S

    # inputs: analytic data evaluated on the library's own grid (gh_domain_coords) for the base subdomain set,
    # replicated (reading S13); every rank builds the same arrays (replicas)
    coords = dom.coords()[:nbase]
    us_b, Hs_b = base_inputs(base, coords)
    u_host = torch.zeros(50, S, dtype=torch.float64).pin_memory()
    H_host = np.zeros((4, S))
    un = u_host.numpy()
    for s in range(len(descs)):
        o, n = dom.offsets[s], dom.sizes[s]
        un[:, o:o + n] = us_b[s % nbase]
        H_host[:, o:o + n] = Hs_b[s % nbase]
    dom.set_gauge_source(H_host)
    u_dev = torch.empty(50, S, dtype=torch.float64, device=dev)
    u_dev.copy_(u_host)
    dt = float(cfg["dt"])
    work = kernel_work(descs)

    def sync_all():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    def step():
        # A2-A8 in one call: the constraint norms (of the state the step starts from) are an epilogue of the first stage's
        # fused RHS kernel (gh_rk_step_norms); --unfused-norms times the round-1 path (gh_rk_step + stand-alone gh_constraint_norms)
        if args.unfused_norms:
            dom.rk_step(dt)
            return dom.constraint_norms()
        return dom.rk_step_norms(dt)

    fp64 = dom.fp64_peak()      # (DMMA, DFMA) TFLOP/s of this GPU, now

    # ---- device-resident timing: per-launch events OFF; one CUDA event between steps on the library's stream (= torch's current) ----
    dom.set_fields(u_dev, 0.0)
    for _ in range(args.warmup):
        step()
    dom.set_fields(u_dev, 0.0)
    dom.set_profiling(False)
    l0 = dom.launch_count()
    sampler = ClockSampler(local_rank)
    sampler.start()
    sync_all()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    ev[0].record(dom.stream)          # the library's stream (the domain's own), which is where its kernels run
    for i in range(args.steps):
        norms = step()
        ev[i + 1].record(dom.stream)
    sync_all()
    ms = ev[0].elapsed_time(ev[-1])
    per_step = [ev[i].elapsed_time(ev[i + 1]) for i in range(args.steps)]
    clocks = sampler.stop()
    launches = dom.launch_count() - l0
    if not np.all(np.isfinite(norms)):
        raise SystemExit("bench.py: non-finite constraint norms after the timed region")

    # ---- second pass, per-launch events ON: the per-kernel split (not part of `value`) -------------------------------------
    prof_steps = max(1, min(args.steps, args.profile_steps))
    dom.set_fields(u_dev, 0.0)
    dom.set_profiling(True)
    dom.profile_reset()
    for _ in range(prof_steps):
        step()
    prof = dom.profile_read()
    dom.set_profiling(False)

    # ---- end to end through the C ABI with HOST buffers (pinned): H2D of the state, step, D2H of the state --------
    out_host = torch.empty(50, S, dtype=torch.float64).pin_memory()
    e2e_steps = max(2, min(args.steps, args.e2e_steps))
    for _ in range(2):
        dom.set_fields(u_host, 0.0); step(); dom.get_fields(out_host)
    sync_all()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        dom.set_fields(u_host, 0.0)
        step()
        dom.get_fields(out_host)
    torch.cuda.synchronize()
    e2e_single_s = (time.perf_counter() - t0) / e2e_steps
    if not bool(torch.isfinite(out_host).all()):
        raise SystemExit("bench.py: non-finite state after the e2e region")
    # what the two copies alone cost (the PCIe floor of one un-overlapped step)
    t0 = time.perf_counter(); dom.set_fields(u_host, 0.0); torch.cuda.synchronize(); h2d_s = time.perf_counter() - t0
    t0 = time.perf_counter(); dom.get_fields(out_host); torch.cuda.synchronize(); d2h_s = time.perf_counter() - t0
    pcie = {"h2d_GBps": 50 * S * 8 / h2d_s / 1e9, "d2h_GBps": 50 * S * 8 / d2h_s / 1e9, "copies_only_ms": (h2d_s + d2h_s) * 1e3,
            "single_domain_ms_per_step": e2e_single_s * 1e3}
    # The same e2e steps with SEVERAL domains in flight (handles of the same public API on their own streams, each driven by a host
    # thread; every step still copies its own 1.94 GB in and out): one domain's H2D overlaps another's D2H (PCIe is full
    # duplex) and both overlap the kernels.  One domain's chain is H2D + step + D2H (35 + 19 + 35 ms on C4): two in flight can reach
    # half of that at best, three are bounded by one PCIe direction, max(H2D, D2H, compute).
    e2e_s, e2e_mode = e2e_single_s, "one domain: copy in, step, copy out, one after the other"
    if not args.no_e2e_overlap:
        try:
            doms = [(dom, out_host)]
            for _ in range(max(1, args.e2e_domains) - 1):
                dom2 = gh.Domain(descs, device=dev)
                if args.no_graph:
                    dom2.set_option(gh.GH_OPT_NO_GRAPH, 1)
                dom2.set_gauge_source(H_host)
                doms.append((dom2, torch.empty(50, S, dtype=torch.float64).pin_memory()))
            nd = len(doms)

            def worker(dm, oh, n):
                torch.cuda.set_device(local_rank)
                with torch.cuda.stream(dm.stream):      # the thread's current stream IS the domain's: no cross-stream waits through torch's default stream
                    for _ in range(n):
                        dm.set_fields(u_host, 0.0)
                        if args.unfused_norms:
                            dm.rk_step(dt); dm.constraint_norms()
                        else:
                            dm.rk_step_norms(dt)
                        dm.get_fields(oh)

            def run_pair(n):
                th = [threading.Thread(target=worker, args=(dm, oh, n)) for dm, oh in doms]
                for t in th:
                    t.start()
                for t in th:
                    t.join()
                torch.cuda.synchronize()

            run_pair(1)
            sync_all()
            n_each = max(2, -(-e2e_steps // nd))
            t0 = time.perf_counter()
            run_pair(n_each)
            e2e_s = (time.perf_counter() - t0) / (nd * n_each)
            e2e_steps = nd * n_each
            e2e_mode = f"{nd} domains in flight on {nd} streams (host threads): H2D, kernels and D2H of different steps overlap"
            for dm, oh in doms[1:]:
                if not (bool(torch.isfinite(oh).all()) and torch.equal(out_host, oh)):
                    raise SystemExit("bench.py: the e2e domains disagree")
                dm.close()
            del doms
        except torch.OutOfMemoryError:
            pass
    pcie["mode"] = e2e_mode

    filt = time_filter(dom, u_dev, descs) if rank == 0 and not args.no_extras else None
    dp5 = time_dp5(dom, u_dev, dt, P) if rank == 0 and not args.no_extras else None
    scj = time_scj(dom, u_dev, P) if rank == 0 and not args.no_extras else None

    tmax, e2emax, med = max_over_ranks([ms, e2e_s, float(np.median(per_step))], dist, dev)
    if rank != 0:
        dom.close()
        if dist is not None:
            dist.barrier(); dist.destroy_process_group()
        return
    return finish_ours(args, world, label, cfg, descs, reps, P, S, tmax, e2emax, e2e_steps, launches, prof, prof_steps, work, clocks,
                       norms, base, dom, dist, filt, dp5, scj, fp64, med, per_step, pcie)


def time_scj(dom, u_dev, P, reps: int = 5):
    """NEXT-4 (outside the timed step): gh_spatial_coord_jac_state with a rotation-about-z Jacobian field; HBM-bound,
    (2 x 50 + 9) doubles per point."""
    import torch

    J = torch.zeros(9, dom.S, dtype=torch.float64, device=u_dev.device)
    c, s = float(np.cos(0.3)), float(np.sin(0.3))
    J[0], J[1], J[3], J[4], J[8] = c, -s, s, c, 1.0
    dom.set_jacobian(J)
    dom.set_fields(u_dev, 0.0)
    for _ in range(2):
        dom.spatial_coord_jac_state()
    dom.set_profiling(True)
    dom.profile_reset()
    for _ in range(reps):
        dom.spatial_coord_jac_state()
    prof = dom.profile_read()
    dom.set_profiling(False)
    ms = prof["k_scj"][0] / reps
    return {"ms_per_call": ms, "achieved_GBps": 109 * 8.0 * P / (ms * 1e-3) / 1e9, "bound": "hbm", "bytes_per_point": 109 * 8}


def time_filter(dom, u_dev, descs, reps: int = 5):
    """NEXT-1 (outside the timed step): gh_apply_filter with the exponential filter on every block axis and in l on every
    shell; per-kernel device time from the library's CUDA events, mean of `reps` calls after 2 warm-ups."""
    from paper_1804_09101_b200 import configs

    f = {"kind": "exp", "alpha": 36.0, "p": 32}
    dom.set_filter(block_axes=f, shell_angular=f)
    dom.set_fields(u_dev, 0.0)
    for _ in range(2):
        dom.apply_filter()
    dom.set_profiling(True)
    dom.profile_reset()
    for _ in range(reps):
        dom.apply_filter()
    prof = dom.profile_read()
    dom.set_profiling(False)
    dom.set_filter(None, None)
    Ps = sum(configs.num_points(d) for d in descs if d["kind"] == "shell")
    Pb = sum(configs.num_points(d) for d in descs if d["kind"] == "block")
    ms_c = prof["k_cheb(filter)"][0] / reps
    ms_a = prof["k_ang(filter)"][0] / reps
    out = {"filter": "exp(-36 (k/kmax)^64) on the 3 Chebyshev axes of every block and in l on every shell", "ms_per_call": ms_c + ms_a}
    if ms_c > 0:   # three passes, each reads and writes the 50 block components once
        out["k_cheb(filter)"] = {"ms_per_call": ms_c, "achieved_GBps": 3 * 2 * 50 * 8.0 * Pb / (ms_c * 1e-3) / 1e9, "bound": "hbm"}
    if ms_a > 0:   # analysis + filtered projector + one synthesis: about 5 (2L+1) flop per point and component unfolded
        fl = sum(50.0 * configs.num_points(d) * 5 * (2 * d["n"][1] + 1) for d in descs if d["kind"] == "shell")
        out["k_ang(filter)"] = {"ms_per_call": ms_a, "achieved_GBps": 2 * 50 * 8.0 * Ps / (ms_a * 1e-3) / 1e9,
                                "achieved_TFLOPs": fl / (ms_a * 1e-3) / 1e12, "bound": "alu"}
    return out


def time_dp5(dom, u_dev, dt, P, reps: int = 3):
    """NEXT-3 (outside the timed step): gh_dp5_step, 6 new RHS evaluations per step (the 7th stage is reused as the next
    step's first).  Wall time around `reps` steps after one warm-up step (the call synchronises: it returns the error norms)."""
    import torch

    try:
        dom.dp5_attach()
    except Exception as e:          # not enough device memory for the 7 stage arrays
        return {"unavailable": str(e)}
    dom.set_fields(u_dev, 0.0)
    dom.dp5_step(dt)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(reps):
        rms, mx, acc = dom.dp5_step(dt)
    torch.cuda.synchronize()
    s_per = (time.perf_counter() - t0) / reps
    return {"ms_per_step": s_per * 1e3, "rhs_evals_per_step": 6, "points_per_s": 6.0 * P / s_per, "err_rms": rms, "err_max": mx}


def finish_ours(args, world, label, cfg, descs, reps, P, S, ms, e2e_step_s, e2e_steps, launches, prof, prof_steps, work, clocks,
                norms, base, dom, dist, filt, dp5, scj, fp64, ms_median, per_step, pcie):
    hbm_peak, peak_src = load_peaks()
    steps = args.steps
    value = whole_job_value(world, P, steps, ms)
    # per-kernel numbers from the SECOND pass (library CUDA events around each launch on its own stream)
    total_kernel_ms = sum(v[0] for v in prof.values()) or 1.0
    nd = 3.8 if args.unfused_norms else 3.0     # derivative passes per step (the stand-alone constraint pass differentiates 40 of 50 components)
    calls_per_step = {"k_rhs": 3, "k_con": 1, "k_cheb": nd, "k_ang": nd}   # library calls that run the kernel
    kernels = {}
    for name, (kms, cnt) in prof.items():
        if cnt == 0 or "filter" in name or name.startswith("k_dp") or name == "k_scj":
            continue
        e = {"launches_per_step": cnt / prof_steps, "ms_per_launch": kms / cnt, "ms_per_step": kms / prof_steps,
             "share_of_kernel_time": kms / total_kernel_ms}
        w = work.get(name)
        if w:
            # one "call" = all launches of this kernel inside one RHS evaluation (K_ang: one launch per shared-memory class);
            # work is per call, time is the measured total over the profiled pass
            per_call_s = kms * 1e-3 / (prof_steps * calls_per_step[name])
            e["ms_per_call"] = per_call_s * 1e3
            e["achieved_GBps"] = w["bytes"] / per_call_s / 1e9
            e["achieved_TFLOPs"] = w["flop"] / per_call_s / 1e12
            e["bound"] = w["bound"]
            if "flop_executed" in w:      # symmetry folds: fewer flop issued than the unfolded factored map counts
                e["executed_TFLOPs"] = w["flop_executed"] / per_call_s / 1e12
        kernels[name] = e
    top = max((k for k in kernels if k in work), key=lambda k: kernels[k]["share_of_kernel_time"])
    fp64_peak = fp64[0]
    if work[top]["bound"] == "hbm":
        roof = {"kernel": top, "bound": "hbm", "achieved": kernels[top]["achieved_GBps"], "peak": hbm_peak, "unit": "GB/s",
                "frac": kernels[top]["achieved_GBps"] / hbm_peak, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": work[top]["bytes"], "traffic": read_traffic(top, P)}
    else:
        roof = {"kernel": top, "bound": "alu", "achieved": kernels[top]["achieved_TFLOPs"], "peak": fp64_peak, "unit": "TFLOP/s",
                "frac": kernels[top]["achieved_TFLOPs"] / fp64_peak,
                "peak_source": "measured in this run (gh_fp64_peak: register-resident DMMA m8n8k4 kernel on this GPU)",
                "algorithmic_flop_per_launch": work[top]["flop"], "traffic": read_traffic(top, P)}
        if "executed_TFLOPs" in kernels[top]:
            roof["issued_frac"] = kernels[top]["executed_TFLOPs"] / fp64_peak
    # the fused RHS kernel is the one north_star sets a target for: always report it too
    roof_rhs = None
    if "k_rhs" in kernels:
        roof_rhs = {"achieved": kernels["k_rhs"]["achieved_GBps"], "peak": hbm_peak, "unit": "GB/s",
                    "frac": kernels["k_rhs"]["achieved_GBps"] / hbm_peak, "frac_of_8TBps_nominal": kernels["k_rhs"]["achieved_GBps"] / 8000.0,
                    "traffic": read_traffic("k_rhs", P)}

    cpu = None
    if not args.no_cpu_baseline:
        pick, _ = oracle_sample(base, args.cpu_points)
        v, s_per, cores, pts = time_oracle(base, pick, 1, 1)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"one oracle RHS evaluation (Real=double build, OpenMP) of subdomains {pick} of the workload's base set "
                         f"({pts} points, {s_per:.1f} s)"}
        # the paper's own comparisons are against ONE CPU core: the same oracle on one thread, smaller sample
        pick1, _ = oracle_sample(base, max(20_000, args.cpu_points // 20))
        v1, s1, _, pts1 = time_oracle(base, pick1, 1, 0, threads=1)
        cpu["single_core"] = {"value": v1, "unit": UNIT, "cores": 1,
                              "sample": f"subdomains {pick1} ({pts1} points, {s1:.1f} s), one thread"}

    h2d = 50 * S * 8
    d2h = 50 * S * 8 + 6 * 8
    step_name = "gh_rk_step + gh_constraint_norms" if args.unfused_norms else "gh_rk_step_norms (RK3 step, constraint norms fused into stage 1)"
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": args.warmup,
        "ms_per_step": ms / steps, "ms_per_step_median": ms_median, "ms_per_step_min": float(min(per_step)), "ms_per_step_max": float(max(per_step)),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": label, "points_per_gpu": P, "subdomains": len(descs), "replicas_of_base_set": reps,
                   "components": 50, "dt": float(cfg["dt"]), "rhs_evals_per_step": 3,
                   "step": step_name, "parallelism": "replicas only" if world > 1 else "single GPU",
                   "l2": f"inputs larger than L2: the step streams {316 * S * 8 / 1e9:.2f} GB of state/derivative arrays (L2 126 MB)",
                   "per_launch_events": f"off in the timed region; the per-kernel split is from a second pass of {prof_steps} steps with them on",
                   "cuda_graph": "off (--no-graph)" if args.no_graph else "each step replays one captured CUDA graph (gpu_launches counts its kernel nodes)"},
        "rk_steps_per_s": world * steps / (ms * 1e-3),
        "gpu_launches": int(launches),
        "roofline": roof, "roofline_k_rhs": roof_rhs, "kernels": kernels,
        "fp64_peak_measured_TFLOPs": {"dmma_m8n8k4": fp64[0], "dfma": fp64[1]},
        "cpu_baseline": cpu,
        "e2e": {"value": world * 3.0 * P / e2e_step_s, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "steps": e2e_steps, "ms_per_step": e2e_step_s * 1e3,
                "path": "gh_set_fields(HOST pinned) + the step + gh_get_fields(HOST pinned), every step; " + pcie["mode"],
                "pcie": pcie},
        "clocks": clocks,
        "constraint_norms_of_last_step_input": [[float(x) for x in r] for r in np.asarray(norms)],
        "spectral_filter": filt,
        "dormand_prince_5_4": dp5,
        "spatial_coord_jac_state": scj,
    }
    print(json.dumps(out))
    sys.stdout.flush()
    dom.close()
    if dist is not None:
        dist.barrier(); dist.destroy_process_group()
    return out


# ------------------------------------------------------------------------------------------------------------------
# the size sweep (BASELINE.json configs[4]): one JSON line per member
# ------------------------------------------------------------------------------------------------------------------
def sweep_members(max_points, paper_members=False):
    from paper_1804_09101_b200 import configs

    out = []
    for n in (8, 16, 32, 64, 128, 256):
        out.append((f"shell n={n} (N_r={n}, L={n - 1})", configs.c5_shell(n)))
    for N in (10, 20, 40, 80, 160, 320):
        out.append((f"block {N}^3", configs.c5_block(N)))
    if paper_members:      # the paper's own grid prescriptions for this sweep and its whole-code test shell
        out.append(("paper test shell (10,19,38)", {**configs.paper_two_shells(), "descs": configs.paper_two_shells()["descs"][:1]}))
        for k in range(0, 11):
            out.append((f"SingleBH k={k}", configs.single_bh(k)))
        for k in range(1, 17):
            out.append((f"BBH k={k}", configs.bbh(k)))
    return [(lbl, cfg) for lbl, cfg in out if configs.num_points(cfg["descs"][0]) <= max_points]


def run_sweep(args, dev):
    """gh_rhs on every member: median of `reps` calls after 3 warm-ups, per-kernel times from the library's events; the derivative
    rate counts the algorithmic flop of the factored maps, and the paper's dense-matrix convention beside it."""
    import torch

    from paper_1804_09101_b200 import configs, gh, inputs, opcount

    hbm_peak, _ = load_peaks()
    for label, cfg in sweep_members(args.sweep_max_points, args.sweep_paper_members):
        if args.sweep_only and args.sweep_only not in label:
            continue
        d = cfg["descs"][0]
        dom = gh.Domain([d], device=dev)
        P, S = dom.P, dom.S
        xyz = np.zeros((3, S)); gh.gh_domain_coords(dom.h, xyz)
        u = torch.zeros(50, S, dtype=torch.float64).pin_memory()
        H = np.zeros((4, S))
        inputs.initial_data_chunked(d, xyz[:, :P], cfg["spin"], cfg["amplitude"], cfg["id"], 0, u.numpy()[:, :P], H[:, :P])
        del xyz
        dom.set_gauge_source(H)
        dom.set_fields(u, 0.0)
        del u, H
        out = dom.empty(50)
        fp64 = dom.fp64_peak()
        reps = args.sweep_reps if P < 5_000_000 else max(3, args.sweep_reps // 4)
        for _ in range(3):
            dom.rhs(out)
        dom.set_profiling(True)
        tot, der, rhs = [], [], []
        for _ in range(reps):
            dom.profile_reset()
            dom.rhs(out)
            prof = dom.profile_read()
            t_der = prof["k_cheb"][0] + prof["k_ang"][0]
            tot.append(t_der + prof["k_rhs"][0]); der.append(t_der); rhs.append(prof["k_rhs"][0])
        dom.set_profiling(False)
        # wall time of the call with events off (launch overhead included: the latency regime of the small members)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        wall = []
        for _ in range(reps):
            e0.record(dom.stream); dom.rhs(out); e1.record(dom.stream); torch.cuda.synchronize()
            wall.append(e0.elapsed_time(e1))
        if not bool(torch.isfinite(out).all()):
            raise SystemExit(f"bench.py: non-finite RHS on {label}")
        if d["kind"] == "shell":
            flop = opcount.shell_factored_flop(50, d["n"][0], d["n"][1])
            flop_paper = opcount.shell_deriv_dense(50, d["n"][0], d["n"][1] + 1, 2 * d["n"][1] + 2)[1]
        else:
            flop = flop_paper = opcount.block_deriv(50, *d["n"])[1]
        ms, ms_d, ms_r, ms_w = (float(np.median(x)) for x in (tot, der, rhs, wall))
        line = {"metric": "gh_rhs_points_per_s", "workload": "c5", "member": label, "points": P, "reps": reps,
                "gh_rhs_ms_kernels": ms, "gh_rhs_ms_call": ms_w, "points_per_s": P / (ms_w * 1e-3), "unit": UNIT,
                "deriv_ms": ms_d, "deriv_TFLOPs": flop / (ms_d * 1e-3) / 1e12, "deriv_frac_of_fp64_peak": flop / (ms_d * 1e-3) / 1e12 / fp64[0],
                "deriv_TFLOPs_paper_dense_convention": flop_paper / (ms_d * 1e-3) / 1e12,
                "k_rhs_ms": ms_r, "k_rhs_GBps": float(BYTES_RHS_PT) * P / (ms_r * 1e-3) / 1e9,
                "k_rhs_frac_of_hbm": float(BYTES_RHS_PT) * P / (ms_r * 1e-3) / 1e9 / hbm_peak,
                "fp64_peak_measured_TFLOPs": fp64[0], "dtype": "f64", "data": "synthetic",
                "regime": "single subdomain (latency-bound below ~1e5 points: the call is 3-7 launches)"}
        print(json.dumps(line))
        sys.stdout.flush()
        dom.close()
        del dom, out
        torch.cuda.empty_cache()


# ------------------------------------------------------------------------------------------------------------------
# reference arm: the CPU oracle as it stands
# ------------------------------------------------------------------------------------------------------------------
def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import gh_oracle

    gh_oracle.build()
    cfg, base, label = make_config(args.workload, args.min_points)
    pick, _ = oracle_sample(base, args.ref_points)
    v, s_per, cores, pts = time_oracle(base, pick, args.steps, min(args.warmup, 1))
    sample = (f"each step = one oracle RHS evaluation (Real=double build, OpenMP) of subdomains {pick} of the workload's base set "
              f"({pts} points)")
    out = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": s_per * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f64", "data": "synthetic", "config": {"workload": label, "sample": sample},
           "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
           "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c4", choices=["c1", "c2", "c3", "c4", "c5"])
    ap.add_argument("--profile-steps", type=int, default=10, help="steps of the second (per-launch events on) pass")
    ap.add_argument("--sweep-reps", type=int, default=20, help="c5: repetitions per member")
    ap.add_argument("--sweep-max-points", type=int, default=40_000_000, help="c5: skip members above this size")
    ap.add_argument("--sweep-only", default="", help="c5: only the members whose label contains this text (e.g. 'block 160' for an ncu capture)")
    ap.add_argument("--sweep-paper-members", action="store_true", help="c5: also the paper's SingleBH / BBH shell prescriptions (PAPER.md:436)")
    ap.add_argument("--min-points", type=int, default=4_000_000, help="C4: replicate the base set until P >= this")
    ap.add_argument("--e2e-steps", type=int, default=9)
    ap.add_argument("--cpu-points", type=int, default=1_300_000,
                    help="points in the cpu_baseline sample (default: the whole 64-subdomain base set, ~10 s on 16 cores)")
    ap.add_argument("--ref-points", type=int, default=60_000, help="points per step of --impl reference")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e-overlap", action="store_true", help="e2e leg with one domain only (no second domain in flight)")
    ap.add_argument("--e2e-domains", type=int, default=3, help="domains in flight in the e2e leg (each with its own stream and host thread)")
    ap.add_argument("--no-graph", action="store_true", help="enqueue the step's kernels one by one instead of replaying the captured CUDA graph")
    ap.add_argument("--unfused-norms", action="store_true", help="step = gh_rk_step + stand-alone gh_constraint_norms (the round-1 path)")
    ap.add_argument("--no-extras", action="store_true", help="skip the spectral-filter and Dormand-Prince legs (run after the timed step)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
