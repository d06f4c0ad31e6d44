#!/usr/bin/env python
"""bench.py -- NUFFT forward+adjoint pairs/s on one B200 (BASELINE.json metric), with roofline and CPU baseline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--batch B] [--no-extra]

A "step" is one pass of the whole hot path over one batch: y = A x (nufft_forward: S + zero-pad + F + V) followed by
x' = A^H y (nufft_adjoint: V^H + F^H + crop + S^H) for a batch of B independent images that share one trajectory
(the paper's batch mode).  Workload at N = 1: BASELINE config 2 (configs[1]): 2-D golden-angle radial,
Nd = 256^2, Kd = 512^2, Jd = 6^2, M = 131072, complex64, synthetic seeded inputs (workloads.py).

  value      pairs/s, inputs resident in HBM, device time from CUDA events around each step on the launch stream;
             L2 is flushed (256 MiB memset) between steps, outside the event brackets.
  e2e        same metric through the host-buffer call: pinned host x -> H2D -> forward -> adjoint -> D2H x'.
  roofline   the dominant kernel of the step: ALGORITHMIC bytes per launch / its average
             duration measured live with CUDA events by the library (nufft_profile_*), against the measured HBM copy
             bandwidth in MEASURED_PEAKS.json.
  cpu_baseline  the float64 oracle, as it stands, timed on this box's host cores on a bounded sample.

N > 1 (torchrun): replicas only -- every rank runs the same independent job on its own GPU, no collective in the data
path; value = total pairs over the max-over-ranks time; scaling = weak.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads as wl  # noqa: E402

METRIC = "nufft_fwd_adj_pairs_per_s"
UNIT = "pairs/s"
WORKLOAD = "cfg2_2d_radial: Nd=256x256 Kd=512x512 Jd=6x6 golden-angle radial 256x512 (M=131072), complex64"


# ----------------------------------------------------------------------------------------------------------------
def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            v = float(json.load(f)["hbm_gbs"])
        return v, "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


def algorithmic_bytes(d, N, K, M, B, cov=1.0):
    """Per-launch algorithmic bytes of every kernel label."""
    rec = 4 + 4 * d
    if d == 2:
        return {
            "fft_rows_fwd": 8 * B * (N * N + N * K),
            "fft_cols_fwd": 8 * B * (N * K + K * K),
            "interp": B * (8 * K * K * cov + 8 * M) + M * rec,
            "gridding": B * (8 * M + 8 * K * K) + M * rec,
            "fft_cols_adj": 8 * B * (K * K + N * K),
            "fft_rows_adj": 8 * B * (N * K + N * N),
        }
    return {
        "fft_rows_fwd": 8 * B * (N ** 3 + N * N * K),
        "fft_cols_fwd_axis1": 8 * B * (N * N * K + N * K * K),
        "fft_cols_fwd_axis0": 8 * B * (N * K * K + K ** 3),
        "interp": B * (8 * K ** 3 * cov + 8 * M) + M * rec,
        "gridding": B * (8 * M + 8 * K ** 3) + M * rec,
        "fft_cols_adj_axis0": 8 * B * (K ** 3 + N * K * K),
        "fft_cols_adj_axis1": 8 * B * (N * K * K + N * N * K),
        "fft_rows_adj": 8 * B * (N * N * K + N ** 3),
    }


def max_over_ranks(values, world, device):
    """Replicas-only multi-GPU timing rule: every rank times its own replica on its device, the job's time is the MAX
    over ranks (one all-reduce of a few scalars, outside the timed region; no collective in the data path)."""
    if world <= 1:
        return [float(v) for v in values]
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.cpu()]


def aggregate_pairs_per_s(world, batch, ms_per_step):
    """Whole-job throughput of `world` independent replicas that each process `batch` pairs per step (weak scaling)."""
    return world * batch / (ms_per_step * 1e-3)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 50 ms while the timed region runs."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.gpu = str(gpu_index)
        self.lines = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                                          "-lms", "50", "-i", self.gpu], stdout=subprocess.PIPE, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1]))
                mx.append(float(f[2]))
            except ValueError:
                continue
            for name, val in zip(["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"], f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ----------------------------------------------------------------------------------------------------------------
# the oracle legs (CPU)
# ----------------------------------------------------------------------------------------------------------------
def oracle_pair_seconds(cfg, x, min_seconds, max_pairs):
    from oracle import nufft_oracle as orc
    Nd, Kd, Jd, om = cfg["Nd"], cfg["Kd"], cfg["Jd"], cfg["om"]
    x128 = x.astype(np.complex128)
    n, t0, c0 = 0, time.perf_counter(), time.process_time()
    while True:
        y = orc.forward(x128, om, Nd, Kd, Jd)
        orc.adjoint(y, om, Nd, Kd, Jd)
        n += 1
        el = time.perf_counter() - t0
        if el >= min_seconds or n >= max_pairs:
            return el / n, n, cores_used(time.process_time() - c0, el)


def cores_used(cpu_seconds, wall_seconds):
    """Threads the oracle actually kept busy: process CPU time / wall time, rounded (numpy's FFT and the vectorised
    stencil loops are single-threaded, so this is normally 1)."""
    return max(1, int(round(cpu_seconds / max(wall_seconds, 1e-9))))


def run_reference(args):
    """--impl reference: the float64 oracle (oracle/), as it stands, on the host cores.  One step = one
    forward+adjoint pair on ONE image of the workload (a bounded sample of the batch the CUDA arm processes)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cfg = wl.config(1)
    x = wl.image_gaussian(cfg["Nd"])
    from oracle import nufft_oracle as orc
    Nd, Kd, Jd, om = cfg["Nd"], cfg["Kd"], cfg["Jd"], cfg["om"]
    x128 = x.astype(np.complex128)
    steps = max(1, min(args.steps, 40))
    for _ in range(max(1, min(args.warmup, 3))):
        orc.adjoint(orc.forward(x128, om, Nd, Kd, Jd), om, Nd, Kd, Jd)
    t0, c0 = time.perf_counter(), time.process_time()
    for _ in range(steps):
        orc.adjoint(orc.forward(x128, om, Nd, Kd, Jd), om, Nd, Kd, Jd)
    el = time.perf_counter() - t0
    ncores = cores_used(time.process_time() - c0, el)
    v = steps / el
    sample = "1 image (batch element 0) of the workload per step, %d steps" % steps
    out = {
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * el / steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "complex128", "data": "synthetic",
        "config": {"workload": WORKLOAD, "batch": 1, "sample": sample},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": ncores, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(out))
    return 0


# ----------------------------------------------------------------------------------------------------------------
# the CUDA arm
# ----------------------------------------------------------------------------------------------------------------
def kernel_table(prof, bytes_per_launch, peak):
    rows = {}
    for name, (ms, n) in prof.items():
        if n == 0:
            continue
        avg_ms = ms / n
        b = bytes_per_launch.get(name)
        rows[name] = {"ms_per_launch": avg_ms, "launches": n}
        if b is not None and avg_ms > 0:
            gbs = b / (avg_ms * 1e-3) / 1e9
            rows[name].update({"alg_bytes": int(b), "gbs": gbs, "frac": gbs / peak})
    return rows


def stage_of(rows, keys):
    return sum(rows[k]["ms_per_launch"] for k in keys if k in rows)


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_1710_03197_b200 as nb

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    nb.lib()   # fail loudly here if the extension is missing

    B, K_steps, W = args.batch, args.steps, max(args.warmup, 3)
    cfg = wl.config(1)
    Nd, Kd, Jd, om = cfg["Nd"], cfg["Kd"], cfg["Jd"], cfg["om"]
    M = om.shape[0]
    plan = nb.NufftPlan(Nd, Kd, Jd, om, max_batch=B)
    x_host = torch.from_numpy(wl.image_gaussian(Nd, seed=wl.SEED_IMAGE + rank, batch=B)).pin_memory()
    x = x_host.cuda()
    y = torch.empty((B, M), dtype=torch.complex64, device="cuda")
    xo = torch.empty((B,) + tuple(Nd), dtype=torch.complex64, device="cuda")
    xo_host = torch.empty((B,) + tuple(Nd), dtype=torch.complex64).pin_memory()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream()

    def step():
        plan.forward(x, y)
        plan.adjoint(y, xo)

    def step_e2e():
        # the pair through the host-buffer C-ABI call: pinned x -> H2D -> A -> A^H -> D2H x' (y stays on the device),
        # chunked copy/compute pipeline inside the library (nufft_selfadjoint_host)
        plan.selfadjoint_host(x_host, xo_host)

    def timed(fn, nsteps):
        evs = []
        for _ in range(nsteps):
            flush.zero_()                     # L2 flush, outside the event bracket
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            fn()
            b.record(stream)
            evs.append((a, b))
        torch.cuda.synchronize()
        return sum(a.elapsed_time(b) for a, b in evs)

    def timed_median(fn, min_ms=50.0, reps=5):
        """ms per call: `reps` repetitions of >= min_ms of timed calls each (L2 flushed before every call), the median."""
        est = max(timed(fn, 5) / 5, 1e-3)
        n = max(5, int(np.ceil(min_ms / est)))
        return float(np.median([timed(fn, n) / n for _ in range(reps)]))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(W):
        step()
    torch.cuda.synchronize()

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    barrier()
    l0 = plan.launch_count()
    total_ms = timed(step, K_steps)
    l1 = plan.launch_count()
    # the timed region of this workload lasts ~10 ms, less than nvidia-smi's sampling period: keep running the SAME step
    # (untimed) for ~0.6 s so that the sampler, started before the timed region, sees the clocks under this load
    t_load = time.perf_counter()
    while time.perf_counter() - t_load < 0.6:
        for _ in range(20):
            step()
        torch.cuda.synchronize()
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    if clocks is not None:
        clocks["note"] = ("sampled every 50 ms from the start of the timed region through a 0.6 s untimed continuation of "
                          "the same step (the timed region itself is ~10 ms)")

    # e2e, STRICT stream order (the headline e2e number): every copy in is ordered after the L2 flush and the start event
    # on the caller's stream, so no byte of a step's H2D traffic can move outside that step's event bracket
    y_host = torch.empty((B, M), dtype=torch.complex64).pin_memory()

    def step_e2e_two_calls():
        # the same pair as two host-buffer calls: y goes back to the host and comes in again (what a caller who keeps y does)
        plan.forward_host(x_host, y_host)
        plan.adjoint_host(y_host, xo_host)

    plan.host_input_ready(False)
    for _ in range(2):
        step_e2e()
    barrier()
    e2e_ms = timed(step_e2e, K_steps)
    barrier()
    for _ in range(2):
        step_e2e_two_calls()
    e2e2_ms = timed(step_e2e_two_calls, K_steps)
    barrier()
    # relaxed: the caller promises the host input is final at call time (nufft_host_input_ready), so the copy in of step k + 1
    # may overlap the copy back of step k -- and, in this loop, the untimed flush between the brackets: context only
    plan.host_input_ready(True)
    for _ in range(2):
        step_e2e()
    e2e_relaxed_ms = timed(step_e2e, K_steps)
    plan.host_input_ready(False)
    barrier()

    total_ms, e2e_ms, e2e2_ms, e2e_relaxed_ms = max_over_ranks([total_ms, e2e_ms, e2e2_ms, e2e_relaxed_ms], world, "cuda")

    # per-kernel device times of the same step (library-side CUDA events on the launch stream)
    peak, peak_src = measured_peak()
    plan.profile_enable(True)
    plan.profile_reset()
    timed(step, K_steps)
    rows = kernel_table(plan.profile(), algorithmic_bytes(2, Nd[0], Kd[0], M, B), peak)
    plan.profile_enable(False)

    # forward, adjoint and A^H A alone (north star: absolute transforms/s and fraction of the HBM roofline), same batch,
    # L2 flushed between calls, median of 5 repetitions of >= 50 ms each; A^H A keeps y on the device in the interleaved
    # layout (no layout pass either way)
    ab = algorithmic_bytes(2, Nd[0], Kd[0], M, B)
    fwd_bytes = ab["fft_rows_fwd"] + ab["fft_cols_fwd"] + ab["interp"]
    adj_bytes = ab["gridding"] + ab["fft_cols_adj"] + ab["fft_rows_adj"]
    transforms = {}
    for name, fn, nbytes in (("forward", lambda: plan.forward(x, y), fwd_bytes),
                             ("adjoint", lambda: plan.adjoint(y, xo), adj_bytes),
                             ("selfadjoint", lambda: plan.selfadjoint(x, xo), fwd_bytes + adj_bytes)):
        fn()
        ms = timed_median(fn)
        transforms[name] = {"transforms_per_s": world * B / (ms * 1e-3), "ms_per_call": ms, "alg_bytes_per_call": int(nbytes),
                            "frac_of_hbm_roofline": (nbytes / (ms * 1e-3) / 1e9) / peak}

    # the batch-32 point (one interleaved group) of the same workload
    batch32 = None
    if world == 1 and B != 32 and not args.no_extra:
        p32 = nb.NufftPlan(Nd, Kd, Jd, om, max_batch=32)
        x32, y32, xo32 = x[:32].contiguous(), y[:32].contiguous(), xo[:32].contiguous()

        def step32():
            p32.forward(x32, y32)
            p32.adjoint(y32, xo32)

        for _ in range(3):
            step32()
        ms32 = timed_median(step32)
        b32 = algorithmic_bytes(2, Nd[0], Kd[0], M, 32)
        batch32 = {"batch": 32, "ms_per_step": ms32, "pairs_per_s": 32 / (ms32 * 1e-3),
                   "step_frac_of_roofline": (sum(b32.values()) / (ms32 * 1e-3) / 1e9) / peak}
        p32.destroy()

    result = None
    if rank == 0:
        ms_per_step = total_ms / K_steps
        value = aggregate_pairs_per_s(world, B, ms_per_step)
        timed_kernels = {k: v for k, v in rows.items() if "alg_bytes" in v}
        dom = max(timed_kernels, key=lambda k: timed_kernels[k]["ms_per_launch"])
        traffic = dram_traffic("cfg2_batch%d" % B, dom)     # from the committed ncu --set full capture of this workload
        step_bytes = sum(v["alg_bytes"] for v in timed_kernels.values())
        roofline = {
            "bound": "hbm", "kernel": dom, "achieved": timed_kernels[dom]["gbs"], "peak": peak, "unit": "GB/s",
            "frac": timed_kernels[dom]["frac"], "traffic": traffic, "peak_source": peak_src,
            "alg_bytes_per_launch": timed_kernels[dom]["alg_bytes"],
            "ms_per_launch": timed_kernels[dom]["ms_per_launch"],
            "step_alg_bytes": int(step_bytes),
            "step_frac_of_roofline": (step_bytes / (ms_per_step * 1e-3) / 1e9) / peak,
            "kernels": rows,
            "stages_ms": {
                "F (S+pad+FFT)": stage_of(rows, ["fft_rows_fwd", "fft_cols_fwd"]),
                "V": stage_of(rows, ["interp", "y_from_il"]),
                "V^H": stage_of(rows, ["y_to_il", "grid_zero", "gridding", "gridding_merge"]),
                "F^H (IFFT+crop+S^H)": stage_of(rows, ["fft_cols_adj", "fft_rows_adj"]),
            },
            "note": "2-D grids of this batch are partly L2-resident between kernels of one step; V and V^H are "
                    "bound by shared-memory/L1 gather bandwidth before HBM (SURVEY.md 7.3-1)",
        }
        cpu_s, cpu_n, cpu_cores = oracle_pair_seconds(cfg, wl.image_gaussian(Nd), args.cpu_seconds, 200)
        result = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K_steps, "warmup": W,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "complex64 (f32 arithmetic)", "data": "synthetic",
            "config": {"workload": WORKLOAD, "batch": B, "pairs_per_step": B, "l2": "flushed between steps (256 MiB memset)",
                       "parallelism": "replicas x%d" % world, "adjoint_mode": 0,
                       "batch_layout": "interleaved [group][K0][K1][32] (batch >= 12)" if B >= 12 else "planar"},
            "clocks": clocks,
            "e2e": {"value": world * B / (e2e_ms / K_steps * 1e-3), "unit": UNIT,
                    "h2d_bytes_per_step": int(x_host.numel() * 8), "d2h_bytes_per_step": int(xo_host.numel() * 8),
                    "ms_per_step": e2e_ms / K_steps,
                    "order": "strict: copies in are ordered after the caller's stream (flush + start event), nothing moves "
                             "outside the event bracket",
                    "call": "nufft_selfadjoint_host: the forward+adjoint pair A^H(A x) per image with y kept on the device "
                            "(sorted-walk V, no layout pass), 16-image chunks pipelined H2D / kernels / D2H",
                    "relaxed_input_ready": {"value": world * B / (e2e_relaxed_ms / K_steps * 1e-3),
                                            "note": "nufft_host_input_ready(1): the copy in of a call may start before the "
                                                    "previous work on the caller's stream ends (here: during the untimed "
                                                    "flush) -- context, not the e2e number"},
                    "forward_host_plus_adjoint_host": {
                        "value": world * B / (e2e2_ms / K_steps * 1e-3), "ms_per_step": e2e2_ms / K_steps,
                        "h2d_bytes_per_step": int(x_host.numel() * 8 + y_host.numel() * 8),
                        "d2h_bytes_per_step": int(y_host.numel() * 8 + xo_host.numel() * 8),
                        "note": "the same kernels as `value` (nufft_forward + nufft_adjoint), y through the host"}},
            "gpu_launches": int(l1 - l0),
            "roofline": roofline,
            "transforms": transforms,
            "batch32": batch32,
            "cpu_baseline": {"value": 1.0 / cpu_s, "unit": UNIT, "cores": cpu_cores, "kind": "oracle",
                             "sample": "%d forward+adjoint pairs on one image of the workload (batch element 0)" % cpu_n},
            "paper_context": "PAPER.md Table 1 (:299-300): forward 6 ms + adjoint 6 ms on one K80 GK210 (PyCUDA), "
                             "workload sizes not stated by the paper",
        }
        if world == 1 and not args.no_extra:
            # the 3-D half of the metric (BASELINE: "(2D 256^2, 3D 128^3)"), a record of its own next to the headline
            try:
                result["cfg4_3d"] = cfg4_record(nb, torch, peak, peak_src, args.cpu_seconds)
            except Exception as e:
                result["cfg4_3d"] = {"error": repr(e)}
            try:
                result["parity"] = parity_block(nb, torch)
            except Exception as e:
                result["parity"] = {"error": repr(e)}
        if world == 1 and not args.no_extra:
            try:
                result["extra"] = extra_legs(nb, torch, peak, args)
            except Exception as e:  # extras never break the contract line
                result["extra"] = {"error": repr(e)}
    plan.destroy()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(result))
    return 0


def dram_traffic(config, kernel):
    """DRAM bytes per launch of `kernel` from the committed ncu --set full capture (profiles/dram_traffic.csv), or None."""
    try:
        import csv
        with open(os.path.join(ROOT, "profiles", "dram_traffic.csv")) as f:
            for row in csv.DictReader(f):
                if row["config"] == config and row["kernel"] == kernel:
                    return int(row["dram_bytes_per_launch"])
    except Exception:
        pass
    return None


def _events_ms(torch, fn, n, flush):
    evs = []
    for _ in range(n):
        flush.zero_()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        fn()
        b.record()
        evs.append((a, b))
    torch.cuda.synchronize()
    return [a.elapsed_time(b) for a, b in evs]


def cfg4_record(nb, torch, peak, peak_src, cpu_seconds):
    """The 3-D half of the metric (BASELINE config 4: Nd = 128^3, Kd = 256^3, Jd = 6^3, M = 2 097 152 kooshball), batch 1:
    pairs/s, per-kernel roofline, e2e through the host-buffer calls, the oracle on a bounded sample."""
    cfg = wl.config(3)
    Nd, Kd, Jd, om = cfg["Nd"], cfg["Kd"], cfg["Jd"], cfg["om"]
    N, K, M = Nd[0], Kd[0], om.shape[0]
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    p = nb.NufftPlan(Nd, Kd, Jd, om, max_batch=1)
    x_host = torch.from_numpy(wl.image_gaussian(Nd)).reshape(1, *Nd).pin_memory()
    x = x_host.cuda()
    y = p.forward(x)
    xo = p.adjoint(y)

    def step():
        p.forward(x, y)
        p.adjoint(y, xo)

    for _ in range(3):
        step()
    est = max(float(np.median(_events_ms(torch, step, 5, flush))), 1e-3)
    n = max(5, int(np.ceil(50.0 / est)))
    l0 = p.launch_count()
    ms_pair = float(np.median([np.sum(_events_ms(torch, step, n, flush)) / n for _ in range(5)]))
    launches = (p.launch_count() - l0) // (5 * n)
    f_ms = float(np.median(_events_ms(torch, lambda: p.forward(x, y), 10, flush)))
    a_ms = float(np.median(_events_ms(torch, lambda: p.adjoint(y, xo), 10, flush)))
    s_ms = float(np.median(_events_ms(torch, lambda: p.selfadjoint(x, xo), 10, flush)))
    p.profile_enable(True)
    p.profile_reset()
    _events_ms(torch, step, 5, flush)
    ab = algorithmic_bytes(3, N, K, M, 1, cov=0.55)
    rows = kernel_table(p.profile(), ab, peak)
    p.profile_enable(False)
    timed_k = {k: v for k, v in rows.items() if "alg_bytes" in v}
    dom = max(timed_k, key=lambda k: timed_k[k]["ms_per_launch"])
    step_bytes = sum(v["alg_bytes"] for v in timed_k.values())
    # e2e: pinned x -> H2D -> A -> D2H y ; pinned y -> H2D -> A^H -> D2H x'  (strict stream order)
    y_host = torch.empty((1, M), dtype=torch.complex64).pin_memory()
    xo_host = torch.empty((1,) + tuple(Nd), dtype=torch.complex64).pin_memory()

    def step_e2e():
        p.forward_host(x_host, y_host)
        p.adjoint_host(y_host, xo_host)

    for _ in range(2):
        step_e2e()
    e2e_ms = float(np.median(_events_ms(torch, step_e2e, 5, flush)))
    info = p.info()
    p.destroy()
    # the oracle on a bounded sample of the same workload: the first 512 of the 4096 spokes on the full 128^3 / 256^3 geometry
    sub = om[: 512 * 512]
    x128 = wl.image_gaussian(Nd).astype(np.complex128)
    from oracle import nufft_oracle as orc
    t0, c0 = time.perf_counter(), time.process_time()
    orc.adjoint(orc.forward(x128, sub, Nd, Kd, Jd), sub, Nd, Kd, Jd)
    el = time.perf_counter() - t0
    return {
        "metric": METRIC, "unit": UNIT, "value": 1e3 / ms_pair, "ms_per_step": ms_pair, "gpu_launches_per_step": int(launches),
        "config": {"workload": "cfg4_3d_kooshball: Nd=128^3 Kd=256^3 Jd=6^3 M=2097152 (4096 spokes x 512), complex64",
                   "batch": 1, "l2": "flushed between steps (256 MiB memset); the 134 MB grid exceeds L2 anyway",
                   "timing": "median of 5 repetitions of >= 50 ms of event-bracketed steps"},
        "forward_ms": f_ms, "adjoint_ms": a_ms, "selfadjoint_ms": s_ms,
        "roofline": {"bound": "hbm", "kernel": dom, "achieved": timed_k[dom]["gbs"], "peak": peak, "unit": "GB/s",
                     "frac": timed_k[dom]["frac"], "traffic": dram_traffic("cfg4_batch1", dom), "peak_source": peak_src,
                     "alg_bytes_per_launch": timed_k[dom]["alg_bytes"], "ms_per_launch": timed_k[dom]["ms_per_launch"],
                     "step_alg_bytes": int(step_bytes),
                     "step_frac_of_roofline": (step_bytes / (ms_pair * 1e-3) / 1e9) / peak, "kernels": rows,
                     "traffic_by_kernel": {k: dram_traffic("cfg4_batch1", k) for k in timed_k},
                     "note": "interp alg_bytes use coverage 0.55 of the 256^3 grid (SURVEY.md 8(d)); V and V^H are bound by "
                             "issue slots / shared-memory traffic of the 216-point stencil before HBM (SURVEY 7.3-1: ceiling "
                             "16-20 % of HBM peak)"},
        "e2e": {"value": 1e3 / e2e_ms, "unit": UNIT, "ms_per_step": e2e_ms,
                "h2d_bytes_per_step": int(x_host.numel() * 8 + y_host.numel() * 8),
                "d2h_bytes_per_step": int(y_host.numel() * 8 + xo_host.numel() * 8),
                "call": "nufft_forward_host + nufft_adjoint_host, pinned buffers, strict stream order"},
        "cpu_baseline": {"value": 1.0 / el, "unit": UNIT, "cores": cores_used(time.process_time() - c0, el), "kind": "oracle",
                         "sample": "one forward+adjoint pair on the first 512 of the 4096 spokes (M = 262144) with the full "
                                   "128^3 / 256^3 geometry: %.1f s" % el},
        "plan": info,
    }


def coef_mode_table(nb, torch):
    """North star item 3 / SURVEY 8(b) coef_mode: V (and the 3-D V^H) with weights recomputed on the fly from the kernel
    polynomial (mode 0: 4 + 4 d bytes of plan data per sample) against weights precomputed by the plan in a coalesced
    per-sample layout (mode 1: 64 B per sample on the interleaved 2-D path, 112 B in 3-D), on config 2 batch 64 and config 4.
    Device ms per launch (library-side events, L2 flushed between steps) and plan bytes; parity of mode 1 vs the oracle."""
    from oracle import nufft_oracle as orc
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    out = {}
    for name, cfg, B in (("cfg2_batch64", wl.config(1), 64), ("cfg4_batch1", wl.config(3), 1)):
        Nd, Kd, Jd, om = cfg["Nd"], cfg["Kd"], cfg["Jd"], cfg["om"]
        x = torch.from_numpy(wl.image_gaussian(Nd, batch=B)).cuda()
        rows = {}
        for mode in (0, 1):
            p = nb.NufftPlan(Nd, Kd, Jd, om, max_batch=B, coef_mode=mode)
            y = p.forward(x)
            xo = p.adjoint(y)
            for _ in range(3):
                p.forward(x, y), p.adjoint(y, xo), p.selfadjoint(x, xo)
            p.profile_enable(True)
            p.profile_reset()
            for _ in range(10):
                flush.zero_()
                p.forward(x, y)
                p.adjoint(y, xo)
            torch.cuda.synchronize()
            pr = p.profile()
            fa = {k: v[0] / v[1] for k, v in pr.items() if v[1] and k in ("interp", "gridding")}
            p.profile_reset()
            for _ in range(10):
                flush.zero_()
                p.selfadjoint(x, xo)
            torch.cuda.synchronize()
            sa = {k: v[0] / v[1] for k, v in p.profile().items() if v[1] and k in ("interp", "gridding")}
            rows["coef_mode_%d" % mode] = {"interp_ms": fa.get("interp"), "gridding_ms": fa.get("gridding"),
                                           "interp_ms_in_selfadjoint": sa.get("interp"), "plan_bytes": p.info()["bytes_plan"]}
            p.destroy()
        out[name] = rows
    cfg = wl.config(3, scale=4)
    Nd, Kd, Jd, om = cfg["Nd"], cfg["Kd"], cfg["Jd"], cfg["om"]
    xs, ys = wl.image_gaussian(Nd), wl.data_gaussian(om.shape[0])
    p = nb.NufftPlan(Nd, Kd, Jd, om, coef_mode=1)
    rel = lambda a, b: float(np.linalg.norm(a.ravel() - b.ravel()) / np.linalg.norm(b.ravel()))
    out["parity_coef_mode_1_cfg4_scaled"] = {
        "forward": rel(p.forward(torch.from_numpy(xs).cuda()).cpu().numpy()[0], orc.forward(xs.astype(np.complex128), om, Nd, Kd, Jd)),
        "adjoint": rel(p.adjoint(torch.from_numpy(ys).cuda()).cpu().numpy()[0], orc.adjoint(ys.astype(np.complex128), om, Nd, Kd, Jd))}
    p.destroy()
    return out


def parity_block(nb, torch):
    """Relative L2 and max-abs (of the largest reference value) of forward / adjoint / A^H A against the float64 oracle,
    on config 1 and the scaled config 4, computed in this very run (SURVEY section 5 "Metrics")."""
    from oracle import nufft_oracle as orc
    out = {}
    for name, cfg in (("cfg1_2d_64", wl.config(0)), ("cfg4_3d_scaled_32", wl.config(3, scale=4))):
        Nd, Kd, Jd, om = cfg["Nd"], cfg["Kd"], cfg["Jd"], cfg["om"]
        x = wl.image_gaussian(Nd)
        y = wl.data_gaussian(om.shape[0])
        p = nb.NufftPlan(Nd, Kd, Jd, om)
        dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
        got = (p.forward(dev(x)).cpu().numpy()[0], p.adjoint(dev(y)).cpu().numpy()[0], p.selfadjoint(dev(x)).cpu().numpy()[0])
        p.destroy()
        yo = orc.forward(x.astype(np.complex128), om, Nd, Kd, Jd)
        ref = (yo, orc.adjoint(y.astype(np.complex128), om, Nd, Kd, Jd), orc.adjoint(yo, om, Nd, Kd, Jd))
        out[name] = {k: {"rel_l2": float(np.linalg.norm(g.ravel() - r.ravel()) / np.linalg.norm(r.ravel())),
                         "max_abs_over_max_ref": float(np.abs(g.ravel() - r.ravel()).max() / np.abs(r).max())}
                     for k, g, r in zip(("forward", "adjoint", "selfadjoint"), got, ref)}
    out["bounds"] = {"rel_l2": 2e-5, "max_abs_over_max_ref": "50 eps32 sqrt(prod J): 3.6e-5 (2-D), 8.8e-5 (3-D)"}
    return out


def extra_legs(nb, torch, peak, args):
    """Other BASELINE configs on one GPU: batch-1 latency of config 2, config 3 (CG), config 5 (L1TV-OLS), variants."""
    out = {}

    def time_calls(fn, n, flush):
        evs = []
        for _ in range(n):
            flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            fn()
            b.record()
            evs.append((a, b))
        torch.cuda.synchronize()
        return float(np.median([a.elapsed_time(b) for a, b in evs]))

    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    # config 2, batch 1 (latency)
    cfg = wl.config(1)
    p = nb.NufftPlan(cfg["Nd"], cfg["Kd"], cfg["Jd"], cfg["om"], max_batch=1)
    x = torch.from_numpy(wl.image_gaussian(cfg["Nd"])).cuda().reshape(1, *cfg["Nd"])
    y = p.forward(x)
    xo = p.adjoint(y)
    for _ in range(3):
        p.forward(x, y), p.adjoint(y, xo)
    out["cfg2_batch1"] = {"forward_ms": time_calls(lambda: p.forward(x, y), 20, flush),
                          "adjoint_ms": time_calls(lambda: p.adjoint(y, xo), 20, flush),
                          "selfadjoint_ms": time_calls(lambda: p.selfadjoint(x, xo), 20, flush)}
    p.destroy()
    # the same with opts.use_graphs (repeated calls with fixed pointers replayed as CUDA graphs; non-default stream)
    pg = nb.NufftPlan(cfg["Nd"], cfg["Kd"], cfg["Jd"], cfg["om"], max_batch=1, use_graphs=1)
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())

    def time_side(fn, n):
        evs = []
        with torch.cuda.stream(side):
            for _ in range(3):
                fn()
            for _ in range(n):
                flush.zero_()
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(side)
                fn()
                b.record(side)
                evs.append((a, b))
        side.synchronize()
        return float(np.median([a.elapsed_time(b) for a, b in evs]))

    out["cfg2_batch1"].update({"forward_graph_ms": time_side(lambda: pg.forward(x, y), 20),
                               "adjoint_graph_ms": time_side(lambda: pg.adjoint(y, xo), 20),
                               "selfadjoint_graph_ms": time_side(lambda: pg.selfadjoint(x, xo), 20)})
    torch.cuda.current_stream().wait_stream(side)
    pg.destroy()
    # config 3: 2-D variable-density spiral 512^2, 50 CG iterations on A^H A x = A^H y (batch 1, planar path)
    cfg = wl.config(2)
    p = nb.NufftPlan(cfg["Nd"], cfg["Kd"], cfg["Jd"], cfg["om"], max_batch=1)
    xt = torch.from_numpy(wl.phantom(cfg["Nd"])).cuda().reshape(1, *cfg["Nd"])
    y3 = p.forward(xt)
    y3 = y3 + 0.01 * y3.abs().pow(2).mean().sqrt() * torch.randn_like(y3)
    xs = p.solve_cg(y3, 3)
    cg_ms = time_calls(lambda: p.solve_cg(y3, 50, x=xs), 3, flush)
    sa_ms = time_calls(lambda: p.selfadjoint(xt, xt.clone()), 10, flush)
    out["cfg3_2d_spiral_cg50"] = {"workload": "Nd=512^2 Kd=1024^2 M=262144 VD spiral, batch 1", "cg50_ms": cg_ms,
                                  "ms_per_iteration": cg_ms / 50, "selfadjoint_ms": sa_ms,
                                  "note": "linear CG on A^H A x = A^H y, x0 = 0, scalars float64 on device (R12)"}
    p.destroy()
    # the same 50 iterations with opts.use_graphs (one CUDA graph per CG iteration), on a non-default stream
    pg = nb.NufftPlan(cfg["Nd"], cfg["Kd"], cfg["Jd"], cfg["om"], max_batch=1, use_graphs=1)
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        xs = pg.solve_cg(y3, 5)
        evs = []
        for _ in range(3):
            flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(side)
            pg.solve_cg(y3, 50, x=xs)
            b.record(side)
            evs.append((a, b))
    side.synchronize()
    out["cfg3_2d_spiral_cg50"]["cg50_graph_ms"] = float(np.median([a.elapsed_time(b) for a, b in evs]))
    # next row 8(f)-1 on config 3: the same 50 iterations with A^H A in Toeplitz form (no V / V^H per iteration)
    pg.toeplitz_build()
    pg.toeplitz_enable(True)
    with torch.cuda.stream(side):
        pg.solve_cg(y3, 5, x=xs)
        evs = []
        for _ in range(3):
            flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(side)
            pg.solve_cg(y3, 50, x=xs)
            b.record(side)
            evs.append((a, b))
    side.synchronize()
    out["cfg3_2d_spiral_cg50"]["cg50_toeplitz_graph_ms"] = float(np.median([a.elapsed_time(b) for a, b in evs]))
    torch.cuda.current_stream().wait_stream(side)
    pg.destroy()
    # config 5: 32-coil 2-D radial, multi-coil A^H A and 20 split-Bregman L1TV-OLS iterations (interleaved path)
    cfg = wl.config(4)
    nc = cfg["ncoil"]
    p = nb.NufftPlan(cfg["Nd"], cfg["Kd"], cfg["Jd"], cfg["om"], max_batch=nc)
    c = torch.from_numpy(wl.coil_maps(nc, cfg["Nd"])).cuda()
    p.set_coils(c)
    xt = torch.from_numpy(wl.phantom(cfg["Nd"])).cuda()
    y5 = p.forward_coils(xt)
    y5 = y5 + 0.01 * y5.abs().pow(2).mean().sqrt() * torch.randn_like(y5)
    xo5 = p.selfadjoint_coils(xt)
    xs = p.solve_l1tv_ols(y5, 1.0, 0.02, 1, 1, 1, use_coils=True)
    sac_ms = time_calls(lambda: p.selfadjoint_coils(xt, xo5), 10, flush)
    fwc_ms = time_calls(lambda: p.forward_coils(xt, y5), 10, flush)
    adc_ms = time_calls(lambda: p.adjoint_coils(y5, xo5), 10, flush)
    tv_ms = time_calls(lambda: p.solve_l1tv_ols(y5, 1.0, 0.02, 4, 5, 3, use_coils=True, x=xs), 3, flush)
    # next row 8(f)-1: Toeplitz A^H A (no V / V^H per application) on the same 32-coil problem
    p.toeplitz_build()
    toep_ms = time_calls(lambda: p.selfadjoint_toeplitz_coils(xt, xo5), 10, flush)
    p.toeplitz_enable(True)
    xs = p.solve_l1tv_ols(y5, 1.0, 0.02, 1, 1, 1, use_coils=True, x=xs)
    tv_toep_ms = time_calls(lambda: p.solve_l1tv_ols(y5, 1.0, 0.02, 4, 5, 3, use_coils=True, x=xs), 3, flush)
    p.toeplitz_enable(False)
    # next row 8(f)-3: density compensation, 4 iterations of eq. (6) + the weighted adjoint of eq. (7)
    wdc = p.density_weights(1)
    dcf_ms = time_calls(lambda: p.density_weights(4, wdc), 5, flush)
    out["next_rows"] = {
        "toeplitz_selfadjoint_coils_ms": toep_ms, "l1tv_ols_20it_toeplitz_ms": tv_toep_ms,
        "density_weights_4it_ms": dcf_ms,
        "note": "cfg5 problem; Toeplitz: crop(F^H(T^ . F(pad c_i x))) summed over 32 coils, T^ built once per plan"}
    # the same 20 iterations with the inner CG steps replayed as CUDA graphs (opts.use_graphs; non-default stream)
    pg = nb.NufftPlan(cfg["Nd"], cfg["Kd"], cfg["Jd"], cfg["om"], max_batch=nc, use_graphs=1)
    pg.set_coils(c)
    pg.toeplitz_build()
    pg.toeplitz_enable(True)
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        xs2 = pg.solve_l1tv_ols(y5, 1.0, 0.02, 1, 1, 3, use_coils=True)
        evs = []
        for _ in range(3):
            flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(side)
            pg.solve_l1tv_ols(y5, 1.0, 0.02, 4, 5, 3, use_coils=True, x=xs2)
            b.record(side)
            evs.append((a, b))
    side.synchronize()
    torch.cuda.current_stream().wait_stream(side)
    out["next_rows"]["l1tv_ols_20it_toeplitz_graph_ms"] = float(np.median([a.elapsed_time(b) for a, b in evs]))
    pg.destroy()
    out["cfg5_2d_multicoil_l1tv"] = {
        "workload": "Nd=256^2 Kd=512^2 M=65536 radial 128x512, 32 coils", "forward_coils_ms": fwc_ms,
        "adjoint_coils_ms": adc_ms, "selfadjoint_coils_ms": sac_ms, "l1tv_ols_20it_ms": tv_ms,
        "coil_pairs_per_s": 32 * 1e3 / (fwc_ms + adc_ms),
        "note": "n_outer=4, n_inner=5, n_cg=3, mu=1, lam=0.02 (R17); 32-coil batch on the interleaved grid"}
    p.destroy()
    # the paper's own experiment shape (512^2 image, non-Cartesian k-space of its ref. [15]) on a synthetic
    # PROPELLER stand-in, batch 1: the operations of Table 1, whose workload the paper does not state
    cfg = wl.config_propeller()
    pp = nb.NufftPlan(cfg["Nd"], cfg["Kd"], cfg["Jd"], cfg["om"], max_batch=1)
    xt = torch.from_numpy(wl.phantom(cfg["Nd"])).cuda().reshape(1, *cfg["Nd"])
    yp = pp.forward(xt)
    xop = pp.adjoint(yp)
    for _ in range(3):
        pp.forward(xt, yp), pp.adjoint(yp, xop), pp.selfadjoint(xt, xop)
    xs = pp.solve_cg(yp, 2)
    xl = pp.solve_l1tv_ols(yp, 1.0, 0.02, 1, 1, 1)
    xd = pp.solve_l1tv_lad(yp, 1.0, 0.02, 1, 1, 1)
    out["paper_2_3_propeller_512"] = {
        "workload": "Nd=512^2 Kd=1024^2 Jd=6^2, PROPELLER 24 blades x 32 lines x 512 (M=393216), batch 1, synthetic",
        "forward_ms": time_calls(lambda: pp.forward(xt, yp), 10, flush),
        "adjoint_ms": time_calls(lambda: pp.adjoint(yp, xop), 10, flush),
        "selfadjoint_ms": time_calls(lambda: pp.selfadjoint(xt, xop), 10, flush),
        "cg_20it_ms": time_calls(lambda: pp.solve_cg(yp, 20, x=xs), 3, flush),
        "l1tv_ols_20it_ms": time_calls(lambda: pp.solve_l1tv_ols(yp, 1.0, 0.02, 4, 5, 3, x=xl), 3, flush),
        "l1tv_lad_20it_ms": time_calls(lambda: pp.solve_l1tv_lad(yp, 1.0, 0.02, 4, 5, 3, x=xd), 3, flush),
        "paper_table1_k80_pycuda": "A 6 ms, A^H 6 ms, A^H A 8 ms; CG 1.89 s, L1TV-OLS 1.68 s, L1TV-LAD 1.78 s "
                                   "(PAPER.md:299-305; sizes and iteration counts not stated: context only)"}
    pp.destroy()
    # SURVEY 8(f)-4 variants on config 2's trajectory, batch 1 (functional paths next to the tuned one)
    cfg = wl.config(1)
    var = {}
    for name, Nd_v, Jd_v, kern in (("kb_J6", (256, 256), (6, 6), "kb"), ("minmax_J6", (256, 256), (6, 6), "minmax"),
                                   ("kb_J4", (256, 256), (4, 4), "kb"), ("kb_J8", (256, 256), (8, 8), "kb"),
                                   ("kb_J6_sigma1.6", (320, 320), (6, 6), "kb")):
        pv = nb.NufftPlan(Nd_v, cfg["Kd"], Jd_v, cfg["om"], max_batch=1, kernel=kern)
        xv = torch.from_numpy(wl.image_gaussian(Nd_v)).cuda().reshape(1, *Nd_v)
        yv = pv.forward(xv)
        xov = pv.adjoint(yv)
        for _ in range(3):
            pv.forward(xv, yv), pv.adjoint(yv, xov)
        var[name] = {"forward_ms": time_calls(lambda: pv.forward(xv, yv), 10, flush),
                     "adjoint_ms": time_calls(lambda: pv.adjoint(yv, xov), 10, flush)}
        pv.destroy()
    var["note"] = ("Kd=512^2, radial 256x512; min-max runs the same kernels as Kaiser-Bessel; J != 6 runs the direct V / atomic "
                   "V^H kernels; sigma != 2 (Nd=320^2) runs the unpruned FFT with pad / crop fused into its contiguous-axis pass")
    out["variants_cfg2_batch1"] = var
    # cuFFT reference point for F alone (never linked into the product): full 512^2 FFT of 64 grids via torch.fft
    gref = torch.randn(64, 512, 512, dtype=torch.complex64, device="cuda")
    torch.fft.fftn(gref, dim=(1, 2))
    out["cufft_reference"] = {"what": "torch.fft.fftn (cuFFT) on [64][512][512] complex64, unpruned, no scaling/pad fused",
                              "ms": time_calls(lambda: torch.fft.fftn(gref, dim=(1, 2)), 10, flush),
                              "ours_F_ms": "roofline.stages_ms['F (S+pad+FFT)'] (pruned, S and zero-pad fused)"}
    del gref
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--batch", type=int, default=64)
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    ap.add_argument("--no-extra", action="store_true",
                    help="headline workload only: skip the cfg4_3d record, the parity block, the batch-32 point and the extra "
                         "legs (used by the ncu commands in profiles/)")
    ap.add_argument("--only", default="", choices=["", "cfg4", "coef"],
                    help="cfg4: measure only the 3-D config 4 record and print it as the JSON line (used by the ncu "
                         "commands in profiles/)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.only == "coef":
        import torch
        import paper_1710_03197_b200 as nb
        torch.cuda.set_device(0)
        print(json.dumps({"coef_mode_table": coef_mode_table(nb, torch)}))
        return 0
    if args.only == "cfg4":
        import torch
        import paper_1710_03197_b200 as nb
        torch.cuda.set_device(0)
        peak, peak_src = measured_peak()
        rec = cfg4_record(nb, torch, peak, peak_src, args.cpu_seconds)
        rec.update({"n_gpus": 1, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                    "dtype": "complex64 (f32 arithmetic)", "data": "synthetic"})
        print(json.dumps(rec))
        return 0
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
               "--master-addr", "127.0.0.1", "--master-port", "29533", os.path.abspath(__file__)] + sys.argv[1:]
        return subprocess.call(cmd)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
