#!/usr/bin/env python
"""bench.py -- demagnetization-field evaluations per second of hfft_demag on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl reference]

A "step" is one pass of the whole hot path (S1 x-FFT, S2 y-FFT, S3 layer coupling, S4 inverse
y-FFT, S5 inverse x-FFT) over one batch of synthetic magnetisation, i.e. one
hfft_demag call (B field evaluations; B = 1 except config 5).  Default workload: BASELINE.json
configs[3], the 256 x 256 x 64 non-equidistant fp32 stack that north_star's target is quoted on
(tensor bank 12.9 GB, far larger than L2, so every step streams it from HBM).

Prints ONE JSON line (contract in the task statement).  Multi-GPU: the method does not shard
(north_star: one GPU, no collectives) -- N ranks run N independent replicas ("replicas only").
`--impl reference` times the CPU oracle (oracle/, T1 hybrid with numpy FFT) on the host cores.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1910_07054_b200 import workloads as W  # noqa: E402

METRIC = "demag_field_evals_per_sec"
UNIT = "evals/s"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--config", default="4", help="BASELINE.json config 1..5, '2f64', '4eq'")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sweep-nz", action="store_true",
                    help="layer-count scaling at 256 x 256 fp32 (the experiment of PAPER.md:189-203, Fig.3/4): one JSON "
                         "line per (nz, method) instead of the bench line")
    ap.add_argument("--mirror", type=int, default=None, help="hfft_plan_set_mirror mode (default: the library's, 1)")
    ap.add_argument("--recip", type=int, default=None, help="hfft_plan_set_recip (default: the library's)")
    ap.add_argument("--dedup", type=int, default=None, help="hfft_plan_set_dedup mode (default: the library's, 1)")
    return ap.parse_args()


def get_workload(name):
    if name == "2f64":
        return W.config(2, "f64")
    if name == "4eq":
        return W.config(4, "equal")
    return W.config(int(name))


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as fh:
            d = json.load(fh)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def algorithmic_bytes(w, n_slots=None, mirror=False):
    """what the shipped storage must move per hfft_demag call.
    n_slots: bank slots per wavevector (nz^2 pairs, or the tensor classes of a deduplicated bank);
    mirror: ky-mirror storage, one bank entry per (kx, ky <= ny)."""
    s = 4 if w.precision == "f32" else 8
    n_k = 2 * w.ny * (w.nx + 1)
    planes = 3 * w.nz * w.B
    bank = 6 * (n_slots if n_slots else w.nz * w.nz) * ((w.nx + 1) * (w.ny + 1) if mirror else n_k) * s
    spec = planes * n_k * 2 * s            # M^ (= H^)
    xhat = planes * w.ny * (w.nx + 1) * 2 * s
    field = planes * w.ny * w.nx * s
    coupling = bank + 2 * spec
    whole = 2 * field + 4 * xhat + 4 * spec + bank
    return {"bank": bank, "coupling": coupling, "whole": whole}


class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index):
        self.index = index
        self.proc = None
        self.out = None

    def start(self):
        self.out = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.FIELDS,
                 "--format=csv,noheader,nounits", "-lms", "50"], stdout=self.out, stderr=subprocess.DEVNULL)
        except OSError:
            self.proc = None

    def stop(self):
        res = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return res
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.out.flush()
        self.out.seek(0)
        sm, mx, reasons = [], [], set()
        for ln in self.out:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except ValueError:
                continue
            for name, val in zip(self.NAMES, f[3:7]):
                if val == "Active":
                    reasons.add(name)
        self.out.close()
        os.unlink(self.out.name)
        if sm:
            res.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons),
                       samples=len(sm))
        return res


def cpu_baseline(w, budget_s=20.0):
    """The oracle's hybrid tier (T1, numpy FFT) on target layer 0 of the workload, tensor row
    prebuilt (setup, like hfft_build_tensor for the GPU).  evals/s = 1 / (nz * t_layer)."""
    import oracle as O
    m = w.m_rounded([0])[0]
    t0 = time.perf_counter()
    row = O.tensor_row(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, 0)
    setup = time.perf_counter() - t0
    times = []
    while len(times) < 3 or (sum(times) < budget_s and len(times) < 20):
        t0 = time.perf_counter()
        O.hybrid_layers(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, m, w.Ms, [0], dft="fft", rows={0: row})
        times.append(time.perf_counter() - t0)
        if sum(times) > 4 * budget_s:
            break
    t_layer = float(np.median(times))
    return {"value": 1.0 / (w.nz * t_layer), "unit": UNIT, "cores": O.threads(), "kind": "oracle",
            "sample": "target layer 0 of %d, one state (oracle.hybrid_layers, numpy FFT, fp64), tensor row "
                      "prebuilt; median of %d runs of %.3f s; value = 1/(nz*t_layer); numpy's FFT and einsum "
                      "run on 1 thread, the binary128 tensor row (setup, %.1f s) on `cores` OpenMP threads"
                      % (w.nz, len(times), t_layer, setup),
            "oracle_tensor_row_s": setup}


def run_reference(args, w):
    """--impl reference: the oracle, as it stands, on the host cores.  One step = target layer 0."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle as O
    m = w.m_rounded([0])[0]
    row = O.tensor_row(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, 0)
    Ms = np.broadcast_to(np.asarray(w.Ms, dtype=np.float64), (w.nz,))

    def make_step(nzs):
        """Target layer 0 of the stack cut to its first nzs layers (N_0j depends on the layers 0..j only, so the
        tensor row of the cut stack is the head of the full row)."""
        mm, dz, ms, rows = np.ascontiguousarray(m[:, :nzs]), w.dz[:nzs], Ms[:nzs], {0: row[:nzs]}
        return lambda: O.hybrid_layers(w.nx, w.ny, nzs, w.dx, w.dy, dz, mm, ms, [0], dft="fft", rows=rows)

    # size the per-step sample so that the whole run stays within a few minutes whatever K and W are
    budget_s = 120.0
    step = make_step(w.nz)
    t0 = time.perf_counter()
    step()
    t_probe = time.perf_counter() - t0
    nzs = w.nz
    if (args.steps + args.warmup) * t_probe > budget_s:
        nzs = max(1, min(w.nz, int(w.nz * budget_s / ((args.steps + args.warmup) * t_probe))))
        step = make_step(nzs)
    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = time.perf_counter() - t0
    # one step = 1 target layer x nzs source layers; a whole evaluation = nz target layers x nz source layers
    t_layer = dt / args.steps * (w.nz / nzs)
    value = 1.0 / (w.nz * t_layer)                          # one state; evals/s of a whole-stack evaluation
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(w, "host memory; no GPU"),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": O.threads(), "kind": "oracle",
                         "sample": "each step = target layer 0 of %d, summed over the first %d of %d source layers, of one "
                                   "state (oracle.hybrid_layers, numpy FFT, fp64, tensor row prebuilt); value = "
                                   "1 / (nz * s_per_step * nz / source layers per step)" % (w.nz, nzs, w.nz)},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def max_over_ranks(times_ms, device="cpu"):
    """The timed regions of all ranks, reduced with MAX (the slowest replica sets the job's time).
    Works on any initialised process group (nccl on the GPUs, gloo in the CPU tests); identity for one process."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(times_ms), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def whole_job_value(world, batch, steps, ms_total):
    """Evaluations per second of the whole job: every rank ran `steps` calls of `batch` states (weak scaling)."""
    return world * batch * steps / (ms_total * 1e-3)


def sweep_nz():
    """evaluation time against the number of layers at nx = ny = 256, non-equidistant hybrid method
    (fit a x^2 + b x + c) against the equidistant methods (a x log x + b).  Synthetic: dz log-uniform in [0.3, 3] nm
    (hybrid) or 1 nm (equidistant), random unit vectors, fp32, mean of 20-50 back-to-back calls, best of 3."""
    import torch
    from paper_1910_07054_b200 import binding as hb
    nx = ny = 256
    for nz in [2, 4, 8, 16, 32, 64, 96, 128]:
        m = torch.randn(1, 3, nz, ny, nx, device="cuda", dtype=torch.float32)
        m /= m.norm(dim=1, keepdim=True)
        h = torch.empty_like(m)
        dz_var = np.exp(np.random.default_rng(SEED_SWEEP + nz).uniform(np.log(0.3), np.log(3.0), size=nz))
        for name, dz, kw in [("hybrid (ky-mirror bank)", dz_var, dict(dedup=0)),
                             ("hybrid (plain bank)", dz_var, dict(dedup=0, mirror=0)),
                             ("equidistant, Toeplitz classes", np.full(nz, 1.0), dict(dedup=2)),
                             ("equidistant, z-FFT (Eq.25)", np.full(nz, 1.0), dict(dedup=3))]:
            if kw.get("mirror") == 0 and nz > 64:
                continue                                     # plain bank of 29 / 52 GB: not needed for the comparison
            plan = hb.Plan(nx, ny, nz, 2.0, 2.0, dz, "f32", **kw)
            t0 = time.perf_counter()
            plan.build_tensor()
            torch.cuda.synchronize()
            setup = time.perf_counter() - t0
            info = hb.plan_info(plan.handle)
            for _ in range(5):
                plan.demag(m, 8e5, h)
            n = 50 if nz <= 32 else 20
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            best = 1e30
            for _ in range(3):
                e0.record()
                for _ in range(n):
                    plan.demag(m, 8e5, h)
                e1.record()
                torch.cuda.synchronize()
                best = min(best, e0.elapsed_time(e1) / n)
            print(json.dumps({"nz": nz, "method": name, "ms_per_eval": best, "setup_s": setup,
                              "bank_GB": info.bank_bytes / 1e9, "dedup": info.dedup, "mirror": info.mirror}), flush=True)
            plan.close()
            del plan
            torch.cuda.empty_cache()


SEED_SWEEP = 191007054


def workload_config(w, l2):
    return {"workload": w.name, "nx": w.nx, "ny": w.ny, "nz": w.nz, "batch": w.B, "precision": w.precision,
            "dz_nm": [round(float(v), 6) for v in w.dz[:8]] + (["..."] if w.nz > 8 else []),
            "m": w.m_kind, "seed": w.seed, "l2": l2, "parallelism": "replicas only (no sharding, no collective)"}


def main():
    args = parse_args()
    if args.sweep_nz:
        sweep_nz()
        return
    w = get_workload(args.config)
    if args.impl == "reference":
        run_reference(args, w)
        return

    import torch
    import torch.distributed as dist
    from paper_1910_07054_b200 import binding as hb

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: hfft has no CPU path")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    steps, warmup = max(1, args.steps), max(3, args.warmup)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    plan = hb.Plan(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, w.precision, batch=w.B, dedup=args.dedup, mirror=args.mirror,
                   recip=args.recip)
    t0 = time.perf_counter()
    plan.build_tensor()
    torch.cuda.synchronize()
    setup_s = time.perf_counter() - t0

    dt = torch.float32 if w.precision == "f32" else torch.float64
    m_host = torch.from_numpy(w.m_rounded()).to(dt).pin_memory()
    m = m_host.cuda()
    h = torch.empty_like(m)
    h_host = torch.empty_like(m_host).pin_memory()
    Ms = w.Ms
    nbytes = m.numel() * m.element_size()
    dedup = int(plan.info.dedup)
    # bank slots per wavevector: nz^2 pairs, tensor classes, or the Lz values of kz in the z-FFT mode
    mirror = bool(plan.info.mirror)
    slots = int(plan.info.bank_bytes // (6 * (plan.info.n_k_padded // (2 if mirror else 1)) * (4 if w.precision == "f32" else 8)))
    ab = algorithmic_bytes(w, slots if (dedup or int(plan.info.mirror) == 2) else None, mirror)
    # inputs larger than L2?  otherwise flush L2 between steps (and say so)
    flush = None
    if ab["whole"] < 512 << 20:
        flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

    def step():
        if flush is not None:
            flush.zero_()
        plan.demag(m, Ms, h)

    for _ in range(warmup):
        step()
    sampler = ClockSampler(local_rank)
    barrier()
    sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    # ---- timed region 1: device-resident inputs ----
    if flush is None:
        ev0.record()
        for _ in range(steps):
            step()
        ev1.record()
        torch.cuda.synchronize()
        ms_total = ev0.elapsed_time(ev1)
    else:   # time each step alone so that the flush is outside the timed intervals
        ms_total = 0.0
        for _ in range(steps):
            flush.zero_()
            ev0.record()
            plan.demag(m, Ms, h)
            ev1.record()
            torch.cuda.synchronize()
            ms_total += ev0.elapsed_time(ev1)
    barrier()
    # ---- small (launch-bound) configs only: the same step replayed from a CUDA graph (hfft_demag is capturable) ----
    ms_graph = None
    if flush is not None or ab["whole"] < (2 << 30):
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            plan.demag(m, Ms, h)
        torch.cuda.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=side):
            plan.demag(m, Ms, h)
        if flush is not None:
            ms_graph = 0.0
            for _ in range(steps):
                flush.zero_()
                ev0.record()
                graph.replay()
                ev1.record()
                torch.cuda.synchronize()
                ms_graph += ev0.elapsed_time(ev1)
            ms_graph /= steps
        else:                                            # inputs larger than L2: back to back, as the main region
            graph.replay()
            ev0.record()
            for _ in range(steps):
                graph.replay()
            ev1.record()
            torch.cuda.synchronize()
            ms_graph = ev0.elapsed_time(ev1) / steps
        del graph
    barrier()
    # ---- timed region 2: same steps with per-stage CUDA events (hfft_profile_*) ----
    hb.profile_enable(plan.handle, True)
    stage_ms = np.zeros(hb.NUM_STAGES)
    calls = 0
    done = 0
    while done < steps:
        n = min(200, steps - done)
        for _ in range(n):
            step()
        ms, c = hb.profile_read(plan.handle)
        stage_ms += ms
        calls += c
        done += n
    hb.profile_enable(plan.handle, False)
    stage_ms /= max(calls, 1)
    # ---- timed region 3: end to end through the host-buffer API (pinned host buffers).  Every step copies its
    # input host -> device and its result device -> host inside the timed region; hfft_demag_host_async pipelines
    # the copies of neighbouring steps with the kernels (two staging slots, three streams), hfft_host_join + the
    # final synchronisation close the region.  Also timed: the plain, serialised hfft_demag_host.
    for _ in range(3):
        plan.demag_host(m_host, Ms, h_host)
    barrier()
    e2e_steps = max(1, min(steps, 50))
    ev0.record()
    for _ in range(e2e_steps):
        plan.demag_host(m_host, Ms, h_host)
    ev1.record()
    torch.cuda.synchronize()
    ms_e2e_serial = ev0.elapsed_time(ev1)
    for _ in range(3):
        plan.demag_host_async(m_host, Ms, h_host)
    plan.host_join()
    barrier()
    ev0.record()
    for _ in range(e2e_steps):
        plan.demag_host_async(m_host, Ms, h_host)
    plan.host_join()
    ev1.record()
    torch.cuda.synchronize()
    ms_e2e = ev0.elapsed_time(ev1)
    barrier()
    clocks = sampler.stop()

    assert bool(torch.isfinite(h).all()) and bool(torch.isfinite(h_host).all())
    ms_total, ms_e2e, ms_e2e_serial = max_over_ranks([ms_total, ms_e2e, ms_e2e_serial], device="cuda")

    if rank == 0:
        peak, peak_src = measured_peaks()
        ms_step = ms_total / steps
        value = whole_job_value(world, w.B, steps, ms_total)
        coup_ms = float(stage_ms[hb.STAGE_NAMES.index("coupling")])
        achieved = ab["coupling"] / (coup_ms * 1e-3) / 1e9 if coup_ms > 0 else None
        traffic = None
        tp = os.path.join(ROOT, "profiles", "traffic.json")
        if os.path.exists(tp):
            with open(tp) as fh:
                traffic = json.load(fh).get(w.name, {}).get("coupling_dram_bytes_per_launch")
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warmup,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": w.precision, "data": "synthetic",
            "config": workload_config(
                w, "inputs larger than L2 (tensor bank %.2f GB streamed every step)" % (ab["bank"] / 1e9)
                if flush is None else "L2 flushed (256 MiB memset) before every timed step"),
            "clocks": {"sm_mhz": clocks["sm_mhz"], "sm_max_mhz": clocks["sm_max_mhz"], "reasons": clocks["reasons"],
                       "samples": clocks["samples"]},
            "e2e": {"value": whole_job_value(world, w.B, e2e_steps, ms_e2e), "unit": UNIT,
                    "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes, "steps": e2e_steps,
                    "api": "hfft_demag_host_async + hfft_host_join (per step: pinned host m -> device, 5 kernels, "
                           "device h -> pinned host; copies of neighbouring steps overlap the kernels)",
                    "serialised_hfft_demag_host": whole_job_value(world, w.B, e2e_steps, ms_e2e_serial)},
            "gpu_launches": plan.info.launches_per_demag * steps,
            "roofline": {"bound": "hbm", "kernel": "coupling_kernel (S3)", "achieved": achieved, "peak": peak,
                         "peak_source": peak_src, "unit": "GB/s", "frac": achieved / peak if achieved else None,
                         "frac_of_nominal_8TBs": achieved / 8000.0 if achieved else None,
                         "algorithmic_bytes_per_launch": ab["coupling"], "avg_launch_ms": coup_ms,
                         "traffic": traffic},
            "stages_ms": {n: float(v) for n, v in zip(hb.STAGE_NAMES, stage_ms)},
            "whole_eval": {"algorithmic_bytes": ab["whole"], "roofline_ms_at_peak": ab["whole"] / peak / 1e6,
                           "ms_per_step": ms_step, "ratio_to_roofline": ms_step / (ab["whole"] / peak / 1e6)},
            "setup_s": setup_s,
        }
        if ms_graph is not None:
            line["cuda_graph"] = {"ms_per_step": ms_graph, "evals_per_s": w.B / (ms_graph * 1e-3),
                                  "note": "the same hfft_demag captured once and replayed (timed like the main region)"}
        if dedup == 4:
            line["roofline"]["kernel"] = "coupling_zfft_kernel (S3, z-convolution by FFT, PAPER.md:182 Eq.25)"
        if dedup in (2, 3):
            # deduplicated bank held in shared memory: the coupling is bound by the FP32/FP64 FMA pipe, not by HBM
            # (18 nz^2 n_k B real FMAs; peak = SMs x 128 (fp32) or 64 (fp64) FMA lanes x 2 x clock)
            flops = 2.0 * 18 * w.nz * w.nz * (2 * w.ny * (w.nx + 1)) * w.B
            lanes = 128 if w.precision == "f32" else 64
            alu_peak = 148 * lanes * 2 * clocks["sm_max_mhz"] * 1e6 / 1e12
            tf = flops / (coup_ms * 1e-3) / 1e12 if coup_ms > 0 else None
            line["roofline"] = {"bound": "alu", "kernel": "coupling_class_kernel (S3, deduplicated bank)",
                                "achieved": tf, "peak": alu_peak,
                                "peak_source": "derived: 148 SMs x %d FMA lanes x 2 flop x sm_max_mhz (DESIGN.md)" % lanes,
                                "unit": "TFLOP/s", "frac": tf / alu_peak if tf else None,
                                "algorithmic_flops_per_launch": flops, "avg_launch_ms": coup_ms,
                                "hbm_gbs": achieved, "traffic": None}
        line["config"]["bank"] = {"dedup": dedup, "ky_mirror": mirror, "reciprocity": int(plan.info.mirror) == 2, "slots_per_k": slots,
                                  "bytes": int(plan.info.bank_bytes)}
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(w)
        print(json.dumps(line))
    plan.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
