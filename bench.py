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
    ap.add_argument("--fusion", type=int, default=None, help="hfft_plan_set_fusion mode (default: the library's, 1)")
    ap.add_argument("--update-dz", action="store_true",
                    help="time one thickness update (hfft_update_dz / hfft_update_dz_static) against the full tensor build")
    ap.add_argument("--all-configs", action="store_true",
                    help="run every config (1, 2, 2f64, 3, 4, 4eq, 5) in a process of its own and write the bench lines, "
                         "with their clocks, as a markdown table + JSON lines to --out")
    ap.add_argument("--out", default=os.path.join("gpurun_out", "bench_all.md"), help="file --all-configs writes")
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


def algorithmic_bytes(w, n_slots=None, mirror=False, recip=False, fused=False):
    """what the method must move per hfft_demag call with the symmetries the storage
    uses.  n_slots: bank slots per wavevector (nz^2 pairs, or the tensor classes of a deduplicated bank);
    mirror: ky-mirror storage, one bank entry per (kx, ky <= ny); recip: reciprocity, one block per unordered
    layer pair, nz (nz + 1) / 2 (the padding of the symv layout is NOT counted: it is overhead, not algorithm)."""
    s = 4 if w.precision == "f32" else 8
    n_k = 2 * w.ny * (w.nx + 1)
    planes = 3 * w.nz * w.B
    if recip:
        n_slots = w.nz * (w.nz + 1) // 2
    bank = 6 * (n_slots if n_slots else w.nz * w.nz) * ((w.nx + 1) * (w.ny + 1) if mirror else n_k) * s
    spec = planes * n_k * 2 * s            # M^ (= H^)
    xhat = planes * w.ny * (w.nx + 1) * 2 * s
    field = planes * w.ny * w.nx * s
    coupling = bank + 2 * spec
    whole = 2 * field + 4 * xhat + 4 * spec + bank
    if fused:                              # S2 + S3 + S4 in one kernel: X^ in, X^ out, the spectra stay in shared memory
        coupling = bank + 2 * xhat
        whole = 2 * field + 4 * xhat + bank
    return {"bank": bank, "coupling": coupling, "whole": whole}


class ClockSampler:
    """SM clock and throttle reasons of one GPU while the timed regions run.  Reads NVML in this process (a thread
    that samples every 10 ms; the first sample is taken synchronously in start(), so that even a timed region of a
    few milliseconds has its record); where NVML cannot be loaded it falls back to `nvidia-smi -lms 50`, whose output
    is block-buffered and can therefore miss short runs -- `source` and `why` say which path ran and why a record is
    empty."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
    # NVML clocks-event (throttle) reason bits
    BITS = {"sw_power_cap": 0x4, "hw_slowdown": 0x8, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40}

    def __init__(self, index, pci_bus_id=None):
        self.index = index
        self.pci_bus_id = pci_bus_id
        self.proc = None
        self.out = None
        self.nvml = None
        self.handle = None
        self.thread = None
        self.stop_flag = False
        self.sm, self.mx, self.reasons = [], [], set()
        self.why = None

    def _sample(self):
        n = self.nvml
        self.sm.append(float(n.nvmlDeviceGetClockInfo(self.handle, n.NVML_CLOCK_SM)))
        self.mx.append(float(n.nvmlDeviceGetMaxClockInfo(self.handle, n.NVML_CLOCK_SM)))
        get = getattr(n, "nvmlDeviceGetCurrentClocksEventReasons", None) or n.nvmlDeviceGetCurrentClocksThrottleReasons
        mask = int(get(self.handle))
        for name, bit in self.BITS.items():
            if mask & bit:
                self.reasons.add(name)

    def _loop(self):
        while not self.stop_flag:
            try:
                self._sample()
            except Exception as exc:  # keep what was sampled so far
                self.why = "NVML sampling stopped: %r" % (exc,)
                return
            time.sleep(0.01)

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nvml = pynvml
            try:
                self.handle = pynvml.nvmlDeviceGetHandleByPciBusId(self.pci_bus_id.encode() if self.pci_bus_id else b"")
            except Exception:
                self.handle = pynvml.nvmlDeviceGetHandleByIndex(self.index)
            self._sample()
            import threading
            self.thread = threading.Thread(target=self._loop, daemon=True)
            self.thread.start()
            return
        except Exception as exc:
            self.nvml = None
            self.why = "NVML unavailable (%r); fell back to nvidia-smi -lms 50" % (exc,)
        self.out = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.FIELDS,
                 "--format=csv,noheader,nounits", "-lms", "50"], stdout=self.out, stderr=subprocess.DEVNULL)
        except OSError as exc:
            self.proc = None
            self.why += "; nvidia-smi could not be started (%r)" % (exc,)

    def stop(self):
        res = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0, "source": None, "why": None}
        if self.nvml is not None:
            try:
                self._sample()                               # one more under the last timed region's tail
            except Exception:
                pass
            self.stop_flag = True
            if self.thread is not None:
                self.thread.join(timeout=2)
            res["source"] = "nvml (in-process, 10 ms)"
            sm, mx, reasons = self.sm, self.mx, self.reasons
        else:
            res["source"] = "nvidia-smi -lms 50"
            sm, mx, reasons = [], [], set()
            if self.proc is not None:
                self.proc.terminate()
                try:
                    self.proc.wait(timeout=5)
                except subprocess.TimeoutExpired:
                    self.proc.kill()
                self.out.flush()
                self.out.seek(0)
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
        res["why"] = self.why if sm else (self.why or "no sample arrived before the timed regions ended")
        return res


def _full_eval_on_host(w):
    """Whether the CPU oracle times a whole evaluation (C1-C3) or a bounded sample of target layers (C4, C5)."""
    return w.nx * w.ny * w.nz * w.B <= 256 * 256 * 16


def _host_threads_for(w, cores):
    """Threads of the all-cores run: bounded by the host memory one hybrid_layers call needs (padded tensor row, its
    spectrum, the spectrum of M: ~ (6 nz (8 + 16) + 3 nz 16) * 4 nx ny bytes)."""
    per = (6 * w.nz * 24 + 3 * w.nz * 16) * 4 * w.nx * w.ny * 1.3
    try:
        import psutil
        avail = psutil.virtual_memory().available
    except Exception:
        avail = 32 << 30
    return max(1, min(cores, w.nz, int(0.5 * avail / per)))


def oracle_timing(w, budget_s=20.0, steps=None, warmup=0):
    """The oracle's hybrid tier (T1, Eq.24; oracle.hybrid_layers with numpy's FFT, fp64), AS IT STANDS,
    on the host cores, one state -- like for like with the GPU arm ("tensor bank pre-built, setup
    excluded"): the binary128 tensor rows AND their in-plane spectra (oracle.tensor_spectrum, what hfft_build_tensor
    does on the GPU) are built before the timing and handed over through `nhat=`; inside the timing are the forward
    FFT of M (once per call) and, per target layer, the z-sum of Eq.24 and the inverse FFT.  The figure that also pays
    the tensor planes' 2-D FFT on every evaluation (hybrid_layers called with `rows=` only, as rounds 1-2 timed it)
    is reported beside it as `with_tensor_fft`.  numpy's FFT and einsum run on ONE thread (`cores_timed`); the
    all-cores figure runs the same calls, one target-layer chunk per thread.

    C1-C3: whole evaluations (every target layer).  C4 / C5: a bounded sample, EXTRAPOLATED -- calls with target layers
    [0] and [0, 1] give the per-layer and the once-per-evaluation time; evaluation = once + nz * per_layer (the tensor
    row of layer 0 stands in for both sampled layers: the timing does not depend on the values)."""
    import oracle as O
    from concurrent.futures import ThreadPoolExecutor
    m = w.m_rounded([0])[0]
    cores = os.cpu_count() or 1
    full = _full_eval_on_host(w)
    t0 = time.perf_counter()
    if full:
        rows = {i: O.tensor_row(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, i) for i in range(w.nz)}
    else:
        row0 = O.tensor_row(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, 0)
        rows = {i: row0 for i in range(w.nz)}
    setup = time.perf_counter() - t0
    t0 = time.perf_counter()
    if full:
        nhat = {i: O.tensor_spectrum(rows[i], w.nx, w.ny, "fft") for i in range(w.nz)}
    else:
        nhat0 = O.tensor_spectrum(row0, w.nx, w.ny, "fft")
        nhat = {i: nhat0 for i in range(w.nz)}
    setup_fft = time.perf_counter() - t0

    def call(layers, prebuilt=True):
        kw = {"nhat": nhat} if prebuilt else {"rows": rows}
        t = time.perf_counter()
        O.hybrid_layers(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, m, w.Ms, list(layers), dft="fft", **kw)
        return time.perf_counter() - t

    def repeat(fn, n_fixed):
        for _ in range(warmup):
            fn()
        ts = []
        if n_fixed is not None:
            for _ in range(n_fixed):
                ts.append(fn())
            return ts
        while len(ts) < 3 or (sum(ts) < budget_s and len(ts) < 1000):
            ts.append(fn())
            if sum(ts) > 3 * budget_s:
                break
        return ts

    nthr = _host_threads_for(w, cores)
    if full:
        ts = repeat(lambda: call(range(w.nz)), steps)
        t_eval = float(np.mean(ts))
        t_eval_fft = float(np.mean([call(range(w.nz), False) for _ in range(max(1, min(3, len(ts))))]))
        chunks = [list(range(w.nz))[t::nthr] for t in range(nthr)]

        def par():
            t = time.perf_counter()
            with ThreadPoolExecutor(nthr) as ex:
                list(ex.map(call, chunks))
            return time.perf_counter() - t
        tp = [par() for _ in range(max(1, min(3, len(ts))))]
        t_eval_all = float(np.mean(tp))
        sample = ("whole evaluations (all %d target layers) of one state: mean of %d runs of %.4f s"
                  % (w.nz, len(ts), t_eval))
        formula = None
        runs, s_timed = len(ts), float(np.sum(ts))
    else:
        n = steps if steps is not None else 3
        a1, a2 = repeat(lambda: call([0]), n), repeat(lambda: call([0, 1]), n)
        t1, t2 = float(np.median(a1)), float(np.median(a2))
        per = max(t2 - t1, 1e-9)
        once = max(t1 - per, 0.0)
        t_eval = once + w.nz * per
        f1, f2 = call([0], False), call([0, 1], False)
        per_f = max(f2 - f1, 1e-9)
        t_eval_fft = max(f1 - per_f, 0.0) + w.nz * per_f

        def par():
            t = time.perf_counter()
            with ThreadPoolExecutor(nthr) as ex:
                list(ex.map(call, [[0]] * nthr))
            return time.perf_counter() - t
        t_par = par()
        # nthr layers (each with its own forward FFT of M, as the call stands) in t_par seconds
        t_eval_all = t_par * w.nz / nthr
        sample = ("target layers [0] (%.3f s) and [0, 1] (%.3f s) of %d, one state, median of %d calls each"
                  % (t1, t2, w.nz, n))
        formula = ("s_per_eval = once + nz * per_layer, per_layer = t[0,1] - t[0] = %.4f s, once = t[0] - per_layer = %.4f s, "
                   "nz = %d: the %.1f s evaluation was not run" % (per, once, w.nz, t_eval))
        runs, s_timed = 2 * n, float(np.sum(a1) + np.sum(a2))
    return {"value": 1.0 / t_eval, "unit": UNIT, "cores": 1, "cores_timed": 1, "cores_available": cores,
            "kind": "oracle", "s_per_eval": t_eval, "extrapolated": not full, "extrapolation": formula,
            "timed_work": "bank_prebuilt: forward FFT of M, z-sum of Eq.24, inverse FFT (tensor rows and their spectra built "
                          "beforehand, as hfft_build_tensor does for the GPU arm)",
            "with_tensor_fft": {"value": 1.0 / t_eval_fft, "unit": UNIT, "s_per_eval": t_eval_fft, "extrapolated": not full,
                                "what": "hybrid_layers given the tensor rows only: it also transforms the 6 nz padded "
                                        "tensor planes of every target layer on every evaluation (the figure rounds 1-2 "
                                        "printed as `value`)"},
            "sample": sample + "; oracle.hybrid_layers (numpy FFT, fp64) as it stands; untimed setup: tensor rows (binary128, "
                      "%.1f s on %d OpenMP threads) and their in-plane spectra (oracle.tensor_spectrum, %.1f s)"
                      % (setup, O.threads(), setup_fft),
            "all_cores": {"value": 1.0 / t_eval_all, "unit": UNIT, "cores": nthr, "s_per_eval": t_eval_all,
                          "extrapolated": not full,
                          "how": "the same calls, one chunk of target layers per thread (numpy releases the GIL)"},
            "oracle_tensor_rows_s": setup, "oracle_tensor_spectra_s": setup_fft, "_runs": runs, "_s_timed": s_timed}


def cpu_baseline(w, budget_s=20.0):
    r = oracle_timing(w, budget_s)
    r.pop("_runs"); r.pop("_s_timed")
    return r


def traffic_entry(workload_name, storage, root=None):
    """(DRAM bytes per launch of the coupling kernel, where the figure comes from) out of profiles/traffic.json, or
    (None, why).  An entry counts only while the source files that define its kernel still hash to what they did at
    the capture: a changed kernel prints traffic = null (with the reason) instead of a stale number."""
    import hashlib
    root = root or ROOT
    tp = os.path.join(root, "profiles", "traffic.json")
    if not os.path.exists(tp):
        return None, "no profiles/traffic.json"
    with open(tp) as fh:
        ent = json.load(fh).get(workload_name, {}).get(storage)
    if not isinstance(ent, dict):
        return None, "no ncu --set full capture of this workload with the %s storage" % storage
    files = ent.get("source_files") or []
    hsh = hashlib.sha256()
    try:
        for f in files:
            with open(os.path.join(root, f), "rb") as fh:
                hsh.update(fh.read())
    except OSError as exc:
        return None, "stale: %s (%r)" % (ent.get("source"), exc)
    if not files or hsh.hexdigest()[:16] != ent.get("source_sha16"):
        return None, ("stale: %s changed since the capture of %s at commit %s (%s); capture again"
                      % (", ".join(files) or "kernel sources", ent.get("kernel"), ent.get("git"), ent.get("source")))
    return ent.get("coupling_dram_bytes_per_launch"), "%s; kernel %s, commit %s" % (ent.get("source"), ent.get("kernel"), ent.get("git"))


def l2_mode(w):
    """How the timed steps keep L2 from serving the inputs -- a function of the workload alone, so that both arms
    print the same `config`.  Workloads whose smallest storage (reciprocity + ky-mirror bank) exceeds twice the L2
    stream it every step; the small ones get a 256 MiB memset before every timed step."""
    small = algorithmic_bytes(w, None, True, True)["whole"] < (256 << 20)
    if small:
        return "L2 flushed (256 MiB memset) before every timed step"
    # the bank is larger than L2 in every such workload; the spectra M^ / H^ (one complex plane set) may or may not be
    elem = 4 if w.precision == "f32" else 8
    spectra = 3 * w.nz * w.B * 2 * w.ny * (w.nx + 1) * 2 * elem
    if spectra < (126 << 20):
        return ("inputs larger than L2 (126 MB): the tensor bank is streamed from HBM every step; the spectra (%d MB) fit L2 "
                "and are served from it between the stages, so the coupling's achieved GB/s on algorithmic bytes is L2-assisted"
                % (spectra // 1000000))
    return ("inputs larger than L2 (126 MB): the tensor bank and the spectra (%d MB) are streamed from HBM every step"
            % (spectra // 1000000))


def run_reference(args, w):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    full = _full_eval_on_host(w)
    # C1-C3: every step is a whole evaluation.  C4 / C5: each step is the bounded sample (target layers [0] and [0, 1]);
    # the number of sampled calls is cut so that the run stays within a few minutes whatever K and W are.
    steps, warmup = args.steps, args.warmup
    if not full:
        steps, warmup = max(1, min(args.steps, 3)), min(args.warmup, 1)
    elif w.nx * w.ny * w.nz > 64 * 64 * 6:
        steps, warmup = max(1, min(args.steps, 5)), min(args.warmup, 1)
    r = oracle_timing(w, steps=steps, warmup=warmup)
    runs, s_timed = r.pop("_runs"), r.pop("_s_timed")
    value = r["value"]
    # One line, one meaning per key: `steps` / `warmup` are what RAN (the request is echoed beside them), `value` and
    # `ms_per_step` describe one whole evaluation (value = 1000 / ms_per_step); where that evaluation is extrapolated
    # from a bounded sample (C4, C5) the line says so and `timed_s` is the wall time of the calls actually timed.
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": steps if full else runs, "warmup": warmup, "ms_per_step": 1e3 * r["s_per_eval"], "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(w),
        "cpu_baseline": r,
        "extrapolated": r["extrapolated"], "extrapolation": r["extrapolation"],
        "step_is": "one whole evaluation" if full else "one sampled oracle call (target layers [0] or [0, 1]); ms_per_step is "
                   "the extrapolated whole evaluation, not the duration of such a call",
        "steps_requested": args.steps, "warmup_requested": args.warmup, "oracle_calls_timed": runs, "timed_s": s_timed,
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def measure_pcie(torch, m_host, m, h, h_host, nbytes):
    """What the PCIe link gives for the end-to-end step's own transfers, without any kernel: the pinned host -> device
    copy of m and the device -> pinned host copy of h, the sizes and buffers of the e2e region, issued back to back on
    two streams so that both directions run at once (as they do in the hfft_demag_host_async pipeline).  Returns GB/s
    per direction with both directions busy, and each direction alone."""
    cur = torch.cuda.current_stream()
    s_in, s_out = torch.cuda.Stream(), torch.cuda.Stream()
    iters = int(max(5, min(200, (1 << 30) // max(nbytes, 1))))

    def run(do_in, do_out):
        torch.cuda.synchronize()
        e0 = torch.cuda.Event(enable_timing=True)
        e1 = torch.cuda.Event(enable_timing=True)
        e0.record(cur)
        ends = []
        for on, st, fn in ((do_in, s_in, lambda: m.copy_(m_host, non_blocking=True)),
                           (do_out, s_out, lambda: h_host.copy_(h, non_blocking=True))):
            if not on:
                continue
            st.wait_event(e0)
            with torch.cuda.stream(st):
                for _ in range(iters):
                    fn()
                ev = torch.cuda.Event()
                ev.record(st)
                ends.append(ev)
        for ev in ends:
            cur.wait_event(ev)
        e1.record(cur)
        torch.cuda.synchronize()
        return iters * nbytes / (e0.elapsed_time(e1) * 1e-3) / 1e9

    run(True, True)                                      # warm-up
    return {"both_directions_gbs_per_direction": run(True, True), "h2d_alone_gbs": run(True, False),
            "d2h_alone_gbs": run(False, True), "bytes_per_copy": nbytes, "copies_per_direction": iters,
            "how": "pinned cudaMemcpyAsync of the step's own buffers on two streams, no kernels, CUDA events"}


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
        for name, dz, kw in [("hybrid, automatic (reciprocity / ky-mirror bank)", dz_var, dict()),
                             ("hybrid, ky-mirror bank (recip 0)", dz_var, dict(dedup=0, recip=0)),
                             ("hybrid, plain bank (mirror 0)", dz_var, dict(dedup=0, mirror=0)),
                             ("equidistant, automatic", np.full(nz, 1.0), dict()),
                             ("equidistant, Toeplitz classes (dedup 2)", np.full(nz, 1.0), dict(dedup=2)),
                             ("equidistant, z-FFT of Eq.25 (dedup 3)", np.full(nz, 1.0), dict(dedup=3))]:
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


def update_dz_timing():
    """SURVEY 8f-1 / PAPER.md:205-211 (the tensor is rebuilt at every Newton step of the thickness optimisation): wall
    time of one thickness update -- hfft_update_dz (scratch from cudaMalloc / cudaFree per call) and, where the plan fits
    the fixed 32 MiB scratch, hfft_update_dz_static (no allocation) -- against the full hfft_build_tensor, per bank
    storage.  Both update calls synchronise their stream, so host wall time is the time of the call.  Median of 5."""
    import torch
    from paper_1910_07054_b200 import binding as hb
    saf = W.small(64, 64, 5, precision="f64", seed=1, dz=np.array([5.0, 1.0, 5.0, 1.0, 3.0]))
    cases = [("SAF disc grid 64x64x5 f64 (PAPER.md:205-211)", saf, 2, dict()),
             ("C2 64x64x6 f32", W.config(2), 3, dict()),
             ("C3 256x256x16 f32, reciprocity bank (default)", W.config(3), 8, dict()),
             ("C3 256x256x16 f32, ky-mirror bank (recip 0)", W.config(3), 8, dict(recip=0)),
             ("C4 256x256x64 f32, reciprocity bank (default), middle layer", W.config(4), 32, dict()),
             ("C4 256x256x64 f32, reciprocity bank (default), bottom layer", W.config(4), 0, dict()),
             ("C4 256x256x64 f32, ky-mirror bank (recip 0), middle layer", W.config(4), 32, dict(recip=0))]
    for name, w, k, kw in cases:
        plan = hb.Plan(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, w.precision, dedup=0, **kw)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        plan.build_tensor()
        torch.cuda.synchronize()
        build_s = time.perf_counter() - t0
        info = hb.plan_info(plan.handle)

        def med(fn):
            ts = []
            for r in range(6):
                dz_new = w.dz[k] * (1.1 if r % 2 == 0 else 1.0)
                torch.cuda.synchronize()
                t = time.perf_counter()
                fn(k, dz_new)
                ts.append(time.perf_counter() - t)
            return float(np.median(ts[1:]))
        upd = med(plan.update_dz)
        fits = info.setup_scratch_bytes <= hb.STATIC_SCRATCH_BYTES
        sta = med(plan.update_dz_static) if fits else None
        changed = sum(1 for i in range(w.nz) for j in range(i, w.nz) if i <= k <= j)
        print(json.dumps({"case": name, "layer": k, "mirror": info.mirror, "bank_GB": info.bank_bytes / 1e9,
                          "setup_scratch_MB": info.setup_scratch_bytes / 1e6, "build_tensor_s": build_s,
                          "update_dz_s": upd, "update_dz_static_s": sta,
                          "unordered_pairs_changed": changed, "unordered_pairs": w.nz * (w.nz + 1) // 2}), flush=True)
        plan.close()
        del plan
        torch.cuda.empty_cache()


def workload_config(w):
    l2 = l2_mode(w)
    return {"workload": w.name, "nx": w.nx, "ny": w.ny, "nz": w.nz, "batch": w.B, "precision": w.precision,
            "dz_nm": [round(float(v), 6) for v in w.dz[:8]] + (["..."] if w.nz > 8 else []),
            "m": w.m_kind, "seed": w.seed, "l2": l2, "parallelism": "replicas only (no sharding, no collective)"}


ALL_CONFIGS = ["1", "2", "2f64", "3", "4", "4eq", "5"]


def all_configs(args):
    """north_star: "evaluations/sec and achieved HBM GB/s as a fraction of peak for each config".  Every config runs in
    a bench.py process of its own (same flags); the JSON lines, each with its `clocks`, go to --out as a table."""
    lines = []
    for c in ALL_CONFIGS:
        cmd = [sys.executable, os.path.abspath(__file__), "--config", c, "--steps", str(args.steps), "--warmup",
               str(args.warmup), "--no-cpu-baseline"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        out = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
        if r.returncode != 0 or not out:
            raise SystemExit("bench.py --config %s failed:\n%s" % (c, r.stderr[-4000:]))
        lines.append(json.loads(out[-1]))
        print(out[-1], flush=True)
    os.makedirs(os.path.dirname(os.path.abspath(args.out)) or ".", exist_ok=True)
    with open(args.out, "w") as fh:
        fh.write("# bench.py --all-configs --steps %d --warmup %d\n\n" % (args.steps, args.warmup))
        fh.write("Command: `python bench.py --all-configs --steps %d --warmup %d --out %s` (one B200; every config in a "
                 "process of its own; clocks sampled through NVML from the warm-up on, bench.ClockSampler).\n\n" % (args.steps, args.warmup, args.out))
        fh.write("| config | ms / call | evals/s | e2e evals/s | S1 / S2 / S3 / S4 / S5 ms | S3 roofline (bound, achieved / peak = frac) "
                 "| whole / roofline | bank | SM MHz (median / max) | throttle reasons |\n|---|---:|---:|---:|---|---|---:|---|---|---|\n")
        for d in lines:
            r, st, ck, bk = d["roofline"], d["stages_ms"], d["clocks"], d["bank"]
            kind = ("fused S2+S3+S4, plain" if bk.get("fused_s2s3s4") else "z-FFT" if bk["dedup"] == 4 else "classes" if bk["dedup"] else "symv" if bk["symv_layout"] else
                    "recip" if bk["reciprocity"] else "mirror" if bk["ky_mirror"] else "plain")
            fh.write("| %s | %.4f | %.1f | %.1f | %s | %s %.4g / %.4g %s = %.2f | %.2f | %s, %.3f GB | %s / %s | %s |\n" % (
                d["config"]["workload"], d["ms_per_step"], d["value"], d["e2e"]["value"],
                " / ".join("%.4f" % st[n] for n in ("fftx_fwd", "ffty_fwd", "coupling", "iffty", "ifftx")),
                r["bound"], r["achieved"], r["peak"], r["unit"], r["frac"], d["whole_eval"]["ratio_to_roofline"],
                kind, bk["bytes"] / 1e9, ck["sm_mhz"], ck["sm_max_mhz"], ", ".join(ck["reasons"]) or "none"))
        fh.write("\nJSON lines:\n\n```\n" + "\n".join(json.dumps(d) for d in lines) + "\n```\n")


def main():
    args = parse_args()
    if args.sweep_nz:
        sweep_nz()
        return
    if args.update_dz:
        update_dz_timing()
        return
    if args.all_configs:
        all_configs(args)
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
    steps, warmup = max(1, args.steps), max(0, args.warmup)    # W >= 3 is the caller's contract: not clamped

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    plan = hb.Plan(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, w.precision, batch=w.B, dedup=args.dedup, mirror=args.mirror,
                   recip=args.recip, fusion=args.fusion)
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
    recip = int(plan.info.mirror) >= 2                     # 2: p <= q storage read twice, 3: symv layout read once
    symv = int(plan.info.mirror) == 3
    slots = int(plan.info.bank_bytes // (6 * (plan.info.n_k_padded // (2 if mirror else 1)) * (4 if w.precision == "f32" else 8)))
    fused = bool(plan.info.fused)
    ab = algorithmic_bytes(w, slots if dedup else None, mirror, recip, fused)
    # inputs larger than L2?  otherwise flush L2 between steps (l2_mode: the same rule, printed in `config`)
    flush = None
    if l2_mode(w).startswith("L2 flushed") or ab["whole"] < (256 << 20):
        flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

    def step():
        if flush is not None:
            flush.zero_()
        plan.demag(m, Ms, h)

    # clocks are sampled from the warm-up on (under load), through every timed region
    props = torch.cuda.get_device_properties(local_rank)
    try:
        bus = "%08x:%02x:%02x.0" % (props.pci_domain_id, props.pci_bus_id, props.pci_device_id)
    except AttributeError:
        bus = None
    sampler = ClockSampler(local_rank, bus)
    if warmup > 0:                                       # the first sample is taken with the GPU already at work
        step()
        torch.cuda.synchronize()
    sampler.start()
    for _ in range(max(0, warmup - 1)):
        step()
    barrier()
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
    pcie = measure_pcie(torch, m_host, m, h, h_host, nbytes)     # after the timed regions; h_host keeps the same field

    assert bool(torch.isfinite(h).all()) and bool(torch.isfinite(h_host).all())
    ms_total, ms_e2e, ms_e2e_serial = max_over_ranks([ms_total, ms_e2e, ms_e2e_serial], device="cuda")

    if rank == 0:
        peak, peak_src = measured_peaks()
        ms_step = ms_total / steps
        value = whole_job_value(world, w.B, steps, ms_total)
        coup_ms = float(stage_ms[hb.STAGE_NAMES.index("coupling")])
        achieved = ab["coupling"] / (coup_ms * 1e-3) / 1e9 if coup_ms > 0 else None
        # DRAM bytes per launch of the coupling kernel from the committed ncu --set full capture of this workload and
        # storage (not re-measured here: ncu cannot run inside a timed bench); null once the kernel's sources changed
        storage = ("zfft" if dedup == 4 else "class" if dedup else "batched" if w.B > 1 else
                   "symv" if symv else "recip" if recip else "mirror" if mirror else "plain")
        traffic, traffic_src = traffic_entry(w.name, storage)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warmup,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": w.precision, "data": "synthetic",
            "config": workload_config(w),
            "clocks": {"sm_mhz": clocks["sm_mhz"], "sm_max_mhz": clocks["sm_max_mhz"], "reasons": clocks["reasons"],
                       "samples": clocks["samples"], "source": clocks["source"], "why": clocks["why"]},
            "e2e": {"value": whole_job_value(world, w.B, e2e_steps, ms_e2e), "unit": UNIT,
                    "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes, "steps": e2e_steps,
                    "api": "hfft_demag_host_async + hfft_host_join (per step: pinned host m -> device, 5 kernels, "
                           "device h -> pinned host; copies of neighbouring steps overlap the kernels)",
                    "serialised_hfft_demag_host": whole_job_value(world, w.B, e2e_steps, ms_e2e_serial),
                    # "PCIe-bound" as a number: bytes per second and direction of the e2e region over what the link
                    # gives for the same copies with no kernels in between (rank 0's link)
                    "gbs_per_direction": nbytes * e2e_steps / (ms_e2e * 1e-3) / 1e9,
                    "pcie_gbs_measured": pcie["both_directions_gbs_per_direction"],
                    "frac_of_pcie": nbytes * e2e_steps / (ms_e2e * 1e-3) / 1e9 / pcie["both_directions_gbs_per_direction"],
                    "pcie": pcie},
            "gpu_launches": plan.info.launches_per_demag * steps,
            "roofline": {"bound": "hbm", "kernel": "coupling_symv_kernel (S3, reciprocity + ky-mirror bank read once)" if symv
                         else "coupling_kernel (S3)", "achieved": achieved, "peak": peak,
                         "peak_source": peak_src, "unit": "GB/s", "frac": achieved / peak if achieved else None,
                         "frac_of_nominal_8TBs": achieved / 8000.0 if achieved else None,
                         "algorithmic_bytes_per_launch": ab["coupling"], "avg_launch_ms": coup_ms,
                         "stored_bank_bytes": int(plan.info.bank_bytes),
                         "traffic": traffic, "traffic_source": traffic_src,
                         # the same launch time against the DRAM bytes ncu counted (cold L2) instead of the bytes the
                         # method needs: where they differ, L2 serves part of the stream in a running evaluation
                         "achieved_dram": traffic / (coup_ms * 1e-3) / 1e9 if traffic and coup_ms > 0 else None,
                         "frac_dram": traffic / (coup_ms * 1e-3) / 1e9 / peak if traffic and coup_ms > 0 else None,
                         "achieved_is": "algorithmic bytes / launch time" + ("" if ab["whole"] >= (2 << 30) else
                                        " (L2-assisted: bank + spectra are within a few L2 sizes, part of M^ / H^ never leaves L2)")},
            "stages_ms": {n: float(v) for n, v in zip(hb.STAGE_NAMES, stage_ms)},
            "whole_eval": {"algorithmic_bytes": ab["whole"], "roofline_ms_at_peak": ab["whole"] / peak / 1e6,
                           "ms_per_step": ms_step, "ratio_to_roofline": ms_step / (ab["whole"] / peak / 1e6)},
            "setup_s": setup_s,
        }
        if fused:
            line["roofline"]["kernel"] = ("fused_ycy_kernel (S2 + S3 + S4 in one launch: y transforms and coupling of one kx "
                                          "column of all planes, spectra in shared memory; stages_ms charges it to `coupling`)")
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
        line["bank"] = {"dedup": dedup, "ky_mirror": mirror, "reciprocity": recip, "symv_layout": symv, "fused_s2s3s4": fused,
                        "slots_per_k": slots, "bytes": int(plan.info.bank_bytes)}
        line["l2_flush_between_steps"] = flush is not None
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(w)
        print(json.dumps(line))
    plan.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
