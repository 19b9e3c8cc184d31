#!/usr/bin/env python
"""bench.py -- Jacobian evaluations per second of the batched analytical kinetics Jacobian on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]
                    [--also 2,3] [--sweep short|full|off] [--no-cpu-baseline] [--no-e2e] [--peaks]
    python bench.py --ncu-target CFG:KERNEL:N[:SHAPE]      # the short command the ncu captures of profiles/ wrap
    python bench.py --ncu-import REPORT --ncu-label WORKLOAD:KERNEL:N    # one row of profiles/r3_ncu_counters.csv

A "step" is one pass of the whole hot path (thermo -> rates -> source term -> Jacobian -> store;
SURVEY.md section 8(a) rows S0-S10, one kernel launch) over one batch of seeded synthetic states.
At N = 1 the workload is BASELINE.json configs[1] (53 species, 325 reactions, 100,000 states).
Rank 0 prints ONE JSON line.  Under torchrun (N > 1) every rank evaluates the same batch on its own
GPU (states are independent: no data-path collective, "scaling": "weak").

`--impl reference` times the CPU oracle (oracle/) on the host cores instead -- the only other place
this file executes anything under oracle/ besides the cpu_baseline leg.
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

METRIC = "jacobian_evals_per_sec"
UNIT = "states/s"
FALLBACK_HBM_GBS = 6650.0          # /opt/skills/guides/B200_PROFILING.md fallback
# oracle sample sizes per config (about 10-30 s of CPU work on 8-32 cores)
CPU_SAMPLE = {0: 1024, 1: 8192, 2: 2048, 3: 256}
# Counters of the committed `ncu` captures (profiles/r2_ncu_counters.csv, written from the reports the .md
# beside it names): DRAM bytes and fp64 flops per state of each kernel.  They describe the kernels whose
# source hash they carry; with different sources the bench reports null instead of a stale number.
NCU_COUNTERS = [os.path.join(ROOT, "profiles", f) for f in ("r3_ncu_counters.csv", "r2_ncu_counters.csv")]
KERNEL_SOURCES = ("kernels.cu", "mech_pack.cu", "device_mech.h", "api.cu", "dispatch.cu")
FP64_PEAK_TFLOPS = 33.74        # measured: bench.py --peaks, profiles/r1_machine_peaks.md (8 FMA chains per thread)


def kernel_source_sha16() -> str:
    import hashlib
    h = hashlib.sha256()
    for f in KERNEL_SOURCES:
        with open(os.path.join(ROOT, "paper_1605_03262_b200", "csrc", f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def ncu_counters():
    """({workload: {kernel: {dram_bytes_per_state, fp64_flop_per_state}}}, source) of the committed captures
    that belong to these kernel sources."""
    import csv
    out, src = {}, None
    try:
        sha = kernel_source_sha16()
        for path in NCU_COUNTERS:
            if not os.path.exists(path) or out:
                continue
            rel = os.path.relpath(path, ROOT)
            for row in csv.DictReader(open(path)):
                if row["kernel_source_sha16"] != sha:
                    src = src or "%s describes other kernel sources (%s)" % (rel, row["kernel_source_sha16"])
                    continue
                out.setdefault(row["workload"], {})[row["kernel"]] = {
                    "dram_bytes_per_state": float(row["dram_bytes_per_state"]),
                    "fp64_flop_per_state": float(row["fp64_flop_per_state"]), "n_states": int(row["n_states"]),
                    "lsu_wavefronts_per_state": float(row["lsu_wavefronts_per_state"])}
                src = "%s (ncu --set full captures of kernel sources %s, %s)" % (rel, sha, rel[:-4] + ".md")
    except Exception:
        return {}, None
    return out, src


_FP64_PEAK = {"tflops": FP64_PEAK_TFLOPS,
              "source": "round-1 measurement (bench.py --peaks, profiles/r1_machine_peaks.md), not re-measured in this run"}


def fp64_peak():
    return _FP64_PEAK["tflops"]


def measure_fp64_peak(torch):
    """The fp64 FMA probe of `--peaks` (8 independent chains per thread, 3 warm-up + 10 timed launches, best),
    run inside this bench run so that the fp64 roofline entries divide by a peak of the same box and clocks."""
    try:
        from paper_1605_03262_b200 import binding
        sms = torch.cuda.get_device_properties(torch.cuda.current_device()).multi_processor_count
        out = torch.empty(sms * 4096, dtype=torch.float64, device="cuda")
        sp = torch.cuda.current_stream().cuda_stream
        flops = [0]
        for _ in range(3):
            flops[0] = binding.peak_dfma(out, 1 << 16, sp)
        torch.cuda.synchronize()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(11)]
        ev[0].record()
        for i in range(10):
            binding.peak_dfma(out, 1 << 16, sp)
            ev[i + 1].record()
        torch.cuda.synchronize()
        best = min(ev[i].elapsed_time(ev[i + 1]) for i in range(10))
        _FP64_PEAK["tflops"] = flops[0] / best / 1e9
        _FP64_PEAK["source"] = "fp64 FMA probe of the tools library, measured in this run (best of 10 launches)"
    except Exception as e:      # the probe is a helper, not the product: fall back to the recorded figure
        _FP64_PEAK["source"] += " (probe failed: %s)" % type(e).__name__


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown",
                                "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def algorithmic_bytes(ns: int, n: int) -> int:
    """per state the method must read (Ns+2) and write (Ns+1)^2 doubles."""
    return n * ((ns + 2) + (ns + 1) * (ns + 1)) * 8


def cpu_model() -> str:
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


def time_oracle(cfg: int, n_sample: int, steps: int = 3, warmup: int = 1, single_thread: bool = False):
    """The oracle as it stands on the host cores: `warmup` untimed passes over 64 states, then `steps`
    timed passes over the first n_sample states of the workload (1 warm-up + 3
    repetitions); optionally also one pass on ONE thread over n_sample / cores states -- the paper's CPU
    numbers are single-thread."""
    import numpy as np  # noqa: F401
    from oracle.oracle import Oracle
    from paper_1605_03262_b200 import synth
    m = synth.make_mechanism(cfg)
    o = Oracle(m)
    n_sample = min(n_sample, synth.CONFIGS[cfg].n_states)
    T, P, Y = synth.config_states(cfg, n_sample)
    for _ in range(warmup):
        o.jacobian(T[:64], P[:64], Y[:64])
    per = []
    for _ in range(steps):
        t0 = time.perf_counter()
        o.jacobian(T, P, Y)
        per.append(time.perf_counter() - t0)
    dt = sum(per) / len(per)
    res = {"value": n_sample / dt, "unit": UNIT, "cores": o.threads, "kind": "oracle", "cpu": cpu_model(),
           "best_value": n_sample / min(per),
           "sample": "analytical Jacobian (oracle/oracle.c, Algorithm-1 order, OpenMP static over states) on "
                     "the first %d states of the workload, %d warm-up + %d timed pass(es), %.2f s per pass"
                     % (n_sample, warmup, steps, dt)}
    if single_thread:
        n1 = max(16, n_sample // max(o.threads, 1))
        o1 = Oracle(m, threads=1)
        o1.jacobian(T[:16], P[:16], Y[:16])
        t0 = time.perf_counter()
        o1.jacobian(T[:n1], P[:n1], Y[:n1])
        res["single_thread"] = {"value": n1 / (time.perf_counter() - t0), "unit": UNIT, "cores": 1,
                                "sample": "first %d states, one pass" % n1}
    return res, dt


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_1605_03262_b200 import synth
    cfg = args.config
    c = synth.CONFIGS[cfg]
    steps = max(1, args.steps)
    # bounded: the whole run stays within a few minutes
    n_sample = CPU_SAMPLE[cfg] if steps <= 2 else max(256, CPU_SAMPLE[cfg] // steps)
    base, dt = time_oracle(cfg, n_sample, steps=steps, warmup=min(args.warmup, 1))
    line = {"impl": "reference", "metric": METRIC, "value": base["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": c.name, "n_species": c.n_species, "n_reactions": c.n_reactions,
                       "n_states": c.n_states, "sampled_states_per_step": n_sample},
            "cpu_baseline": base,
            "e2e": {"value": base["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def time_gpu(pj, torch, dT, dP, dY, out, steps, warmup, fn=None):
    """CUDA events on torch's current stream (the stream the library launches on)."""
    fn = fn or (lambda: pj.eval_jacobian(dT, dP, dY, out=out))
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
    ev[0].record()
    for i in range(steps):
        fn()
        ev[i + 1].record()
    torch.cuda.synchronize()
    per = [ev[i].elapsed_time(ev[i + 1]) for i in range(steps)]
    return ev[0].elapsed_time(ev[steps]), per


def bench_config(torch, cfg, steps, warmup, n_states=None, chunk=None):
    """One configuration on the current device; returns a dict of results."""
    from paper_1605_03262_b200 import synth
    from paper_1605_03262_b200.binding import PyJac
    c = synth.CONFIGS[cfg]
    m = synth.make_mechanism(cfg)
    n = c.n_states if n_states is None else n_states
    T, P, Y = synth.config_states(cfg, n)
    per_launch = n if chunk is None else min(chunk, n)
    pj = PyJac(m, device=torch.cuda.current_device())
    ld = c.n_species + 1
    dT, dP, dY = (torch.from_numpy(a).cuda() for a in (T, P, Y))
    out = torch.empty((per_launch, ld * ld), dtype=torch.float64, device="cuda")
    views = [(dT[a:a + per_launch].contiguous(), dP[a:a + per_launch].contiguous(),
              dY[a:a + per_launch].contiguous()) for a in range(0, n, per_launch)]

    def step():
        for (a, b, c_) in views:
            pj.eval_jacobian(a, b, c_, out=out)

    l0 = pj.kernel_launches()
    total_ms, per = time_gpu(pj, torch, dT, dP, dY, out, steps, warmup, fn=step)
    launches = pj.kernel_launches() - l0 - warmup * len(views)
    return dict(pj=pj, mech=m, cfg=c, n=n, T=T, P=P, Y=Y, dT=dT, dP=dP, dY=dY, out=out, total_ms=total_ms,
                per_step_ms=per, launches=launches, launches_per_step=len(views), per_launch=per_launch)


def run_peaks():
    """The two machine peaks SURVEY.md section 8(d) asks for beside MEASURED_PEAKS.json's copy bandwidth:
    a write-only stream with the DENSE pass's store instruction, and the fp64 FMA rate (8 independent
    chains per thread, full occupancy).  CUDA events, 3 warm-up + 10 timed launches, best and mean."""
    import torch
    from paper_1605_03262_b200 import build, binding
    build.build()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(0)
    sp = torch.cuda.current_stream().cuda_stream
    buf = torch.empty(1 << 29, dtype=torch.float64, device="cuda")          # 4 GiB, far beyond L2
    out = torch.empty(torch.cuda.get_device_properties(0).multi_processor_count * 4096, dtype=torch.float64, device="cuda")

    def timed(fn):
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(11)]
        ev[0].record()
        for i in range(10):
            fn()
            ev[i + 1].record()
        torch.cuda.synchronize()
        per = [ev[i].elapsed_time(ev[i + 1]) for i in range(10)]
        return min(per), sum(per) / len(per)

    best, mean = timed(lambda: binding.peak_store_stream(buf, sp))
    nbytes = buf.numel() * 8
    flops = [0]
    iters = 1 << 16

    def dfma():
        flops[0] = binding.peak_dfma(out, iters, sp)
    fbest, fmean = timed(dfma)
    # the output path of a tile kernel: per-state tiles filled in shared memory, one bulk copy each (mode 0) or a read-back
    # through the LSU pipe (mode 1); tile = one state's (N_s+1)^2 matrix of the 53- and 111-species mechanisms
    tiles = {}
    for ns, ctas_list in ((53, (1, 2, 4)), (111, (1, 2))):
        td = (ns + 1) * (ns + 1)
        nt = min(100_000, buf.numel() // td)
        for mode in (0, 1):
            for ctas in ctas_list:
                tb, tm = timed(lambda: binding.peak_tile_store(buf, nt, td, mode, ctas, sp))
                tiles["%dsp_%s_%dcta" % (ns, "bulk" if mode == 0 else "lds_stg", ctas)] = {
                    "tile_bytes": td * 8, "tiles": nt, "ctas_per_sm": ctas, "best_gbs": nt * td * 8 / tb / 1e6,
                    "mean_gbs": nt * td * 8 / tm / 1e6}
    # the buffer must hold what the probe wrote: tile t, element i = t + i (checked on the last configuration run)
    td = 112 * 112
    chk = buf[: 3 * td].cpu()
    tiles["last_run_verified"] = bool(chk[0] == 0.0 and chk[td - 1] == td - 1 and chk[td] == 1.0 and chk[3 * td - 1] == 2 + td - 1)
    peak, src = measured_peaks()
    print(json.dumps({"tile_store": tiles, "store_stream": {"bytes": nbytes, "best_gbs": nbytes / best / 1e6, "mean_gbs": nbytes / mean / 1e6,
                                       "instruction": "st.global.cs.v2.f64"},
                      "fp64_fma": {"flops": flops[0], "best_tflops": flops[0] / fbest / 1e9, "mean_tflops": flops[0] / fmean / 1e9,
                                   "chains_per_thread": 8},
                      "hbm_copy_gbs": peak, "hbm_copy_source": src}))


def rates_buffers(torch, pj, n):
    """the four outputs of pyjac_eval_rates (R_f, R_r, c_i [n][N_reac], wdot [n][N_sp]), allocated once"""
    return {k: torch.empty((n, pj.ns if k == "wdot" else pj.nr), dtype=torch.float64, device="cuda")
            for k in ("rf", "rr", "cmod", "wdot")}


def run_gather_probe(n_states: int = 100_000):
    """profiles/r3_gather_probe.md: the timing prototype of unpadded, length-balanced gathers into a per-state tile +
    one bulk copy per state (tools library, real cell lists of the 53- and 111-species mechanisms, stand-in values),
    for several shapes; every launch's output is compared with the expected tile."""
    import numpy as np
    import torch
    from paper_1605_03262_b200 import build, binding, synth
    build.build()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(0)
    sp = torch.cuda.current_stream().cuda_stream
    res = []
    for cfg, shapes in ((1, ((3, 512, 1, 1), (2, 512, 1, 2), (2, 256, 2, 1), (1, 256, 2, 2), (1, 128, 4, 1), (1, 256, 3, 1))),
                        (2, ((1, 512, 1, 1), (1, 256, 1, 1)))):
        m = synth.make_mechanism(cfg)
        ld = m.n_species + 1
        n = min(n_states, (3 << 30) // (ld * ld * 8))
        out = torch.empty((n, ld * ld), dtype=torch.float64, device="cuda")
        for S, threads, ctas, nbuf in shapes:
            out.fill_(-1.0)
            try:
                r = binding.gather_probe(m, out, n, S, threads, ctas, nbuf, 10, sp)
            except binding.PyJacError as e:
                res.append({"workload": synth.CONFIGS[cfg].name, "S": S, "threads": threads, "ctas_per_sm": ctas, "n_buf": nbuf,
                            "error": str(e)})
                continue
            torch.cuda.synchronize()
            exp = torch.from_numpy(r.pop("expected")).cuda()
            err = float(((out - exp[None, :]).abs() / exp.abs().clamp_min(1e-300)).max())
            alg = algorithmic_bytes(m.n_species, n)
            res.append({"workload": synth.CONFIGS[cfg].name, "n_states": n, "S": S, "threads": threads, "ctas_per_sm": ctas,
                        "n_buf": nbuf, **r, "max_rel_err_vs_expected": err,
                        "states_per_s": n / (r["ms_best"] * 1e-3), "gbs": alg / (r["ms_best"] * 1e-3) / 1e9})
        del out
        torch.cuda.empty_cache()
    peak, src = measured_peaks()
    print(json.dumps({"gather_probe": res, "hbm_copy_gbs": peak, "hbm_copy_source": src,
                      "note": "timing prototype (stand-in values, real cell lists); not an evaluation"}))


def run_ncu_target(spec: str):
    """CFG:KERNEL:N[:SHAPE] -- three launches (two warm-up) of one kernel on the first N states of a configuration and
    nothing else: what `ncu --set full -s 2 -c 1` wraps for the captures under profiles/."""
    import torch
    from paper_1605_03262_b200 import build, synth
    from paper_1605_03262_b200.binding import PyJac
    build.build()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    parts = spec.split(":")
    cfg, kernel, n = int(parts[0]), parts[1], int(parts[2])
    # optional fourth field: an explicit launch shape, e.g. states_per_cta=1,threads=128 (pyjac_launch_shape)
    shape = dict((k, int(v)) for k, v in (kv.split("=") for kv in parts[3].split(","))) if len(parts) > 3 else None
    m = synth.make_mechanism(cfg)
    T, P, Y = synth.config_states(cfg, min(n, synth.CONFIGS[cfg].n_states))
    n = len(T)
    pj = PyJac(m, device=0, shape=shape)
    dT, dP, dY = (torch.from_numpy(a).cuda() for a in (T, P, Y))
    ld = m.n_species + 1
    out = torch.empty((n, ld * ld if kernel in ("jacobian", "jacobian_fd") else ld), dtype=torch.float64, device="cuda")
    rates_out = rates_buffers(torch, pj, n)
    fn = {"jacobian": lambda: pj.eval_jacobian(dT, dP, dY, out=out),
          "jacobian_fd": lambda: pj.eval_jacobian_fd(dT, dP, dY, out=out, chunk_states=256),
          "dydt": lambda: pj.eval_dydt(dT, dP, dY, out=out),
          "rates": lambda: pj.eval_rates(dT, dP, dY, out=rates_out),
          "rates_wdot": lambda: pj.eval_rates(dT, dP, dY, out={"wdot": rates_out["wdot"]})}[kernel]
    total, per = time_gpu(pj, torch, dT, dP, dY, out, 1, 2, fn=fn)
    print(json.dumps({"workload": synth.CONFIGS[cfg].name, "kernel": kernel, "n_states": n, "launch_ms": per[0],
                      "launch_config": pj.launch_config(n)}))


NCU_CSV_FIELDS = ("workload", "kernel", "n_states", "kernel_source_sha16", "duration_us", "dram_bytes_per_state",
                  "fp64_flop_per_state", "fp64_inst_per_state", "warp_inst_per_state", "lsu_wavefronts_per_state",
                  "shared_wavefronts_per_state", "lsu_data_pipe_pct", "fp64_pipe_pct", "issue_active_pct",
                  "registers", "source")


def run_ncu_import(report: str, label: str):
    """Reads one kernel from an `.ncu-rep` (`ncu -i REPORT --page raw --csv`, no GPU needed) and prints the row
    of profiles/r2_ncu_counters.csv that describes it: per-state DRAM bytes, fp64 operations (DFMA counts two
    flops), warp instructions and L1TEX LSU data-pipe wavefronts, with the hash of the kernel sources."""
    import csv
    import io
    workload, kernel, n = label.split(":")
    n = float(n)
    txt = subprocess.run(["ncu", "-i", report, "--page", "raw", "--csv"], capture_output=True, text=True).stdout
    rows = list(csv.reader(io.StringIO(txt)))
    d = dict(zip(rows[0], rows[2]))
    units = dict(zip(rows[0], rows[1]))

    def g(k):
        v = float(d[k].replace(",", ""))
        u = units.get(k, "")
        return v * {"Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}.get(u, 1.0)

    dur_us = g("gpu__time_duration.sum") * {"ns": 1e-3, "nsecond": 1e-3, "us": 1.0, "usecond": 1.0, "ms": 1e3, "msecond": 1e3,
                                            "s": 1e6, "second": 1e6}[units["gpu__time_duration.sum"]]
    cyc = g("smsp__cycles_elapsed.max") if "smsp__cycles_elapsed.max" in d else g("sm__cycles_elapsed.max")
    ops = {k: g("smsp__sass_thread_inst_executed_op_%s_pred_on.sum.per_cycle_elapsed" % k) * cyc for k in ("dfma", "dmul", "dadd")}
    # all LSU data-pipe wavefronts (shared + global + local): the shared count scaled by the ratio of the two
    # utilisation figures the report carries for the same pipe
    lsu = g("l1tex__data_pipe_lsu_wavefronts_mem_shared.sum") * \
        g("l1tex__data_pipe_lsu_wavefronts.sum.pct_of_peak_sustained_elapsed") / \
        g("l1tex__data_pipe_lsu_wavefronts_mem_shared.sum.pct_of_peak_sustained_elapsed")
    row = {"workload": workload, "kernel": kernel, "n_states": int(n), "kernel_source_sha16": kernel_source_sha16(),
           "duration_us": "%.1f" % dur_us,
           "dram_bytes_per_state": "%.1f" % ((g("dram__bytes_read.sum") + g("dram__bytes_write.sum")) / n),
           "fp64_flop_per_state": "%.1f" % ((2 * ops["dfma"] + ops["dmul"] + ops["dadd"]) / n),
           "fp64_inst_per_state": "%.1f" % ((ops["dfma"] + ops["dmul"] + ops["dadd"]) / n),
           "warp_inst_per_state": "%.1f" % (g("smsp__inst_executed.sum") / n),
           "lsu_wavefronts_per_state": "%.1f" % (lsu / n),
           "shared_wavefronts_per_state": "%.1f" % (g("l1tex__data_pipe_lsu_wavefronts_mem_shared.sum") / n),
           "lsu_data_pipe_pct": "%.1f" % g("l1tex__data_pipe_lsu_wavefronts.sum.pct_of_peak_sustained_elapsed"),
           "fp64_pipe_pct": "%.1f" % g("sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active"),
           "issue_active_pct": "%.1f" % g("smsp__issue_active.avg.pct_of_peak_sustained_active"),
           "registers": int(g("launch__registers_per_thread")), "source": os.path.basename(report)}
    w = csv.DictWriter(sys.stdout, fieldnames=NCU_CSV_FIELDS)
    if os.environ.get("NCU_CSV_HEADER"):
        w.writeheader()
    w.writerow(row)


def max_over_ranks(ms: float, dist, device: str) -> float:
    """Device-timed milliseconds of the timed region, MAX over the ranks (the only collective of the
    run: states are independent, every rank evaluates its own replica)."""
    if dist is None:
        return float(ms)
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world: int, n_states_per_rank: int, ms_per_step: float) -> float:
    """States all ranks evaluated per second ("scaling": "weak": n per rank is fixed)."""
    return world * n_states_per_rank / (ms_per_step * 1e-3)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=1, choices=[0, 1, 2, 3])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--also", default="2,3", help="comma list of further configs reported under per_config")
    ap.add_argument("--sweep", default="short", choices=["short", "full", "off"],
                    help="config 4: state-count sweep of the three kernels (short: 4^5, 4^7, 4^9; full: 4^5 .. 4^10)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--peaks", action="store_true",
                    help="measure the write-only store stream and the fp64 FMA rate (SURVEY.md 8(d)) and exit")
    ap.add_argument("--gather-probe", action="store_true",
                    help="run the gather timing prototype of the tools library (profiles/r3_gather_probe.md) and exit")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-fd", action="store_true", help="skip the finite-difference / analytical time ratio")
    ap.add_argument("--ncu-target", default=None, help="CFG:KERNEL:N (KERNEL = jacobian | jacobian_fd | dydt | rates | rates_wdot): three launches, for ncu")
    ap.add_argument("--ncu-import", default=None, help="an .ncu-rep to turn into a row of profiles/r2_ncu_counters.csv")
    ap.add_argument("--ncu-label", default=None, help="WORKLOAD:KERNEL:N of the imported report")
    args = ap.parse_args()
    if args.ncu_target:
        run_ncu_target(args.ncu_target)
        return
    if args.ncu_import:
        run_ncu_import(args.ncu_import, args.ncu_label)
        return
    if args.impl == "reference":
        run_reference(args)
        return
    if args.peaks:
        run_peaks()
        return
    if args.gather_probe:
        run_gather_probe()
        return
    args.warmup = max(3, args.warmup)

    import numpy as np
    import torch
    from paper_1605_03262_b200 import build
    build.build()                       # no-op when the in-tree .so is current
    from paper_1605_03262_b200 import synth

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    cfg = args.config
    chunk = 8192 if cfg == 3 else None           # config 3: 34 GB of output, evaluated in chunks
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    r = bench_config(torch, cfg, args.steps, args.warmup, chunk=chunk)
    barrier()
    clocks = sampler.stop()
    total_ms = max_over_ranks(r["total_ms"], dist, "cuda")
    c, n, pj = r["cfg"], r["n"], r["pj"]
    ms_per_step = total_ms / args.steps
    value = whole_job_value(world, n, ms_per_step)
    peak, peak_src = measured_peaks()
    launch_ms = r["total_ms"] / (args.steps * r["launches_per_step"])
    alg_bytes = algorithmic_bytes(c.n_species, r["per_launch"])
    achieved = alg_bytes / (launch_ms * 1e-3) / 1e9
    counters, counters_src = ncu_counters()
    n_sm = torch.cuda.get_device_properties(local).multi_processor_count
    measure_fp64_peak(torch)

    def traffic_of(name, states):
        """EXTRAPOLATED: DRAM bytes per state of the committed ncu capture (taken at fewer states, see
        `traffic_capture_states`) times the states of this launch; lines still dirty in L2 when the captured kernel
        ended are not in it, so it can sit a few per cent below the bytes the kernel stores"""
        c = counters.get(name, {}).get("jacobian")
        return None if not c else int(round(c["dram_bytes_per_state"] * states))

    def capture_states(name):
        c = counters.get(name, {}).get("jacobian")
        return None if not c else c.get("n_states")

    def fp64_of(name, kernel, states, ms):
        """achieved fp64 FLOP/s of one launch from the counted DFMA / DADD / DMUL per state (ncu), against the
        measured FMA peak: the second roofline SURVEY.md 8(d) asks for"""
        c = counters.get(name, {}).get(kernel)
        if not c:
            return None
        tf = c["fp64_flop_per_state"] * states / (ms * 1e-3) / 1e12
        return {"bound": "alu", "achieved": tf, "peak": fp64_peak(), "unit": "TFLOP/s", "frac": tf / fp64_peak(),
                "flop_per_state": c["fp64_flop_per_state"], "peak_source": _FP64_PEAK["source"]}

    def lsu_of(name, kernel, states, ms, sm_mhz):
        """the pipe that binds the Jacobian kernel: L1TEX LSU data-pipe wavefronts (shared
        and global accesses; one per SM and clock at best), counted by ncu per state, over this launch's time"""
        c = counters.get(name, {}).get(kernel)
        if not c or not sm_mhz:
            return None
        rate = c["lsu_wavefronts_per_state"] * states / (ms * 1e-3) / 1e9
        peak = n_sm * sm_mhz * 1e6 / 1e9
        return {"bound": "lsu", "diagnostic": True,
                "note": "a diagnosis, not a roofline: the wavefront count is derived (shared-memory count scaled by the "
                        "ratio of two utilisation figures of the same ncu report) and the peak is nominal, not measured",
                "achieved": rate, "peak": peak, "unit": "Gwavefront/s", "frac": rate / peak,
                "wavefronts_per_state": c["lsu_wavefronts_per_state"],
                "peak_source": "one L1TEX data-pipe wavefront per SM and clock, %d SMs at the SM clock sampled during the run" % n_sm}

    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": traffic_of(c.name, r["per_launch"]), "traffic_source": counters_src,
                "traffic_kind": "extrapolated from a smaller capture (per-state DRAM bytes x states of this launch)",
                "traffic_capture_states": capture_states(c.name),
                "peak_source": peak_src,
                "kernel": "pyjac::eval_kernel<2 (Jacobian), S = %d states per CTA iteration>" % pj.launch_config(r["per_launch"])["states_per_cta"],
                "algorithmic_bytes_per_launch": alg_bytes,
                "algorithmic_bytes_note": "(Ns+2) doubles read + (Ns+1)^2 doubles written per state, the placeholder "
                                          "row and the zero column of the (Ns+1)^2 layout included",
                "launch_ms": launch_ms, "launch_config": pj.launch_config(r["per_launch"]),
                "fp64": fp64_of(c.name, "jacobian", r["per_launch"], launch_ms),
                "lsu": lsu_of(c.name, "jacobian", r["per_launch"], launch_ms, clocks.get("sm_mhz"))}
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": c.name, "n_species": c.n_species, "n_reactions": c.n_reactions,
                       "n_states": n, "states_per_launch": r["per_launch"],
                       "jacobian": "%dx%d fp64 column-major per state" % (c.n_species + 1, c.n_species + 1),
                       "parallelism": "replicas x%d" % world if world > 1 else "single GPU",
                       "cache": "output (%.2f GB per launch) and inputs exceed the 126 MB L2; no flush needed"
                                % (r["per_launch"] * (c.n_species + 1) ** 2 * 8 / 1e9)},
            "roofline": roofline, "clocks": clocks, "gpu_launches": int(r["launches"]),
            "step_ms_min_max": [min(r["per_step_ms"]), max(r["per_step_ms"])]}

    if rank == 0 and world == 1:
        # ---- end to end through the host-buffer C-ABI call (pinned host memory, copies timed)
        if not args.no_e2e:
            ld = c.n_species + 1
            n_e = n if cfg != 3 else 8192
            hT, hP, hY = (torch.from_numpy(a[:n_e].copy()).pin_memory() for a in (r["T"], r["P"], r["Y"]))
            hout = torch.empty((n_e, ld * ld), dtype=torch.float64).pin_memory()
            e_steps = max(2, min(args.steps, 5))
            pj.eval_jacobian_host(hT, hP, hY, hout)              # warm-up (also pages in the pinned buffer)
            t0 = time.perf_counter()
            for _ in range(e_steps):
                pj.eval_jacobian_host(hT, hP, hY, hout)
            dt = (time.perf_counter() - t0) / e_steps
            line["e2e"] = {"value": n_e / dt, "unit": UNIT, "h2d_bytes_per_step": n_e * (c.n_species + 2) * 8,
                           "d2h_bytes_per_step": n_e * ld * ld * 8, "ms_per_step": dt * 1e3, "steps": e_steps,
                           "call": "pyjac_eval_jacobian_host (pinned host buffers, double-buffered chunks)",
                           "n_states": n_e}
            del hout
        # ---- further configs (same timing rules), reported beside the headline
        per = {}
        del r["out"]
        torch.cuda.empty_cache()
        for extra in [int(x) for x in args.also.split(",") if x.strip() != ""]:
            if extra == cfg:
                continue
            ch = 8192 if extra == 3 else None
            st = max(3, args.steps // (2 if extra == 2 else 4))
            rr = bench_config(torch, extra, st, args.warmup, chunk=ch)
            cc = rr["cfg"]
            lm = rr["total_ms"] / (st * rr["launches_per_step"])
            ab = algorithmic_bytes(cc.n_species, rr["per_launch"])
            per[cc.name] = {"value": rr["n"] / (rr["total_ms"] / st * 1e-3), "unit": UNIT, "steps": st,
                            "n_states": rr["n"], "states_per_launch": rr["per_launch"], "launch_ms": lm,
                            "roofline": {"bound": "hbm", "achieved": ab / (lm * 1e-3) / 1e9, "peak": peak,
                                         "unit": "GB/s", "frac": ab / (lm * 1e-3) / 1e9 / peak,
                                         "traffic": traffic_of(cc.name, rr["per_launch"]),
                                         "fp64": fp64_of(cc.name, "jacobian", rr["per_launch"], lm),
                                         "lsu": lsu_of(cc.name, "jacobian", rr["per_launch"], lm, clocks.get("sm_mhz"))},
                            "launch_config": rr["pj"].launch_config(rr["per_launch"])}
            del rr
            torch.cuda.empty_cache()
        if per:
            line["per_config"] = per
            # north_star names two target configurations: the other one (and the 360-species one) inside the
            # headline's roofline object, with the same definition of `frac`
            line["roofline"]["other_configs"] = {
                k: {"launch_ms": v["launch_ms"], "states_per_launch": v["states_per_launch"],
                    "achieved": v["roofline"]["achieved"], "frac": v["roofline"]["frac"], "value": v["value"]}
                for k, v in per.items()}
        if args.sweep != "off":
            line["sweep_53sp"] = sweep(torch, args, fp64_of)
        if not args.no_fd:
            line["fd_vs_analytical"] = fd_ratio(torch)
            line["jvp_on_chip"] = jvp_rates(torch)
        if not args.no_cpu_baseline:
            line["cpu_baseline"], _ = time_oracle(cfg, CPU_SAMPLE[cfg], steps=3, warmup=1, single_thread=True)
    if rank == 0:
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def fd_ratio(torch):
    """The paper's own comparison (Table 5): the first-order forward-difference
    Jacobian built on the source-term kernel (pyjac_eval_jacobian_fd, 1 + N_sp source-term evaluations per
    state) against the analytical one, same states, CUDA events, per mechanism.  The paper's GPU ratios
    (Tesla C2075, one thread per state) are 1.37 - 2.73; context, not a target."""
    from paper_1605_03262_b200 import synth
    from paper_1605_03262_b200.binding import PyJac
    out = {}
    for cfg, n in ((0, 1024), (1, 8192), (2, 4096), (3, 512)):
        m = synth.make_mechanism(cfg)
        T, P, Y = synth.config_states(cfg, n)
        pj = PyJac(m, device=torch.cuda.current_device())
        ld = m.n_species + 1
        dT, dP, dY = (torch.from_numpy(a).cuda() for a in (T, P, Y))
        jac = torch.empty((n, ld * ld), dtype=torch.float64, device="cuda")
        chunk = max(1, min(n, (1 << 28) // pj.fd_workspace_doubles(1)))           # 2 GiB of scratch at most
        work = torch.empty(pj.fd_workspace_doubles(chunk), dtype=torch.float64, device="cuda")
        ta, _ = time_gpu(pj, torch, dT, dP, dY, jac, 5, 3)
        tf, _ = time_gpu(pj, torch, dT, dP, dY, jac, 3, 3,
                         fn=lambda: pj.eval_jacobian_fd(dT, dP, dY, out=jac, work=work))
        out[synth.CONFIGS[cfg].name] = {"n_states": n, "analytical_ms": ta / 5, "fd_ms": tf / 3,
                                        "fd_over_analytical": (tf / 3) / (ta / 5)}
        del jac, work
        torch.cuda.empty_cache()
    out["paper_gpu_ratio_range"] = [1.37, 2.73]
    out["note"] = ("cost of THIS forward-difference path, not of the method: pyjac_eval_jacobian_fd writes N_sp perturbed "
                   "copies of every state (N_sp^2 doubles) to HBM, reads them back through 1 + N_sp source-term "
                   "evaluations and a difference kernel (csrc/fd.cu); not comparable with the paper's ratios")
    return out


def jvp_rates(torch):
    """the Jacobian consumed on chip.  pyjac_eval_jvp evaluates J v per state without
    forming J (the (N_sp+1)^2 store that sets the HBM roof disappears); states/s per mechanism, next to the
    time the full Jacobian takes for the same states."""
    import numpy as np
    from paper_1605_03262_b200 import synth
    from paper_1605_03262_b200.binding import PyJac
    out = {}
    for cfg, n in ((1, 100_000), (2, 50_000), (3, 8192)):
        m = synth.make_mechanism(cfg)
        T, P, Y = synth.config_states(cfg, n)
        pj = PyJac(m, device=torch.cuda.current_device())
        ld = m.n_species + 1
        dT, dP, dY = (torch.from_numpy(a).cuda() for a in (T, P, Y))
        v = torch.from_numpy(np.random.default_rng(1).standard_normal((n, ld))).cuda()      # host-made: no library kernel
        jv = torch.empty((n, ld), dtype=torch.float64, device="cuda")
        t, _ = time_gpu(pj, torch, dT, dP, dY, None, 10, 3, fn=lambda: pj.eval_jvp(dT, dP, dY, v, out=jv))
        out[synth.CONFIGS[cfg].name] = {"n_states": n, "jvp_ms": t / 10, "jvp_states_per_s": n / (t / 10 * 1e-3),
                                        "bytes_per_state": (2 * ld + m.n_species + 2) * 8}
    return out


def sweep(torch, args, fp64_of):
    """BASELINE.json configs[4]: 53-species mechanism, 4^5 .. 4^10 states (short: three of them), the three
    kernels separately, each with its fp64 roofline entry (rates and dPhi/dt move few bytes: fp64-bound)."""
    from paper_1605_03262_b200 import synth
    from paper_1605_03262_b200.binding import PyJac
    m = synth.make_mechanism(1)
    pj = PyJac(m, device=torch.cuda.current_device())
    ld = m.n_species + 1
    res = []
    counts = synth.SWEEP_STATES if args.sweep == "full" else (4 ** 5, 4 ** 7, 4 ** 9)
    for n in counts:
        T, P, Y = synth.make_states(m.n_species, n, synth.CONFIGS[1].seed + 2000 + n)
        dT, dP, dY = (torch.from_numpy(a).cuda() for a in (T, P, Y))
        out = torch.empty((n, ld * ld), dtype=torch.float64, device="cuda")
        dy = torch.empty((n, ld), dtype=torch.float64, device="cuda")
        steps = 10
        tj, _ = time_gpu(pj, torch, dT, dP, dY, out, steps, 3)
        td, _ = time_gpu(pj, torch, dT, dP, dY, None, steps, 3, fn=lambda: pj.eval_dydt(dT, dP, dY, out=dy))
        ro = rates_buffers(torch, pj, n)
        # all four outputs (8.2 KB per state for the rate arrays); the wdot-only figure beside it
        tr, _ = time_gpu(pj, torch, dT, dP, dY, None, steps, 3, fn=lambda: pj.eval_rates(dT, dP, dY, out=ro))
        tw, _ = time_gpu(pj, torch, dT, dP, dY, None, steps, 3,
                         fn=lambda: pj.eval_rates(dT, dP, dY, out={"wdot": ro["wdot"]}))
        name = synth.CONFIGS[1].name
        res.append({"n_states": n, "jacobian_states_per_s": n / (tj / steps * 1e-3),
                    "dydt_states_per_s": n / (td / steps * 1e-3), "rates_states_per_s": n / (tr / steps * 1e-3),
                    "rates_outputs": "rf, rr, cmod, wdot (%d B per state)" % ((3 * pj.nr + pj.ns) * 8),
                    "rates_wdot_only_states_per_s": n / (tw / steps * 1e-3),
                    "fp64": {"jacobian": fp64_of(name, "jacobian", n, tj / steps),
                             "dydt": fp64_of(name, "dydt", n, td / steps),
                             "rates": fp64_of(name, "rates", n, tr / steps)}})
        del out, dy, ro
        torch.cuda.empty_cache()
    return res


if __name__ == "__main__":
    main()
