#!/usr/bin/env python
"""bench.py -- headline benchmark of cwo-b200: propagations/s for the 4096^2 angular spectrum method.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

A step is one pass of the whole hot path (plan tables for a NEW z, row pass, fused column pass,
inverse row pass) over one 4096 x 4096 complex64 field of BASELINE.json config c3; z cycles through
{0.01, 0.1, 0.5} m so every step is the paper's "re-calculation" case.  Prints ONE JSON line.

  value      whole-job propagations/s, inputs resident in HBM, CUDA events on the launching stream
  e2e        same metric through the public binding with HOST (pinned) buffers: H2D of u1 and D2H of
             u2 inside the timed region
  roofline   the dominant kernel (c3: the fused column pass): algorithmic bytes (or nominal flops) per launch / its
             average duration from CUDA events recorded by the library (include/cwo_debug.h timing mode)
  cpu_baseline  the fp64 oracle as it stands on the host cores (reported baseline, not the target): c3 on all threads
             and on one thread, the CPU model, and one propagation of every other BASELINE config
  extra      (default run, N = 1 only) the other sizes the throughput target names -- asm8192, fresnel4096, fresnel8192,
             c4, c5 -- each timed briefly after the headline: ms per call against its target, effective GB/s, the
             dominant kernel's roofline fraction, clocks.  --no-extra skips them (profiling runs).

--impl reference times the oracle itself (this tier has no installable reference implementation).
N > 1: the path does not shard (replicas only) -- every rank propagates its own field.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "propagations/sec (4096^2 ASM, new z per call); effective HBM GB/s for 48*N^2 algorithmic bytes"
UNIT = "propagations/s"
C3_DESC = ("c3: ASM 4096x4096 complex64 speckle field, lambda 633 nm, pitch 4 um, z cycling {0.01,0.1,0.5} m "
           "(new z every call)")
NOMINAL_HBM_GBS = 8000.0          # BASELINE.json's "~8 TB/s peak" (the target's denominator)
FALLBACK_HBM_GBS = 6650.0         # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent


def _peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def _ncu_traffic(workload: str, kernel_key: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of a kernel, as MEASURED BY THE COMMITTED ncu --set full
    capture (profiles/traffic.csv names the capture); a constant of the repository, not something this run measures.
    None when no capture of that kernel of that workload is committed."""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    try:
        for line in open(p):
            t = [x.strip() for x in line.split(",")]
            if len(t) >= 4 and t[0] == workload and t[1] == kernel_key:
                return float(t[2]) + float(t[3])
    except Exception:
        pass
    return None


FP32_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12      # 148 SMs x 128 fp32 lanes x 2 flop (FMA) x 1965 MHz


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx = float(r[1])
                for nme, v in zip(names, r[2:6]):
                    if v.lower().startswith("active"):
                        reasons.add(nme)
            except Exception:
                continue
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


def _dist():
    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


# ------------------------------------------------------------------------------------------------------
# oracle arm (--impl reference) and the cpu_baseline leg: the ONLY places that touch oracle/
# ------------------------------------------------------------------------------------------------------

def _oracle_time_props(cfg, n_props: int, size: int):
    """Seconds for n_props oracle ASM propagations of a size x size field (same pitch/lambda/z cycle)."""
    from oracle import oracle as O
    from paper_1107_5578_b200 import workloads as W
    threads = O.max_threads()
    O.set_threads(threads)
    u1 = W.make_field(cfg.scaled(size) if size != cfg.N else cfg)
    t0 = time.perf_counter()
    for i in range(n_props):
        O.asm(u1, cfg.pitch, cfg.pitch, cfg.lam, cfg.zs[i % len(cfg.zs)])
    return time.perf_counter() - t0, threads


def _cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


def _mem_available_gb():
    try:
        for line in open("/proc/meminfo"):
            if line.startswith("MemAvailable"):
                return float(line.split()[1]) / 1e6
    except Exception:
        pass
    return 0.0


_C5_INPUTS = {}


def _gs_inputs_c5(W):
    """c5's amplitudes and start phase (7 s of host work at 8192^2): drawn once per process."""
    if "v" not in _C5_INPUTS:
        _C5_INPUTS["v"] = W.gs_inputs_c5(W.CONFIGS["c5"])
    return _C5_INPUTS["v"]


def cpu_baseline_per_config(budget_s: float = 60.0):
    """the oracle's time for ONE propagation of each BASELINE config (c4: one plane; c5: one Fresnel
    propagation and one GS iteration), all host threads.  The c5 entries (three fp64 FFTs of 16384^2 per propagation,
    ~9 GB) run only if their estimate fits the remaining budget and the host has the memory; otherwise they say so."""
    from oracle import oracle as O
    from paper_1107_5578_b200 import workloads as W
    threads = O.max_threads()
    O.set_threads(threads)
    out, t_begin = {}, time.perf_counter()

    def timed(f):
        t0 = time.perf_counter(); f(); return time.perf_counter() - t0
    for name in ("c1", "c2", "c4"):
        cfg = W.CONFIGS[name]
        u1 = W.make_field(cfg)
        f = O.asm if cfg.op != "fresnel" else O.fresnel_conv
        key = name if name != "c4" else "c4_one_plane"
        out[key] = {"what": "%s %dx%d, one propagation" % ("Fresnel convolution" if f is O.fresnel_conv else "ASM", cfg.N, cfg.N),
                    "seconds": timed(lambda: f(u1, cfg.pitch, cfg.pitch, cfg.lam, cfg.zs[0])), "threads": threads}
    c5 = W.CONFIGS["c5"]
    # one c5 propagation = three 2-D FFTs of (2 * 8192)^2 against three of (2 * 1024)^2 for c2
    est = out["c2"]["seconds"] * (16384.0 ** 2 * 28) / (2048.0 ** 2 * 22)
    for key, mult in (("c5_fresnel_propagation", 1.0), ("c5_gs_iteration", 2.0)):
        left = budget_s - (time.perf_counter() - t_begin)
        if est * mult > left or _mem_available_gb() < 40.0:
            out[key] = {"skipped": "estimated %.0f s against %.0f s of budget left, %.0f GB of host memory available"
                                   % (est * mult, left, _mem_available_gb())}
            continue
        if key == "c5_fresnel_propagation":
            u1 = W.field_c3(W.Config("c5f", "fresnel", c5.N, c5.lam, c5.pitch, c5.zs, index=c5.index + 100))
            sec = timed(lambda: O.fresnel_conv(u1, c5.pitch, c5.pitch, c5.lam, c5.zs[0]))
            what = "Fresnel convolution 8192x8192 (transforms of 16384x16384), one propagation"
            est = sec
        else:
            a_src, a_dst, _ = _gs_inputs_c5(W)
            pz = W.random_phasor(c5)
            sec = timed(lambda: O.gs_iter(0, a_src, a_dst, pz, c5.pitch, c5.pitch, c5.lam, c5.zs[0]))
            what = "one Gerchberg-Saxton iteration at 8192x8192 (two Fresnel propagations + constraints)"
        out[key] = {"what": what, "seconds": sec, "threads": threads}
    return out


def cpu_baseline(cfg, budget_s: float = 20.0, per_config: bool = True):
    """The oracle as it stands, on a bounded sample: whole 4096^2 propagations while they fit the budget; then (SURVEY.md
    8(d)) the same propagation on ONE thread and one propagation of each of the other configs."""
    from oracle import oracle as O
    t1, threads = _oracle_time_props(cfg, 1, cfg.N)
    n = int(max(1, min(8, budget_s // max(t1, 1e-3))))
    t, _ = _oracle_time_props(cfg, n, cfg.N)
    out = {"value": n / t, "unit": UNIT, "cores": threads, "kind": "oracle", "cpu_model": _cpu_model(),
           "sample": "%d full %dx%d fp64 oracle propagation(s), %d OpenMP threads, %.2f s" % (n, cfg.N, cfg.N, threads, t)}
    if per_config:
        from paper_1107_5578_b200 import workloads as W
        u1 = W.make_field(cfg)
        O.set_threads(1)
        t0 = time.perf_counter()
        O.asm(u1, cfg.pitch, cfg.pitch, cfg.lam, cfg.zs[0])
        ts = time.perf_counter() - t0
        O.set_threads(threads)
        out["one_thread"] = {"value": 1.0 / ts, "unit": UNIT, "cores": 1,
                             "sample": "1 full %dx%d fp64 oracle propagation on one thread, %.2f s" % (cfg.N, cfg.N, ts)}
        out["per_config"] = cpu_baseline_per_config()
        out["per_config"]["c3"] = {"what": "ASM %dx%d, one propagation" % (cfg.N, cfg.N), "seconds": t / n, "threads": threads}
    return out


def run_reference(args):
    rank, world, _ = _dist()
    if rank != 0:
        return
    from paper_1107_5578_b200 import workloads as W
    cfg = W.CONFIGS["c3"]
    t_full, threads = _oracle_time_props(cfg, 1, cfg.N)
    total = args.steps + args.warmup
    size, scale = cfg.N, 1.0
    while size > 512 and t_full * scale * total > 150.0:     # keep the whole run within a few minutes
        size //= 2
        scale = (size * size * np.log2(size)) / (cfg.N * cfg.N * np.log2(cfg.N))
    _oracle_time_props(cfg, args.warmup, size)
    t, _ = _oracle_time_props(cfg, args.steps, size)
    value = args.steps / t * scale                            # 4096^2-equivalent propagations/s
    sample = ("each step = one fp64 oracle ASM propagation of %dx%d (same pitch/lambda/z cycle)%s, %d threads"
              % (size, size, "" if size == cfg.N else "; value scaled by N^2 log2 N to 4096^2", threads))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": t / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": C3_DESC,
                       "l2": "working set 403 MB per step, rotating over 3 field pairs (larger than the 126 MB L2); no flush",
                       "parallelism": "single GPU", "bytes_per_step": 48 * cfg.N * cfg.N, "propagations_per_step": 1},
            "arm_note": "oracle on the host cores (this tier has no installable reference); config keys mirror the CUDA arm",
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------------
# workloads: c3 is the headline (BASELINE.json); the others time the same C-ABI calls on other configs
# ------------------------------------------------------------------------------------------------------

WORKLOADS = {"c1": ("asm", 256), "c3": ("asm", 4096), "asm8192": ("asm", 8192), "asm2048": ("asm", 2048), "asm16384": ("asm", 16384),
             "c2": ("fresnel", 1024), "fresnel2048": ("fresnel", 2048), "fresnel4096": ("fresnel", 4096),
             "fresnel8192": ("fresnel", 8192), "c4": ("stack", 2048), "c4_intensity": ("stack_i", 2048), "c5": ("gs", 8192),
             "asm_pad2x_2048": ("asm_pad", 2048), "asm_pad2x_4096": ("asm_pad", 4096),
             "fourier4096": ("fourier", 4096), "fourier8192": ("fourier", 8192), "shifted4096": ("shifted", 4096),
             "pls2048": ("pls", 2048), "gs_asm2048": ("gs_asm", 2048)}


def make_workload(name, rank, torch, api, W, nbuf=3):
    """Device-resident inputs, the step function and the algorithmic byte counts of a workload.
    nbuf: field pairs the steps rotate over (the `extra` legs use one: a single 4096^2 / 8192^2 step already touches
    403 MB / 1.6 GB, more than the 126 MB L2)."""
    op, N = WORKLOADS[name]
    NBUF = nbuf
    n2 = float(N) * N
    pad2x = op == "asm_pad"                                  # cwo_asm on the zero-expanded grid
    if pad2x:
        op = "asm"
    if op == "pls":
        # the paper's List 3: 2048 x 2048 hologram of 11 646 point light sources (the dinosaur model is not
        # in the container: seeded uniform points in the same +-4 mm box, offset (1 cm, -2 mm), 0.2 m away), pitch 4 um
        npts = 11646
        r = np.random.default_rng(11075578 * 10 + 6 + rank)
        pts = np.stack([r.uniform(-4e-3, 4e-3, npts) + 1e-2, r.uniform(-4e-3, 4e-3, npts) - 2e-3,
                        0.2 + r.uniform(-4e-3, 4e-3, npts), r.uniform(0.2, 1.0, npts)], axis=1)
        d_pts = torch.from_numpy(pts).cuda()
        out = torch.empty((N, N), dtype=torch.float32, device="cuda")
        plan = api.cwo_plan(N, N, 4e-6, 633e-9)

        def step(i):
            api.cwo_pls_cgh(plan, d_pts, out)

        def e2e():
            pin_in = torch.from_numpy(pts).pin_memory()
            pin_out = torch.empty((N, N), dtype=torch.float32).pin_memory()

            def f(i):
                d_pts.copy_(pin_in, non_blocking=True)
                api.cwo_pls_cgh(plan, d_pts, out)
                pin_out.copy_(out, non_blocking=True)
            return f, 32 * npts, 4 * n2
        return dict(plan=plan, step=step, N=N, props_per_step=1, bytes_per_step=4 * n2 + 32 * npts,
                    kind_bytes={10: 4 * n2 + 32 * npts}, kind_flops={10: 4.0 * npts * n2}, e2e=e2e,
                    scheme_bytes_per_step=4 * n2 + 32 * npts,
                    desc="pls2048: CGH of %d point light sources on a 2048x2048 hologram (Eq.(23)), lambda 633 nm, pitch 4 um, "
                         "z 0.2 m" % npts,
                    l2="16.8 MB output; everything on chip; ALU-bound", metric="holograms/sec (PLS CGH, Eq.(23)); fp32 FMA rate")
    other = op in ("fourier", "shifted")          # same host loop as the convolution form
    if other:
        call_other = api.cwo_fresnel_fourier if op == "fourier" else api.cwo_fresnel_shifted
        op_name, op = op, "fresnel"
    if op in ("asm", "fresnel"):
        base = (W.CONFIGS["c1"] if name == "c1" else W.CONFIGS["c3"]) if op == "asm" else (
            W.CONFIGS["c2"] if N <= 2048 else W.CONFIGS["c5"])
        zs = base.zs if op == "asm" else (base.zs[0], 1.07 * base.zs[0], 0.93 * base.zs[0])
        hosts = [W.field_c3(W.Config(name, op, N, base.lam, base.pitch, zs, index=base.index + 100 * (i + rank * NBUF)))
                 for i in range(NBUF)]
        u1 = [torch.from_numpy(h).cuda() for h in hosts]
        u2 = [torch.empty_like(u1[0]) for _ in range(NBUF)]
        plan = api.cwo_plan(N, N, base.pitch, base.lam)
        call = api.cwo_asm if op == "asm" else api.cwo_fresnel_conv
        if other:
            call = call_other
            if op_name == "shifted":          # 1.5 x magnification, window displaced by a quarter of its width
                plan.set_dst_pitch_xy(1.5 * base.pitch, 1.5 * base.pitch)
                plan.set_offset(0.25 * N * base.pitch, -0.25 * N * base.pitch)
        if pad2x:
            plan.set_option(api.CWO_OPT_ASM_PAD2X, 1)
        plan.ensure_workspace(api.CWO_OP_ASM if op == "asm" else api.CWO_OP_FRESNEL)
        if other:
            op = op_name

        def step(i):
            call(plan, u1[i % NBUF], u2[i % NBUF], zs[i % len(zs)])

        def e2e():
            # the public host-buffer API: every step copies its input from pinned host memory and its result
            # back; api.HostPipeline overlaps the copies of neighbouring steps with the kernels
            pin_in = [torch.from_numpy(h).pin_memory() for h in hosts]
            pin_out = [torch.empty((N, N), dtype=torch.complex64).pin_memory() for _ in range(NBUF)]
            if other:
                d_in = torch.empty_like(u1[0])

                def g(i):
                    d_in.copy_(pin_in[i % NBUF], non_blocking=True)
                    call(plan, d_in, u2[i % NBUF], zs[i % len(zs)])
                    pin_out[i % NBUF].copy_(u2[i % NBUF], non_blocking=True)
                return g, 8 * n2, 8 * n2
            hp = api.HostPipeline(plan, op)

            def f(i):
                hp.submit(pin_in[i % NBUF], pin_out[i % NBUF], zs[i % len(zs)])
            f.begin = hp.start_after
            f.end = hp.join
            return f, 8 * n2, 8 * n2
        if op == "asm" and not pad2x:
            kb = {0: 16 * n2, 3: 16 * n2, 1: 16 * n2}
            bps = 48 * n2
            desc = ("%s: ASM %dx%d complex64 speckle field, lambda %g nm, pitch %g um, z cycling %s m (new z every call)"
                    % (name, N, N, base.lam * 1e9, base.pitch * 1e6, "{" + ",".join("%g" % z for z in zs) + "}"))
            assert name != "c3" or desc == C3_DESC, desc
        else:
            # two-dimensional form: R: 8 rd + 16 wr; C: 16 + 16; R': 16 rd + 8 wr.  Separable form (Fresnel, 256..8192):
            # kind 5 = one line-convolution pass (8 rd + 8 wr), kind 6 = one transpose (8 + 8)
            kb = {0: 24 * n2, 3: 32 * n2, 1: 24 * n2, 5: 16 * n2, 6: 16 * n2, 7: 16 * n2}
            bps = 80 * n2
            what = "zero-expanded ASM" if pad2x else "Fresnel convolution"
            if other:      # one 2-D transform (Fourier form: 2 passes of 8 rd + 8 wr) / the scaled convolution (as the convolution form)
                what = "Fresnel diffraction, Fourier form" if op_name == "fourier" else "shifted Fresnel diffraction"
                bps = (32 if op_name == "fourier" else 80) * n2
            desc = ("%s: %s %dx%d complex64 speckle field (virtual %dx%d), lambda %g nm, pitch %g um, "
                    "z cycling %s m (new z every call)" % (name, what,
                                                           N, N, 2 * N, 2 * N, base.lam * 1e9, base.pitch * 1e6,
                                                           "{" + ",".join("%.4g" % z for z in zs) + "}"))
        ws = (24 if (op == "asm" and not pad2x) else 32) * n2   # u1 + u2 + workspace touched per step
        l2 = ("working set %.0f MB per step, rotating over %d field pair%s (%s the 126 MB L2); no flush"
              % (ws / 1e6, NBUF, "s" if NBUF > 1 else "", "larger than" if ws > 126e6 else "FITS in"))
        # nominal flops of one line-convolution launch: N lines x (4 N-point FFTs at 5 n log2 n + ~30 flops per sample for
        # the modulation, the spectrum multiply and the recombination)
        kf = {5: N * (20.0 * N * np.log2(N) + 30.0 * N)}
        scheme = bps if (op == "asm") else 64 * n2          # separable Fresnel: 2 x (conv 16 + transpose 16) N^2
        return dict(plan=plan, step=step, N=N, props_per_step=1, bytes_per_step=bps, kind_bytes=kb, kind_flops=kf, e2e=e2e,
                    desc=desc, l2=l2, scheme_bytes_per_step=scheme,
                    metric="propagations/sec (%s); effective HBM GB/s for the algorithmic bytes" % name)
    if op in ("stack", "stack_i"):
        cfg = W.CONFIGS["c4"]
        n = len(cfg.zs)
        host = W.make_field(cfg)
        u1 = torch.from_numpy(host).cuda()
        inten = op == "stack_i"              # float |u|^2 planes (CWO_OPT_STACK_INTENSITY), half the output
        odt = torch.float32 if inten else torch.complex64
        out = torch.empty((n, N, N), dtype=odt, device="cuda")
        plan = api.cwo_plan(N, N, cfg.pitch, cfg.lam)
        if inten:
            plan.set_option(api.CWO_OPT_STACK_INTENSITY, 1)
        plan.ensure_workspace(api.CWO_OP_STACK, n)

        def step(i):
            api.cwo_propagate_stack(plan, u1, cfg.zs, out)

        def e2e():
            pin_in = torch.from_numpy(host).pin_memory()
            pin_out = torch.empty((n, N, N), dtype=odt).pin_memory()
            d_in = torch.empty_like(u1)

            def f(i):
                d_in.copy_(pin_in, non_blocking=True)
                api.cwo_propagate_stack(plan, d_in, cfg.zs, out)
                pin_out.copy_(out, non_blocking=True)
            return f, 8 * n2, (4 if inten else 8) * n2 * n
        per_plane = 28 if inten else 32      # C': 8 rd + 8 wr, R': 8 rd + 8 (4) wr
        return dict(plan=plan, step=step, N=N, props_per_step=n, bytes_per_step=32 * n2 + n * per_plane * n2,
                    kind_bytes={0: 16 * n2, 2: 16 * n2, 4: min(n, 64) * 16 * n2, 1: min(n, 64) * (per_plane - 16) * n2}, kind_flops={},   # C' / R' launches cover up to 64 planes
                    scheme_bytes_per_step=32 * n2 + n * per_plane * n2, e2e=e2e,
                    desc="%s: depth stack, one 2048x2048 random-phase field to 64 planes z = 1..64 mm by ASM, lambda 633 nm, "
                         "pitch 6.4 um, out 64x2048x2048 %s" % (name, "float32 intensity" if inten else "complex64"),
                    l2="spectrum (34 MB) stays in L2; the 2.1 GB output stack streams to HBM; no flush",
                    metric="planes/sec (c4 depth stack); effective HBM GB/s for 32 N^2 + n 32 N^2 bytes")
    if op == "gs_asm":
        # the paper's own GS experiment (Listing 8 / Table 7): angular spectrum propagator, 2048 x 2048, its
        # default wavelength and pitch (633 nm, 10 um), 0.1 m, 20 iterations; inputs drawn like c5's
        lam, pitch, z, iters = 633e-9, 10e-6, 0.1, 20
        a_src, a_dst, phi0 = W.gs_inputs((N, N), 11 + rank)
        d_src, d_dst = torch.from_numpy(a_src).cuda(), torch.from_numpy(a_dst).cuda()
        d_phi0 = torch.from_numpy(phi0).cuda()
        d_phi = torch.empty_like(d_phi0)
        plan = api.cwo_plan(N, N, pitch, lam)
        plan.set_option(api.CWO_OPT_GS_METHOD, api.CWO_GS_ASM)
        plan.ensure_workspace(api.CWO_OP_GS)

        def step(i):
            d_phi.copy_(d_phi0)
            api.cwo_gs(plan, d_src, d_dst, z, iters, d_phi)

        def e2e():
            pins = [torch.from_numpy(x).pin_memory() for x in (a_src, a_dst, phi0)]
            pin_out = torch.empty((N, N), dtype=torch.float32).pin_memory()

            def f(i):
                d_src.copy_(pins[0], non_blocking=True); d_dst.copy_(pins[1], non_blocking=True)
                d_phi.copy_(pins[2], non_blocking=True)
                api.cwo_gs(plan, d_src, d_dst, z, iters, d_phi)
                pin_out.copy_(d_phi, non_blocking=True)
            return f, 12 * n2, 4 * n2
        bps = iters * 2 * (48 + 4) * n2 + 52 * n2          # per propagation 48 N^2 + one amplitude read
        return dict(plan=plan, step=step, N=N, props_per_step=2 * iters + 1, bytes_per_step=bps,
                    kind_bytes={0: 16 * n2, 3: 16 * n2, 1: 20 * n2}, kind_flops={}, scheme_bytes_per_step=bps, e2e=e2e,
                    desc="gs_asm2048: Gerchberg-Saxton with the angular spectrum propagator (the paper's Listing 8), 2048x2048, "
                         "lambda 633 nm, pitch 10 um, z 0.1 m, 20 iterations (41 propagations per call)",
                    l2="34 MB field + 34 MB workspace (L2-resident); no flush",
                    metric="propagations/sec inside cwo_gs (ASM propagator, 41 per call)")
    cfg = W.CONFIGS["c5"]
    a_src, a_dst, phi0 = _gs_inputs_c5(W)
    d_src, d_dst = torch.from_numpy(a_src).cuda(), torch.from_numpy(a_dst).cuda()
    d_phi0 = torch.from_numpy(phi0).cuda()
    d_phi = torch.empty_like(d_phi0)
    plan = api.cwo_plan(N, N, cfg.pitch, cfg.lam)
    plan.ensure_workspace(api.CWO_OP_GS)

    def step(i):
        d_phi.copy_(d_phi0)
        api.cwo_gs(plan, d_src, d_dst, cfg.zs[0], cfg.iters, d_phi)

    def e2e():
        pins = [torch.from_numpy(x).pin_memory() for x in (a_src, a_dst, phi0)]
        pin_out = torch.empty((N, N), dtype=torch.float32).pin_memory()

        def f(i):
            d_src.copy_(pins[0], non_blocking=True); d_dst.copy_(pins[1], non_blocking=True)
            d_phi.copy_(pins[2], non_blocking=True)
            api.cwo_gs(plan, d_src, d_dst, cfg.zs[0], cfg.iters, d_phi)
            pin_out.copy_(d_phi, non_blocking=True)
        return f, 12 * n2, 4 * n2
    props = 2 * cfg.iters + 1
    # separable form: 2 iters + 2 convolution passes (2 iters of them fuse two convolutions and read one amplitude:
    # 8 rd + 4 rd + 8 wr) and 2 iters + 1 field transposes (+ 2 real ones)
    scheme = (2 * cfg.iters) * (20 + 16) * n2 + (16 + 16 + 12 + 16 + 8 + 8) * n2
    return dict(plan=plan, step=step, N=N, props_per_step=props, bytes_per_step=cfg.iters * 168 * n2 + 84 * n2,
                kind_bytes={0: 24 * n2, 3: 32 * n2, 1: 28 * n2, 5: 20 * n2, 6: 16 * n2},
                kind_flops={5: 2 * N * (20.0 * N * np.log2(N) + 30.0 * N)}, scheme_bytes_per_step=scheme, e2e=e2e,
                desc="c5: Gerchberg-Saxton, 8192x8192, Fresnel convolution forward/back, lambda 532 nm, pitch 3.74 um, z 0.3 m, "
                     "20 iterations (41 propagations per call)",
                l2="537 MB field + 1074 MB workspace per propagation (>> 126 MB L2); no flush",
                metric="propagations/sec inside cwo_gs (c5, 41 per call); effective HBM GB/s for 168 N^2 bytes per iteration")


KIND_NAMES = {0: "pass_R (row FFT)", 1: "pass_R' (row IFFT)", 2: "pass_C0 (column FFT)",
              3: "pass_C (fused column FFT*H*IFFT)", 4: "pass_C' (H * column IFFT)",
              5: "line convolution pass (FFT*C*IFFT per line, separable Fresnel)", 6: "transpose",
              7: "line transform pass (pre * FFT * post per line, Fourier-form Fresnel)", 10: "point-light-source CGH (Eq.(23))"}
KIND_KEYS = {0: "pass_R", 1: "pass_Rinv", 2: "pass_C0", 3: "pass_C", 4: "pass_Cmidinv", 5: "lineconv", 6: "transpose",
             7: "linefft", 10: "pls"}


def _roofline(wl, tm, workload):
    """The roofline object of the dominant kernel from the library-recorded per-launch times `tm` ([(tag, ms), ...])."""
    per_kind = {}
    for tag, t_ms in tm:
        per_kind.setdefault(tag & 15, []).append(t_ms)
    names = KIND_NAMES
    passes = {names[k]: float(np.mean(v)) for k, v in per_kind.items() if k in names}
    dom_kind = max(per_kind, key=lambda k: np.sum(per_kind[k]))
    dom_ms = float(np.mean(per_kind[dom_kind]))
    peak, peak_src = _peak()
    tot = sum(float(np.sum(v)) for v in per_kind.values())
    alg_bytes = wl["kind_bytes"][dom_kind]         # algorithmic bytes one launch of that pass moves
    hbm_gbs = alg_bytes / (dom_ms * 1e-3) / 1e9
    traffic = _ncu_traffic(workload, KIND_KEYS.get(dom_kind, "-"))
    common = {"kernel": names[dom_kind], "traffic": traffic,
              "traffic_source": "profiles/traffic.csv (committed ncu --set full capture; not measured by this run)" if traffic else None,
              "algorithmic_bytes_per_launch": alg_bytes, "kernel_ms": dom_ms, "pass_ms": passes,
              "step_share": float(np.sum(per_kind[dom_kind])) / tot,
              "hbm_gbs": hbm_gbs, "hbm_frac": hbm_gbs / peak, "hbm_peak": peak, "hbm_peak_source": peak_src}
    if dom_kind in wl.get("kind_flops", {}):
        # the line-convolution passes are bound by the fp32 pipes, not by HBM: nominal flops per launch
        # over the live duration against 148 SMs x 128 lanes x 2 x 1965 MHz
        fl = wl["kind_flops"][dom_kind]
        ach = fl / (dom_ms * 1e-3) / 1e12
        return dict(common, bound="alu", achieved=ach, peak=FP32_PEAK_TFLOPS, unit="TFLOP/s", frac=ach / FP32_PEAK_TFLOPS,
                    peak_source="148 SMs x 128 fp32 lanes x 2 flop x 1.965 GHz (B200_PROFILING.md unit counts and clocks)",
                    nominal_flops_per_launch=fl)
    return dict(common, bound="hbm", achieved=hbm_gbs, peak=peak, unit="GB/s", frac=hbm_gbs / peak, peak_source=peak_src)


# the other sizes north_star's target names (time at 60 % of 8 TB/s for the algorithmic bytes), timed
# briefly after the headline so that the driver's one JSON line carries them: (workload, timed steps, target ms per call)
EXTRA_WORKLOADS = (("asm8192", 30, 0.671), ("fresnel4096", 40, 0.280), ("fresnel8192", 15, 1.118), ("c4", 6, 1.818),
                   ("c5", 2, 48.0))


def time_extra(name, steps, target_ms, local, torch, api, W):
    """One extra workload, device-resident, CUDA events on the launching stream: a compact record for the `extra` object."""
    wl = make_workload(name, 0, torch, api, W, nbuf=1)
    plan, step = wl["plan"], wl["step"]
    stream = torch.cuda.current_stream()
    sampler = ClockSampler(local)
    sampler.start()
    for i in range(3):
        step(i)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for i in range(steps):
        step(i)
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    plan.set_timing(True)
    for i in range(6 if wl["props_per_step"] == 1 else 1):
        step(i)
    tm = plan.timings(65536)
    plan.set_timing(False)
    t_end, i = time.time() + 1.5, 0
    while len(sampler.rows) < 4 and time.time() < t_end and sampler.proc is not None:
        step(i); i += 1
        torch.cuda.synchronize()
    clocks = sampler.stop()
    r = _roofline(wl, tm, name)
    peak, _ = _peak()
    eff = wl["bytes_per_step"] / (ms * 1e-3) / 1e9
    rec = {"workload": wl["desc"], "steps": steps, "warmup": 3, "ms_per_call": ms, "target_ms_per_call": target_ms,
           "value": wl["props_per_step"] / (ms * 1e-3), "unit": "propagations/s" if name != "c4" else "planes/s",
           "bytes_per_call": int(wl["bytes_per_step"]), "effective_gbs": eff, "pct_of_8TBs": 100.0 * eff / NOMINAL_HBM_GBS,
           "pct_of_measured_copy": 100.0 * eff / peak,
           "roofline": {k: r[k] for k in ("kernel", "bound", "achieved", "peak", "unit", "frac", "kernel_ms", "step_share")},
           "clocks": clocks}
    del wl, plan, step
    torch.cuda.empty_cache()
    return rec


# ------------------------------------------------------------------------------------------------------
# the CUDA arm
# ------------------------------------------------------------------------------------------------------

def run_cuda(args):
    import torch
    from paper_1107_5578_b200 import api, sharding as S, workloads as W

    rank, world, local = _dist()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    use_dist = world > 1
    if use_dist:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if use_dist:
            dist.barrier()
        torch.cuda.synchronize()

    wl = make_workload(args.workload, rank, torch, api, W)
    plan, step, N = wl["plan"], wl["step"], wl["N"]
    if args.no_pipeline:
        plan.set_option(api.CWO_OPT_PIPELINE, 0)
    if args.fresnel_2d:
        plan.set_fresnel_2d(True)
    NBUF = 3
    stream = torch.cuda.current_stream()

    # ---- device-resident timing -----------------------------------------------------------------
    # clocks are sampled every 20 ms from the warm-up to the end of the per-kernel timing below: the timed region
    # proper lasts only ~60 ms at the default step count, the GPU is under the same load throughout
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    for i in range(max(args.warmup, 3)):
        step(i)
    barrier()
    l0 = plan.launch_count
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    marks = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    barrier()
    e0.record(stream)
    marks[0].record(stream)
    for i in range(args.steps):
        step(i)
        marks[i + 1].record(stream)      # per-step times (median); the bracket e0..e1 gives the mean the value uses
    e1.record(stream)
    barrier()
    ms = e0.elapsed_time(e1)
    step_ms = [marks[i].elapsed_time(marks[i + 1]) for i in range(args.steps)]
    launches = plan.launch_count - l0
    ms = S.max_over_ranks(ms, device="cuda")
    value = S.whole_job_rate([args.steps * wl["props_per_step"]] * world, ms)

    # ---- launch-bound workloads: the same steps replayed from a CUDA graph (no Python / launch overhead) ----
    graph_ms = None
    if N <= 1024 and not use_dist:
        try:
            gs = torch.cuda.Stream()
            gs.wait_stream(stream)
            with torch.cuda.stream(gs):
                step(0); gs.synchronize()
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g, stream=gs):
                    for i in range(20):
                        step(i)
                g.replay()
                g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                g0.record(gs)
                for _ in range(10):
                    g.replay()
                g1.record(gs); gs.synchronize()
                graph_ms = g0.elapsed_time(g1) / 200.0
            stream.wait_stream(gs)
        except Exception:
            graph_ms = None
        torch.cuda.synchronize()

    # ---- per-kernel durations (library-recorded CUDA events on the same stream) -------------------
    plan.set_timing(True)
    reps = min(max(args.steps, 6), 60) if wl["props_per_step"] == 1 else 2
    for i in range(reps):
        step(i)
    tm = plan.timings(65536)
    plan.set_timing(False)
    if rank == 0:
        # nvidia-smi needs ~0.1-0.3 s to deliver its first sample: a short run (the driver's 20 steps last 4 ms) keeps the
        # GPU under the same load, untimed, until a few samples are in
        t_end = time.time() + 2.0
        i = 0
        while len(sampler.rows) < 5 and time.time() < t_end and sampler.proc is not None:
            step(i); i += 1
            if i % 16 == 0:
                torch.cuda.synchronize()
        torch.cuda.synchronize()
    clocks = sampler.stop() if rank == 0 else None
    roofline = _roofline(wl, tm, args.workload)

    # ---- end to end: host (pinned) buffers, H2D + propagate + D2H every step -----------------------
    e2e_step, h2d, d2h = wl["e2e"]()

    e2e_steps = max(3, min(args.steps, 20))
    for i in range(3):
        e2e_step(i)
    if hasattr(e2e_step, "end"):
        e2e_step.end(stream)
    barrier()
    e0.record(stream)
    if hasattr(e2e_step, "begin"):
        e2e_step.begin(stream)                      # side streams start after e0 ...
    for i in range(e2e_steps):
        e2e_step(i)
    if hasattr(e2e_step, "end"):
        e2e_step.end(stream)                        # ... and e1 is recorded after all of them
    e1.record(stream)
    barrier()
    ms_e2e = e0.elapsed_time(e1)
    ms_e2e = S.max_over_ranks(ms_e2e, device="cuda")
    e2e = {"value": S.whole_job_rate([e2e_steps * wl["props_per_step"]] * world, ms_e2e), "unit": UNIT, "steps": e2e_steps,
           "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h)}

    if rank == 0:
        peak, _ = _peak()
        ms_step = ms / args.steps
        eff = wl["bytes_per_step"] / (ms_step * 1e-3) / 1e9
        line = {"metric": METRIC if args.workload == "c3" else wl["metric"], "value": value, "unit": UNIT, "n_gpus": world,
                "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_step,
                "ms_per_step_median": float(np.median(step_ms)), "ms_per_step_min": float(np.min(step_ms)),
                "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": wl["desc"], "l2": wl["l2"],
                           "parallelism": "replicas" if world > 1 else "single GPU",
                           "bytes_per_step": int(wl["bytes_per_step"]), "propagations_per_step": wl["props_per_step"]},
                "effective_gbs": eff, "pct_of_8TBs": 100.0 * eff / NOMINAL_HBM_GBS, "pct_of_measured_copy": 100.0 * eff / peak,
                "scheme_bytes_per_step": int(wl["scheme_bytes_per_step"]),
                "roofline": roofline, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks}
        if graph_ms is not None:
            line["ms_per_step_cuda_graph"] = graph_ms       # the step is launch-bound through the Python binding
        if args.fresnel_2d or args.no_pipeline:
            line["not_a_benchmark"] = "fresnel_2d=%d no_pipeline=%d" % (int(args.fresnel_2d), int(args.no_pipeline))
        if world == 1 and not args.no_extra and args.workload == "c3":
            # the headline's buffers are no longer needed: release them before the 8192^2 workloads allocate theirs
            del wl, plan, step, e2e_step
            torch.cuda.empty_cache()
            line["extra"] = {}
            for name, k, target in EXTRA_WORKLOADS:
                try:
                    line["extra"][name] = time_extra(name, k, target, local, torch, api, W)
                except Exception as ex:       # the headline must still be printed
                    line["extra"][name] = {"error": repr(ex)}
        if world == 1 and not args.no_cpu_baseline and args.workload == "c3":
            line["cpu_baseline"] = cpu_baseline(W.CONFIGS["c3"], per_config=not args.no_extra)
        print(json.dumps(line), flush=True)
    if use_dist:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None, help="default: 300 for c3, fewer for the long workloads")
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra", action="store_true",
                    help="skip the `extra` legs (asm8192, fresnel4096, fresnel8192, c4, c5 timed briefly after c3) and the "
                         "per-config / one-thread oracle timings (profiling runs)")
    ap.add_argument("--no-pipeline", action="store_true",
                    help="CWO_OPT_PIPELINE = 0: one CTA per tile everywhere (comparison runs only)")
    ap.add_argument("--fresnel-2d", action="store_true",
                    help="cwo_debug_set_fresnel_2d: three-pass two-dimensional Fresnel form (comparison runs only)")
    ap.add_argument("--workload", default="c3", choices=sorted(WORKLOADS),
                    help="c3 (default) is the headline; the others are extra measurements of the same calls")
    args = ap.parse_args()
    if args.steps is None:
        args.steps = {"c5": 3, "gs_asm2048": 10, "c4": 20, "c4_intensity": 20, "fresnel8192": 50, "asm8192": 100, "asm16384": 10, "pls2048": 20}.get(args.workload, 300)
    if args.impl == "reference":
        run_reference(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
