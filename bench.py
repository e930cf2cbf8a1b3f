#!/usr/bin/env python
"""bench.py -- throughput of the TVB-AdEx sweep hot path on B200 (BASELINE.json metric:
simulated region-steps/s = sims x regions x steps / s, and % of the binding roofline).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl tvbx|reference] [--config 2]

One "step" = one pass of the whole hot path over one batch of synthetic input: the full sweep of the
chosen BASELINE.json config (default configs[1]: 1,024 simulations x 68 regions x 50,000 Euler steps,
noise on, 1-ms downsample, 1 s discarded) integrated from t = 0 and reduced to mean rates + FC.
  value  : device-resident -- connectome, tables and state already in HBM; the timed region is
           reset -> tvbx_run -> tvbx_fc_readout (device buffers), K times, CUDA events.
  per_config : the same measurement (value, e2e, ms_per_step, kernel ms, its own roofline) for the other four
           BASELINE.json configs at their full sizes, with a fixed small number of repeats each.
  e2e    : the same through the C ABI from HOST buffers: tvbx_create_connectome + tvbx_sweep_create
           (host W, L, axes) -> tvbx_run -> tvbx_fc_readout into pinned host arrays -> destroy.
  roofline / cpu_baseline : see DESIGN.md section 7.
N > 1 (torchrun): simulations are independent, so every rank runs its own replica of the sweep
(noise seed + rank) with no data-path collective; value = all ranks' region-steps / max time (weak).
`--impl reference` times the FP64 CPU oracle (oracle/) on a bounded sample of the same workload.
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

METRIC = "simulated region-steps/s (sims x regions x steps / s)"
UNIT = "region-steps/s"

# DESIGN.md section 7 (frozen there, not re-derived from the binary): algorithmic FP32 floating-point operations of one
# region-step = both closed-form transfer functions with first and second derivatives + Eqs. (1)-(3) + OU / Box-Muller
# share = 757 (115 packed FMA x 4 + 111 packed MUL x 2 + 23 packed ADD x 2 + 8 FMA x 2 + 10 MUL/ADD + 3), plus 2 flops
# per non-zero edge of the coupling sum; FP32 peak of the chip: 148 SMs x 128 lanes x 2 flop x sm_max_mhz.
KERNEL_FLOPS_BASE = 757.0
FLOPS_PER_EDGE = 2.0
SM_COUNT, LANES_PER_SM = 148, 128
# ncu --set full captures of the integrator, committed as text under profiles/ (each names its command).  bench.py
# PARSES them at run time (DRAM bytes, L2 -> SM bytes, pipe counters of the captured launch) and records path + sha256,
# so a stale profile is visible in the line instead of hiding behind typed-in constants.  First existing file wins.
PROFILES = {
    1: ["profiles/r2_integrate2_kernel_cfg1_ncu.txt"],
    2: ["profiles/r2_integrate2_kernel_cfg2_ncu.txt", "profiles/r1_integrate2_kernel_cfg2_ncu.txt"],
    3: ["profiles/r2_integrate2_kernel_cfg3_ncu.txt"],
    4: ["profiles/r2_integrate2_kernel_cfg4_ncu.txt", "profiles/r1_integrate2_kernel_cfg4_small_ncu.txt"],
    5: ["profiles/r2_integrate2_kernel_cfg5_ncu.txt", "profiles/r1_integrate2_kernel_cfg5_cluster_ncu.txt"],
}
NCU_KEYS = ("sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active", "smsp__issue_active.avg.pct_of_peak_sustained_active",
            "sm__throughput.avg.pct_of_peak_sustained_elapsed", "lts__t_sector_hit_rate.pct",
            "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed", "sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active",
            "smsp__average_warps_issue_stalled_long_scoreboard_per_issue_active.ratio", "launch__registers_per_thread")
_UNIT = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}


def read_profile(cfg_id):
    """Parse the committed ncu raw-page extract of this config's integrator capture -> dict or None."""
    import hashlib
    import re
    for rel in PROFILES.get(cfg_id, []):
        path = os.path.join(ROOT, rel)
        if not os.path.exists(path):
            continue
        txt = open(path).read()
        m = re.search(r"=\s*([0-9.]+e[+-]?[0-9]+|[0-9.]+)\s*region-steps", txt)
        if not m:
            continue
        units = float(m.group(1))
        vals = {}
        for line in txt.splitlines():
            parts = line.split()
            if len(parts) >= 2 and re.match(r"^[a-z0-9_]+__", parts[0]):
                try:
                    vals[parts[0]] = (float(parts[1].replace(",", "")), parts[2] if len(parts) > 2 else "")
                except ValueError:
                    pass

        def nbytes(key):
            if key not in vals:
                return None
            v, u = vals[key]
            return v * _UNIT.get(u, 1.0)

        rd, wr, l2 = nbytes("dram__bytes_read.sum"), nbytes("dram__bytes_write.sum"), nbytes("l1tex__m_xbar2l1tex_read_bytes.sum")
        return {"source": rel, "sha256_16": hashlib.sha256(txt.encode()).hexdigest()[:16], "captured_region_steps": units,
                "dram_bytes_per_region_step": (rd + wr) / units if rd is not None and wr is not None else None,
                "l2_to_sm_bytes_per_region_step": l2 / units if l2 is not None else None,
                "counters": {k: vals[k][0] for k in NCU_KEYS if k in vals}}
    return None


class Probes:
    """bench_probes.cu: measurement-only micro-benchmarks (L2 / HBM read bandwidth, FP32-lane throughput of the
    instruction forms the integrator is made of), built here into bench_probes.so -- not part of libtvbx.so."""

    KINDS = ("ffma2_3reg", "ffma2_bcast", "fmul2", "fadd2", "ffma", "mufu_rcp")

    @staticmethod
    def build():
        src, so = os.path.join(ROOT, "bench_probes.cu"), os.path.join(ROOT, "bench_probes.so")
        if not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(src):
            subprocess.check_call(["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-shared",
                                   "-Xcompiler", "-fPIC", "-o", so, src])
        return so

    def __init__(self):
        import ctypes as C
        self.C, self.L = C, C.CDLL(self.build())
        self.L.probe_read_bandwidth.argtypes = [C.c_longlong, C.c_int, C.POINTER(C.c_double)]
        self.L.probe_alu.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_double)]

    def read_bandwidth(self, nbytes, passes=20):
        out = self.C.c_double()
        rc = self.L.probe_read_bandwidth(int(nbytes), int(passes), self.C.byref(out))
        if rc != 0:
            raise RuntimeError(f"probe_read_bandwidth rc={rc}")
        return out.value

    def alu_lanes_per_clk_per_sm(self, sm_mhz, iters=400):
        res = {}
        for kind, name in enumerate(self.KINDS):
            out = self.C.c_double()
            rc = self.L.probe_alu(kind, int(iters), self.C.byref(out))
            if rc != 0:
                raise RuntimeError(f"probe_alu({name}) rc={rc}")
            res[name] = out.value / (SM_COUNT * sm_mhz * 1e6)
        return res


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return d, "measured"
    return dict(hbm_gbs=6650.0, bf16_tflops=1590.0, sm_max_mhz=1965.0), "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "100"], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=max(mx) if mx else None,
                    reasons=sorted(reasons), samples=len(sm))


def workload(cfg_id):
    cfg = wl.config(cfg_id)
    W, L = wl.config_connectome(cfg)
    S = int(np.prod([a["n"] for a in cfg["axes"]]))
    return cfg, W, L, S


def config_dict(cfg_id, cfg, S, extra=None):
    d = {"workload": f"BASELINE.json configs[{cfg_id - 1}] ({cfg['name']}): {S} sims x {cfg['n']} regions x "
                     f"{cfg['steps']} steps, dt {cfg['dt']} ms, noise on (seed {cfg['seed']}), ds {cfg['ds']}, "
                     f"discard {cfg['discard_steps']} steps, outputs mean_E/mean_I/FC",
         "sims": S, "regions": cfg["n"], "steps_per_sim": cfg["steps"],
         "l2": "working set (history ring + 1-ms sample chunks) larger than the 126 MB L2; ring and accumulators re-initialised every step"}
    if extra:
        d.update(extra)
    return d


# ------------------------------------------------------------------------------------------------
def run_reference(args):
    """--impl reference: the FP64 oracle as it stands, on the host cores, on a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oracle as orc
    cfg, W, L, S = workload(args.config)
    cores = orc.max_threads()
    n_s = min(S, max(1, cores))
    sims = [int(x) for x in np.linspace(0, S - 1, n_s).round()]
    steps = args.ref_steps
    P = wl.grid_params(cfg, sims=sims)
    times = []
    for it in range(args.warmup + args.steps):
        o = orc.OracleSweep(W, L, P, seed=cfg["seed"], ext_ids=sims)
        t0 = time.perf_counter()
        o.run(steps, cfg["dt"], noise_on=True, ds=cfg["ds"], discard_steps=0)
        o.fc_readout()
        t1 = time.perf_counter()
        o.close()
        if it >= args.warmup:
            times.append(t1 - t0)
    total = sum(times)
    value = n_s * cfg["n"] * steps * len(times) / total
    sample = f"{n_s} sims (stratified over the grid) x {cfg['n']} regions x {steps} steps per step, FP64, OpenMP over sims"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * total / len(times), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(args.config, cfg, S, {"reference_sample": sample}),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def cpu_baseline(cfg_id):
    """The oracle as it stands on the host cores, on a bounded sample of the workload (~15 s)."""
    from oracle import oracle as orc
    cfg, W, L, S = workload(cfg_id)
    cores = orc.max_threads()
    N = cfg["n"]

    def strat(n_s):
        return [int(x) for x in np.linspace(0, S - 1, n_s).round()]

    n_s = int(min(S, 4 * cores))
    sims = strat(n_s)
    o = orc.OracleSweep(W, L, wl.grid_params(cfg, sims=sims), seed=cfg["seed"], ext_ids=sims)
    steps, piece, dt = 0, 2000, 0.0
    t0 = time.perf_counter()
    while steps < cfg["steps"] and dt < 12.0:        # time-boxed: ~12-20 s of CPU work
        take = min(piece, cfg["steps"] - steps)
        o.run(take, cfg["dt"], noise_on=True, ds=cfg["ds"], discard_steps=0)
        steps += take
        dt = time.perf_counter() - t0
    o.fc_readout()
    dt = time.perf_counter() - t0
    return {"value": n_s * N * steps / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{n_s} sims (stratified over the grid) x {N} regions x {steps} steps, FP64, "
                      f"OpenMP over sims, {dt:.1f} s"}


# ------------------------------------------------------------------------------------------------
def measure_config(tvbx, torch, dist, cfg_id, steps, warmup, e2e_steps, sim_steps, rank, world, local, stream, pk, probes, clocks=None,
                   sim_slice=None):
    """One config: device-resident arm (value), end-to-end arm through the C ABI from host buffers (e2e), roofline.
    Returns a dict (rank 0 uses it)."""
    cfg, W, L, S = workload(cfg_id)
    sim_ids = None
    if sim_slice:                                # profiling runs only: every STEP-th simulation from START (cfg 3: one speed class)
        start, stride = (int(x) for x in sim_slice.split(":"))
        sim_ids = list(range(start, S, stride))
        S = len(sim_ids)
    N, steps_sim = cfg["n"], (sim_steps or cfg["steps"])
    if steps_sim != cfg["steps"]:                # profiling runs only: keep the discard proportionate
        cfg["discard_steps"] = min(cfg["discard_steps"], (steps_sim // 5) // cfg["ds"] * cfg["ds"])
    seed = cfg["seed"] + rank                    # replica r of the sweep: same grid, its own noise

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def maxr(x):
        t = torch.tensor([x], device="cuda", dtype=torch.float64)
        if world > 1:
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    # ---- device-resident arm --------------------------------------------------------------------
    conn, sw = tvbx.sweep_from_config(cfg, W, L, seed=seed, sim_ids=sim_ids)
    fc = torch.empty((S, N, N), device="cuda", dtype=torch.float32)
    me = torch.empty((S, N), device="cuda", dtype=torch.float32)
    mi = torch.empty((S, N), device="cuda", dtype=torch.float32)

    def one_step():
        sw.reset(stream)
        sw.run(steps_sim, cfg["dt"], noise_on=True, ds=cfg["ds"], discard_steps=cfg["discard_steps"], stream=stream)
        sw.fc_readout(device=True, stream=stream, out=(fc, me, mi))

    sw.run(1, cfg["dt"], noise_on=True, ds=cfg["ds"], discard_steps=cfg["discard_steps"], stream=stream)   # allocate
    for _ in range(warmup):
        one_step()
    barrier()
    sw.profile_enable(os.environ.get("TVBX_BENCH_NOPROF") is None)
    sw.profile_read()
    l0 = sw.launch_count()
    if clocks is not None:
        clocks.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    with torch.cuda.stream(stream):
        e0.record(stream)
        for _ in range(steps):
            one_step()
        e1.record(stream)
    stream.synchronize()
    barrier()
    ms = e0.elapsed_time(e1)
    clk = clocks.stop() if clocks is not None else None
    launches = sw.launch_count() - l0
    prof = sw.profile_read()
    sw.profile_enable(False)
    info = sw.launch_info()
    ms_max = maxr(ms)
    units_per_step = S * N * steps_sim
    value = world * units_per_step * steps / (ms_max * 1e-3)
    finite = bool(torch.isfinite(fc).all().item() and torch.isfinite(me).all().item())
    rec = {"cfg": cfg_id, "value": value, "unit": UNIT, "steps": steps, "warmup": warmup, "ms_per_step": ms_max / steps,
           "gpu_launches": int(launches), "config": config_dict(cfg_id, cfg, S, {"launch": info, "sim_steps": steps_sim,
                                                                                "replicas": world, "results_finite": finite}),
           "clocks": clk}

    # ---- f3 (not part of the step): FCSC / mean FC per simulation from the resident accumulators ----
    sw.fc_scores(device=True, stream=stream)
    stream.synchronize()
    sw.profile_enable(True)
    sw.profile_read()
    s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    per_call = []
    for _ in range(3):
        s0.record(stream)
        sw.fc_scores(device=True, stream=stream)
        s1.record(stream)
        stream.synchronize()
        per_call.append(s0.elapsed_time(s1))
    scores_ms = sorted(per_call)[len(per_call) // 2]
    sprof = sw.profile_read()
    sw.profile_enable(False)
    scores_kernel_ms = sprof["readout"][0] / max(sprof["readout"][1], 1)      # fc_scores_kernel alone
    scores_bytes = S * N * N * 8.0          # the FP64 co-moments, read once
    kname = sw.kernel_name()
    sw.close(); conn.close()
    del fc, me, mi

    # ---- end-to-end arm: host buffers through the C ABI ---------------------------------------------
    hfc = torch.empty((S, N, N), dtype=torch.float32).pin_memory().numpy()
    hme = torch.empty((S, N), dtype=torch.float32).pin_memory().numpy()
    hmi = torch.empty((S, N), dtype=torch.float32).pin_memory().numpy()
    h2d = d2h = 0
    e2e_phases = []

    def e2e_step():
        nonlocal h2d, d2h
        ta = time.perf_counter()
        c2, s2 = tvbx.sweep_from_config(cfg, W, L, seed=seed, sim_ids=sim_ids)
        tb = time.perf_counter()
        s2.run(steps_sim, cfg["dt"], noise_on=True, ds=cfg["ds"], discard_steps=cfg["discard_steps"], stream=stream)
        tc = time.perf_counter()
        s2.fc_readout(device=False, stream=stream, out=(hfc, hme, hmi))
        td = time.perf_counter()
        h2d, d2h = s2.bytes_copied()
        s2.close(); c2.close()
        te = time.perf_counter()
        e2e_phases.append([round(1e3 * x, 2) for x in (tb - ta, tc - tb, td - tc, te - td)])

    e2e_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        e2e_step()
    torch.cuda.synchronize()
    e2e_s = maxr(time.perf_counter() - t0)
    rec["e2e"] = {"value": world * units_per_step * e2e_steps / e2e_s, "unit": UNIT, "steps": e2e_steps,
                  "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                  "phases_ms": {"order": ["create", "run_enqueue", "readout_sync", "destroy"], "steps": e2e_phases[1:]}}
    del hfc, hme, hmi
    tvbx.trim_memory()

    # ---- roofline of the dominant kernel (the integrator) ----------------------------------------------
    if rank == 0:
        nnz_row = float((W != 0).sum()) / N
        flops_unit = KERNEL_FLOPS_BASE + FLOPS_PER_EDGE * nnz_row
        alg_bytes = 4.0 * nnz_row + 4.0 + 4.0 / cfg["ds"]        # gathered ring values + ring write + 1-ms sample
        int_ms, int_n = prof["integrate"]
        clk_mhz = pk.get("sm_max_mhz", 1965.0)
        peak_tflops = SM_COUNT * LANES_PER_SM * 2 * clk_mhz * 1e6 / 1e12
        achieved = flops_unit * units_per_step * steps / (int_ms * 1e-3) / 1e12 if int_ms > 0 else None
        ncu = read_profile(cfg_id)
        per_launch_units = units_per_step * steps / max(int_n, 1)
        roof = {"bound": "alu", "kernel": kname, "achieved": achieved, "peak": peak_tflops, "unit": "TFLOP/s",
                "frac": (achieved / peak_tflops) if achieved else None,
                "peak_kind": f"nominal: 148 SMs x 128 FP32 lanes x 2 x sm_max_mhz ({pk['_kind']} clock)",
                "flops_per_region_step": flops_unit, "algorithmic_bytes_per_region_step": alg_bytes,
                "kernel_ms_per_launch": int_ms / max(int_n, 1), "kernel_launches": int_n,
                "kernel_share_of_step": int_ms / ms if ms > 0 else None,
                "other_kernels_ms": {k: prof[k][0] for k in ("fc", "readout", "reset")},
                "traffic": (ncu["dram_bytes_per_region_step"] * per_launch_units
                            if ncu and ncu["dram_bytes_per_region_step"] is not None else None),
                "traffic_note": "DRAM bytes per launch = (dram__bytes_read.sum + dram__bytes_write.sum) / region-steps of the ncu "
                                "capture parsed from `ncu.source`, x region-steps of one bench launch",
                "ncu": ncu, "hbm_peak_gbs": pk.get("hbm_gbs")}
        if probes is not None:
            alu = probes["alu"]
            # the measured ceiling of register-operand packed FMA code on this box (FFMA2, three register pairs)
            peak_meas = SM_COUNT * alu["ffma2_3reg"] * 2 * clk_mhz * 1e6 / 1e12
            roof.update({"peak_measured": peak_meas, "frac_measured": (achieved / peak_meas) if achieved else None,
                         "peak_measured_kind": "bench_probes.cu FFMA2 chain, three distinct register-pair operands, lanes/clk/SM x 148 x 2 x clock",
                         "alu_lanes_per_clk_per_sm_measured": alu, "l2_peak_gbs_measured": probes["l2_gbs"],
                         "hbm_read_gbs_measured": probes["hbm_read_gbs"]})
            if N > 120 and int_ms > 0:      # N = 360: the delay gather is bound by the L2 -> SM read bandwidth
                gather_gbs = alg_bytes * units_per_step * steps / (int_ms * 1e-3) / 1e9
                roof.update({"bound": "l2", "achieved": gather_gbs, "peak": probes["l2_gbs"], "unit": "GB/s",
                             "frac": gather_gbs / probes["l2_gbs"],
                             "peak_kind": "L2 -> SM read bandwidth measured in this run (bench_probes.cu: 64 MiB buffer, 16-byte ld.global.cg)",
                             "l2_traffic_gbs_ncu": (ncu["l2_to_sm_bytes_per_region_step"] * units_per_step * steps / (int_ms * 1e-3) / 1e9
                                                    if ncu and ncu["l2_to_sm_bytes_per_region_step"] else None),
                             "alu_frac": (achieved / peak_tflops) if achieved else None})
        rec["roofline"] = roof
        rec["fc_scores"] = {"ms": scores_ms, "kernel_ms": scores_kernel_ms,
                            "kernel_achieved_gbs": scores_bytes / (scores_kernel_ms * 1e-3) / 1e9 if scores_kernel_ms > 0 else None,
                            "note": "tvbx_fc_scores (FCSC + mean FC per simulation, P:113), outside the timed step"}
    return rec


def run_tvbx(args):
    import torch
    import torch.distributed as dist
    import paper_2311_13337_b200 as tvbx

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    tvbx.lib()                                   # fails loudly if libtvbx.so is missing
    stream = torch.cuda.Stream()
    pk, pk_kind = peaks()
    pk["_kind"] = pk_kind
    probes = None
    if rank == 0 and not args.no_probes:
        P = Probes()
        probes = {"alu": P.alu_lanes_per_clk_per_sm(pk.get("sm_max_mhz", 1965.0)), "l2_gbs": P.read_bandwidth(64 << 20, 30),
                  "hbm_read_gbs": P.read_bandwidth(4 << 30, 3)}
    clocks = ClockSampler(local) if rank == 0 else None
    head = measure_config(tvbx, torch, dist, args.config, args.steps, args.warmup, args.steps, args.sim_steps, rank, world, local,
                          stream, pk, probes, clocks, args.sim_slice)
    # the other BASELINE.json configs, each its own record (fewer repeats: the 1.5-3 s configs would not fit a default run)
    per_config = {}
    if world == 1 and not args.headline_only and not args.sim_steps and not args.sim_slice:
        plan = {1: (5, 3), 2: (3, 3), 3: (2, 3), 4: (1, 3), 5: (1, 3)}      # cfg -> (timed steps, warm-up steps)
        for cid, (k, w) in plan.items():
            if cid == args.config:
                continue
            r = measure_config(tvbx, torch, dist, cid, k, w, 1, 0, rank, world, local, stream, pk, probes, ClockSampler(local))
            per_config[f"cfg{cid}"] = r
    if rank == 0:
        line = {"metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": head["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32", "data": "synthetic", "config": head["config"], "clocks": head["clocks"], "e2e": head["e2e"],
                "gpu_launches": head["gpu_launches"], "roofline": head["roofline"], "fc_scores": head["fc_scores"]}
        if per_config:
            line["per_config"] = per_config
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(args.config)
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="tvbx", choices=["tvbx", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config number (1-5); the metric is quoted on 2")
    ap.add_argument("--sim-steps", type=int, default=0, help="override the Euler steps per simulation (profiling only)")
    ap.add_argument("--sim-slice", default="", help="START:STEP -- only every STEP-th simulation from START (profiling only; cfg 3: one speed class = i:8)")
    ap.add_argument("--ref-steps", type=int, default=4000, help="Euler steps per oracle sample (--impl reference)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-probes", action="store_true", help="skip the ALU / L2 micro-benchmarks (bench_probes.cu)")
    ap.add_argument("--headline-only", action="store_true", help="only the --config line, no per_config records")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_tvbx(args)


if __name__ == "__main__":
    main()
