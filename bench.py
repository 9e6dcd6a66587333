#!/usr/bin/env python
"""bench.py -- throughput of the short-range PP hot path on B200 (contract: see the round prompt / DESIGN.md).

A "step" is one pass of the whole hot path over one batch of synthetic input:
    srpp_build_mesh (A1-A4)  ->  srpp_accel_kick (A5 force, A6 write-back with the A7 kick fused into it)
on the workload BASELINE.json's target is quoted on: configs[3], the clustered 2^25-particle per-node load
(`--config 4`; configs are numbered 1..5 as in SURVEY.md).  Metric: candidate pair interactions per second,
W / t_step with W = sum_c n_c * sum_{c' in 27-stencil(c)} n_c' (depends on the input only).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl reference]

N > 1 (torchrun): the path has no exchange step (BASELINE.json: one GPU, no sharding) -> N independent
replicas of the same workload, barrier + max-over-ranks timing, value = N * K * W / t.
`--impl reference` times the fp64 CPU oracle (oracle/), as it stands, on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1411_3396_b200 import workloads  # noqa: E402  (input generators only; no arithmetic of the method)

METRIC = "short_range_pair_interactions_per_s"
UNIT = "pairs/s"
FLOP_PER_PAIR = 30.0          # 11 FMA x 2 + 4 add + 3 mul + 1 rsqrt
FP32_LANES_PER_SM = 128       # SMs x 128 lanes x 2 flop x f_max
BIN_BYTES_PER_PARTICLE = 52   # 16 read (ids) + 16 read + 16 write (sorted) + 4 write (perm)


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            return json.load(fh), "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


FORCE_PROFILE = os.path.join("profiles", "r02_force_config4_ncu_full.txt")
FORCE_SOURCE = os.path.join("paper_1411_3396_b200", "csrc", "srpp_force.cu")


def _git_blob_hash(path):
    """git's blob hash of a file (sha1 of 'blob <len>\0' + content), computed without calling git."""
    import hashlib
    with open(path, "rb") as fh:
        data = fh.read()
    return hashlib.sha1(b"blob %d\0" % len(data) + data).hexdigest()


def _profiled_traffic():
    """DRAM bytes per launch of the force kernel from the committed `ncu --set full` summary under profiles/
    (dram__bytes_read.sum + dram__bytes_write.sum; text file, never executed), plus the git blob hash of srpp_force.cu
    the capture was made from (its header line `source-blob: <hash>`) and whether the shipped source still has it."""
    path = os.path.join(ROOT, FORCE_PROFILE)
    unit = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
    total, seen, blob = 0.0, 0, None
    try:
        with open(path) as fh:
            for line in fh:
                if line.startswith("source-blob:"):
                    blob = line.split(":", 1)[1].strip()
                for key in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
                    if line.startswith(key + " ["):
                        u = line.split("[")[1].split("]")[0]
                        total += float(line.split("=")[1]) * unit[u]
                        seen += 1
    except OSError:
        return None, None, None
    cur = _git_blob_hash(os.path.join(ROOT, FORCE_SOURCE))
    return (total if seen == 2 else None), blob, (blob == cur)


# --------------------------------------------------------------------------------------- clocks --
class ClockSampler:
    """Samples SM clock + throttle reasons of one GPU every 200 ms through NVML while the timed region runs."""

    REASONS = (("sw_power_cap", 0x4), ("hw_slowdown", 0x8), ("sw_thermal_slowdown", 0x20),
               ("hw_thermal_slowdown", 0x40), ("hw_power_brake", 0x80))

    def __init__(self, index: int):
        self.samples, self.reasons, self.power = [], set(), []
        self.max_mhz = None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception as exc:  # NVML missing: report that, never invent clocks
            self._nv = None
            self.error = repr(exc)

    def _run(self):
        nv = self._nv
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
                self.power.append(nv.nvmlDeviceGetPowerUsage(self._h) / 1000.0)
                mask = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self._h)) if hasattr(
                    nv, "nvmlDeviceGetCurrentClocksEventReasons") else int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h))
                for name, bit in self.REASONS:
                    if mask & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop.wait(0.2)

    def __enter__(self):
        if self._nv is not None:
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thread is not None:
            self._thread.join()

    def summary(self) -> dict:
        if self._nv is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvml_unavailable"]}
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples), "power_w_max": max(self.power) if self.power else None}


# ------------------------------------------------------------------------------ CPU oracle legs --
def _mesh_candidates(oracle, pos, w):
    """Per-cell chaining-mesh candidate counts of the workload's own mesh (oracle's counting sort)."""
    cs, perm, _ = oracle.build_mesh(pos, w.box, w.ncell)
    nz, ny, nx = w.ncell[2], w.ncell[1], w.ncell[0]
    cnt = np.diff(cs.astype(np.int64)).reshape(nz, ny, nx)
    sten = sum(np.roll(cnt, (dz, dy, dx), axis=(0, 1, 2)) for dz in (-1, 0, 1) for dy in (-1, 0, 1) for dx in (-1, 0, 1))
    return cs, perm, cnt, sten


def _oracle_sample(oracle, pos, w, n_targets, seed):
    """half uniform over particles, half drawn in proportion to candidate count (halo cores).
    Returns (targets, chaining-mesh candidates of those targets)."""
    rng = np.random.default_rng(seed)
    cs, perm, cnt, sten = _mesh_candidates(oracle, pos, w)
    w_cell = (cnt * sten).ravel().astype(np.float64)
    nw = n_targets // 2
    cells = rng.choice(w_cell.size, size=nw, p=w_cell / w_cell.sum())
    k = cs[cells].astype(np.int64) + (rng.random(nw) * np.diff(cs)[cells]).astype(np.int64)
    t = np.concatenate([rng.integers(0, pos.shape[0], n_targets - nw), perm[k].astype(np.int64)])
    # candidates of target i in the WORKLOAD's mesh = stencil sum of its cell
    cid = oracle.cell_ids(pos[t], w.box, w.ncell)
    cand = sten.ravel()[cid].astype(np.int64)
    # the harness logs how many cells hold half of W (the clustered W values are heavy-tail dominated)
    ws = np.sort(w_cell)[::-1]
    _oracle_sample.cells_half_w = int(np.searchsorted(np.cumsum(ws), 0.5 * ws.sum()) + 1)
    return t, cand


def oracle_rate(oracle, pos, w, budget_s: float, seed: int = 0):
    """Marginal rate of the oracle in the bench's unit: (candidates_B - candidates_A) / (t_B - t_A) for two nested
    target samples A < B, which removes the fixed cost of the oracle's own cell-list build (paid once per call and
    amortised over all N targets in a full evaluation).  Sample B is sized from A's timing to fill `budget_s`."""
    prm = oracle.make_params(w.box, w.rcut, w.eps)
    t_all, cand_all = _oracle_sample(oracle, pos, w, 4096, seed)
    order = np.random.default_rng(seed + 1).permutation(t_all.shape[0])
    t_all, cand_all = t_all[order], cand_all[order]
    n_a = 64
    t0 = time.perf_counter()
    oracle.accel(pos, prm, targets=t_all[:8])
    t_fixed = time.perf_counter() - t0                       # ~ the cell-list build
    t0 = time.perf_counter()
    oracle.accel(pos, prm, targets=t_all[:n_a])
    t_a = time.perf_counter() - t0
    per_cand = max(t_a - t_fixed, 1e-4) / max(int(cand_all[:n_a].sum()), 1)
    csum = np.cumsum(cand_all)
    n_b = int(np.searchsorted(csum, budget_s / per_cand)) + 1
    n_b = int(min(max(n_b, 2 * n_a), t_all.shape[0]))
    t0 = time.perf_counter()
    _, st_b = oracle.accel(pos, prm, targets=t_all[:n_b], stats=True)
    t_b = time.perf_counter() - t0
    # in-cutoff share of the candidate pairs, W-weighted: for targets drawn with probability proportional to their
    # candidate count, E[n_in_i / cand_i] = sum_i n_in_i / W exactly (the work-weighted half of the sample)
    wt = order[:n_b] >= (4096 - 4096 // 2)
    frac_in = float(np.mean(st_b["n_in"][wt] / np.maximum(cand_all[:n_b][wt], 1))) if wt.any() else None
    d_c = int(cand_all[:n_b].sum() - cand_all[:n_a].sum())
    rate = d_c / max(t_b - t_a, 1e-9)
    return {"value": rate, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", "in_cutoff_fraction": frac_in,
            "cells_holding_half_of_W": getattr(_oracle_sample, "cells_half_w", None),
            "sample": "%s: %d targets (half uniform, half work-weighted; SURVEY.md 8(d)), %d chaining-mesh candidate "
                      "pairs in %.1f s of fp64 oracle time; marginal rate between nested samples of %d and %d targets "
                      "(fixed cell-list build of %.1f s per call excluded)"
                      % (w.name, n_b, d_c, t_b - t_a, n_a, n_b, t_fixed)}


def run_reference(args, w):
    """--impl reference: the oracle, as it stands, on the host cores; each step = one bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    oracle.build()
    pos = workloads.generate(w)
    prm = oracle.make_params(w.box, w.rcut, w.eps)
    t_all, cand_all = _oracle_sample(oracle, pos, w, 4096, 0)
    order = np.random.default_rng(1).permutation(t_all.shape[0])
    t_all, cand_all = t_all[order], cand_all[order]
    total_budget = args.ref_budget
    t0 = time.perf_counter()
    oracle.accel(pos, prm, targets=t_all[:8])
    t_fixed = time.perf_counter() - t0
    t0 = time.perf_counter()
    oracle.accel(pos, prm, targets=t_all[:64])
    t_a = time.perf_counter() - t0
    per_cand = max(t_a - t_fixed, 1e-4) / max(int(cand_all[:64].sum()), 1)
    per_step = max(total_budget / (args.steps + args.warmup) - t_fixed, 1.0)
    n_s = int(min(max(int(np.searchsorted(np.cumsum(cand_all), per_step / per_cand)) + 1, 16), t_all.shape[0]))
    tgt, cand = t_all[:n_s], int(cand_all[:n_s].sum())
    for _ in range(args.warmup):
        oracle.accel(pos, prm, targets=tgt)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.accel(pos, prm, targets=tgt)
    dt = time.perf_counter() - t0
    value = cand * args.steps / dt
    sample = ("%s: each step = %d targets (half uniform, half work-weighted), %d chaining-mesh candidate pairs; the "
              "oracle's own cell-list build (%.1f s per call) is inside every step" % (w.name, n_s, cand, t_fixed))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "n_particles": w.n, "sample_targets": n_s},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------------- product arm --
def run_product(args, w):
    import torch
    from paper_1411_3396_b200 import binding
    from paper_1411_3396_b200.replicas import Replicas

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the srpp path has no CPU fallback (use --impl reference for the oracle)")
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    rep = Replicas(backend="nccl", device=dev)        # replicas only: barrier + max-over-ranks, no data collective
    world, rank = rep.world, rep.rank

    def barrier():
        rep.barrier()
        torch.cuda.synchronize()

    max_over_ranks = rep.max_over_ranks

    binding.load()                                    # fail loudly if libsrpp.so is missing
    pos = workloads.generate(w)                       # replicas: every rank runs the same workload
    n = pos.shape[0]
    sol = binding.Solver(w.box, w.ncell, w.rcut, w.eps, n_max=n, device=dev)
    sol.set_timing(True)
    d_pos = torch.from_numpy(pos).to(dev)
    d_acc = torch.empty_like(d_pos)
    d_vel = torch.zeros_like(d_pos)
    kdt = w.dt if w.dt else 0.01

    def step():
        sol.build_mesh(d_pos)
        sol.accel_kick(d_vel, kdt, acc=d_acc)       # A5 + A6 + A7: accelerations in the caller's order and v += kdt * a

    for _ in range(args.warmup):
        step()
    stats0 = sol.get_stats()
    W = stats0["candidate_pairs"]
    mesh_ms, accel_ms, force_ms = [], [], []
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    with ClockSampler(local) as clocks:
        ev0.record()
        for _ in range(args.steps):
            step()
            if args.phase_timing:                      # reads events of this step (one extra stream sync per step)
                t = sol.get_timings()
                mesh_ms.append(t["mesh_ms"]); accel_ms.append(t["accel_ms"]); force_ms.append(t["force_ms"])
        ev1.record()
        barrier()
    t_ms = max_over_ranks(ev0.elapsed_time(ev1))
    stats1 = sol.get_stats()
    launches = (stats1["kernel_launches"] - stats0["kernel_launches"])
    value = world * args.steps * W / (t_ms * 1e-3)

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    e2e = None
    if args.e2e_steps > 0:
        h_pos = torch.from_numpy(pos).pin_memory()
        h_vel = torch.zeros((n, 4), dtype=torch.float32).pin_memory()
        h_acc = torch.empty((n, 4), dtype=torch.float32).pin_memory()
        scratch = torch.empty(48 * n, dtype=torch.uint8, device=dev)
        sol.step_host(h_pos, h_vel, h_acc, kdt, scratch)            # warm-up
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            sol.step_host(h_pos, h_vel, h_acc, kdt, scratch)        # synchronises: results are in host memory on return
        barrier()
        e2e_s = max_over_ranks(time.perf_counter() - t0)
        e2e = {"value": world * args.e2e_steps * W / e2e_s, "unit": UNIT, "h2d_bytes_per_step": 2 * 16 * n,
               "d2h_bytes_per_step": 2 * 16 * n, "steps": args.e2e_steps, "ms_per_step": 1e3 * e2e_s / args.e2e_steps,
               "api": "srpp_step_host (pinned host pos/vel in, acc/vel out)"}

    if rank != 0:
        rep.close()
        return

    peaks, peak_kind = _peaks()
    traffic, traffic_blob, traffic_ok = _profiled_traffic()
    props = torch.cuda.get_device_properties(dev)
    sms = props.multi_processor_count
    clk = clocks.summary()
    f_max_hz = 1e6 * float(peaks.get("sm_max_mhz") or clk.get("sm_max_mhz") or 1965.0)
    peak_tflops = sms * FP32_LANES_PER_SM * 2 * f_max_hz / 1e12
    force_avg_ms = float(np.mean(force_ms)) if force_ms else None
    achieved = FLOP_PER_PAIR * W / (force_avg_ms * 1e-3) / 1e12 if force_avg_ms else None
    probe = {"ffma_tflops": sol.probe_fp32(0, 4000) / 1e12, "ffma2_tflops": sol.probe_fp32(1, 4000) / 1e12,
             "ffma2_2_vector_operands_tflops": sol.probe_fp32(2, 4000) / 1e12,
             "ffma2_3_vector_operands_tflops": sol.probe_fp32(3, 4000) / 1e12}
    ncells = w.ncell[0] * w.ncell[1] * w.ncell[2]
    bin_bytes = BIN_BYTES_PER_PARTICLE * n + 8 * ncells
    mesh_avg_ms = float(np.mean(mesh_ms)) if mesh_ms else None
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": t_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": w.name, "baseline_config": "BASELINE.json configs[%d]" % (args.config - 1),
                   "n_particles": n, "box": list(w.box), "ncell": list(w.ncell), "rcut": w.rcut, "eps": w.eps,
                   "candidate_pairs_W": W, "max_cell_count": stats1["max_cell_count"],
                   "step": "build_mesh + accel_kick (force, write-back and kick; same results as accel + kick)", "parallelism": "replicas only (no exchange step)",
                   "l2": "inputs larger than L2 (16 B x N = %d MiB per array)" % (16 * n >> 20)},
        "clocks": clk, "e2e": e2e, "gpu_launches": launches,
        "roofline": {"bound": "alu", "kernel": "k_pp_force", "achieved": achieved, "peak": peak_tflops,
                     "unit": "TFLOP/s", "frac": (achieved / peak_tflops) if achieved else None,
                     "traffic": traffic if args.config == 4 else None,
                     "traffic_kind": "DRAM bytes per launch, ncu --set full capture %s (the kernel is ALU-bound: "
                                     "algorithmic bytes are 2 x 16 B x N + cell tables, re-reads are served by L2)" % FORCE_PROFILE,
                     "traffic_capture_source_blob": traffic_blob, "traffic_capture_matches_shipped_source": traffic_ok,
                     "peak_kind": "nominal: %d SMs x 128 FP32 lanes x 2 flop x %.0f MHz (sm_max_mhz, %s); "
                                  "30 flop per candidate pair" % (sms, f_max_hz / 1e6, peak_kind),
                     "launch_ms": force_avg_ms, "fp32_probe": probe,
                     "frac_of_probe_ffma2": (achieved / probe["ffma2_tflops"]) if achieved else None},
        "phases": {"mesh_ms": mesh_avg_ms, "accel_ms": float(np.mean(accel_ms)) if accel_ms else None,
                   "force_ms": force_avg_ms,
                   "plan_write_back_kick_ms": float(np.mean(accel_ms) - np.mean(force_ms)) if accel_ms else None,
                   "write_back_kick_kind": "accel_ms - force_ms: work plan (4 small kernels) + bucketed write-back with the "
                                           "kick fused in; algorithmic bytes 28 read + 16 written (A6) + 32 (A7) per particle",
                   "accel_pairs_per_s": W / (np.mean(accel_ms) * 1e-3) if accel_ms else None,
                   "binning_gbs": bin_bytes / (mesh_avg_ms * 1e-3) / 1e9 if mesh_avg_ms else None,
                   "binning_frac_of_hbm": (bin_bytes / (mesh_avg_ms * 1e-3) / 1e9 / peaks["hbm_gbs"]) if mesh_avg_ms else None,
                   "hbm_gbs_peak": peaks["hbm_gbs"], "hbm_peak_kind": peak_kind},
    }
    if world == 1 and not args.no_cpu_baseline:
        import oracle                                  # cpu_baseline leg: the one place the product arm may run it
        oracle.build()
        cb = oracle_rate(oracle, pos, w, args.cpu_budget)
        line["cpu_baseline"] = cb
        # oracle binning timed in full; in-cutoff pairs beside candidate pairs; the full-config oracle
        # time as a labelled extrapolation
        t0 = time.perf_counter()
        oracle.build_mesh(pos, w.box, w.ncell)
        line["phases"]["oracle_mesh_ms"] = 1e3 * (time.perf_counter() - t0)
        line["phases"]["oracle_mesh_kind"] = "orc_build_mesh, all %d particles, one host thread (plain counting sort)" % n
        frac = cb.pop("in_cutoff_fraction")
        line["config"]["cells_holding_half_of_W"] = cb.pop("cells_holding_half_of_W")
        line["in_cutoff"] = {"fraction_of_candidates": frac, "pairs_per_s": value * frac,
                             "kind": "mean of n_in_i / candidates_i over the oracle's work-weighted target sample (= sum n_in / W in expectation)"}
        cb["full_config_extrapolated_s"] = W / cb["value"]
        cb["full_config_extrapolated_kind"] = "EXTRAPOLATION: W / marginal oracle rate, not a measured run"
    if world == 1 and not args.no_extras:
        # the sub-cycle call on the headline workload: two sub-steps, velocities drawn so that a few per
        # cent of the particles change cell per sub-step (kdt = 0 keeps them: with G = m = 1 the halo cores would
        # otherwise fly apart, R16); reports the incremental re-bin beside the full build
        g = torch.Generator(device=dev); g.manual_seed(1)
        d_vel.normal_(0.0, 1.0, generator=g)
        d_vel[:, 3] = 0
        x_sub = d_pos.clone()
        dt_sub = 0.2
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        sol.subcycle(x_sub, d_vel, dt_sub, 0.0, 2, acc=d_acc)
        ev1.record()
        torch.cuda.synchronize()
        tt, st_sub = sol.get_timings(), sol.get_stats()
        wb_ms = None
        if accel_ms and force_ms:
            wb_ms = float(np.mean(accel_ms) - np.mean(force_ms))
        line["subcycle"] = {"workload": w.name, "nsub": 2, "dt": dt_sub, "ms_per_substep": ev0.elapsed_time(ev1) / 2,
                            "movers_last_pass": st_sub["last_movers"], "mover_fraction_last_pass": st_sub["last_movers"] / n,
                            "rebins_incremental": st_sub["rebins_incremental"], "rebins_full": st_sub["rebins_full"],
                            "incremental_rebin_ms": tt["rebin_ms"], "full_build_ms": mesh_avg_ms,
                            "rebin_over_full_build": tt["rebin_ms"] / mesh_avg_ms if mesh_avg_ms else None,
                            "fused_kick_stream_ms": tt["kick_stream_ms"],
                            "plan_plus_write_back_ms_of_srpp_accel": wb_ms,
                            "note": "the incremental re-bin carries positions, velocities and perm (36 B per particle read "
                                    "+ 36 B written, plus the movers' own sort and merge); the full build carries positions "
                                    "and perm only.  fused_kick_stream_ms replaces write-back + kick + two streams of the "
                                    "caller-order path"}
        del x_sub
        del d_pos, d_acc, d_vel, sol
        torch.cuda.empty_cache()
        line["other"] = run_extras(args, torch, binding, dev, peak_tflops, peaks)
    print(json.dumps(line), flush=True)
    rep.close()


def run_extras(args, torch, binding, dev, peak_tflops, peaks):
    """Short device-timed passes that are NOT the headline (outside its timed region): BASELINE.json configs 1-3
    (force fraction of FP32 peak, binning GB/s), the sub-cycle call, and srpp_mbp with its own roofline."""
    out = {}
    for cfg, reps in ((1, 20), (2, 10), (3, 1)):
        wc = workloads.CONFIGS[cfg]
        pos = workloads.generate(wc)
        n = pos.shape[0]
        sol = binding.Solver(wc.box, wc.ncell, wc.rcut, wc.eps, n_max=n, device=dev)
        sol.set_timing(True)
        d_pos = torch.from_numpy(pos).to(dev)
        d_acc = torch.empty_like(d_pos)
        sol.build_mesh(d_pos); sol.accel(d_acc)                        # warm-up
        mesh, force, accel = [], [], []
        for _ in range(reps):
            sol.build_mesh(d_pos)
            sol.accel(d_acc)
            t = sol.get_timings()
            mesh.append(t["mesh_ms"]); force.append(t["force_ms"]); accel.append(t["accel_ms"])
        st = sol.get_stats()
        W = st["candidate_pairs"]
        ncells = wc.ncell[0] * wc.ncell[1] * wc.ncell[2]
        fm, mm = float(np.median(force)), float(np.median(mesh))
        rec = {"workload": wc.name, "n_particles": n, "candidate_pairs_W": W, "reps": reps, "force_ms": fm,
               "accel_ms": float(np.median(accel)), "mesh_ms": mm,
               "pairs_per_s_force_kernel": W / (fm * 1e-3),
               "frac_of_fp32_peak": FLOP_PER_PAIR * W / (fm * 1e-3) / 1e12 / peak_tflops,
               "pair_slots_per_candidate_pair": st["pair_slots"] / max(W, 1),
               "binning_gbs": (BIN_BYTES_PER_PARTICLE * n + 8 * ncells) / (mm * 1e-3) / 1e9}
        rec["binning_frac_of_hbm"] = rec["binning_gbs"] / peaks["hbm_gbs"]
        if cfg == 2:   # the sub-cycle call: stream - accel - kick - stream, re-bin included
            d_vel = torch.zeros_like(d_pos)
            ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            sol.subcycle(d_pos, d_vel, 1e-3, 1e-3, 1, acc=d_acc)
            torch.cuda.synchronize()
            ev0.record()
            sol.subcycle(d_pos, d_vel, 1e-3, 1e-3, 4, acc=d_acc)
            ev1.record()
            torch.cuda.synchronize()
            rec["subcycle_ms_per_substep"] = ev0.elapsed_time(ev1) / 4
            del d_vel
        if not args.no_cpu_baseline:
            # oracle binning timed in full at every config; configs 1-2: the oracle evaluated in full
            # (pairs/s = W / t and the exact in-cutoff pair count).  cpu_baseline leg: the one place this arm runs oracle/.
            import oracle
            oracle.build()
            t0 = time.perf_counter()
            oracle.build_mesh(pos, wc.box, wc.ncell)
            rec["oracle_mesh_ms"] = 1e3 * (time.perf_counter() - t0)
            if cfg <= 2:
                t0 = time.perf_counter()
                _, st_o = oracle.accel(pos, oracle.make_params(wc.box, wc.rcut, wc.eps), stats=True)
                t_o = time.perf_counter() - t0
                n_in = int(st_o["n_in"].sum())
                rec["oracle_full"] = {"seconds": t_o, "pairs_per_s": W / t_o, "cores": oracle.num_threads(),
                                      "in_cutoff_pairs": n_in, "in_cutoff_fraction_of_W": n_in / W,
                                      "gpu_in_cutoff_pairs_per_s": n_in / (fm * 1e-3)}
        out["config%d" % cfg] = rec
        del sol, d_pos, d_acc
        torch.cuda.empty_cache()
    # most bound particle (the paper's Thrust version ran 45x faster on K20X than on the CPU; context)
    rng = np.random.default_rng(7)
    sizes = [2_000_000] + [200_000] * 10 + [2000] * 500
    tot = int(sum(sizes))
    hs = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
    p = np.ones((tot, 4), dtype=np.float32)
    p[:, :3] = rng.normal(0, 1.0, (tot, 3)).astype(np.float32) + np.repeat(rng.uniform(10, 500, (len(sizes), 3)), sizes, axis=0).astype(np.float32)
    sol = binding.Solver((512.0,) * 3, (16,) * 3, 3.0, 0.05, n_max=16, device=dev)
    d = torch.from_numpy(p).to(dev)
    sol.mbp(d, hs, want_phi=False)
    torch.cuda.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(3):
        sol.mbp(d, hs, want_phi=False)
    ev1.record()
    torch.cuda.synchronize()
    ms = ev0.elapsed_time(ev1) / 3
    pairs = float(sum(float(k) * float(k) for k in sizes))
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    xu_peak = sms * 16 * 1e6 * float(peaks.get("sm_max_mhz") or 1965.0)       # one MUFU.RSQ per pair, 16 per SM and clock
    out["mbp"] = {"halos": len(sizes), "members": tot, "ordered_pairs": pairs, "ms": ms, "pairs_per_s": pairs / (ms * 1e-3),
                  "roofline": {"bound": "xu", "peak_pairs_per_s": xu_peak, "frac": pairs / (ms * 1e-3) / xu_peak,
                               "peak_kind": "%d SMs x 16 MUFU.RSQ per clock x sm_max_mhz, one rsqrt per pair (DESIGN.md 5.4)" % sms},
                  "paper_context": "PAPER.md:97: the PISTON/Thrust centre finder ran ~45x faster on a K20X than on the CPU"}
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, choices=sorted(workloads.CONFIGS))
    ap.add_argument("--impl", default="srpp", choices=["srpp", "reference"])
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--cpu-budget", type=float, default=15.0, help="seconds of oracle time for cpu_baseline")
    ap.add_argument("--ref-budget", type=float, default=150.0, help="seconds for the whole --impl reference run")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the configs 1-3 / sub-cycle / MBP passes")
    ap.add_argument("--no-phase-timing", dest="phase_timing", action="store_false")
    args = ap.parse_args()
    w = workloads.CONFIGS[args.config]
    if args.impl == "reference":
        run_reference(args, w)
    else:
        run_product(args, w)


if __name__ == "__main__":
    main()
