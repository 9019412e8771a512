#!/usr/bin/env python
"""bench.py -- timesteps/s and pair-interactions/s of the short-range force pipeline on the
1,000,000-bead Kremer-Grest melt (BASELINE.json configs[2], "C3"), one B200 per rank.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--config C3] [--inner 500]

A bench "step" is one gm_step(inner) call: `inner` MD timesteps of the whole hot path (a1..a8 of
SURVEY.md section 8(a): displacement test, device-gated cell binning + Verlet-list rebuild, fused
pair+bond force and velocity-Verlet kernel, and the SFC reorder when it falls due).  The default
inner = 500 is one SFC period of C3, so every step holds the same mix of rebuilds and one reorder.
Prints ONE JSON line (see DESIGN.md "Measurement" for every field).

--impl reference times the fp64 CPU oracle (oracle/, test infrastructure) on the host cores; each
of its steps is ONE MD timestep of the same workload (a bounded sample).  Under torchrun only rank
0 runs it.

Multi-GPU: the path does not shard (single-GPU method, "replicas only"): with
--gpus N every rank steps an independent replica of the same melt; value is the sum over replicas.
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

METRIC = "timesteps/s"
L2_BYTES = 126e6


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler(threading.Thread):
    """SM clock and throttle reasons DURING the timed region (NVML; same fields as the recipe's
    nvidia-smi clocks line)."""
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown",
               0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting"}

    def __init__(self, torch_device):
        super().__init__(daemon=True)
        self.samples, self.reasons, self.max_mhz, self.power = [], set(), None, []
        self._stop_evt = threading.Event()
        self.h = None
        try:
            import pynvml
            import torch
            pynvml.nvmlInit()
            self.nv = pynvml
            try:
                uuid = str(torch.cuda.get_device_properties(torch_device).uuid)
                self.h = pynvml.nvmlDeviceGetHandleByUUID(("GPU-" + uuid) if not uuid.startswith("GPU-") else uuid)
            except Exception:
                vis = os.environ.get("CUDA_VISIBLE_DEVICES")
                idx = torch_device.index or 0
                if vis:
                    idx = int(vis.split(",")[idx])
                self.h = pynvml.nvmlDeviceGetHandleByIndex(idx)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception as e:          # no NVML: the clocks record says so instead of inventing numbers
            self.err = repr(e)
            self.h = None

    def run(self):
        if self.h is None:
            return
        nv = self.nv
        while not self._stop_evt.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)) if hasattr(nv, "nvmlDeviceGetCurrentClocksEventReasons") \
                    else int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for bit, name in self.REASONS.items():
                    if r & bit:
                        self.reasons.add(name)
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
            except Exception:
                pass
            time.sleep(0.02)

    def stop(self) -> dict:
        self._stop_evt.set()
        if self.h is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvml unavailable"]}
        self.join(timeout=2)
        s = self.samples[1:] if len(self.samples) > 2 else self.samples
        return {"sm_mhz": float(np.median(s)) if s else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s),
                "power_w_max": round(max(self.power), 1) if self.power else None}


def oracle_timesteps(w, n_steps, n_threads):
    """Time n_steps MD timesteps of the oracle as it stands (cell-list mode, OpenMP over beads)."""
    from oracle import oracle as orc
    o = orc.Oracle(w, use_cells=True, n_threads=n_threads)
    o.compute_forces()
    o.run(1)                                    # warm-up (page faults, thread pool)
    t0 = time.perf_counter()
    o.run(n_steps)
    dt = time.perf_counter() - t0
    return dt, orc.lib().orc_num_threads() if n_threads <= 0 else n_threads


def run_reference(args, w):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oracle as orc
    cores = os.cpu_count() or 1
    o = orc.Oracle(w, use_cells=True, n_threads=cores)
    o.compute_forces()
    if w.equil_steps:
        pass    # the oracle is timed at the start state: per-timestep cost does not depend on the thermostat
    for _ in range(args.warmup):
        o.run(1)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.run(1)
    dt = time.perf_counter() - t0
    tps = args.steps / dt
    sample = f"{args.steps} single MD timesteps of {w.name} (N={w.n}), fp64 cell-list oracle, OpenMP"
    line = {
        "impl": "reference", "metric": METRIC, "value": tps, "unit": "timesteps/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": describe(w), "timesteps_per_step": 1},
        "cpu_baseline": {"value": tps, "unit": "timesteps/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": tps, "unit": "timesteps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def max_over_ranks(ms: float, world: int, device) -> float:
    """Device-timed milliseconds of the slowest rank (replicas only: no data-path collective)."""
    if world > 1:
        import torch
        import torch.distributed as dist
        t = torch.tensor([ms], device=device, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    return ms


def whole_job_value(world: int, timesteps_per_rank: int, ms: float) -> float:
    """Whole-job timesteps/s of `world` independent replicas that each ran timesteps_per_rank in (max) ms."""
    return world * timesteps_per_rank / (ms * 1e-3)


def describe(w) -> str:
    rc = float(np.max(w.pair["rc"]))
    return (f"{w.name}: {w.n} beads, chains of {w.chain_len}, box {float(w.box[0]):.3f}, {w.pair_style} rc={rc:.4f}, "
            f"{w.bond_style} bonds, {w.integrator}, dt={w.dt}, skin={w.r_skin}, sfc_period={w.sfc_period}")


def src_sha16() -> str:
    """Hash of the step kernel's CUDA sources: the ncu-derived figures under profiles/ carry the hash of the code they were
    taken on and are only quoted while it still matches (otherwise the field is null)."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_1310_2041_b200", "csrc")
    for f in ("gm_internal.cuh", "gm_force_impl.cuh", "gm_force.cu", "gm_force_dpd.cu"):
        with open(os.path.join(d, f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def profile_row(config: str):
    """Row of profiles/kernels_r02.csv for this config's step kernel, or None if absent or taken on other code."""
    path = os.path.join(ROOT, "profiles", "kernels_r02.csv")
    if not os.path.exists(path):
        return None
    import csv
    sha = src_sha16()
    with open(path) as f:
        for row in csv.DictReader(f):
            if row["config"] == config and row["src_sha16"] == sha:
                return row
    return None


def measure(gm, torch, w, local, stream, inner, steps, warmup, flags, tune, barrier, world, dev, clocks=None,
            pair_samples=5):
    """Set-up by the config's own protocol (untimed), W warm-up bench steps, exactly K timed ones (CUDA events on the
    library's stream), then the step kernel alone (gm_step_timed) and the in-cutoff pair count averaged over
    `pair_samples` states."""
    import copy
    w_run = w
    if w.equil_steps:
        w_run = copy.copy(w)
        w_run.integrator = "langevin"
    s = gm.System(w_run, device=local, flags=flags, tune=tune)
    if w.equil_steps:
        s.step(w.equil_steps)                   # C3: 1,000 Langevin steps (kT=1, gamma=1), then NVE
        if w.integrator in ("nph", "npt"):
            s.set_barostat(float(w.p_ext), float(w.piston_mass))
        s.set_integrator(w.integrator, w.kT, 0.0)
    for _ in range(warmup):
        s.step(inner)
    barrier()
    st1 = s.stats()
    if clocks is not None:
        clocks.start()
        time.sleep(0.05)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    for _ in range(steps):
        s.step(inner)
    e1.record(stream)
    barrier()
    ms = e0.elapsed_time(e1)
    clk = clocks.stop() if clocks is not None else {}
    st2 = s.stats()
    ms = max_over_ranks(ms, world, dev)
    n_ts = steps * inner
    rebuilds = st2["rebuilds"] - st1["rebuilds"]
    # the dominant kernel alone: CUDA events around every launch (gm_step_timed)
    tk = s.step_timed(min(inner, 200))
    k_ms = tk["force_ms"] / max(1, tk["force_launches"])
    # unique pairs inside r_cut, averaged over several states (>= 5 samples)
    pairs, en = [], None
    for _ in range(pair_samples):
        s.step(max(1, min(inner, 100) // pair_samples))
        en = s.energies()
        pairs.append(en["n_pairs"])
    st3 = s.stats()
    nbar_l = st3["sum_nn"] / w.n
    bbar = 2.0 * len(w.bonds) / w.n
    dpd = w.pair_style == "dpd"
    bytes_kernel = w.n * ((48 + 48 if dpd else 32 + 32) + 16 + 4 + 4 * nbar_l + 4 + 4 * bbar)
    m_interval = n_ts / max(1, rebuilds)
    bytes_step = bytes_kernel + w.n * (80 + 4 * nbar_l) / m_interval
    # kernels launched inside the timed region: per timestep the gate + the fused force/integrate kernel; per rebuild
    # keys, scan, scatter, permute (= SFC sort of all particle arrays), NL build, and with bonds the BL remap
    launches = n_ts * 2 + rebuilds * (6 if len(w.bonds) else 5)
    return dict(system=s, ms=ms, n_ts=n_ts, tps=whole_job_value(world, n_ts, ms), ms_ts=ms / n_ts, k_ms=k_ms,
                rebuilds=rebuilds, reorders=st2["reorders"] - st1["reorders"], m_interval=m_interval, nbar_l=nbar_l,
                max_nn=st3["max_nn"], sum_nn=st3["sum_nn"], pairs_in_rc=float(np.mean(pairs)), energies=en,
                bytes_kernel=bytes_kernel, bytes_step=bytes_step, launches=int(launches), clocks=clk,
                rebuild_ms_direct=tk["rebuild_ms"] / max(1, tk["force_launches"]), tuning=s.tuning())


def rooflines(config, w, m, hbm_gbs, peak_src, sm_mhz):
    """HBM roofline of the step kernel (algorithmic bytes of SURVEY.md 8(d) / CUDA-event time) and of the whole timestep,
    plus -- from the ncu capture of the same code, profiles/kernels_r02.csv -- measured DRAM traffic, the issue-slot
    ("alu") roofline and L2 throughput.  DESIGN.md 7 derives the peaks."""
    k_s, ts_s = m["k_ms"] * 1e-3, m["ms_ts"] * 1e-3
    achieved = m["bytes_kernel"] / k_s / 1e9
    whole = m["bytes_step"] / ts_s / 1e9
    roof = {"bound": "hbm", "kernel": "k_step (fused a4+a5/a6+a7+a8)", "achieved": achieved, "peak": hbm_gbs,
            "unit": "GB/s", "frac": achieved / hbm_gbs, "traffic": None, "peak_source": peak_src,
            "what": "achieved = ALGORITHMIC bytes per launch / CUDA-event time of the kernel (not a DRAM counter)",
            "kernel_ms": m["k_ms"], "algorithmic_bytes_per_launch": m["bytes_kernel"],
            "kernel_share_of_step": m["k_ms"] / m["ms_ts"],
            "whole_step": {"algorithmic_bytes_per_timestep": m["bytes_step"], "achieved": whole,
                           "frac": whole / hbm_gbs, "frac_of_nominal_8TBs": whole / 8000.0},
            "target": {"what": "whole timestep >= 0.50 of the HBM roofline (BASELINE.json north_star; C3)",
                       "value": whole / hbm_gbs, "met": bool(whole / hbm_gbs >= 0.5)} if config == "C3" else None}
    row = profile_row(config)
    if row is not None:
        traffic = float(row["dram_bytes_per_launch"])
        tinst = float(row["thread_inst_per_launch"])
        # issue-slot peak: 148 SMs x 4 schedulers x 1 warp instruction per clock x 32 lanes at the SM clock seen under load
        peak_alu = 148 * 4 * 32 * sm_mhz * 1e6
        roof["traffic"] = traffic
        roof["dram_gbs_measured"] = traffic / k_s / 1e9
        roof["alu"] = {"bound": "alu", "achieved": tinst / k_s / 1e12, "peak": peak_alu / 1e12,
                       "unit": "T thread-instructions/s", "frac": tinst / k_s / peak_alu,
                       "thread_inst_per_bead": tinst / w.n, "source": "ncu smsp__thread_inst_executed.sum, same code"}
        roof["l2"] = {"lts_throughput_pct": float(row["lts_throughput_pct"]), "lts_hit_pct": float(row["lts_hit_pct"]),
                      "l1_lsu_wavefronts_pct": float(row["l1_lsu_wavefronts_pct"])}
    return roof


def compact(name, w, m, hbm_gbs, peak_src, sm_mhz):
    r = rooflines(name, w, m, hbm_gbs, peak_src, sm_mhz)
    out = {"workload": describe(w), "tps": m["tps"], "ms_per_timestep": m["ms_ts"], "mean_nn": m["nbar_l"],
           "rebuild_interval": m["m_interval"], "k_step_ms": m["k_ms"], "k_step_frac": r["frac"],
           "whole_step_frac": r["whole_step"]["frac"], "pair_interactions_per_s": m["tps"] * m["pairs_in_rc"],
           "timesteps": m["n_ts"], "tiles_not_windowed": m["tuning"]["tiles_not_windowed"], "tiles": m["tuning"]["tiles"]}
    for k in ("traffic", "dram_gbs_measured", "alu", "l2"):
        if k in r and r[k] is not None:
            out[k] = r[k]
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="C3")
    ap.add_argument("--scale", type=float, default=None, help="shrink the config (debugging only)")
    ap.add_argument("--beads", type=int, default=None,
                    help="bead count of the paper's Fig. 4 liquids (--config F4LJ | F4DPD; default 1,000,000)")
    ap.add_argument("--inner", type=int, default=0, help="MD timesteps per bench step (0: one SFC period)")
    ap.add_argument("--no-cond-nodes", action="store_true",
                    help="gate the rebuild with early-exit kernels instead of a conditional graph node "
                         "(ncu cannot profile kernel nodes of graphs that hold conditional nodes)")
    ap.add_argument("--no-graph", action="store_true",
                    help="GM_FLAG_NO_GRAPH: launch kernel by kernel (for ncu: it does not profile graph kernel nodes that can "
                         "set a conditional handle, which the step kernel can)")
    ap.add_argument("--skin", type=float, default=None,
                    help="override the config's neighbor skin (a tuning knob that never changes results; "
                         "BASELINE.json gives none for C4)")
    ap.add_argument("--tune", action="append", default=[], metavar="FIELD=INT",
                    help="gm_config tuning override (x_cell_div, nl_scan_trip, step_shape, win_capacity); never changes results")
    ap.add_argument("--no-windows", action="store_true", help="GM_FLAG_NO_WINDOWS: 32-bit neighbor rows and L1/L2 gathers")
    ap.add_argument("--barostat", default=None, metavar="P_EXT,PISTON_MASS",
                    help="run the config under the Andersen barostat (NPH; information only: two plain kernels per timestep, "
                         "no CUDA graph, no tile windows -- the roofline block then describes the barostat's force kernel)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true",
                    help="skip the short runs of C1, C2, C4, C5 that the default C3 line carries in `configs`")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3

    from workloads import make_config
    w = make_config(args.config, scale=args.scale, n=args.beads)
    if args.skin is not None:
        w.r_skin = float(args.skin)
    if args.barostat:
        p_ext, piston = (float(x) for x in args.barostat.split(","))
        w.integrator, w.p_ext, w.piston_mass = "nph", p_ext, piston
    if args.impl == "reference":
        run_reference(args, w)
        return

    import torch
    import torch.distributed as dist
    from paper_1310_2041_b200 import gm

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    inner = args.inner or (w.sfc_period if w.sfc_period > 0 else 500)
    hbm_gbs, peak_src = load_peaks()
    flags = (gm.GM_FLAG_NO_COND_NODES if args.no_cond_nodes else 0) | (gm.GM_FLAG_NO_WINDOWS if args.no_windows else 0) | \
            (gm.GM_FLAG_NO_GRAPH if args.no_graph else 0)
    tune = {k: int(v) for k, v in (kv.split("=") for kv in args.tune)}
    flags |= tune.pop("flags", 0)
    stream = torch.cuda.current_stream(dev)

    # ---- device-resident throughput: W warm-up steps, then exactly K timed steps -------------------
    clocks = ClockSampler(dev)
    m = measure(gm, torch, w, local, stream, inner, args.steps, args.warmup, flags, tune, barrier, world, dev, clocks)
    s, ms, tps, n_ts, ms_ts, k_ms = m["system"], m["ms"], m["tps"], m["n_ts"], m["ms_ts"], m["k_ms"]
    clk = m["clocks"]
    sm_mhz = clk.get("sm_mhz") or clk.get("sm_max_mhz") or 1965.0
    roof = rooflines(args.config, w, m, hbm_gbs, peak_src, sm_mhz)
    launches = m["launches"]

    # ---- end to end through the C ABI with HOST buffers ---------------------------------------------
    e2e = None
    if not args.no_e2e:
        n = w.n
        hp = torch.empty((n, 3), dtype=torch.float32).pin_memory()
        hv = torch.empty((n, 3), dtype=torch.float32).pin_memory()
        ht = torch.from_numpy(np.ascontiguousarray(w.type, np.int32)).pin_memory()
        gm.gm_get_particles(s.h, hp, hv, None)
        k_e2e = max(2, min(args.steps, 5))
        for _ in range(1):
            gm.gm_set_particles(s.h, hp, hv, ht, None); s.step(inner); gm.gm_get_particles(s.h, hp, hv, None)
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(k_e2e):
            gm.gm_set_particles(s.h, hp, hv, ht, None)      # H2D: pos, vel, type (pinned host memory)
            s.step(inner)
            gm.gm_get_particles(s.h, hp, hv, None)          # D2H: pos, vel; synchronises
        e1.record(stream)
        barrier()
        ms_e = e0.elapsed_time(e1)
        if world > 1:
            t = torch.tensor([ms_e], device=dev, dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms_e = float(t.item())
        e2e = {"value": world * k_e2e * inner / (ms_e * 1e-3), "unit": "timesteps/s",
               "h2d_bytes_per_step": n * (12 + 12 + 4), "d2h_bytes_per_step": n * 24, "steps": k_e2e,
               "what": "gm_set_particles(host) + gm_step(inner) + gm_get_particles(host) per step"}

    # ---- the oracle beside it (rank 0, N=1 only) ----------------------------------------------------
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cores = os.cpu_count() or 1
        t1, _ = oracle_timesteps(w, 1, cores)
        k = int(max(2, min(200, 15.0 / max(t1, 1e-3))))       # about 15 s of CPU work
        tt, thr = oracle_timesteps(w, k, cores)
        k1 = int(max(1, min(50, 5.0 / max(t1 * thr, 1e-3))))   # about 5 s more on ONE thread
        t1t, _ = oracle_timesteps(w, k1, 1)
        cpu = {"value": k / tt, "unit": "timesteps/s", "cores": thr, "kind": "oracle",
               "sample": f"{k} MD timesteps of {w.name} (N={w.n}) from the start state, fp64 cell-list oracle, OpenMP over beads",
               "one_thread": {"value": k1 / t1t, "unit": "timesteps/s", "cores": 1, "sample": f"{k1} MD timesteps"}}

    s.close()
    # ---- the other configs of BASELINE.json, short runs (rank 0, N=1 only): one line carries all five -------------
    others = None
    if rank == 0 and world == 1 and args.config == "C3" and not args.no_other_configs and args.scale is None:
        others = {}
        for name in ("C1", "C2", "C4", "C5"):
            wo = make_config(name)
            io = min(200, wo.sfc_period if wo.sfc_period > 0 else 200)
            mo = measure(gm, torch, wo, local, stream, io, 3, 3, flags, {}, barrier, 1, dev)
            mo["system"].close()
            others[name] = compact(name, wo, mo, hbm_gbs, peak_src, sm_mhz)
            del mo, wo
            torch.cuda.empty_cache()

    if rank == 0:
        en = m["energies"]
        line = {
            "metric": METRIC, "value": tps, "unit": "timesteps/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": describe(w), "timesteps_per_step": inner, "parallelism": f"replicas x{world}",
                       "l2": f"no flush: successive timesteps are data-dependent; per-timestep working set "
                             f"{(m['bytes_kernel'] + 16 * w.n) / 1e6:.0f} MB vs L2 {L2_BYTES / 1e6:.0f} MB",
                       "equilibration": f"{w.equil_steps} Langevin steps (untimed set-up)" if w.equil_steps else "none"},
            "ms_per_timestep": ms_ts,
            "pair_interactions_per_s": tps * m["pairs_in_rc"],
            "list_entries_per_s": tps * m["sum_nn"],
            "pairs_in_rc": m["pairs_in_rc"], "pairs_in_rc_samples": 5, "mean_nn": m["nbar_l"], "max_nn": m["max_nn"],
            "rebuilds": m["rebuilds"], "rebuild_interval": m["m_interval"], "reorders": m["reorders"],
            "rebuild_ms_per_timestep_direct": m["rebuild_ms_direct"],
            "energy_per_bead": en["etot"] / w.n, "temperature": en["T"], "tuning": m["tuning"],
            "roofline": roof, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches), "clocks": clk,
            "configs": others,
        }
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
