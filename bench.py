"""bench.py — throughput of the hot path (CFL dt + one RK2 step of the 3D Euler finite-volume update, and the
VJP of that step) on synthetic workloads shaped like the paper's, through the C ABI of include/dh.h.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--n 1024] [--impl dh|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P \
        bench.py --gpus N --steps K --warmup W

One JSON line on stdout (rank 0).  Contract and the meaning of every key: DESIGN.md §"Measurement".

* workload (default): BASELINE.json configs[4] — 1024^3 fp32 periodic decaying turbulence, rms Mach 2, no
  cooling (21.5 GB per state, far larger than the 126 MB L2, so no L2 flush is needed between iterations).
* a "step" = CFL reduction + dt epilogue + predictor stage + corrector stage; the K timed steps are one
  dh_advance(U, K) call (dt never leaves the device; --no-chain issues dh_cfl_dt_async + dh_step_devdt per step
  instead).  `value` = cells * K / time, inputs resident in HBM.  The VJP of the step (dh_step_vjp) is timed in the
  same run and reported under "vjp".
* "e2e" = the same steps through dh_stream_host: pinned HOST state -> device, CFL + step, device -> HOST every step, all
  inside the timed region.
* N > 1: the path does not shard in this build ("replicas only"): every rank runs the same-shaped
  workload (its own seed) on its own GPU, no data-path collective; value = sum of the ranks' cells / max time.
* --impl reference: the CPU oracle (oracle/), as it stands, on the host cores, on a bounded sample of the same
  workload.  This and the `cpu_baseline` leg are the only places this file touches oracle/.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "cell-updates/s per RK2 step (forward: CFL dt + predictor + corrector)"
UNIT = "cell-updates/s"
FWD_WORDS, VJP_WORDS = 25, 45          # algorithmic words per cell: SURVEY.md §8(d), DESIGN.md §"Kernels"
STAGE_WORDS = {"stage1": 10, "stage2": 15, "rev2": 15, "rev1": 20, "cfl_reduce": 5, "lincomb": 15, "cool": 6}
FALLBACK_HBM_GBS = 6650.0              # /opt/skills/guides/B200_PROFILING.md, used only without MEASURED_PEAKS.json


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="dh", choices=["dh", "reference"])
    ap.add_argument("--n", "--grid", dest="n", type=int, default=1024, help="grid size per axis (default 1024: BASELINE configs[4])")
    ap.add_argument("--cooling", type=int, default=0, help="1: configs[3]'s cooling source in the corrector epilogue")
    ap.add_argument("--cool-mode", choices=["euler", "trapezoid"], default="euler", help="DH_OPT_COOL_MODE (PAPER.md:318-325), with --cooling 1")
    ap.add_argument("--cool-nsub", type=int, default=1, help="DH_OPT_COOL_NSUB: substeps of Eq. 23, with --cooling 1")
    ap.add_argument("--c-cool", type=float, default=0.0, help="DH_OPT_C_COOL: c_cool of Eq. 21 (PAPER.md:314), with --cooling 1; 0 = no cooling-time limit")
    ap.add_argument("--mach", type=float, default=2.0)
    ap.add_argument("--kernel", default="fused", choices=["fused", "gather"])
    ap.add_argument("--no-chain", action="store_true", help="one dh_cfl_dt_async + dh_step_devdt pair per step instead of one dh_advance call")
    ap.add_argument("--riemann", choices=["hllc", "hll", "rusanov"], default="hllc", help="DH_OPT_RIEMANN (PAPER.md:828, 835); default HLLC")
    ap.add_argument("--limiter", choices=["minmod", "vanleer", "mc"], default="minmod", help="DH_OPT_LIMITER (PAPER.md:820)")
    ap.add_argument("--integrator", choices=["vl2", "heun", "ssprk3"], default="vl2",
                    help="vl2 = the predictor / corrector of Eqs. A6-A7 (BASELINE's metric); heun, ssprk3: SURVEY 8(f) item 2")
    ap.add_argument("--adjoint", type=int, default=0, help="also time dh_adjoint over this many steps (checkpointed multi-step adjoint)")
    ap.add_argument("--poisson", type=int, default=0, metavar="N",
                    help="instead of the hydro step: time multigrid cycles of the periodic Poisson solver on an N^3 grid (SURVEY 8(f) item 3)")
    ap.add_argument("--mg-cycle", choices=["V", "W"], default="V")
    ap.add_argument("--mg-subtree", type=int, default=1, help="DH_MG_SUBTREE: 1 (default) the levels of <= 4096 cells in one block, 0 one launch per operator")
    ap.add_argument("--issue-probe", action="store_true",
                    help="instead of the hydro step: dh_issue_probe, the issue cost of the instruction mixes the stage kernels are made of "
                         "(SM cycles per group per scheduler at 2 and 4 warps per scheduler; DESIGN.md section 7b)")
    ap.add_argument("--no-vjp", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--cpu-sample", type=int, default=192, help="edge of the periodic sub-block the oracle is timed on")
    return ap.parse_args()


def workload_name(a) -> str:
    if a.cooling:
        return f"cooling_turbulence_{a.n}^3_fp32_mach{a.mach:g} (BASELINE configs[3] recipe)"
    return f"decaying_turbulence_{a.n}^3_fp32_mach{a.mach:g} (BASELINE configs[4] recipe)"


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy bandwidth)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md, MEASURED_PEAKS.json absent)"


def committed_capture(n: int):
    """What the committed `ncu --set full` capture of the stage kernel says for an n^3 grid (profiles/traffic.json, written
    from the .ncu-rep by hand-run commands named in the profiles/*.md beside it; the entry records the commit it was
    taken at): DRAM bytes per launch averaged over the predictor and corrector launches (like `achieved`), and the
    hardware counters of the same launches.  None when no capture of this size is committed."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            d = json.load(f)
        e = d.get("stage", {}).get(str(n))
        if not e:
            return None, None
        traffic = 0.5 * (e["predictor"]["dram_bytes"] + e["corrector"]["dram_bytes"])
        return traffic, {"kind": "ncu hardware counters of the committed capture, not of this run", "source": e.get("source"),
                         "commit": e.get("commit"), "predictor": e["predictor"], "corrector": e["corrector"]}
    except Exception:
        return None, None


def issue_bound(counters: dict, ms_per_launch: float, clocks: dict, N: int, peak: float):
    """The issue-port reading of the stage kernel (profiles/r02d_issue_bound.md): executed warp instructions of the
    committed ncu capture x the issue-port cycles per instruction that `sass_cost` derives from the kernel's SASS under the rule that
    `dh_issue_probe` measures (max(1, register operands read / 2) cycles per instruction), against the port cycles this run's launch had
    (schedulers x measured time x the SM clock sampled during the run).  A cost model over hardware counters: `kind` says so."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            m = json.load(f)["issue_model"]
        mhz = float(clocks.get("sm_mhz") or 0.0) if isinstance(clocks, dict) else 0.0
        ghz = mhz / 1e3 if mhz > 0 else float(m["sm_clock_ghz"])
        ports = m["schedulers_per_sm"] * m["sm_count"]
        need = 0.0
        for stage in ("predictor", "corrector"):
            cpi = m[stage]["static_issue_cycles"] / m[stage]["static_instructions"]
            need += 0.5 * counters[stage]["warp_instructions"] * cpi          # average over the two launches, like `achieved`
        have = ports * ms_per_launch * 1e-3 * ghz * 1e9
        hbm_ms = 0.5 * (STAGE_WORDS["stage1"] + STAGE_WORDS["stage2"]) * 4.0 * N / (peak * 1e9) * 1e3
        return {"kind": "cost model (measured per-instruction issue cost x executed-instruction counter of the committed capture)",
                "rule": m["rule"], "issue_port_cycles_needed_per_launch": need, "issue_port_cycles_available_per_launch": have,
                "utilisation": need / have, "lane_issue_cycles_per_cell_stage": need * 32.0 / N,
                "ms_per_launch_at_full_utilisation": ms_per_launch * need / have,
                "hbm_frac_at_full_utilisation": hbm_ms / (ms_per_launch * need / have)}
    except Exception:
        return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.thread = [], None, None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "200",
                                          "-i", str(index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [x.strip() for x in line.split(",")]))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        rows = [r for t, r in self.rows if t0 <= t <= t1 + 0.2 and len(r) >= 7] or [r for _, r in self.rows if len(r) >= 7]
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [nm for i, nm in enumerate(names) if any(r[3 + i].lower().startswith("active") for r in rows)]
        num = lambda s: float(s) if s.replace(".", "", 1).isdigit() else float("nan")
        return {"sm_mhz": statistics.median(num(r[0]) for r in rows), "sm_max_mhz": num(rows[0][1]),
                "power_w_max": max(num(r[2]) for r in rows), "samples": len(rows), "reasons": reasons}


# --------------------------------------------------------------------------------------------- oracle legs
def _scheme(a) -> dict:
    return {"limiter": a.limiter, "riemann": a.riemann, "integrator": a.integrator, "cool_mode": a.cool_mode, "cool_nsub": a.cool_nsub}


def oracle_sample(U_block, gamma: float, cooling: bool, with_vjp: bool = False, seed: int = 2005, scheme: dict | None = None) -> dict:
    """Time the CPU oracle, as it stands, for one CFL dt + one full step on `U_block` ([5, m, m, m] numpy,
    treated as its own periodic box).  Returns cell-updates/s and what was timed."""
    import numpy as np

    import oracle

    scheme = scheme or {}          # limiter / riemann / integrator of the timed arm
    p = oracle.params(gamma=gamma, shape=tuple(U_block.shape), cooling=cooling, **scheme)
    cells = int(np.prod(U_block.shape[1:]))
    t0 = time.perf_counter()
    dt, _ = oracle.cfl_dt(U_block, p)
    oracle.step(U_block, dt, p)
    t_fwd = time.perf_counter() - t0
    out = {"value": cells / t_fwd, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
           "sample": f"one CFL dt + RK2 step on a {U_block.shape[3]}x{U_block.shape[2]}x{U_block.shape[1]} periodic sub-block "
                     f"of the workload's initial state ({cells} cells, {t_fwd:.2f} s, fp64 oracle, OpenMP)"}
    if with_vjp:
        m = min(96, U_block.shape[1])
        sub = np.ascontiguousarray(U_block[:, :m, :m, :m])
        g = np.random.default_rng(seed).normal(size=sub.shape)
        ps = oracle.params(gamma=gamma, shape=tuple(sub.shape), cooling=cooling, **scheme)
        t0 = time.perf_counter()
        oracle.step_vjp(sub, dt, g, ps)
        t_v = time.perf_counter() - t0
        out["vjp_value"] = m ** 3 / t_v
        out["vjp_sample"] = f"one step VJP on a {m}^3 sub-block ({t_v:.2f} s)"
    return out


def cpu_block(a, m: int, seed: int):
    """The bounded CPU sample: the workload's own recipe generated at edge m (same generator, same spectrum band
    rule) — used when no device state is at hand (--impl reference)."""
    import torch

    from paper_2512_13403_b200 import workloads

    wl = workloads.turbulence(m, seed=seed, mach=a.mach, cooling=bool(a.cooling), dtype=torch.float32)
    return wl.U.numpy(), wl.gamma


def run_reference(a):
    """--impl reference: the oracle on the host cores; each step = one bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    m = min(a.cpu_sample, a.n, 128)
    U, gamma = cpu_block(a, m, 1005 if not a.cooling else 1004)
    import oracle

    oracle.build()
    for _ in range(min(a.warmup, 1)):
        oracle_sample(U, gamma, bool(a.cooling), scheme=_scheme(a))
    times, last = [], None
    for _ in range(a.steps):
        t0 = time.perf_counter()
        last = oracle_sample(U, gamma, bool(a.cooling), scheme=_scheme(a))
        times.append(time.perf_counter() - t0)
    cells = m ** 3
    total = sum(times)
    value = cells * a.steps / total
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": a.gpus, "steps": a.steps,
            "warmup": a.warmup, "ms_per_step": 1e3 * total / a.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(a), "sample": f"{m}^3 periodic box of the same recipe per step",
                       "l2": "CPU run"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": last["cores"], "kind": "oracle",
                             "sample": f"{a.steps} x (CFL dt + RK2 step) on a {m}^3 box generated by the workload's recipe"},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------- multi-rank helpers
def reduce_max_ms(ms: float, world: int, device=None) -> float:
    """Replicas only: the time of a multi-rank run is the slowest rank's device time."""
    if world == 1:
        return ms
    import torch
    import torch.distributed as dist

    t = torch.tensor([ms], device=device if device is not None else "cpu", dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(cells_per_rank: int, steps: int, world: int, ms_max: float) -> float:
    """Whole-job throughput: every rank advances its own replica, so the cells add up and the time is the max."""
    return world * cells_per_rank * steps / (ms_max * 1e-3)


# --------------------------------------------------------------------------------------------------- dh leg
def run_dh(a):
    import torch
    import torch.distributed as dist

    from paper_2512_13403_b200 import dh, workloads

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the dh path has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    n, K, W = a.n, a.steps, max(a.warmup, 0)
    N = n ** 3
    seed = (1004 if a.cooling else 1005) + 17 * rank       # replicas: same recipe, own seed per rank
    wl = workloads.turbulence(n, seed=seed, mach=a.mach, cooling=bool(a.cooling), dtype=torch.float32, device=dev)
    U = wl.U
    torch.cuda.empty_cache()
    # the oracle's bounded sample: a sub-block of the initial state, taken before anything is stepped
    m = min(a.cpu_sample, n)
    U_cpu_block = U[:, :m, :m, :m].contiguous().cpu().numpy() if (rank == 0 and world == 1 and not a.no_cpu) else None

    s = dh.Solver(n, n, n, gamma=wl.gamma, dtype=torch.float32, kernel=a.kernel, cooling=int(a.cooling),
                  lambda0=wl.lambda0, alpha=wl.alpha, t_floor=wl.t_floor, integrator=a.integrator, riemann=a.riemann, limiter=a.limiter,
                  cool_mode=a.cool_mode, cool_nsub=a.cool_nsub, c_cool=a.c_cool)
    # algorithmic words per cell of one step: CFL 5 + per stage (5 in [+ 5 base] + 5 out) + per combination 15
    # words per cell and step with a full CFL pass (5) in front; the combinations of Heun / SSPRK3 are formed inside the stage kernel
    fwd_words = {"vl2": 5 + FWD_WORDS, "heun": 5 + 10 + 15, "ssprk3": 5 + 10 + 15 + 15}[a.integrator]

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def fwd_step(k=1):
        # k x (CFL dt + RK2 step), dt never leaves the device
        if a.no_chain:
            for _ in range(k):
                s.cfl_dt_async(U)
                s.step_devdt(U)
        else:
            s.advance(U, k, sync=False)

    # a state that fits in the 126 MB L2 (n <= 128) is evicted between iterations by writing a 512 MB buffer;
    # the flush is outside the per-iteration event pairs
    fits_l2 = 5 * 4 * N <= 4 * 126e6
    flush = torch.empty(128 * 1024 * 1024, device=dev, dtype=torch.float32) if fits_l2 else None

    def timed(fn, iters, batched=False):
        """K steps bracketed by barrier + synchronize on both sides, CUDA events on the launching stream; the
        max over ranks is taken by the caller.  batched: fn(K) issues all K steps in one library call."""
        barrier()
        l0 = s.launch_count
        t0 = time.time()
        if flush is None:
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            if batched:
                fn(iters)
            else:
                for _ in range(iters):
                    fn()
            e1.record()
            barrier()
            ms = e0.elapsed_time(e1)
        else:
            pairs = []
            for _ in range(iters):
                flush.zero_()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                fn()
                e1.record()
                pairs.append((e0, e1))
            barrier()
            ms = sum(x.elapsed_time(y) for x, y in pairs)
        t1 = time.time()
        return ms, s.launch_count - l0, t0, t1

    def max_over_ranks(ms):
        return reduce_max_ms(ms, world, dev)

    # ---- forward: warm-up, then the timed region with per-kernel events and the clock sampler running
    fwd_step(W) if flush is None else [fwd_step() for _ in range(W)]
    dt_w = s.poll()                                        # raises on a non-finite state
    s.profile(True)
    sampler = ClockSampler(local) if rank == 0 else None
    ms_fwd, launches, t0, t1 = timed(fwd_step, K, batched=True)
    clocks = sampler.stop(t0, t1) if sampler else None
    prof = s.profile_read()
    dt_last = s.poll()
    ms_fwd = max_over_ranks(ms_fwd)
    value = aggregate_value(N, K, world, ms_fwd)

    peak, peak_src = measured_peak()
    gbs = lambda words, ms, cnt: (words * 4.0 * N * cnt) / (ms * 1e-3) / 1e9 if ms > 0 else None
    st_ms = prof["stage1"][0] + prof["stage2"][0]
    st_cnt = prof["stage1"][1] + prof["stage2"][1]
    st_bytes = 4.0 * N * (STAGE_WORDS["stage1"] * prof["stage1"][1] + STAGE_WORDS["stage2"] * prof["stage2"][1])
    achieved = st_bytes / (st_ms * 1e-3) / 1e9
    # bytes the step really has to move: 20 words per cell in the stages; the 5 words of the CFL pass only in the steps
    # whose dt came from a full reduction (first step of a dh_advance call, fallbacks of the candidate path)
    cstats = s.cfl_stats()
    full_passes = prof["cfl_reduce"][1] + (cstats["fallbacks"] if prof["cfl_cand"][1] else 0)
    step_bytes = 4.0 * N * ((fwd_words - 5) * K + 5 * full_passes)
    traffic, counters = committed_capture(n)

    def per_kernel(pr):
        out = {}
        for k, v in pr.items():
            if v[1] == 0:
                continue
            e = {"ms_per_launch": v[0] / v[1], "launches": v[1], "GB/s": gbs(STAGE_WORDS[k], v[0], v[1]) if k in STAGE_WORDS else None}
            if k == "cfl_cand":
                e["note"] = "exact recipe on the listed packs + guarded full pass (returns at once unless a fallback is needed): no fixed byte count"
            out[k] = e
        return out

    roofline = {"bound": "hbm", "kernel": "stage kernel (predictor + corrector launches of the same kernel)",
                "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "peak_source": peak_src,
                "traffic": traffic, "bytes_per_launch": st_bytes / max(st_cnt, 1),
                "ms_per_launch": st_ms / max(st_cnt, 1),
                "per_kernel": per_kernel(prof),
                "step_GB/s": step_bytes / (ms_fwd * 1e-3) / 1e9,
                "step_frac": step_bytes / (ms_fwd * 1e-3) / 1e9 / peak,
                "step_bytes_note": f"{fwd_words - 5} words/cell/step + 5 words/cell for each of the {full_passes} full CFL passes in the {K} timed steps"}
    if counters is not None:
        roofline["counters"] = counters
        issue = issue_bound(counters, st_ms / max(st_cnt, 1), clocks, N, peak)
        if issue is not None:
            roofline["issue"] = issue
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms_fwd / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_name(a), "grid": [n, n, n], "cells_per_gpu": N, "gamma": wl.gamma,
                       "cfl": 0.4, "limiter": a.limiter, "riemann": a.riemann, "integrator": {"vl2": "rk2 predictor/corrector", "heun": "heun rk2", "ssprk3": "ssprk3"}[a.integrator],
                       "cooling": bool(a.cooling), "cool_mode": a.cool_mode, "cool_nsub": a.cool_nsub, "c_cool": a.c_cool, "kernel": a.kernel,
                       "call": "dh_cfl_dt_async + dh_step_devdt per step" if a.no_chain else "dh_advance(U, K): K x (CFL reduce, dt epilogue, predictor, corrector)", "parallelism": f"replicas x{world}",
                       "l2": "state fits in L2: a 512 MB buffer is written between iterations (outside the event pairs)"
                       if fits_l2 else f"inputs larger than L2 ({5 * 4 * N / 1e6:.0f} MB per state vs 126 MB), no flush",
                       "dt_last": dt_last},
            "roofline": roofline, "clocks": clocks, "gpu_launches": launches}
    s.profile(False)
    line["config"]["cfl_candidate_path"] = cstats             # dh_advance: dt's from candidate lists / fallbacks / packs

    # ---- VJP of the step, same state, seeded Gaussian cotangent on all five fields (configs[4])
    if not a.no_vjp:
        g = workloads.cotangent(U.shape, seed=2005 + rank, dtype=torch.float32, device=dev)
        gin = torch.empty_like(U)
        vjp = lambda: s.step_vjp(U, dt_last, g, gin)
        for _ in range(min(W, 2)):
            vjp()
        s.profile(True)
        Kv = max(1, min(K, 5))
        ms_v, launches_v, _, _ = timed(vjp, Kv)
        pv = s.profile_read()
        s.profile(False)
        ms_v = max_over_ranks(ms_v)
        if not bool(torch.isfinite(gin[:, :2]).all()):
            raise RuntimeError("non-finite VJP result")
        vjp_words = {"vl2": VJP_WORDS, "heun": 10 + 15 + 20, "ssprk3": 10 + 15 + 15 + 15 + 15 + 20}[a.integrator]
        line["vjp"] = {"value": world * N * Kv / (ms_v * 1e-3), "unit": "cell-VJPs/s", "steps": Kv, "ms_per_step": ms_v / Kv,
                       "gpu_launches": launches_v,
                       "roofline": {"bound": "hbm", "achieved": vjp_words * 4.0 * N * Kv / (ms_v * 1e-3) / 1e9, "peak": peak,
                                    "unit": "GB/s", "frac": vjp_words * 4.0 * N * Kv / (ms_v * 1e-3) / 1e9 / peak,
                                    "words_per_cell": vjp_words,
                                    "per_kernel": per_kernel(pv)}}
        line["gpu_launches"] += launches_v
        del g, gin
        torch.cuda.empty_cache()

    # ---- multi-step adjoint: forward sweep with checkpoints + reverse sweep with recomputation
    if a.adjoint > 0:
        import math
        every = max(1, int(round(math.sqrt(a.adjoint))))
        Ua = U.clone()
        ga = workloads.cotangent(U.shape, seed=3005 + rank, dtype=torch.float32, device=dev)
        s.adjoint(Ua, ga, a.adjoint, every)                  # warm-up: allocates the checkpoints
        Ua.copy_(U)
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        s.adjoint(Ua, ga, a.adjoint, every)
        e1.record()
        barrier()
        ms_a = max_over_ranks(e0.elapsed_time(e1))
        nck = -(-a.adjoint // every)
        line["adjoint"] = {"steps": a.adjoint, "checkpoint_every": every, "ms": ms_a,
                           "value": world * N * a.adjoint / (ms_a * 1e-3), "unit": "cell-step-adjoints/s",
                           "states_held": nck + every + 1,
                           "work": "forward sweep (CFL + step) + recomputation of every segment + one VJP per step"}
        del Ua, ga
        torch.cuda.empty_cache()

    # ---- end to end: pinned HOST state -> dh_run_host (H2D, CFL + step, D2H) -> HOST, all inside the timed region
    if not a.no_e2e:
        try:
            import psutil
            avail = psutil.virtual_memory().available
        except Exception:
            avail = 1 << 62
        state_bytes = 5 * 4 * N
        if avail < 2.5 * state_bytes:
            line["e2e"] = {"value": None, "unit": UNIT, "h2d_bytes_per_step": state_bytes, "d2h_bytes_per_step": state_bytes,
                           "note": f"skipped: host has {avail / 1e9:.0f} GB available, the pinned state needs {state_bytes / 1e9:.1f} GB"}
        else:
            h = torch.empty(U.shape, dtype=torch.float32, pin_memory=True)
            h.copy_(U)
            torch.cuda.synchronize()
            Ke = max(1, K)
            s.stream_host(h, max(1, W))                       # warm-up (allocates the library's device states, streams, events)
            barrier()
            t0 = time.perf_counter()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            s.stream_host(h, Ke)                              # Ke steps, each reading its input from h and writing its result there
            e1.record()
            barrier()
            wall = time.perf_counter() - t0
            ms_e = max_over_ranks(max(e0.elapsed_time(e1), wall * 1e3))
            # a shorter call, to separate the pipeline fill from the steady state: steady = (T(Ke) - T(K0)) / (Ke - K0)
            K0 = 2
            ms_steady = None
            if Ke > K0:
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                s.stream_host(h, K0)
                torch.cuda.synchronize()
                ms_steady = (ms_e - (time.perf_counter() - t0) * 1e3) / (Ke - K0)
            # the unpipelined call beside it: H2D, CFL + step, D2H, one after the other
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            s.run_host(h, 1)
            torch.cuda.synchronize()
            ms_serial = (time.perf_counter() - t0) * 1e3
            line["e2e"] = {"value": world * N * Ke / (ms_e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": state_bytes,
                           "d2h_bytes_per_step": state_bytes, "steps": Ke, "ms_per_step": ms_e / Ke,
                           "host_link_GB/s": 2 * state_bytes * Ke / (ms_e * 1e-3) / 1e9,
                           "steady_ms_per_step": ms_steady,
                           "steady_host_link_GB/s": (2 * state_bytes / (ms_steady * 1e-3) / 1e9) if ms_steady else None,
                           "serial_ms_per_step": ms_serial,
                           "call": f"dh_stream_host(ctx, U_host, {Ke}, &dt): every step reads the pinned host state (H2D) and writes it back "
                                   "(D2H) in z slabs on two copy streams, CFL + RK2 step between them; the timed call includes the "
                                   "pipeline fill (the first step's H2D overlaps nothing: dt needs the whole state); steady_ms_per_step: the difference to a "
                                   f"{K0}-step call per extra step; serial_ms_per_step: dh_run_host(ctx, U_host, 1)"}
            del h

    # ---- the oracle beside it, on this box's host cores (rank 0, N = 1 only)
    if U_cpu_block is not None:
        import oracle

        oracle.build()
        line["cpu_baseline"] = oracle_sample(U_cpu_block, wl.gamma, bool(a.cooling), with_vjp=not a.no_vjp, scheme=_scheme(a))
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


# ------------------------------------------------------------------------------- multigrid Poisson (--poisson N)
MG_WORDS_PER_CELL_CYCLE = (4 * 3 + 2.125 + 2.125) * 8.0 / 7.0   # nu1 = nu2 = 2 sweeps x (in, F, out) + fused
#   residual/restriction (phi, F, 1/8 out) + prolongation/correction (phi in, phi out, 1/8 in), all levels: x 8/7


def run_poisson(a):
    """K cycles of dh_mg_cycle on an N^3 fp32 grid (one JSON line; single GPU; the oracle's cycle timed on a 64^3 grid)."""
    import numpy as np
    import torch

    from paper_2512_13403_b200 import dh

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py --poisson needs a CUDA device: the path has no CPU fallback")
    n, K, W = a.poisson, a.steps, max(a.warmup, 3)
    torch.cuda.set_device(0)
    gen = torch.Generator(device="cuda").manual_seed(1006)
    F = torch.randn((n, n, n), generator=gen, device="cuda", dtype=torch.float32)
    F -= F.mean()
    phi = torch.zeros_like(F)
    s = dh.Multigrid(n, n, n, 1.0 / n, dtype=torch.float32, cycle=a.mg_cycle, subtree=a.mg_subtree)
    for _ in range(W):
        s.cycle(phi, F)
    phi.zero_()
    torch.cuda.synchronize()
    l0 = s.launches
    sampler = ClockSampler(0)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.time()
    e0.record()
    for _ in range(K):
        s.cycle(phi, F)
    e1.record()
    torch.cuda.synchronize()
    t1 = time.time()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop(t0, t1)
    launches = s.launches - l0
    N = n ** 3
    peak, peak_src = measured_peak()
    gbs = MG_WORDS_PER_CELL_CYCLE * 4.0 * N * K / (ms * 1e-3) / 1e9
    line = {"metric": f"cell-cycles/s (multigrid {a.mg_cycle}-cycle of the periodic Poisson solver, nu1 = nu2 = 2)", "value": N * K / (ms * 1e-3),
            "unit": "cell-cycles/s", "n_gpus": 1, "steps": K, "warmup": W, "ms_per_step": ms / K, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"poisson_multigrid_{n}^3_fp32 (white-noise zero-mean source, seed 1006)", "grid": [n, n, n], "cycle": a.mg_cycle,
                       "levels": s.levels, "nu1": 2, "nu2": 2, "nu_coarse": 64, "omega": 2.0 / 3.0, "call": "dh_mg_cycle(phi, F) x K (CUDA graph replay)",
                       "l2": f"inputs larger than L2 ({2 * 4 * N / 1e6:.0f} MB vs 126 MB), no flush" if 8 * N > 126e6 else "working set fits L2: not an HBM number"},
            "roofline": {"bound": "hbm", "kernel": "whole cycle (Jacobi sweeps dominate: 12 of 16.25 words per fine cell)", "achieved": gbs, "peak": peak,
                         "unit": "GB/s", "frac": gbs / peak, "peak_source": peak_src, "traffic": None,
                         "words_per_cell_cycle": MG_WORDS_PER_CELL_CYCLE},
            "clocks": clocks, "gpu_launches": launches}
    # convergence actually reached by the timed cycles (a property check, not a timing)
    r = F - (sum(torch.roll(phi, sh, d) for d in range(3) for sh in (1, -1)) - 6 * phi) * float(n * n)
    line["config"]["rel_residual_after_K_cycles"] = float(r.norm() / F.norm())
    if not a.no_e2e:
        hF = F.cpu().pin_memory()
        hphi = torch.empty_like(hF).pin_memory()
        dF, dphi = torch.empty_like(F), torch.empty_like(F)
        ncyc = 8
        t_best = None
        for _ in range(3):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            dF.copy_(hF, non_blocking=True)
            dh.dh_mg_solve(s.ctx, dF.data_ptr(), dphi.data_ptr(), ncyc, False)
            hphi.copy_(dphi, non_blocking=True)
            torch.cuda.synchronize()
            dt = time.perf_counter() - t0
            t_best = dt if t_best is None else min(t_best, dt)
        line["e2e"] = {"value": N * ncyc / t_best, "unit": "cell-cycles/s", "h2d_bytes_per_step": 4 * N, "d2h_bytes_per_step": 4 * N,
                       "ms_per_step": t_best * 1e3, "call": f"pinned host F -> device, dh_mg_solve({ncyc} cycles), phi -> pinned host"}
    if not a.no_cpu:
        from oracle import poisson as omg
        m = min(64, n)
        Fc = np.random.default_rng(1006).normal(size=(m, m, m))
        Fc -= Fc.mean()
        t0 = time.perf_counter()
        reps = 0
        x = np.zeros_like(Fc)
        while time.perf_counter() - t0 < 10.0:
            x = omg.cycle(x, Fc, 1.0 / m, gamma={"V": 1, "W": 2}[a.mg_cycle])
            reps += 1
        tc = time.perf_counter() - t0
        line["cpu_baseline"] = {"value": m ** 3 * reps / tc, "unit": "cell-cycles/s", "cores": 1, "kind": "oracle",
                                "sample": f"{reps} cycles of oracle.poisson.cycle on a {m}^3 grid ({tc:.1f} s, numpy fp64)"}
    print(json.dumps(line))


def run_issue_probe(a):
    """A measurement, not a benchmark of the path: prints one JSON line with the dh_issue_probe table."""
    import torch
    from paper_2512_13403_b200 import dh
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py --issue-probe needs a GPU")
    torch.cuda.set_device(0)
    rows = {}
    for wps in (2, 4):
        for r in dh.issue_probe(warps_per_scheduler=wps, iters=4000):
            e = rows.setdefault(r["mix"], {"instructions": r["instructions"]})
            e[f"cycles_per_group_{wps}_warps"] = round(r["cycles_per_group"], 3)
    print(json.dumps({"metric": "issue cost of instruction mixes (dh_issue_probe)", "unit": "SM cycles per group per scheduler",
                      "device": torch.cuda.get_device_name(0), "chains_per_thread": 8, "mixes": rows}))


def main():
    a = parse_args()
    if a.issue_probe:
        run_issue_probe(a)
    elif a.poisson:
        run_poisson(a)
    elif a.impl == "reference":
        run_reference(a)
    else:
        run_dh(a)


if __name__ == "__main__":
    main()
