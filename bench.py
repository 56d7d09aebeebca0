#!/usr/bin/env python3
"""bench.py -- trajectory-epoch evaluations per second of the whole hot path on synthetic DECam-shaped
stacks (BASELINE.json `metric`), one JSON line on stdout (rank 0).

A "step" is one pass of every SURVEY.md section-8(a) row over one stack: kbmod_prepare_psi_phi (a1),
kbmod_search = displacement table + gather + in-line sigma-G + per-pixel top-K (a2-a5), and
kbmod_coadd_stamps on a candidate list (a6).  N = 1 runs BASELINE configs[2] (2048x4096x26, 128x64
velocities, K=8, sigma-G on, min_lh = 10 = the paper's operating point).  N > 1: one
independent CCD stack per rank (replicas: 2580 independent per-CCD searches),
no data-path collective, "scaling": "weak".

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload c3|c2|c1|c4]
                  [--min-lh X] [--algo auto|direct|pruned] [--shard replicas|rows] [--no-extras]
`--impl reference` times the oracle (oracle/, plain C, double) on the host cores on a bounded sample
of the same workload; it is the only leg besides `cpu_baseline` that executes anything under oracle/.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2109_03296_b200 import synth  # noqa: E402  (input generators only: no method arithmetic)

METRIC = "trajectory_epoch_evals_per_s"
UNIT = "evals/s"


def load_peaks():
    """Measured peaks written by the driver; else the fallback B200_PROFILING.md states."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


def make_workload(name: str, seed_shift: int = 0):
    """Returns (stack, vx, vy, params-dict, description).  Recipes: DESIGN.md 'synthetic inputs'."""
    if name == "c3":
        st = synth.config3_decam(seed=2 + seed_shift)
        vx, vy = synth.config3_grid()
        return st, vx, vy, dict(K=8, min_obs=13), "configs[2] DECam-shaped 2048x4096x26, 128x64 velocities, K=8"
    if name == "c4":
        st = synth.config4_heavy(seed=3 + seed_shift)
        vx, vy = synth.config4_grid()
        return st, vx, vy, dict(K=16, min_obs=25), "configs[3] heavy 2048x4096x50, 256x128 velocities, K=16"
    if name == "paper":  # configs[2]'s stack searched with the paper's full 512 x 256 grid
        st = synth.config3_decam(seed=2 + seed_shift)
        vx, vy = synth.paper_grid()
        return st, vx, vy, dict(K=8, min_obs=13), "configs[2] stack x the paper's 512x256 velocity grid (131072), K=8"
    if name == "c2":
        st = synth.config2_medium(seed=1 + seed_shift)
        vx, vy = synth.config2_grid()
        return st, vx, vy, dict(K=8, min_obs=5), "configs[1] 512x512x10, 64x32 velocities, K=8"
    if name == "c1":
        st = synth.config1_tiny(seed=0 + seed_shift)
        vx, vy = synth.config1_grid()
        return st, vx, vy, dict(K=1, min_obs=3), "configs[0] tiny 64x64x5, 16x16 velocities, K=1"
    raise SystemExit(f"unknown workload {name}")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(self.index)], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=lambda: self.lines.extend(self.proc.stdout), daemon=True).start()
        except OSError:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2]))
            except ValueError:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        busy = [s for s in sm if s > 0]
        return dict(sm_mhz=float(np.median(busy)) if busy else None, sm_max_mhz=max(mx) if mx else None,
                    reasons=sorted(reasons), samples=len(sm))


# ----------------------------------------------------------------------------------------- oracle legs
def cpu_model() -> str:
    try:
        for ln in open("/proc/cpuinfo"):
            if ln.lower().startswith("model name"):
                return ln.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


class OracleSample:
    """The oracle (as it stands) on a bounded sample of the workload.  O1 runs once on a crop tall
    enough that most displaced epochs stay on it (real values: movers, masks, artefacts); what is
    timed is the search (O2-O6) on random start pixels of that crop, where the time goes.  (BASELINE.md planned 64
    full rows; random pixels of a crop sample the same trajectories without generating the O1 output of the whole
    stack in double precision, 3.5 GB.)"""

    def __init__(self, st, vx, vy, pd, min_lh):
        from oracle import oracle as O
        self.O, self.vx, self.vy, self.times = O, vx, vy, st.times
        T, H, W = st.img.shape
        self.T, self.ch, self.cw = T, min(H, 2048), min(W, 1024)
        ch, cw = self.ch, self.cw
        t0 = time.time()
        psi, phi, _, _ = O.prepare_psi_phi(st.img[:, :ch, :cw], st.var[:, :ch, :cw], st.mask[:, :ch, :cw], st.psf)
        self.t_prep = time.time() - t0
        self.psiphi = O.interleave(psi, phi)
        self.p = O.Params(K=pd["K"], min_obs=pd["min_obs"], min_lh=min_lh)
        self.rng = np.random.default_rng(123)
        self.rate = None
        self.all_threads = O.num_threads()

    def _run(self, n):
        px = self.rng.integers(0, self.cw, n).astype(np.int32)
        py = self.rng.integers(0, self.ch, n).astype(np.int32)
        t0 = time.time()
        self.O.search_pixels(self.psiphi, self.times, self.vx, self.vy, px, py, self.p)
        return max(time.time() - t0, 1e-6)

    def step(self, target_s):
        """One bounded sample of about target_s seconds.  Returns (evals/s, cores, description, seconds)."""
        if self.rate is None:
            self.rate = 256 / self._run(256)  # pixels per second, probe
        n = int(min(max(256, self.rate * target_s), self.ch * self.cw))
        dt = self._run(n)
        self.rate = n / dt
        evals = float(n) * len(self.vx) * self.T
        desc = (f"oracle search (O2-O6) on {n} random start pixels of a {self.cw}x{self.ch} crop x all {len(self.vx)} "
                f"velocities x {self.T} epochs = {evals:.3g} evals in {dt:.1f} s (O1 on the crop, {self.t_prep:.1f} s, "
                f"not counted)")
        return evals / dt, self.O.num_threads(), desc, dt

    def one_core(self, target_s=4.0):
        """The same on ONE thread ('all cores and 1 core')."""
        self.O.set_num_threads(1)
        try:
            n = int(max(64, (self.rate or 1000.0) / max(1, self.all_threads) * target_s))
            dt = self._run(n)
            return float(n) * len(self.vx) * self.T / dt
        finally:
            self.O.set_num_threads(self.all_threads)


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    peaks = load_peaks()
    st, vx, vy, pd, desc = make_workload(args.workload)
    T, H, W = st.img.shape
    per_step = max(2.0, min(20.0, 150.0 / max(1, args.steps + args.warmup)))
    rates, times_s = [], []
    cores, sample = 0, ""
    smp = OracleSample(st, vx, vy, pd, args.min_lh)
    for i in range(args.warmup + args.steps):
        r, cores, sample, dt = smp.step(per_step)
        if i >= args.warmup:
            rates.append(r); times_s.append(dt)
    value = float(np.mean(rates))
    line = dict(impl="reference", metric=METRIC, value=value, unit=UNIT, n_gpus=args.gpus, steps=args.steps,
                warmup=args.warmup, ms_per_step=1e3 * float(np.mean(times_s)), higher_is_better=True, scaling="weak",
                vs_baseline=None, dtype="f64", data="synthetic",
                config=dict(workload=desc, min_lh=args.min_lh, sigma_g="on", note="each step = a bounded sample"),
                cpu_baseline=dict(value=value, unit=UNIT, cores=cores, kind="oracle", sample=sample, cpu=cpu_model()),
                e2e=dict(value=value, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0,
                peaks_source=peaks["source"])
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------------------- GPU arm
# Algorithmic work per unit for the roofline.
#   direct kernel  : bound "alu" -- every trajectory runs the compare-exchange network; FMNMX, FSETP, LOP3 and SHF
#                    issue on the half-rate ALU pipe (2 warp-instructions per clock per SM, measured live by
#                    kbmod_measure_issue_rate): achieved = ALU-pipe warp-instructions per trajectory (from the
#                    committed ncu capture) x trajectories / live kernel time; peak = 148 SMs x 2 x f_max.
#   pruned path    : bound "smem" -- the dominant kernel, bound_phase_kernel, gathers one packed 32-bit word
#                    (fixed-point psi_+ | low-phi flag | valid flag) per trajectory-epoch evaluation from shared
#                    memory: 4 B algorithmic; peak = 148 SMs x 128 B/clk x f_max.  Its duration is measured live
#                    with CUDA events recorded by the library on the launching stream (kbmod_search_phase_ms).
#                    SURVEY 8(d) counted 8 B per evaluation (psi and phi as float32): reported beside it.
# dram__bytes_read.sum + dram__bytes_write.sum per step of the dominant kernel from the committed ncu --set full
# capture (profiles/); None = not captured for this kernel
TRAFFIC = {"bound_phase_kernel": 15.8e9, "search_direct_kernel": 1.37e12}  # bytes per step: profiles/r2_launches.md, r2_search_direct_kernel_full.md
CE_COUNT = {4: 5, 5: 9, 8: 19, 10: 32, 12: 42, 16: 63, 20: 103, 24: 132, 26: 147, 28: 162, 32: 191, 40: 305,
            48: 384, 50: 403, 56: 464, 64: 543}
N_SM = 148
# executed warp-instructions per warp-trajectory of search_direct_kernel<TP> (ncu smsp__inst_executed / (trajectories / 32),
# profiles/r2_search_direct_kernel_full.md); other TP: scaled by the compare-exchange count
DIRECT_WARP_INSTR_PER_TRAJ = {26: 585.7}
# of which on the half-rate ALU pipe (FMNMX, FSETP, LOP3, SHF ...): sm__inst_executed_pipe_alu of the same capture,
# 74.4 % of 2 per clock over the active cycles
DIRECT_ALU_INSTR_PER_TRAJ = {26: 356.0}
ALU_PIPE_PER_CLK = 2.0  # warp-instructions per clock per SM (16 lanes per scheduler); measured live beside it: issue_rates FMNMX


def direct_roofline(T, tp, n_traj, kernel_ms, f_max, issue):
    """The direct kernel is bound by the half-rate ALU pipe: 2 x 147 FMNMX of the sorting network + 2 FSETP per epoch
    of the clip + the valid-bit shift-adds per trajectory (T = 26: 356 of its 586 warp-instructions)."""
    if T <= max(DIRECT_WARP_INSTR_PER_TRAJ):
        k = min(k for k in DIRECT_WARP_INSTR_PER_TRAJ if k >= T)
        per, per_alu = DIRECT_WARP_INSTR_PER_TRAJ[k], DIRECT_ALU_INSTR_PER_TRAJ[k]
    else:  # other network sizes: scaled by the compare-exchange count
        per = 585.7 * CE_COUNT[tp] / CE_COUNT[26]
        per_alu = 356.0 * CE_COUNT[tp] / CE_COUNT[26]
    warp_traj = n_traj / 32.0
    peak = N_SM * ALU_PIPE_PER_CLK * f_max
    ach = warp_traj * per_alu / (kernel_ms * 1e-3)
    return dict(bound="alu", kernel="search_direct_kernel", achieved=ach / 1e12, peak=peak / 1e12, unit="Twarp-instr/s",
                frac=ach / peak, alu_pipe_warp_instr_per_trajectory=per_alu, warp_instr_per_trajectory=per,
                issue_frac=warp_traj * per / (kernel_ms * 1e-3) / (N_SM * 4 * f_max),
                alu_pipe_rate_measured_live=(issue or {}).get("FMNMX"),
                peak_source="derived: 148 SMs x 2 ALU-pipe warp-instructions per clock x sm_max_mhz; the live FMNMX issue "
                            "rate (kbmod_measure_issue_rate) is beside it",
                source="instruction counts per trajectory from profiles/r2_search_direct_kernel_full.md")


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_2109_03296_b200 as kb

    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    kb.binding.lib()
    kb.kbmod_search_phase_timing(True)
    peaks = load_peaks()
    dev = torch.device("cuda", local)

    shard_rows = args.shard == "rows" and world > 1
    # replicas (default): one CCD stack per rank.  --shard rows: ONE stack, every rank holds all of it and searches its
    # band of start rows; the bands' results concatenate, no collective
    st, vx, vy, pd, desc = make_workload(args.workload, seed_shift=0 if shard_rows else 100 * rank)
    T, H, W = st.img.shape
    algo = dict(auto=kb.ALGO_AUTO, direct=kb.ALGO_DIRECT, pruned=kb.ALGO_PRUNED)[args.algo]
    sp = kb.SearchParams(K=pd["K"], min_obs=pd["min_obs"], min_lh=args.min_lh, algo=algo)
    n_vel = len(vx)
    evals = float(H) * W * n_vel * T

    # inputs resident in HBM before the timed region
    img, var, mask = (torch.from_numpy(a).to(dev) for a in (st.img, st.var, st.mask))
    psiphi = torch.empty((T, H, W, 2), dtype=torch.float32, device=dev)
    rows = row_band(rank, world, H) if shard_rows else None
    n_rows = H if rows is None else rows[1] - rows[0]
    out = tuple(torch.empty((n_rows, W, sp.K), dtype=dt, device=dev)
                for dt in (torch.float32, torch.float32, torch.int32, torch.int32))
    ws = torch.empty(max(256, kb.kbmod_search_workspace_bytes_for(T, H, W, st.times, vx, vy, sp, rows=rows)), dtype=torch.uint8,
                     device=dev)
    if shard_rows:
        evals = float(H) * W * n_vel * T / world  # per rank; whole_job_value multiplies by world
    n_cand = min(100_000, H * W)  # (a6) candidate list: configs[4]'s recipe
    cx0, cy0, cvx, cvy = (torch.from_numpy(a).to(dev) for a in synth.config5_trajectories(4 + rank, H, W, n_cand))

    ev = lambda: torch.cuda.Event(enable_timing=True)
    seg = {"prep": [], "search": [], "coadd": []}
    phases = []  # per timed step: the library's own events between the phases of kbmod_search

    def step(record):
        e = [ev() for _ in range(4)]
        e[0].record()
        kb.kbmod_prepare_psi_phi(img, var, mask, st.psf, out=psiphi)
        e[1].record()
        kb.kbmod_search(psiphi, st.times, vx, vy, sp, out=out, workspace=ws, rows=rows)
        e[2].record()
        kb.kbmod_coadd_stamps_filtered(img, mask, st.times, cx0, cy0, cvx, cvy, 10)  # (a6) + the moment filter (L141)
        e[3].record()
        if record is not None:
            record.append(e)
            phases.append(kb.kbmod_search_phase_ms())  # waits for this step's search: between steps, not inside one

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step(None)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    recs = []
    t_beg, t_end = ev(), ev()
    t_beg.record()
    for _ in range(args.steps):
        step(recs)
    t_end.record()
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    total_ms = t_beg.elapsed_time(t_end)
    for e in recs:
        seg["prep"].append(e[0].elapsed_time(e[1])); seg["search"].append(e[1].elapsed_time(e[2]))
        seg["coadd"].append(e[2].elapsed_time(e[3]))
    stats = kb.kbmod_search_stats(ws)  # [evaluated, nominal, launches, algo]
    smem_gbs = {b: kb.kbmod_measure_smem_gbs(b) for b in (4, 16)}  # after the timed region
    issue = {n: kb.kbmod_measure_issue_rate(i) for i, n in enumerate(("FMNMX", "IADD3", "FADD", "FMNMX+IADD3_exchange"))}
    plan_info = kb.Plan(T, H, W, st.times, vx, vy, sp, rows=rows).info()  # host-only: what the planner staged / skipped
    R = dict(torch=torch, dist=dist, kb=kb, rank=rank, world=world, dev=dev, st=st, vx=vx, vy=vy, pd=pd, sp=sp,
             desc=desc, evals=evals, total_ms=total_ms, seg=seg, stats=stats, clocks=clocks, peaks=peaks, phases=phases,
             n_cand=n_cand, out=out, shard_rows=shard_rows, rows=rows, smem_gbs=smem_gbs, issue=issue, plan_info=plan_info, psiphi=psiphi, ws=ws, extras={})
    # ---- more timed records on the same box, after the headline region (rank 0 of a 1-GPU run, default workload)
    if rank == 0 and world == 1 and args.workload == "c3" and not args.no_extras and args.algo == "auto" and args.min_lh == 10.0:
        R["extras"]["mode_b"] = time_search(R, "configs[2], mode (B): min_lh = -inf, every trajectory filtered (SURVEY 8d)", st, psiphi,
                                            vx, vy, dict(pd), -math.inf, steps=2, warmup=1)
        pvx, pvy = synth.paper_grid()
        R["extras"]["paper_grid"] = time_search(R, "configs[2] stack x the paper's 512 x 256 velocity grid (PAPER.md L167), min_lh = 10",
                                                st, psiphi, pvx, pvy, dict(pd), 10.0, steps=1, warmup=1)
        R["extras"]["postfilter"] = time_postfilter(R)
        del img, var, mask, psiphi, ws
        R["psiphi"] = R["ws"] = None
        torch.cuda.empty_cache()
        R["extras"]["configs2_without_star_residuals"] = time_clean(R)
        R["extras"]["configs3_heavy"] = time_heavy(R)
    return R


def time_search(R, what, st, psiphi, vx, vy, pd, min_lh, steps, warmup):
    """Device time of kbmod_search alone (psi/phi resident) on another grid / mode; events on the launching stream."""
    torch, kb = R["torch"], R["kb"]
    T, H, W = st.img.shape
    sp = kb.SearchParams(K=pd["K"], min_obs=pd["min_obs"], min_lh=min_lh)
    ws = torch.empty(max(256, kb.kbmod_search_workspace_bytes_for(T, H, W, st.times, vx, vy, sp)), dtype=torch.uint8, device=R["dev"])
    out = tuple(torch.empty((H, W, sp.K), dtype=dt, device=R["dev"]) for dt in (torch.float32, torch.float32, torch.int32, torch.int32))
    ms, ph = [], []
    for i in range(warmup + steps):
        b, e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        b.record()
        kb.kbmod_search(psiphi, st.times, vx, vy, sp, out=out, workspace=ws)
        e.record()
        torch.cuda.synchronize()
        if i >= warmup:
            ms.append(b.elapsed_time(e)); ph.append(kb.kbmod_search_phase_ms())
    evaluated, nominal, launches, algo_used, reached = kb.kbmod_search_stats(ws)
    evals = float(H) * W * len(vx) * T
    m = float(np.mean(ms))
    rec = dict(workload=what, search_ms=m, value=evals / (m * 1e-3), unit=UNIT, steps=steps, warmup=warmup,
               algo={1: "direct", 2: "pruned"}.get(algo_used, "?"), evaluated_fraction=evaluated / max(1, nominal),
               trajectories_reaching_min_lh=reached,
               trajectories=float(H) * W * len(vx), workspace_gb=ws.numel() / 1e9,
               search_phases_ms={k: float(np.mean([p[k] for p in ph])) for k in ph[0]},
               filled_result_slots=int((out[2] >= 0).sum()))
    if algo_used == kb.ALGO_DIRECT:
        tp = min(k for k in CE_COUNT if k >= T)
        kern_ms = rec["search_phases_ms"]["gather"]
        rec["roofline"] = direct_roofline(T, tp, float(H) * W * len(vx), kern_ms, R["peaks"]["sm_max_mhz"] * 1e6, R.get("issue"))
        rec["roofline"]["kernel_ms"] = kern_ms
        rec["roofline"]["traffic"] = TRAFFIC["search_direct_kernel"] if T == 26 and len(vx) == 8192 else None
    del ws, out
    return rec


def time_postfilter(R):
    """N1 (the CPU post-filter rejects ~10^6 trajectories in ~60 s on 30 cores -- context, another
    machine): kbmod_sigmag_postfilter (sigma-G, reject L' < 10, ordered survivor list) on 10^6 and 10^7 lightcurves
    of 26 epochs resident on the device."""
    torch, kb = R["torch"], R["kb"]
    out = {}
    g = torch.Generator(device=R["dev"]).manual_seed(7)
    for n in (1_000_000, 10_000_000):
        phi = torch.rand((n, 26), generator=g, device=R["dev"]) * 7e-5 + 5e-5
        psi = (torch.randn((n, 26), generator=g, device=R["dev"]) + 1.5) * phi.sqrt()
        sp = kb.SearchParams(K=1, min_obs=13, min_lh=10.0)
        kb.kbmod_sigmag_postfilter(psi, phi, sp)
        torch.cuda.synchronize()
        b, e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        b.record()
        r = kb.kbmod_sigmag_postfilter(psi, phi, sp)
        e.record()
        torch.cuda.synchronize()
        ms = b.elapsed_time(e)
        out[f"n={n}"] = dict(ms=ms, lightcurves_per_s=n / (ms * 1e-3), survivors=int(r["n_pass"][0]),
                             hbm_gbs=n * 26 * 8 / (ms * 1e-3) / 1e9)
        del phi, psi, r
    out["paper"] = "~1e6 rejections in ~60 s on 30 CPU cores (PAPER.md L123; other hardware: context)"
    return out


def time_clean(R):
    """How much the headline depends on the synthetic artefacts: the configs[2] recipe WITHOUT the 500 star residuals
    (cosmic rays, masks and movers kept).  The bound phase does the same work on any data; the survivors, and with
    them the exact phase, are what the artefacts drive."""
    torch, kb = R["torch"], R["kb"]
    st = synth.decam_stack(2, (7, 6, 7, 6), n_stars=0, name="config3_no_stars")
    vx, vy = synth.config3_grid()
    img, var, mask = (torch.from_numpy(a).to(R["dev"]) for a in (st.img, st.var, st.mask))
    psiphi = kb.kbmod_prepare_psi_phi(img, var, mask, st.psf)
    del img, var, mask
    rec = time_search(R, "configs[2] recipe without the star residuals, min_lh = 10", st, psiphi, vx, vy, dict(K=8, min_obs=13), 10.0,
                      steps=2, warmup=1)
    del psiphi
    torch.cuda.empty_cache()
    return rec


def time_heavy(R):
    """BASELINE configs[3] (2048x4096x50, 256 x 128 velocities, K = 16): prep + search, one warm-up and one timed pass."""
    torch, kb = R["torch"], R["kb"]
    st, vx, vy, pd, desc = make_workload("c4")
    img, var, mask = (torch.from_numpy(a).to(R["dev"]) for a in (st.img, st.var, st.mask))
    psiphi = kb.kbmod_prepare_psi_phi(img, var, mask, st.psf)
    del img, var, mask
    rec = time_search(R, desc + ", min_lh = 10", st, psiphi, vx, vy, pd, 10.0, steps=1, warmup=1)
    del psiphi
    torch.cuda.empty_cache()
    return rec


def in_bounds_fraction(times, vx, vy, H, W) -> float:
    """Share of the nominal trajectory-epoch evaluations whose position is on the image (reported beside
    the nominal count).  Positions follow reading R5: start + floor(v dt + 1/2)."""
    dt = np.asarray(times, np.float64) - float(times[0])
    dx = np.floor(np.asarray(vx, np.float64)[:, None] * dt[None, :] + 0.5)
    dy = np.floor(np.asarray(vy, np.float64)[:, None] * dt[None, :] + 0.5)
    return float((np.clip(W - np.abs(dx), 0, None) * np.clip(H - np.abs(dy), 0, None)).mean() / (float(W) * H))


def max_over_ranks(ms_local: float, dist, device, world: int) -> float:
    """Device time of the timed region: the MAX over ranks (every rank gets it)."""
    import torch
    t = torch.tensor([ms_local], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def row_band(rank: int, world: int, H: int):
    """Start rows [begin, end) of `rank` when one stack is sharded over `world` ranks by row bands."""
    return H * rank // world, H * (rank + 1) // world


def whole_job_value(evals_per_rank: float, world: int, ms_per_step: float) -> float:
    """Replicas only: every rank processes its own stack, so the job did world x evals in ms_per_step."""
    return world * evals_per_rank / (ms_per_step * 1e-3)


def run_e2e(R, steps):
    """Same metric end to end through the C-ABI call with HOST buffers (kbmod_pipeline_host_batch): every step is
    one stack -- its image/variance/mask planes are copied from pinned host memory, prep + search run, and the four
    result arrays are read back; the copies of step i+1 / i-1 overlap the search of step i.  Timed on the device
    with events around the call (the call itself synchronises after the last result has landed)."""
    torch, kb, st, sp = R["torch"], R["kb"], R["st"], R["sp"]
    T, H, W = st.img.shape
    h_in = tuple(torch.from_numpy(a).pin_memory() for a in (st.img, st.var, st.mask))
    h_out = tuple(torch.empty((H, W, sp.K), dtype=dt).pin_memory()
                  for dt in (torch.float32, torch.float32, torch.int32, torch.int32))
    arena = torch.empty(2 * kb.kbmod_pipeline_host_arena_bytes_for(T, H, W, st.times, R["vx"], R["vy"], sp), dtype=torch.uint8,
                        device=R["dev"])
    h2d = sum(a.numel() * a.element_size() for a in h_in)
    d2h = sum(a.numel() * a.element_size() for a in h_out)
    kb.kbmod_pipeline_host_batch([h_in], st.psf, st.times, R["vx"], R["vy"], sp, [h_out], arena)  # warm-up
    b, e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    b.record()
    kb.kbmod_pipeline_host_batch([h_in] * steps, st.psf, st.times, R["vx"], R["vy"], sp, [h_out] * steps, arena)
    e.record()
    torch.cuda.synchronize()
    ms = b.elapsed_time(e) / steps
    # the host result must be the device result of the resident-input run (same inputs)
    same = bool(torch.equal(h_out[2], R["out"][2].cpu()))
    del arena
    return ms, h2d, d2h, same


def report(R, args):
    torch, dist, kb = R["torch"], R["dist"], R["kb"]
    rank, world = R["rank"], R["world"]
    # max over ranks of the device time of the timed region
    total_ms = max_over_ranks(R["total_ms"], dist, R["dev"], world)
    # stacks of one kbmod_pipeline_host_batch call (a pointing group has 60 CCD stacks, L39): the first input copy and the
    # last result copy of a call cannot overlap a search (about 55 ms of fill and drain per call at 55 GB/s)
    e2e_steps = max(10, min(args.steps, 20))
    # (the end-to-end leg is the replica path's: one whole stack per call; a row-band run reports the resident figure only)
    e2e_ms, h2d, d2h, same = run_e2e(R, e2e_steps) if not R["shard_rows"] else (0.0, 0, 0, False)
    e2e_max = max_over_ranks(e2e_ms, dist, R["dev"], world)
    if rank != 0:
        return
    ms_per_step = total_ms / args.steps
    value = whole_job_value(R["evals"], world, ms_per_step)
    st, sp, peaks = R["st"], R["sp"], R["peaks"]
    T, H, W = st.img.shape
    n_vel = len(R["vx"])
    search_ms = float(np.mean(R["seg"]["search"]))
    evaluated, nominal, launches, algo_used, reached = R["stats"]
    f_max = peaks["sm_max_mhz"] * 1e6
    tp = min(k for k in CE_COUNT if k >= T)
    ph = {k: float(np.mean([p[k] for p in R["phases"]])) for k in R["phases"][0]}
    kernel_ms = ph["gather"]  # the dominant kernel alone: bound_phase_kernel launches / the direct kernel
    pi = R["plan_info"]
    if algo_used == kb.ALGO_DIRECT:
        roof = direct_roofline(T, tp, float(H) * W * n_vel, kernel_ms, f_max, R.get("issue"))
    else:
        # one packed 32-bit bound word per trajectory-epoch evaluation.  `frac` counts the words the
        # kernel PHYSICALLY loads from shared memory: the nominal count less the (tile, group, epoch) regions that lie
        # off the image and are skipped, less the epochs at which a whole velocity group shares one displacement
        # (gathered once per pixel) -- both from the host plan (kbmod_plan_info).  The nominal figure is kept beside it.
        nominal_bytes = R["evals"] * 4.0
        phys_bytes = nominal_bytes * (1.0 - pi["off_image_fraction"]) * pi["gather_fraction"]
        # denominator: the shared-memory load bandwidth measured live on this GPU (LDS.128 microbenchmark of the
        # library: the highest of the three widths); the derived figure and the LDS.32 figure are quoted beside it
        peak = R["smem_gbs"][16]
        roof = dict(bound="smem", achieved=phys_bytes / (kernel_ms * 1e-3) / 1e9, peak=peak,
                    unit="GB/s", kernel="bound_phase_kernel",
                    what="shared-memory bytes the kernel loads (in-bounds, unique gathers) / live kernel time",
                    peak_source="measured live: kbmod_measure_smem_gbs(16), conflict-free LDS.128 on all SMs",
                    peak_theoretical=N_SM * 128 * f_max / 1e9, peak_measured_lds32=R["smem_gbs"][4],
                    algorithmic_bytes_per_eval=4, off_image_region_share=pi["off_image_fraction"],
                    gathers_per_nominal_eval=pi["gather_fraction"],
                    nominal_achieved=nominal_bytes / (kernel_ms * 1e-3) / 1e9,
                    nominal_frac=nominal_bytes / (kernel_ms * 1e-3) / 1e9 / peak,
                    # SURVEY 8(d) counted 8 B (psi, phi as float32) per NOMINAL evaluation over the whole search
                    # (a deviation recorded in DESIGN.md section 6); against that figure:
                    whole_search_frac_of_survey_8B_roofline=2.0 * nominal_bytes / (search_ms * 1e-3) / 1e9 / peak,
                    whole_search_frac_4B_nominal=nominal_bytes / (search_ms * 1e-3) / 1e9 / peak)
    roof["frac"] = roof["achieved"] / roof["peak"]
    roof["traffic"] = TRAFFIC.get(roof["kernel"])
    roof["kernel_ms"] = kernel_ms
    roof["kernel_share_of_step"] = kernel_ms / ms_per_step
    roof["search_phases_ms"] = ph
    cpu = None
    if not args.no_cpu_baseline:
        smp = OracleSample(st, R["vx"], R["vy"], R["pd"], args.min_lh)
        r, cores, sample, _ = smp.step(12.0)
        cpu = dict(value=r, unit=UNIT, cores=cores, kind="oracle", sample=sample, value_one_core=smp.one_core(), cpu=cpu_model())
    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=args.warmup,
                ms_per_step=ms_per_step, higher_is_better=True, scaling="strong" if R["shard_rows"] else "weak", vs_baseline=None,
                dtype="f32",
                data="synthetic",
                config=dict(workload=R["desc"], min_lh=args.min_lh, min_obs=sp.min_obs, sigma_g="on",
                            algo={1: "direct", 2: "pruned"}.get(algo_used, "?"), coadd_candidates=R["n_cand"],
                            l2=("inputs larger than L2 (psi/phi stack %.2f GB)" % (T * H * W * 8 / 1e9)) if T * H * W * 8 > 2.6e8 else
                               "inputs SMALLER than L2 and no flush: a parity-test configuration, not a cold-cache measurement",
                            multi_gpu=("one CCD stack sharded by start-row bands, whole stack on every rank, results concatenate, "
                                       "no collective" if R["shard_rows"] else
                                       "one independent CCD stack per rank, no collective") if world > 1 else "single GPU",
                            host_plan="velocity grouping / staging geometry cached after the first (warm-up) step: same grid and times"),
                segments_ms={k: float(np.mean(v)) for k, v in R["seg"].items()},
                evaluated_fraction=evaluated / max(1, nominal), trajectories_reaching_min_lh=reached,
                in_bounds_fraction=in_bounds_fraction(st.times, R["vx"], R["vy"], H, W),
                roofline=roof, cpu_baseline=cpu,
                e2e=dict(value=whole_job_value(R["evals"], world, e2e_max) if e2e_max > 0 else None, unit=UNIT, h2d_bytes_per_step=h2d,
                         d2h_bytes_per_step=d2h, ms_per_step=e2e_max, steps=e2e_steps,
                         matches_resident_run=same, api="kbmod_pipeline_host_batch (prep + search per stack; pinned host buffers; copies overlap the neighbouring searches)"),
                gpu_launches=args.steps * (T + int(launches) + 1), clocks=R["clocks"], peaks_source=peaks["source"],
                issue_rates_warp_instr_per_clk_per_sm=R["issue"],
                planner=dict(n_groups=pi["n_groups"], staged_bytes_per_eval=pi["staged_bytes_per_eval"],
                             canvas=pi["canvas"], workspace_gb=pi["workspace_bytes"] / 1e9),
                **R["extras"])
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c3", choices=["c1", "c2", "c3", "c4", "paper"])
    ap.add_argument("--min-lh", type=float, default=10.0, dest="min_lh")
    ap.add_argument("--algo", default="auto", choices=["auto", "direct", "pruned"])
    ap.add_argument("--shard", default="replicas", choices=["replicas", "rows"],
                    help="N > 1: independent CCD stacks per rank (default) or one stack sharded by start-row bands")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the mode-B / paper-grid / configs[3] / post-filter records")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    R = run_ours(args)
    report(R, args)
    if R["world"] > 1:
        R["dist"].destroy_process_group()


if __name__ == "__main__":
    main()
