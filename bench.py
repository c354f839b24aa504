#!/usr/bin/env python
"""bench.py -- the regular-force step of NBODY6+P3T on B200 (BASELINE.json metric:
regular-force particles/s and interactions/s at N = 1M; ms per force step).

A "step" is one pass of the whole hot path over one synthetic cluster:
p3t_build_tree + p3t_regular_force (cube, keys, sort, octree, moments, groups, walk, p-c / p-p force
with cutoff, neighbour lists, scatter), i.e. what the host integrator asks for once per dt_reg
(PAPER.md:89-94).  Default workload = BASELINE config 3 (Plummer 2^20, Kroupa masses, theta 0.4).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--configs all|none] [--impl ours|reference]

Prints ONE JSON line (rank 0).  `value` times the path with inputs resident in HBM; `e2e` times
p3t_step_host with pinned HOST buffers (H2D of positions, D2H of forces and neighbour lists inside
the timed region).  `roofline` is for the dominant kernel (k_force), an FP32-ALU-bound kernel, with the
algorithmic work stated two ways (SURVEY 8d's formula counts, and the counts of the kernel's own SASS);
`configs` holds the device-resident numbers of the other BASELINE.json configs (1, 2, 4, 5 x theta) from the
same run; `cpu_baseline` is the fp64 oracle on the host cores (full-N tree, 32 768 direct-sum targets, grid
neighbour search).  Multi-GPU: `--gpus N` without a torchrun environment starts N ranks itself; by default
every rank runs an independent replica ("replicas only", weak scaling; north_star is a one-GPU path).
`--mode sharded` splits the target groups of ONE cluster among the ranks
(paper_2110_11658_b200.shard; strong scaling; the all-gather of acc_pot and of the neighbour rows is inside the
timed region); with one GPU, `--mode sharded --sim-ranks R` runs the R shards in turn and reports each rank's time.
"""
from __future__ import annotations

import argparse
import csv
import json
import os
import socket
import subprocess
import sys
import tempfile
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

# FP32-pipe lane-instructions the method needs per interaction, stated two ways:
#  SURVEY.md 8(d)'s estimates from the formulas (what `roofline.frac` has used since round 1), and
#  the counts of the kernel's own SASS (FADD/FMUL/FFMA, packed ones counted twice; ncu's
#  smsp__sass_thread_inst_executed_op_f*_pred_on on an all-p-p launch and on config 3: profiles/r02_sass_counts.md).
INSTR_PP, INSTR_PC = 15, 37
INSTR_PP_SASS, INSTR_PC_SASS = 13.0, 33.0
FLOP_PP, FLOP_PC = 20, 60
# SURVEY.md 8(d) work table (probe: NCRIT = 32 canonical groups): FP32-pipe instructions per particle, 15 pp + 37 pc
SURVEY_INSTR_PER_PARTICLE = {(1, 0.4): 75e3, (2, 0.4): 131e3, (3, 0.4): 158e3, (4, 0.4): 155e3,
                             (5, 0.3): 318e3, (5, 0.5): 95e3, (5, 0.7): 45e3}
NLEAF, NCRIT, KEY_BITS = 16, 64, 63


def peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        return dict(hbm_gbs=float(d.get("hbm_gbs", 6650.0)), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


TRAFFIC_CSV = "r03_traffic.csv"                            # ncu --set full capture of the round's final build (profiles/r03_traffic.md)


def ncu_traffic(workload: str, kernel: str = "k_force"):
    """DRAM bytes per launch of the dominant kernel from the committed ncu capture (profiles/r03_traffic.csv:
    workload, kernel, dram_bytes_read, dram_bytes_write), or None when there is no row for this workload."""
    p = ROOT / "profiles" / TRAFFIC_CSV
    if not p.exists():
        return None
    with p.open() as f:
        for row in csv.DictReader(f):
            if row["workload"] == workload and row["kernel"] == kernel:
                return float(row["dram_bytes_read"]) + float(row["dram_bytes_write"])
    return None


def config_dict(w, world: int = 1) -> dict:
    return {"workload": w.name, "n": w.n, "r_out": w.r_out, "r_in": w.r_in, "theta": w.theta, "key_bits": KEY_BITS,
            "nleaf": NLEAF, "ncrit": NCRIT, "l2": "flushed between timed iterations (512 MiB write)",
            "parallelism": "replicas only" if world > 1 else "1 GPU"}


def stat3(x) -> dict:
    x = [float(v) for v in x]
    return {"mean": float(np.mean(x)), "median": float(np.median(x)), "min": float(np.min(x))}


class ClockSampler:
    """nvidia-smi clocks line of /opt/skills/guides/B200_PROFILING.md, sampled during the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "20",
                                       "-i", str(index)], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self) -> dict:
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush(); self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); mx.append(float(c[2]))
            except ValueError:
                continue
            for name, v in zip(names, c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        self.f.close()
        try:
            os.unlink(self.f.name)
        except OSError:
            pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": float(max(mx)) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------------------------
# the oracle on the host cores: cpu_baseline leg and the --impl reference arm (the only users of oracle/ here)
# ---------------------------------------------------------------------------------------------
def oracle_tree_run(w, group_stride: int = 1):
    """The oracle as it stands: full tree build + fp64 tree force of every group (group_stride 1: the full N,
    SURVEY 8d (i)) or of every k-th group (the bounded sample of the --impl reference arm)."""
    import oracle
    t0 = time.perf_counter()
    T = oracle.Tree(w.pos_mass, KEY_BITS, NLEAF, NCRIT)
    t_build = time.perf_counter() - t0
    g = T.groups()
    cnt = (g["end"] - g["begin"]).astype(np.int64)
    gi = None if group_stride <= 1 else np.arange(0, T.n_groups, group_stride, dtype=np.int64)
    t0 = time.perf_counter()
    f = T.force(w.r_out, w.r_in, w.theta, 0, group_ids=gi)
    t_force = time.perf_counter() - t0
    c = cnt if gi is None else cnt[gi]
    n_s = int(c.sum())
    inter = int(((f["npp"] + f["npc"]) * c).sum())
    t_full = t_build + t_force * w.n / n_s                  # = the measured time when the sample is everything
    return dict(t_build=t_build, t_force=t_force, n_sample=n_s, groups=len(c), stride=max(1, group_stride), interactions=inter,
                particles_per_s=w.n / t_full, interactions_per_s=inter / t_force, t_full=t_full, cores=oracle.omp_threads())


def cpu_baseline(w) -> dict:
    """SURVEY 8(d) / BASELINE.md section 4, on this box's host cores, the oracle untuned:
    (i) the fp64 CPU tree on the full N (N <= 2^20; a group sample above), (ii) eq. 3 by direct summation on 32 768
    stride-sampled targets (all N for N <= 32 768), (iii) the neighbour search (cell grid above 131 072, else brute force)."""
    import oracle
    import workloads
    r = oracle_tree_run(w, 1 if w.n <= (1 << 20) else 8)
    n_t = min(w.n, 32768)
    t0 = time.perf_counter()
    oracle.direct(w.pos_mass, w.r_out, w.r_in, targets=workloads.sample_targets(w.n, n_t))
    t_direct = time.perf_counter() - t0
    t0 = time.perf_counter()
    if w.n > 131072:
        off, _ = oracle.neighbours_grid(w.pos_mass, w.r_out); kind = "uniform cell grid"
    else:
        off, _ = oracle.neighbours(w.pos_mass, w.r_out); kind = "brute force"
    t_nb = time.perf_counter() - t0
    full = r["stride"] == 1
    return {
        "value": r["particles_per_s"], "unit": "particles/s", "cores": r["cores"], "kind": "oracle",
        "interactions_per_s": r["interactions_per_s"], "tree_seconds": r["t_full"], "tree_build_seconds": r["t_build"],
        "direct_sum": {"pairs_per_s": n_t * float(w.n) / t_direct, "targets": n_t, "seconds": t_direct,
                       "full_n2_seconds_extrapolated": t_direct * w.n / n_t},
        "neighbour_search": {"kind": kind, "seconds": t_nb, "entries": int(off[-1]), "targets_per_s": w.n / t_nb,
                             "pairs_per_s_equivalent": float(w.n) * w.n / t_nb},
        "sample": (f"fp64 oracle tree on the {'FULL N' if full else 'groups sampled with stride %d, extrapolated' % r['stride']}: build "
                   f"{r['t_build']:.2f} s + force of {r['groups']} groups / {r['n_sample']} particles {r['t_force']:.2f} s; "
                   f"direct sum of eq. 3 on {n_t} targets x all sources {t_direct:.2f} s; neighbour search ({kind}) {t_nb:.2f} s"),
    }


def run_reference(args, w, rank):
    """--impl reference: the fp64 CPU oracle (there is no other reference implementation: the paper's
    code is not available).  Rank 0 only; every step is a bounded sample of the workload: the full tree build and
    the tree force of every 8th group (about a second per step), extrapolated to the full N."""
    if rank != 0:
        return
    stride = 8 if w.n >= 500000 else 1
    for _ in range(args.warmup):
        oracle_tree_run(w, max(stride, 64))
    t0 = time.perf_counter()
    runs = [oracle_tree_run(w, stride) for _ in range(args.steps)]
    wall = time.perf_counter() - t0
    pps = float(np.mean([r["particles_per_s"] for r in runs]))
    r0 = runs[-1]
    sample = (f"per step: full oracle tree build ({r0['t_build']:.2f} s) + fp64 tree force of every {r0['stride']}th group "
              f"({r0['groups']} groups, {r0['n_sample']} particles, {r0['t_force']:.2f} s); particles/s extrapolated to the "
              f"full N as N / (t_build + t_force * N / n_sample)")
    line = {
        "impl": "reference", "metric": "regular_force_particles_per_s", "value": pps, "unit": "particles/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * wall / max(1, args.steps), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": config_dict(w, args.gpus),
        "interactions_per_s": float(np.mean([r["interactions_per_s"] for r in runs])),
        "cpu_baseline": {"value": pps, "unit": "particles/s", "cores": r0["cores"], "kind": "oracle", "sample": sample},
        "e2e": {"value": pps, "unit": "particles/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def reduce_over_ranks(total_ms: float, units: float, dist) -> tuple:
    """Max of the timed region over ranks and sum of the units processed (host-side logic of the N > 1
    path; covered by a world_size-2 gloo test on CPU)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return total_ms, units
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([total_ms], dtype=torch.float64, device=dev)
    u = torch.tensor([units], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


# ---------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------
def time_steps(torch, ctx, pm_dev, out_dev, w, flush, steps: int, warmup: int) -> dict:
    """W untimed steps, then K steps each between two CUDA events on the context's stream (torch's current stream),
    the L2 flushed before every one; per-phase times from the library's own events (p3t_get_stats)."""
    def step():
        ctx.build_tree(pm_dev, KEY_BITS)
        ctx.regular_force(w.r_out, w.r_in, w.theta, 0, out=out_dev)

    for _ in range(warmup):
        step()
    torch.cuda.synchronize()
    l0 = ctx.stats()["launches"]
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    ph = {k: [] for k in ("ms_build", "ms_sort", "ms_count", "ms_walk", "ms_eval", "ms_force")}
    for k in range(steps):
        flush.zero_()                                     # L2 flush between timed iterations (outside the event pair)
        ev[k][0].record()
        step()
        ev[k][1].record()
        st = ctx.stats()                                  # synchronises; after the closing event
        # a timed step that redid part of its work (undersized buffer, force warps that gave up waiting) is not a measurement
        assert not st["force_flags"] & 6, f"timed step {k} was repaired (force_flags={st['force_flags']}): more warm-up needed"
        for q in ph:
            ph[q].append(st[q])
    torch.cuda.synchronize()
    return dict(step_ms=[a.elapsed_time(b) for a, b in ev], phases=ph, st=st, launches=int(st["launches"] - l0))


def alu_fractions(st, kernel_ms: float, sms: int, sm_mhz: float) -> dict:
    """k_force against the FP32-ALU roofline, the algorithmic work counted both ways."""
    peak = sms * 128 * sm_mhz * 1e6 / 1e12                # Tinstr/s: FP32 lanes x clock
    a_survey = (INSTR_PP * st["n_pp"] + INSTR_PC * st["n_pc"]) / (kernel_ms * 1e-3) / 1e12
    a_sass = (INSTR_PP_SASS * st["n_pp"] + INSTR_PC_SASS * st["n_pc"]) / (kernel_ms * 1e-3) / 1e12
    return dict(peak=peak, achieved=a_survey, frac=a_survey / peak, achieved_sass=a_sass, frac_sass=a_sass / peak)


def config_summary(cfg: int, w, t: dict, sms: int, pk: dict) -> dict:
    st, n = t["st"], w.n
    ms = stat3(t["step_ms"])
    ph = {k: float(np.median(v)) for k, v in t["phases"].items()}
    fr = alu_fractions(st, ph["ms_eval"], sms, pk["sm_max_mhz"])
    n_int = st["n_pp"] + st["n_pc"]
    surv = SURVEY_INSTR_PER_PARTICLE.get((cfg, round(w.theta, 2)))
    mine = (INSTR_PP * st["n_pp"] + INSTR_PC * st["n_pc"]) / n
    return {
        "config": cfg, "workload": w.name, "n": n, "theta": w.theta, "r_out": w.r_out, "steps": len(t["step_ms"]),
        "ms_per_step": ms, "particles_per_s": n / (ms["median"] * 1e-3),
        "ms_build": ph["ms_build"], "ms_sort": ph["ms_sort"], "ms_count": ph["ms_count"], "ms_walk": ph["ms_walk"],
        "ms_eval": ph["ms_eval"], "ms_force": ph["ms_force"],
        "interactions_per_s": n_int / (ph["ms_force"] * 1e-3),                  # over a7-a11
        "interactions_per_s_kernel": n_int / (ph["ms_eval"] * 1e-3),            # over k_force alone
        "pp_per_particle": st["n_pp"] / n, "pc_per_particle": st["n_pc"] / n,
        "frac_alu_survey_counts": fr["frac"], "frac_alu_sass_counts": fr["frac_sass"],
        "work_vs_survey": (mine / surv) if surv else None,
        "frac_vs_survey_work": (fr["frac"] / (mine / surv)) if surv else None,
        "build_gbs": 354.0 * n / (ph["ms_build"] * 1e-3) / 1e9, "build_frac_hbm": 354.0 * n / (ph["ms_build"] * 1e-3) / 1e9 / pk["hbm_gbs"],
        "nodes": st["n_nodes"], "groups": st["n_groups"], "neighbours_total": st["nb_total"], "neighbours_max": st["nb_max"],
        "gpu_launches_per_step": t["launches"] / len(t["step_ms"]),
    }


def run_ours(args, w, rank, world, local_rank, dist):
    import torch
    import workloads
    import paper_2110_11658_b200 as p3t
    from paper_2110_11658_b200 import pipebench

    p3t.lib()                                             # fail loudly when the CUDA library is missing
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    pk = peaks()
    n = w.n
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    pm_dev = torch.from_numpy(w.pos_mass).to(dev)
    out_dev = torch.empty((n, 4), dtype=torch.float32, device=dev)
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)       # > 126 MB of L2
    ctx = p3t.Context(local_rank)
    warm = max(3, args.warmup)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident arm ----
    for _ in range(warm):
        ctx.build_tree(pm_dev, KEY_BITS); ctx.regular_force(w.r_out, w.r_in, w.theta, 0, out=out_dev)
    sampler = ClockSampler(local_rank)
    barrier()
    t = time_steps(torch, ctx, pm_dev, out_dev, w, flush, args.steps, 0)
    barrier()
    clocks = sampler.stop()
    st = t["st"]
    total_ms = float(sum(t["step_ms"]))
    launches = t["launches"]
    ph = t["phases"]

    # ---- the same step with the list walk and the force kernel one after the other (p3t_diag_set_overlap, libp3t_diag.so):
    # the force kernel's duration with the SMs to itself, for the roofline ----
    with p3t.Context(local_rank) as cs:
        pipebench.set_overlap(cs, False)
        ts = time_steps(torch, cs, pm_dev, out_dev, w, flush, min(args.steps, 5), 3)

    # ---- SURVEY 8f NEXT-1 (outside the step): irregular force + jerk over the emitted lists ----
    vel_dev = torch.from_numpy(workloads.velocities_for(w)).to(dev)
    irr_ms = []
    for k in range(5):
        ctx.irregular_force(vel_dev)
        irr_ms.append(ctx.stats()["ms_irregular"])
    irr_ms = float(np.median(irr_ms[1:]))

    # ---- SURVEY 8f NEXT-2 (outside the step): lists out to r_out + r_buff (eq. 20-21: r_buff = 3 tau sigma, r_cut = 4 tau,
    # sigma = 1/sqrt(2) => r_buff = 0.53 r_out) and the leapfrog half-kick fused into the force epilogue ----
    r_buff = float(np.float32(0.75 * 2.0 ** -0.5 * w.r_out))
    kick_dev = vel_dev.clone()
    buf_ms = []
    for k in range(4):
        flush.zero_()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        ctx.build_tree(pm_dev, KEY_BITS)
        ctx.regular_force(w.r_out, w.r_in, w.theta, 0, out=out_dev, r_buff=r_buff, half_dt=1.0e-4, vel=kick_dev)
        e1.record()
        stb = ctx.stats()
        buf_ms.append(e0.elapsed_time(e1))
    buf_ms = float(np.median(buf_ms[1:]))
    ctx.build_tree(pm_dev, KEY_BITS)                      # back to the plain lists for the legs below
    ctx.regular_force(w.r_out, w.r_in, w.theta, 0, out=out_dev)

    # ---- SURVEY 8f NEXT-3 (outside the step): sampled 6-NN core quantities, the paper's sample size ----
    ns = int(min(n, np.sqrt(5000.0 * n)))
    sample_dev = torch.from_numpy(workloads.sample_targets(n, ns).astype(np.int32)).to(dev)
    core_ms = []
    for k in range(5):
        core = ctx.core_quantities(sample_dev, 6)
        core_ms.append(ctx.stats()["ms_core"])
    core_ms = float(np.median(core_ms[1:]))

    # ---- end-to-end arm: HOST buffers through p3t_step_host ----
    pm_host = torch.from_numpy(w.pos_mass).pin_memory()
    acc_host = torch.empty((n, 4), dtype=torch.float32).pin_memory()
    nb_cap = int(st["nb_total"] * 1.25) + 1024
    off_host = torch.empty(n + 1, dtype=torch.int64).pin_memory()
    idx_host = torch.empty(nb_cap, dtype=torch.int32).pin_memory()

    def step_host():
        return ctx.step_host(pm_host, w.r_out, w.r_in, w.theta, 0, KEY_BITS, acc_pot=acc_host, nb_offsets=off_host, nb_indices=idx_host)

    for _ in range(3):
        step_host()
    barrier()
    ev2 = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for k in range(args.steps):
        flush.zero_()
        ev2[k][0].record()
        _, _, _, nb_total = step_host()
        ev2[k][1].record()
    barrier()
    e2e_steps = [a.elapsed_time(b) for a, b in ev2]
    e2e_ms = float(sum(e2e_steps))
    assert torch.isfinite(acc_host).all()

    # ---- the other BASELINE.json configs, device-resident, from the same run (N = 1 only) ----
    others = []
    if world == 1 and args.configs == "all":
        ctx.close()
        del pm_dev, out_dev
        main_cfg = (args.config, round(w.theta, 2))
        for cfg, theta in [(1, 0.4), (2, 0.4), (3, 0.4), (4, 0.4), (5, 0.3), (5, 0.5), (5, 0.7)]:
            if (cfg, theta) == main_cfg or args.n is not None:
                continue
            wc = workloads.make_config(cfg, theta=theta)
            pmc = torch.from_numpy(wc.pos_mass).to(dev)
            outc = torch.empty((wc.n, 4), dtype=torch.float32, device=dev)
            with p3t.Context(local_rank) as cx:
                tc = time_steps(torch, cx, pmc, outc, wc, flush, min(args.steps, 5 if wc.n <= (1 << 20) else 3), 3)
            others.append(config_summary(cfg, wc, tc, sms, pk))
            del pmc, outc
        ctx = None

    total_ms_max, units = reduce_over_ranks(total_ms, float(n) * args.steps, dist)
    e2e_ms_max, _ = reduce_over_ranks(e2e_ms, float(n) * args.steps, dist)
    if rank != 0:
        return
    value = units / (total_ms_max * 1e-3)
    e2e_value = units / (e2e_ms_max * 1e-3)
    n_int = st["n_pp"] + st["n_pc"]
    wms = float(np.mean(ph["ms_eval"]))                   # the dominant kernel: k_force (both launches: beside and behind the list walk)
    fms = float(np.mean(ph["ms_force"]))                  # a7-a11: count walk, offsets, list walk, force kernel, row sort
    fr = alu_fractions(st, wms, sms, pk["sm_max_mhz"])
    pipes = pipebench.pipe_bench(local_rank)              # FFMA chain etc. on this device
    peak_meas = pipes["fp32_lane_instr_per_s"] / 1e12
    surv = SURVEY_INSTR_PER_PARTICLE.get((args.config, round(w.theta, 2))) if args.n is None else None
    mine = (INSTR_PP * st["n_pp"] + INSTR_PC * st["n_pc"]) / n
    alone_ms = float(np.median(ts["phases"]["ms_eval"]))
    alone = alu_fractions(ts["st"], alone_ms, sms, pk["sm_max_mhz"])
    roofline = {
        "bound": "alu", "kernel": "k_force (p-c / p-p force + cutoff + neighbour emission over the interaction lists)",
        "achieved": fr["achieved"], "peak": fr["peak"], "unit": "Tinstr/s (FP32 lane-instructions)", "frac": fr["frac"],
        "algorithmic": f"SURVEY 8(d) estimates: {INSTR_PP} instr per p-p x {st['n_pp']} + {INSTR_PC} per p-c x {st['n_pc']}",
        "achieved_sass_counts": fr["achieved_sass"], "frac_sass_counts": fr["frac_sass"],
        "algorithmic_sass_counts": f"the kernel's own FP32 instructions (profiles/r02_sass_counts.md): {INSTR_PP_SASS:g} per p-p, {INSTR_PC_SASS:g} per p-c",
        "work_vs_survey": (mine / surv) if surv else None,
        "work_vs_survey_note": ("FP32 instructions per particle of this run (15 pp + 37 pc, NCRIT 64 sibling-run groups) over SURVEY 8(d)'s table "
                                "(NCRIT 32 canonical groups): the extra interactions that `achieved` credits as useful"),
        "frac_vs_survey_work": (fr["frac"] / (mine / surv)) if surv else None,
        "traffic": ncu_traffic(w.name), "traffic_unit": "bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum, ncu --set full; profiles/" + TRAFFIC_CSV + ")",
        "peak_source": f"{sms} SMs x 128 FP32 lanes x {pk['sm_max_mhz']:.0f} MHz ({pk['source']} sm_max_mhz)",
        "achieved_tflops": (FLOP_PP * st["n_pp"] + FLOP_PC * st["n_pc"]) / (wms * 1e-3) / 1e12,
        "peak_measured": peak_meas, "frac_of_measured": fr["achieved"] / peak_meas,
        "peak_measured_source": "p3t_diag_pipe_bench: FFMA chain, 32 lanes / %.3f cycles per SM sub-partition" % pipes["cycles"]["FFMA (reuse cache)"],
        "pipe_cycles": pipes["cycles"],
        "kernel_ms": wms, "kernel_share_of_step": wms * args.steps / total_ms,
        # the two kernel numbers side by side: beside the list walk (the step as it runs) and with the SMs to itself
        "kernel_ms_beside_walk": wms, "frac_beside_walk": fr["frac"], "frac_sass_beside_walk": fr["frac_sass"],
        "kernel_ms_alone": alone_ms, "frac_alone": alone["frac"], "frac_sass_alone": alone["frac_sass"],
        "kernel_note": "k_force as it runs in the timed step: beside the list walk (k_walk<LISTS> holds 1 CTA per SM for the first ~40 % of it), so its duration includes that competition",
        "kernel_alone": (lambda a, m: {"kernel_ms": m, "frac": a["frac"], "frac_sass_counts": a["frac_sass"],
                                       "ms_per_step": float(np.median(ts["step_ms"])), "ms_walk": float(np.median(ts["phases"]["ms_walk"])),
                                       "note": "same step without the overlap (p3t_diag_set_overlap 0): list walk, then the force kernel with the SMs to itself"})(
            alu_fractions(ts["st"], float(np.median(ts["phases"]["ms_eval"])), sms, pk["sm_max_mhz"]), float(np.median(ts["phases"]["ms_eval"]))),
        "frac_at_observed_clock": (fr["achieved"] / (sms * 128 * clocks["sm_mhz"] * 1e6 / 1e12)) if clocks.get("sm_mhz") else None,
    }
    # secondary roofline (north_star: "achieved HBM GB/s for build/sort"): a1-a6 against the measured copy bandwidth;
    # algorithmic bytes per particle from SURVEY.md 8(d): cube 16 + keys 28 + radix sort 200 + gather 36 + topology 16 + moments 54 + groups 4
    build_ms_mean = float(np.mean(ph["ms_build"]))
    build_gbs = 354.0 * n / (build_ms_mean * 1e-3) / 1e9
    roofline_build = {"bound": "hbm", "kernels": "a1-a6 (cube, keys, radix sort, permute, topology, moments, groups)",
                      "achieved": build_gbs, "peak": pk["hbm_gbs"], "unit": "GB/s", "frac": build_gbs / pk["hbm_gbs"],
                      "algorithmic": "354 B per particle", "ms": build_ms_mean,
                      "note": "launch/latency-bound below N ~ 2^22 (working set in L2); see configs[] for N = 2^22"}
    line = {
        "metric": "regular_force_particles_per_s", "value": value, "unit": "particles/s", "n_gpus": world,
        "steps": args.steps, "warmup": warm, "ms_per_step": total_ms_max / args.steps, "ms_per_step_stats": stat3(t["step_ms"]),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": config_dict(w, world),
        "interactions_per_s": n_int * world / (fms * 1e-3), "interactions_per_s_note": "over a7-a11 (ms_force), SURVEY 8(d)",
        "interactions_per_s_kernel": n_int * world / (wms * 1e-3), "interactions_per_s_step": n_int * world / (total_ms_max / args.steps * 1e-3),
        "interactions_per_step": n_int,
        "pp_per_particle": st["n_pp"] / n, "pc_per_particle": st["n_pc"] / n,
        "ms_build": build_ms_mean, "ms_sort": float(np.mean(ph["ms_sort"])), "ms_force": fms, "ms_count": float(np.mean(ph["ms_count"])),
        "ms_walk": float(np.mean(ph["ms_walk"])), "ms_eval": wms,
        "ms_note": "ms_walk: the list walk on its own stream, beside the force kernel; ms_eval: the force kernel from its first launch to the end of its second",
        "nodes": st["n_nodes"], "groups": st["n_groups"], "neighbours_total": st["nb_total"], "neighbours_max": st["nb_max"],
        "e2e": {"value": e2e_value, "unit": "particles/s", "ms_per_step": e2e_ms_max / args.steps, "ms_per_step_stats": stat3(e2e_steps),
                "h2d_bytes_per_step": 16 * n, "d2h_bytes_per_step": 16 * n + 8 * (n + 1) + 4 * int(nb_total)},
        "next1_irregular": {"ms": irr_ms, "list_entries_per_s": st["nb_total"] / (irr_ms * 1e-3) if irr_ms > 0 else None,
                            "note": "p3t_irregular_force (F_I, jerk, phi_I over the neighbour lists); not part of the timed step"},
        "next2_buffered_kick": {"ms_per_step": buf_ms, "r_buff": r_buff, "neighbours_total": stb["nb_total"], "neighbours_max": stb["nb_max"],
                                "note": "p3t_regular_force_ex: lists out to r_out + r_buff (eq. 20-21) and the half-kick in the force epilogue; not part of the timed step"},
        "next3_core": {"ms": core_ms, "sample": ns, "k": 6, "r_core": core["r_core"], "rho_core": core["rho_core"], "n_core": core["n_core"],
                       "note": "p3t_core_quantities (k-NN on the octree + Casertano-Hut reductions); not part of the timed step"},
        "gpu_launches": launches, "clocks": clocks, "roofline": roofline, "roofline_build": roofline_build,
        "configs": others,
    }
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(w)
    print(json.dumps(line), flush=True)
    if ctx is not None:
        ctx.close()


def run_sharded(args, w, rank, world, local_rank, dist):
    """One cluster, target groups split among the ranks: every rank builds the whole tree, evaluates
    its own Morton range of groups (cost-balanced from the warm-up step's list lengths) and all-gathers acc_pot."""
    import torch
    import paper_2110_11658_b200 as p3t
    from paper_2110_11658_b200 import shard

    p3t.lib()
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    n = w.n
    pm_dev = torch.from_numpy(w.pos_mass).to(dev)
    out_dev = torch.empty((n, 4), dtype=torch.float32, device=dev)
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)
    sim = world == 1
    nranks = max(2, args.sim_ranks) if sim else world
    ctx = p3t.Context(local_rank)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def step(r):
        ctx.build_tree(pm_dev, KEY_BITS)
        cuts, _ = ctx.shard_cuts()                        # one small D2H after the build
        ctx.regular_force(w.r_out, w.r_in, w.theta, 0, out=out_dev)
        if sim:                                           # the rank's half of the exchange; no peers on one GPU
            ctx.shard_pack(out_dev, chunk)
        else:                                             # one all-gather of acc_pot and of the CSR rows, inside the timed region
            shard.exchange(ctx, out_dev, cuts)
            shard.exchange_neighbours(ctx)
        return cuts

    # step 0 with cuts by particle count, then cuts balanced by the measured cost of every group
    nominal = None
    chunk = torch.empty((n, 4), dtype=torch.float32, device=dev)
    if sim:
        costs = None
        for r in range(nranks):
            ctx.set_shard(r, nranks)
            step(r)
            gb, c = shard.gather_group_costs(ctx)
            costs = c if costs is None else costs + c
    else:
        ctx.set_shard(rank, nranks)
        step(rank)
        gb, costs = shard.gather_group_costs(ctx)
    nominal = shard.balanced_cuts(gb, n, costs, nranks)

    sampler = ClockSampler(local_rank)
    per_rank, launches, n_int = [], 0, 0
    for r in (range(nranks) if sim else [rank]):
        ctx.set_shard(r, nranks, nominal)
        for _ in range(max(3, args.warmup)):
            step(r)
        torch.cuda.synchronize()
        l0 = ctx.stats()["launches"]
        barrier()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        for k in range(args.steps):
            flush.zero_()
            ev[k][0].record()
            step(r)
            ev[k][1].record()
        barrier()
        st = ctx.stats()
        per_rank.append(float(sum(a.elapsed_time(b) for a, b in ev)))
        launches += int(st["launches"] - l0)
        n_int += st["n_pp"] + st["n_pc"]
    clocks = sampler.stop()
    total_ms = float(sum(per_rank))                       # simulated: one GPU did every shard in turn
    total_ms_max, units = reduce_over_ranks(total_ms, float(n) * args.steps / (1 if sim else world), dist)
    if rank != 0:
        return
    line = {
        "metric": "regular_force_particles_per_s", "value": units / (total_ms_max * 1e-3), "unit": "particles/s", "n_gpus": world,
        "steps": args.steps, "warmup": max(3, args.warmup), "ms_per_step": total_ms_max / args.steps,
        "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": dict(config_dict(w, world),
                       parallelism=(f"sharded, {nranks} ranks SIMULATED on one GPU: the shards run in turn, no exchange" if sim
                                    else f"sharded by target group over {world} ranks, all-gather of acc_pot and of the neighbour rows in the timed region")),
        "gpu_launches": launches, "clocks": clocks, "interactions_per_step": n_int if sim else None,
    }
    if sim:
        ms = [t / args.steps for t in per_rank]
        line["simulated"] = {"ranks": nranks, "ms_per_rank": ms, "cuts": [int(c) for c in nominal],
                             "projected_ms_per_step": max(ms), "imbalance": max(ms) / (sum(ms) / nranks),
                             "note": "projection = slowest shard (tree build included on every rank); the all-gather of "
                                     "16 B x n is not included"}
    print(json.dumps(line), flush=True)
    ctx.close()


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def spawn_ranks(n_ranks: int) -> int:
    """`python bench.py --gpus N` outside a torchrun environment: start the N ranks ourselves, exactly as the driver
    does (torch.distributed.run, one process per GPU, rendezvous on 127.0.0.1), and pass their output through."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n_ranks}",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), str(Path(__file__).resolve())] + sys.argv[1:]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")                  # the communicator log (rings / NVLS) stays on, to stderr
    env["P3T_BENCH_SPAWNED"] = "1"
    return subprocess.call(cmd, env=env)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config 1..5 (3 = headline, Plummer 2^20)")
    ap.add_argument("--configs", choices=["all", "none"], default="all",
                    help="also time the other BASELINE.json configs (1, 2, 4, 5 x theta), device-resident, into configs[] (N = 1)")
    ap.add_argument("--n", type=int, default=None, help="override the particle count (debug)")
    ap.add_argument("--theta", type=float, default=None)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--mode", choices=["replicas", "sharded"], default="replicas",
                    help="N > 1: independent replicas (weak scaling, default) or one cluster sharded by target group (strong)")
    ap.add_argument("--sim-ranks", type=int, default=4, help="--mode sharded on ONE GPU: number of ranks whose shards are run in turn")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(spawn_ranks(args.gpus))
    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    import workloads
    if args.impl == "reference":
        if rank == 0:
            run_reference(args, workloads.make_config(args.config, n_override=args.n, theta=args.theta), rank)
        return
    dist = None
    if world > 1:
        import torch
        import torch.distributed as dist
        torch.cuda.set_device(local_rank)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    w = workloads.make_config(args.config, n_override=args.n, theta=args.theta)
    (run_sharded if args.mode == "sharded" else run_ours)(args, w, rank, world, local_rank, dist)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
