#!/usr/bin/env python
"""bench.py -- the regular-force step of NBODY6+P3T on B200 (BASELINE.json metric:
regular-force particles/s and interactions/s at N = 1M; ms per force step).

A "step" is one pass of the whole hot path over one synthetic cluster:
p3t_build_tree + p3t_regular_force (cube, keys, sort, octree, moments, groups, walk, p-c / p-p force
with cutoff, neighbour lists, scatter), i.e. what the host integrator asks for once per dt_reg
(PAPER.md:89-94).  Default workload = BASELINE config 3 (Plummer 2^20, Kroupa masses, theta 0.4).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl ours|reference]

Prints ONE JSON line (rank 0).  `value` times the path with inputs resident in HBM; `e2e` times
p3t_step_host with pinned HOST buffers (H2D of positions, D2H of forces and neighbour lists inside
the timed region).  `roofline` is for the dominant kernel (walk + force), an FP32-ALU-bound kernel;
`cpu_baseline` is the fp64 oracle on the host cores, on a bounded sample.  Multi-GPU: by default every
rank runs an independent replica ("replicas only", weak scaling; north_star is a one-GPU path).
`--mode sharded` splits the target groups of ONE cluster among the ranks
(paper_2110_11658_b200.shard; strong scaling, one all-gather of 16 B per particle); with one GPU,
`--mode sharded --sim-ranks R` runs the R shards in turn and reports each rank's time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

# FP32-pipe instructions the method needs per interaction
INSTR_PP, INSTR_PC = 15, 37
FLOP_PP, FLOP_PC = 20, 60
# DRAM traffic of the dominant kernel from the committed ncu capture (profiles/), per launch, by workload
TRAFFIC_NCU = {"plummer1m_kroupa": 1515.9e6}


def peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        return dict(hbm_gbs=float(d.get("hbm_gbs", 6650.0)), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


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


def oracle_sample_run(w, n_groups_target: int):
    """The oracle as it stands, on a bounded sample: full tree build + force of every k-th group."""
    import oracle
    t0 = time.perf_counter()
    T = oracle.Tree(w.pos_mass, 63, 16, 64)
    t_build = time.perf_counter() - t0
    stride = max(1, T.n_groups // n_groups_target)
    gi = np.arange(0, T.n_groups, stride, dtype=np.int64)
    g = T.groups()
    cnt = (g["end"] - g["begin"]).astype(np.int64)
    t0 = time.perf_counter()
    f = T.force(w.r_out, w.r_in, w.theta, 0, group_ids=gi)
    t_force = time.perf_counter() - t0
    n_s = int(cnt[gi].sum())
    inter = int(((f["npp"] + f["npc"]) * cnt[gi]).sum())
    # whole-path time of the full N, extrapolated from the sample: build + force * N / n_s
    t_full = t_build + t_force * w.n / n_s
    return dict(t_build=t_build, t_force=t_force, n_sample=n_s, groups=len(gi), stride=stride, interactions=inter,
                particles_per_s=w.n / t_full, interactions_per_s=inter / t_force, t_full=t_full, cores=oracle.omp_threads())


def run_reference(args, w, rank):
    """--impl reference: the fp64 CPU oracle (there is no other reference implementation: the paper's
    code is not available).  Rank 0 only; every step is a bounded sample of the workload."""
    if rank != 0:
        return
    n_groups = 1200 if w.n >= 500000 else 100000
    for _ in range(args.warmup):
        oracle_sample_run(w, max(50, n_groups // 20))
    t0 = time.perf_counter()
    runs = [oracle_sample_run(w, n_groups) for _ in range(args.steps)]
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
        "dtype": "f64", "data": "synthetic", "config": {"workload": w.name, "n": w.n, "r_out": w.r_out, "r_in": w.r_in, "theta": w.theta},
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


def run_ours(args, w, rank, world, local_rank, dist):
    import torch
    import workloads
    import paper_2110_11658_b200 as p3t

    p3t.lib()                                             # fail loudly when the CUDA library is missing
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    pk = peaks()
    n = w.n
    pm_dev = torch.from_numpy(w.pos_mass).to(dev)
    out_dev = torch.empty((n, 4), dtype=torch.float32, device=dev)
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)       # > 126 MB of L2
    ctx = p3t.Context(local_rank)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def step_device():
        ctx.build_tree(pm_dev, 63)
        ctx.regular_force(w.r_out, w.r_in, w.theta, 0, out=out_dev)

    for _ in range(max(3, args.warmup)):
        step_device()
    torch.cuda.synchronize()
    st0 = ctx.stats()

    # ---- device-resident arm ----
    sampler = ClockSampler(local_rank)
    barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    walk_ms, build_ms, force_ms, sort_ms, eval_ms, count_ms = [], [], [], [], [], []
    for k in range(args.steps):
        flush.zero_()                                     # L2 flush between timed iterations (outside the event pair)
        ev[k][0].record()
        step_device()
        ev[k][1].record()
        st = ctx.stats()                                  # synchronises; after the closing event
        walk_ms.append(st["ms_walk"]); build_ms.append(st["ms_build"]); force_ms.append(st["ms_force"]); sort_ms.append(st["ms_sort"])
        eval_ms.append(st["ms_eval"]); count_ms.append(st["ms_count"])
    barrier()
    clocks = sampler.stop()
    step_ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = float(sum(step_ms))
    launches = int(st["launches"] - st0["launches"])

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
        ctx.build_tree(pm_dev, 63)
        ctx.regular_force(w.r_out, w.r_in, w.theta, 0, out=out_dev, r_buff=r_buff, half_dt=1.0e-4, vel=kick_dev)
        e1.record()
        stb = ctx.stats()
        buf_ms.append(e0.elapsed_time(e1))
    buf_ms = float(np.median(buf_ms[1:]))
    ctx.build_tree(pm_dev, 63)                            # back to the plain lists for the legs below
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
        return ctx.step_host(pm_host, w.r_out, w.r_in, w.theta, 0, 63, acc_pot=acc_host, nb_offsets=off_host, nb_indices=idx_host)

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
    e2e_ms = float(sum(a.elapsed_time(b) for a, b in ev2))
    assert torch.isfinite(acc_host).all()

    total_ms_max, units = reduce_over_ranks(total_ms, float(n) * args.steps, dist)
    e2e_ms_max, _ = reduce_over_ranks(e2e_ms, float(n) * args.steps, dist)
    if rank != 0:
        return
    value = units / (total_ms_max * 1e-3)
    e2e_value = units / (e2e_ms_max * 1e-3)
    n_int = st["n_pp"] + st["n_pc"]
    wms = float(np.mean(eval_ms))                        # the dominant kernel: k_force
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    alg_instr = INSTR_PP * st["n_pp"] + INSTR_PC * st["n_pc"]
    peak_instr = sms * 128 * pk["sm_max_mhz"] * 1e6 / 1e12            # Tinstr/s, FP32 lanes x clock
    achieved = alg_instr / (wms * 1e-3) / 1e12
    pipes = p3t.pipe_bench(local_rank)                     # FFMA chain etc. on this device
    peak_meas = pipes["fp32_lane_instr_per_s"] / 1e12
    roofline = {
        "bound": "alu", "kernel": "k_force (p-c / p-p force + cutoff + neighbour emission over the interaction lists)",
        "achieved": achieved, "peak": peak_instr, "unit": "Tinstr/s (FP32 lane-instructions)", "frac": achieved / peak_instr,
        "traffic": TRAFFIC_NCU.get(w.name), "traffic_unit": "bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum, ncu --set full, profiles/)",
        "peak_source": f"{sms} SMs x 128 FP32 lanes x {pk['sm_max_mhz']:.0f} MHz ({pk['source']} sm_max_mhz)",
        "algorithmic": f"{INSTR_PP} instr per p-p x {st['n_pp']} + {INSTR_PC} per p-c x {st['n_pc']}",
        "achieved_tflops": (FLOP_PP * st["n_pp"] + FLOP_PC * st["n_pc"]) / (wms * 1e-3) / 1e12,
        "peak_measured": peak_meas, "frac_of_measured": achieved / peak_meas,
        "peak_measured_source": "p3t_pipe_bench: FFMA chain, 32 lanes / %.3f cycles per SM sub-partition" % pipes["cycles"]["FFMA (reuse cache)"],
        "pipe_cycles": pipes["cycles"],
        "kernel_ms": wms, "kernel_share_of_step": wms * args.steps / total_ms,
        "frac_at_observed_clock": (achieved / (sms * 128 * clocks["sm_mhz"] * 1e6 / 1e12)) if clocks.get("sm_mhz") else None,
    }
    # secondary roofline (north_star: "achieved HBM GB/s for build/sort"): a1-a6 against the measured copy bandwidth;
    # algorithmic bytes per particle from SURVEY.md 8(d): cube 16 + keys 28 + radix sort 200 + gather 36 + topology 16 + moments 54 + groups 4
    build_ms_mean = float(np.mean(build_ms))
    build_gbs = 354.0 * n / (build_ms_mean * 1e-3) / 1e9
    roofline_build = {"bound": "hbm", "kernels": "a1-a6 (cube, keys, radix sort, permute, topology, moments, groups)",
                      "achieved": build_gbs, "peak": pk["hbm_gbs"], "unit": "GB/s", "frac": build_gbs / pk["hbm_gbs"],
                      "algorithmic": "354 B per particle", "ms": build_ms_mean,
                      "note": "launch/latency-bound below N ~ 2^22: 34 small kernels, working set in L2"}
    line = {
        "metric": "regular_force_particles_per_s", "value": value, "unit": "particles/s", "n_gpus": world,
        "steps": args.steps, "warmup": max(3, args.warmup), "ms_per_step": total_ms_max / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": w.name, "n": n, "r_out": w.r_out, "r_in": w.r_in, "theta": w.theta, "key_bits": 63,
                   "nleaf": 16, "ncrit": 64, "l2": "flushed between timed iterations (512 MiB write)",
                   "parallelism": "replicas only" if world > 1 else "1 GPU"},
        "interactions_per_s": n_int * world / (wms * 1e-3), "interactions_per_step": n_int,
        "pp_per_particle": st["n_pp"] / n, "pc_per_particle": st["n_pc"] / n,
        "ms_build": float(np.mean(build_ms)), "ms_sort": float(np.mean(sort_ms)), "ms_force": float(np.mean(force_ms)), "ms_count": float(np.mean(count_ms)),
        "ms_walk": float(np.mean(walk_ms)), "ms_eval": wms,
        "nodes": st["n_nodes"], "groups": st["n_groups"], "neighbours_total": st["nb_total"], "neighbours_max": st["nb_max"],
        "e2e": {"value": e2e_value, "unit": "particles/s", "ms_per_step": e2e_ms_max / args.steps,
                "h2d_bytes_per_step": 16 * n, "d2h_bytes_per_step": 16 * n + 8 * (n + 1) + 4 * int(nb_total)},
        "next1_irregular": {"ms": irr_ms, "list_entries_per_s": st["nb_total"] / (irr_ms * 1e-3) if irr_ms > 0 else None,
                            "note": "p3t_irregular_force (F_I, jerk, phi_I over the neighbour lists); not part of the timed step"},
        "next2_buffered_kick": {"ms_per_step": buf_ms, "r_buff": r_buff, "neighbours_total": stb["nb_total"], "neighbours_max": stb["nb_max"],
                                "note": "p3t_regular_force_ex: lists out to r_out + r_buff (eq. 20-21) and the half-kick in the force epilogue; not part of the timed step"},
        "next3_core": {"ms": core_ms, "sample": ns, "k": 6, "r_core": core["r_core"], "rho_core": core["rho_core"], "n_core": core["n_core"],
                       "note": "p3t_core_quantities (k-NN on the octree + Casertano-Hut reductions); not part of the timed step"},
        "gpu_launches": launches, "clocks": clocks, "roofline": roofline, "roofline_build": roofline_build,
    }
    if world == 1 and not args.no_cpu_baseline:
        r = oracle_sample_run(w, 4000 if n >= 500000 else 100000)
        # the plain definition (eq. 3 by direct summation, fp64) on a stride sample of targets
        import oracle
        n_t = 2048
        t0 = time.perf_counter()
        oracle.direct(w.pos_mass, w.r_out, w.r_in, targets=workloads.sample_targets(n, n_t))
        t_direct = time.perf_counter() - t0
        line["cpu_baseline"] = {
            "value": r["particles_per_s"], "unit": "particles/s", "cores": r["cores"], "kind": "oracle",
            "interactions_per_s": r["interactions_per_s"],
            "direct_sum": {"pairs_per_s": n_t * float(n) / t_direct, "targets": n_t, "seconds": t_direct,
                           "full_n2_seconds_extrapolated": t_direct * n / n_t},
            "sample": (f"full oracle tree build ({r['t_build']:.2f} s) + fp64 tree force of every {r['stride']}th group "
                       f"({r['groups']} groups, {r['n_sample']} particles, {r['t_force']:.2f} s); extrapolated to the full N"),
        }
    print(json.dumps(line), flush=True)
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
        ctx.build_tree(pm_dev, 63)
        cuts, _ = ctx.shard_cuts()                        # one small D2H after the build
        ctx.regular_force(w.r_out, w.r_in, w.theta, 0, out=out_dev)
        if sim:                                           # the rank's half of the exchange; no peers on one GPU
            ctx.shard_pack(out_dev, chunk)
        else:
            shard.exchange(ctx, out_dev, cuts)
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
        "config": {"workload": w.name, "n": n, "r_out": w.r_out, "r_in": w.r_in, "theta": w.theta, "key_bits": 63,
                   "l2": "flushed between timed iterations (512 MiB write)",
                   "parallelism": (f"sharded, {nranks} ranks SIMULATED on one GPU: the shards run in turn, no exchange" if sim
                                   else f"sharded by target group over {world} ranks, all-gather of acc_pot")},
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


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config 1..5 (3 = headline, Plummer 2^20)")
    ap.add_argument("--n", type=int, default=None, help="override the particle count (debug)")
    ap.add_argument("--theta", type=float, default=None)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--mode", choices=["replicas", "sharded"], default="replicas",
                    help="N > 1: independent replicas (weak scaling, default) or one cluster sharded by target group (strong)")
    ap.add_argument("--sim-ranks", type=int, default=4, help="--mode sharded on ONE GPU: number of ranks whose shards are run in turn")
    args = ap.parse_args()
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
