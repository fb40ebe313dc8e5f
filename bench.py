#!/usr/bin/env python
"""bench.py -- throughput of the batched MIG-day simulator (BASELINE.json metric: simulated job-events/s and
day-episodes/s on B200, with the fraction of the kernel's roofline).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C5] [--impl ours|reference]
  python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P bench.py --gpus N ...

A "step" is one pass of the whole hot path over one batch of synthetic input: mig_sim_reset + mig_sim_rollout of every
environment of the workload for one simulated day (arrival generation, event loop, scheduling, repartitioning, energy /
tardiness accounting, per-epoch records, totals).  Inputs are synthetic (recipes in DESIGN.md section 4).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

# Algorithmic LANE-instructions per job-event (DESIGN.md section 6 derives them by hand from what the serial method must
# execute per ARRIVE/COMPLETE): arrival generator 136 (gen_arrivals_kernel); event loop 185 = event advance 22 +
# arrival/completion accounting and trace hash 30 + reschedule 128 + taking one list record 5 (the rollout kernel).  The
# roofline numerator uses THESE, not the executed counts, so that neither instruction bloat nor idle lanes can inflate the
# fraction.  Peak = SMs x 128 FP32/INT32 lanes x f_max lane-instructions per second.
ALG_LANE_INSTR = {"gen": 136.0, "sim": 185.0}
# profiles/ncu_summary.json: per-kernel numbers of the committed `ncu --set full` captures (written by
# `python -m paper_2606_25082_b200.ncu_summary`), keyed "kernel|workload|n_envs" and stamped with the hash of csrc/.
NCU_SUMMARY = os.path.join(ROOT, "profiles", "ncu_summary.json")
CPU_SAMPLE_ENVS = 2048


def _peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f), "measured"
    except Exception:
        return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            out, _ = self.p.communicate(timeout=5)
        except Exception:
            self.p.kill()
            out = ""
        clocks, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 6:
                continue
            try:
                clocks.append(float(f[0])); mx = float(f[1])
            except ValueError:
                continue
            for nm, v in zip(names, f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(clocks) if clocks else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(clocks)}


# ------------------------------------------------------------------------------------------------ oracle arm
_ALGO_OVERRIDE = -1


def _oracle_chunk(args):
    name, n_envs, lo, hi = args
    from oracle import oracle as O
    from paper_2606_25082_b200 import workloads as W
    wl = W.CONFIGS[name](n_envs)
    if _ALGO_OVERRIDE >= 0:
        wl.algo[:] = _ALGO_OVERRIDE
    ph = O.ParamsHolder(wl.params)
    qh = O.QNetHolder(wl.qnet) if wl.qnet is not None else None
    ev = 0
    for e in range(lo, hi):
        r = O.rollout(ph, wl.seed, e, algo=int(wl.algo[e]), cfg0=int(wl.cfg0[e]), policy=wl.policy,
                      table=None if wl.table is None else wl.table[e], qnet=qh, epsilon=wl.epsilon)
        ev += int(r.totals["n_jobs"]) + int(r.totals["n_completed"])
    return ev


def time_oracle(name, n_envs, n_sample, pool, cores):
    """One pass of the UNMODIFIED single-threaded oracle over the first n_sample envs, split statically over `cores` processes."""
    bounds = [(name, n_envs, (n_sample * i) // cores, (n_sample * (i + 1)) // cores) for i in range(cores)]
    t0 = time.perf_counter()
    ev = sum(pool.map(_oracle_chunk, bounds))
    dt = time.perf_counter() - t0
    return ev, dt


def run_reference(args):
    import concurrent.futures as cf
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from oracle import build as obuild
    obuild.build()
    cores = os.cpu_count() or 1
    n_envs = args.envs
    n_sample = min(n_envs, CPU_SAMPLE_ENVS)
    with cf.ProcessPoolExecutor(cores) as pool:
        for _ in range(args.warmup):
            time_oracle(args.workload, n_envs, min(n_sample, cores * 4), pool, cores)
        ev_tot, t_tot = 0, 0.0
        for _ in range(args.steps):
            ev, dt = time_oracle(args.workload, n_envs, n_sample, pool, cores)
            ev_tot += ev; t_tot += dt
    value = ev_tot / t_tot
    sample = "first %d of %d envs of %s per step, one simulated day each, env range split statically over %d processes" % (n_sample, n_envs, args.workload, cores)
    line = {
        "impl": "reference", "metric": "job_events_per_s", "value": value, "unit": "job-events/s", "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * t_tot / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int64", "data": "synthetic",
        "config": {"workload": args.workload, "n_envs": n_envs, "sample": sample},
        "day_episodes_per_s": n_sample * args.steps / t_tot,
        "cpu_baseline": {"value": value, "unit": "job-events/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "job-events/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------------ CUDA arm
def run_ours(args):
    import torch
    import torch.distributed as dist

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    if world > 1 or os.environ.get("BENCH_FORCE_DIST") == "1":        # (the flag: a one-rank NCCL group, so that the N > 1 plumbing runs on one GPU)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_2606_25082_b200 import binding as B
    from paper_2606_25082_b200 import workloads as W
    import dataclasses

    peaks, peak_src = _peaks()
    n_envs = args.envs                                   # per GPU (weak scaling: every rank simulates a full batch)
    wl = W.CONFIGS[args.workload](n_envs)
    if args.algo >= 0:
        wl.algo[:] = args.algo
    sp = dataclasses.replace(wl.params, env_offset=rank * n_envs)      # Philox keyed by global env id
    sim = B.MigSim(sp, n_envs, wl.seed, tile=args.tile)
    if args.envs_per_warp:
        sim.set_envs_per_warp(args.envs_per_warp)
    prefetch = bool(args.prefetch) and args.tile in (0, 1)
    if prefetch:                                         # the next step's arrival lists are drawn in the tail of this step's event loop
        sim.set_prefetch(True)
    qnet = B.QNet(wl.qnet) if wl.qnet is not None else None
    d_algo, d_cfg0 = torch.from_numpy(wl.algo).cuda(), torch.from_numpy(wl.cfg0).cuda()
    d_table = None if wl.table is None else torch.from_numpy(wl.table).cuda()
    recs, totals = sim.alloc_recs(), sim.alloc_totals()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream()

    def barrier():
        if dist.is_initialized():
            dist.barrier()
        torch.cuda.synchronize()

    def one_step(episode, ev_pair=None):
        sim.reset(episode, d_algo, d_cfg0)
        if ev_pair:
            ev_pair[0].record(stream)
        sim.rollout(wl.policy, table=d_table, qnet=qnet, epsilon=wl.epsilon, recs_out=recs, totals_out=totals)
        if ev_pair:
            ev_pair[1].record(stream)

    def count_events():                                                                      # one ARRIVE-or-DROP per generated job (n_jobs) + one COMPLETE (n_completed)
        t = totals.view(torch.int32).view(n_envs, 20)
        return (t[:, 8].long() + t[:, 9].long() ).sum()

    job_events = torch.zeros(1, dtype=torch.int64, device="cuda")
    for w in range(args.warmup):                                                             # the same work as a timed step
        one_step(w)
        job_events += count_events()
        flush.fill_(w & 0xFF)
    barrier()
    # ---- timed region: resident inputs --------------------------------------------------------------------------
    sampler = ClockSampler(local) if rank == 0 else None
    pairs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    job_events.zero_()
    launches0 = sim.launch_count()
    e0.record(stream)
    for k in range(args.steps):
        one_step(args.warmup + k, pairs[k])
        job_events += count_events()
        flush.fill_(k & 0xFF)                                                              # L2 flush between iterations
    e1.record(stream)
    barrier()
    launches = sim.launch_count() - launches0
    clocks = sampler.stop() if sampler else None
    t_s, ev_total = W.reduce_over_ranks(e0.elapsed_time(e1) / 1e3, int(job_events.item()), device="cuda")   # max time, summed events
    kern_ms = statistics.mean(a.elapsed_time(b) for a, b in pairs)                  # the whole mig_sim_rollout call: generator + event loop
    ev_per_launch = int(job_events.item()) / args.steps
    sim.kernel_times()                                                             # forget the timed region's spans (profiling was off)
    # ---- per-kernel durations: a second, short region with the library's own event pairs around every launch -------
    sim.set_profiling(True)
    n_prof = max(1, min(args.steps, 3))
    last_episode = args.warmup + args.steps + n_prof - 1                            # the day `recs` / `totals` hold afterwards
    for k in range(n_prof):
        sim.reset(args.warmup + args.steps + k, d_algo, d_cfg0)
        sim.kernel_times()                                                         # (drops the reset launch)
        sim.rollout(wl.policy, table=d_table, qnet=qnet, epsilon=wl.epsilon, recs_out=recs, totals_out=totals)
        ms_k, n_k = sim.kernel_times()
        if k == 0:
            ms_sum, n_sum = dict(ms_k), dict(n_k)
        else:
            for key in ms_sum:
                ms_sum[key] += ms_k[key]; n_sum[key] += n_k[key]
        flush.fill_(k & 0xFF)
    sim.set_profiling(False)
    torch.cuda.synchronize()
    per_day_ms = {key: ms_sum[key] / n_prof for key in ms_sum}                      # per day-batch, all launches of that family
    # ---- the same steps with nothing drawn ahead (mig_sim_set_prefetch off): generator, then event loop, one after the other
    serial = None
    if prefetch:
        sim.set_prefetch(False)
        n_ser = max(1, min(args.steps, 5))
        one_step(0)
        torch.cuda.synchronize()
        z0, z1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev_ser = torch.zeros(1, dtype=torch.int64, device="cuda")
        z0.record(stream)
        for k in range(n_ser):
            one_step(1 + k)
            ev_ser += count_events()
            flush.fill_(k & 0xFF)
        z1.record(stream)
        torch.cuda.synchronize()
        sim.kernel_times()
        sim.set_profiling(True)
        sim.reset(last_episode, d_algo, d_cfg0)
        sim.kernel_times()
        sim.rollout(wl.policy, table=d_table, qnet=qnet, epsilon=wl.epsilon, recs_out=recs, totals_out=totals)   # (leaves `recs` / `totals` on last_episode)
        ms_ser, _ = sim.kernel_times()
        sim.set_profiling(False)
        serial = {"ms_per_step": z0.elapsed_time(z1) / n_ser, "value": int(ev_ser.item()) / (z0.elapsed_time(z1) / 1e3), "unit": "job-events/s", "steps": n_ser,
                  "kernels_ms_per_day": dict(ms_ser), "what": "mig_sim_set_prefetch off: every step draws its own arrivals before its event loop starts"}
        sim.set_prefetch(True)
    # ---- end to end: HOST buffers through the C ABI, copies inside the timed region ---------------------------------
    h_tot = np.zeros(n_envs, dtype=B.TOTALS_DTYPE)
    h_recs = np.zeros((sp.n_epochs + 1, n_envs), dtype=B.REC_DTYPE)
    pin = [torch.from_numpy(a) for a in (wl.algo, wl.cfg0)] + ([torch.from_numpy(wl.table)] if wl.table is not None else [])
    rt = torch.cuda.cudart()
    for a in (h_tot, h_recs, wl.algo, wl.cfg0) + ((wl.table,) if wl.table is not None else ()):
        rt.cudaHostRegister(a.ctypes.data, a.nbytes, 0)
    sim.rollout_host(99, wl.algo, wl.cfg0, wl.policy, wl.table, qnet, wl.epsilon, h_recs, h_tot)    # warm (the episode before the first timed one: like every timed call, that one finds its arrival lists drawn ahead)
    barrier()
    t0 = time.perf_counter()
    ev_e2e = 0
    n_e2e = max(1, min(args.steps, 3))
    for k in range(n_e2e):
        sim.rollout_host(100 + k, wl.algo, wl.cfg0, wl.policy, wl.table, qnet, wl.epsilon, h_recs, h_tot)
        ev_e2e += int(h_tot["n_jobs"].sum() + h_tot["n_completed"].sum())
    torch.cuda.synchronize()
    e2e_t, e2e_ev = W.reduce_over_ranks(time.perf_counter() - t0, ev_e2e, device="cuda")
    h2d = wl.algo.nbytes + wl.cfg0.nbytes + (wl.table.nbytes if wl.table is not None else 0)
    d2h = h_tot.nbytes + h_recs.nbytes
    # ---- secondary number: the same day through mig_sim_step, one launch per decision epoch with the
    # actions given by the caller (here: the configurations the timed rollout chose), state, reward and record outputs on
    step_api = None
    if rank == 0 and not args.no_step_api:
        acts = [recs[k, :, 52].contiguous() for k in range(sp.n_epochs)]             # byte 52 of a record = cfg
        totals_roll = totals.clone()                                                  # of the last rollout (episode last_episode)
        state, reward = sim.alloc_state(), torch.zeros(n_envs, dtype=torch.float32, device="cuda")
        rec1, drain1 = torch.zeros((n_envs, 64), dtype=torch.uint8, device="cuda"), torch.zeros((n_envs, 64), dtype=torch.uint8, device="cuda")
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for it in range(2):                                                           # first day: warm-up
            sim.reset(last_episode, d_algo, d_cfg0, state_out=state)
            s0.record(stream)
            for k in range(sp.n_epochs):
                sim.step(acts[k], state_out=state, reward_out=reward, rec_out=rec1, drain_rec_out=drain1)
            sim.totals(totals)
            s1.record(stream)
            torch.cuda.synchronize()
        ev_step = int(count_events().item())
        step_api = {"value": ev_step / (s0.elapsed_time(s1) / 1e3), "unit": "job-events/s", "ms_per_day": s0.elapsed_time(s1),
                    "launches_per_day": sp.n_epochs + 1, "identical_to_rollout": bool(torch.equal(totals, totals_roll))}
    # ---- roofline of the dominant kernel: plain ALU / issue slots ------------------------------------------------------
    props = torch.cuda.get_device_properties(local)
    sm_mhz = float(peaks.get("sm_max_mhz", 1965.0))
    tile = sim.get_tile()
    kname = sim.kernel_name()
    peak_gips = props.multi_processor_count * 128 * sm_mhz * 1e6 / 1e9           # G lane-instr/s: SMs x 128 lanes x f_max
    sim_ms = per_day_ms["sim"] if per_day_ms["sim"] > 0 else kern_ms
    alg_sim = ALG_LANE_INSTR["sim"] + (0.0 if per_day_ms["gen"] > 0 else ALG_LANE_INSTR["gen"])   # tiles draw arrivals inside the rollout kernel
    drawn_in_tail = None
    if serial and serial["kernels_ms_per_day"].get("gen", 0.0) > 0:                 # the share of the generator's work that the event loop's tail did
        drawn_in_tail = max(0.0, 1.0 - per_day_ms["gen"] / serial["kernels_ms_per_day"]["gen"])
        alg_sim += ALG_LANE_INSTR["gen"] * drawn_in_tail
    achieved_gips = alg_sim * ev_per_launch / (sim_ms / 1e3) / 1e9
    path_gips = (ALG_LANE_INSTR["sim"] + ALG_LANE_INSTR["gen"]) * ev_per_launch / (kern_ms / 1e3) / 1e9
    # algorithmic HBM bytes per launch: the outputs the caller asked for + the per-env inputs, nothing else
    alg_bytes = n_envs * ((sp.n_epochs + 1) * 64 + 80) + d_algo.numel() + d_cfg0.numel() + (d_table.numel() if d_table is not None else 0)
    cap = None
    try:
        with open(NCU_SUMMARY) as f:
            cap = json.load(f).get("%s|%s|%d" % (kname, args.workload, n_envs))
    except Exception:
        cap = None
    from paper_2606_25082_b200 import ncu_summary
    fresh = bool(cap) and cap.get("csrc_sha16") == ncu_summary.csrc_sha16()
    traffic = cap.get("dram_bytes") if fresh else None
    roofline = {"bound": "alu", "achieved": achieved_gips, "peak": peak_gips, "unit": "Glane-instr/s", "frac": achieved_gips / peak_gips,
                "traffic": traffic, "kernel": kname, "kernel_ms": sim_ms, "alg_lane_instr_per_job_event": alg_sim,
                "peak_source": "%d SMs x 128 lanes x %s sm_max_mhz %.0f" % (props.multi_processor_count, peak_src, sm_mhz),
                "hot_path": {"frac": path_gips / peak_gips, "achieved": path_gips, "ms": kern_ms, "alg_lane_instr_per_job_event": ALG_LANE_INSTR["sim"] + ALG_LANE_INSTR["gen"],
                             "what": "generator + event loop: the whole mig_sim_rollout call (round 1's definition of frac)"},
                "drawn_in_tail": drawn_in_tail, "kernels_ms_per_day": per_day_ms, "launches_per_day": {key: n_sum[key] / n_prof for key in n_sum},
                "hbm_algorithmic_bytes_per_launch": alg_bytes, "traffic_over_algorithmic": (traffic / alg_bytes) if traffic else None,
                "hbm_peak_gbs": peaks.get("hbm_gbs"), "hbm_frac": alg_bytes / (sim_ms / 1e3) / 1e9 / float(peaks.get("hbm_gbs", 6650.0)),
                "arrival_list_records_per_env": sim.get_arrival_buffer() if tile == 1 else 0,
                "ncu_capture": None if not cap else {"fresh": fresh, "csrc_sha16": cap.get("csrc_sha16"), "duration_ms": cap.get("duration_ms"),
                                                     "active_threads_per_inst": cap.get("active_threads_per_inst"),
                                                     "issue_frac_executed": (cap.get("issue_pct_of_peak_elapsed") or 0.0) / 100.0 or None,
                                                     "executed_lane_instr_per_job_event": (cap.get("thread_inst_executed_true") / ev_per_launch) if cap.get("thread_inst_executed_true") else None,
                                                     "global_ld_bytes_per_sector": cap.get("global_ld_bytes_per_sector")}}
    line = None
    if rank == 0:
        import concurrent.futures as cf
        cpu = None
        if not args.no_cpu_baseline:
            cores = os.cpu_count() or 1
            n_sample = min(n_envs, CPU_SAMPLE_ENVS)
            with cf.ProcessPoolExecutor(cores) as pool:
                time_oracle(args.workload, n_envs, min(n_sample, cores * 2), pool, cores)
                ev, dt = time_oracle(args.workload, n_envs, n_sample, pool, cores)
            n1 = min(n_envs, 128)                                                        # (i) of SURVEY 8(d): one core
            t1 = time.perf_counter(); ev1 = _oracle_chunk((args.workload, n_envs, 0, n1)); dt1 = time.perf_counter() - t1
            cpu = {"value": ev / dt, "unit": "job-events/s", "cores": cores, "kind": "oracle", "one_core_value": ev1 / dt1,
                   "one_core_sample": "first %d envs, one process (%.1f s)" % (n1, dt1),
                   "sample": "first %d of %d envs of %s, one simulated day each, split statically over %d processes (%.1f s wall)" % (n_sample, n_envs, args.workload, cores, dt)}
        line = {
            "metric": "job_events_per_s", "value": ev_total / t_s, "unit": "job-events/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * t_s / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int64", "data": "synthetic",
            "config": {"workload": args.workload, "n_envs_per_gpu": n_envs, "n_envs_total": n_envs * world, "policy": ["static", "table", "dqn"][wl.policy], "algo": W.ALGO_NAMES[int(wl.algo[0])] if len(set(wl.algo.tolist())) == 1 else "mixed", "lanes_per_env": sim.get_tile(), "envs_per_warp": args.envs_per_warp or "auto",
                       "prefetch": ("on: the arrival lists of step k + 1 are drawn in the tail of step k's event loop; every timed step draws one day of lists and simulates one" if prefetch else "off"),
                       "job_events_per_step": ev_total / args.steps, "l2": "flushed between iterations (256 MiB write)", "parallelism": "env-range sharding, no data-path collective",
                       "dist": ("nccl, world %d" % dist.get_world_size()) if dist.is_initialized() else None},
            "day_episodes_per_s": n_envs * world * args.steps / t_s,
            "e2e": {"value": e2e_ev / e2e_t, "unit": "job-events/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": n_e2e},
            "gpu_launches": launches, "clocks": clocks, "roofline": roofline, "cpu_baseline": cpu, "step_api": step_api, "serial": serial,
        }
        print(json.dumps(line))
    sim.close()
    if dist.is_initialized():
        dist.destroy_process_group()
    return 0


# ------------------------------------------------------------------------------------------------ DQN training step (secondary)
DQN_FLOP_PER_TRANSITION = 647168.0   # algorithmic, H = 256, A = 12: forward of two networks 4 (64H + H^2 + HA), backward through the
                                     # activations 2 (HA + H^2), weight gradients 2 (HA + H^2 + 64H); the 3 x TF32 split is NOT counted


def _dqn_oracle_sample(n):
    from oracle import oracle as O
    from paper_2606_25082_b200 import workloads as W
    net = W.make_qnet(1003, 12, 256)
    rng = np.random.default_rng(0)
    o = O.Dqn(net, 0.9, 0.01)
    s, s2 = rng.normal(0, 1, (n, 64)).astype(np.float32), rng.normal(0, 1, (n, 64)).astype(np.float32)
    a, r = rng.integers(0, 12, n).astype(np.uint8), rng.normal(0, 1, n).astype(np.float32)
    t0 = time.perf_counter()
    o.train_step(s, a, r, s2, None)
    return time.perf_counter() - t0


def run_dqn(args):
    """`--workload DQN`: one step = one mig_dqn_train_step on a batch of --envs transitions (default 32768) sampled from a
    replay ring of 24 x 8192 transitions (one C4 day): sample + forward of the online and the target network + TD error +
    backward + SGD, all products on the tensor cores (3 x TF32).  SURVEY 8(f) #2; a secondary line, not the headline."""
    import torch
    from paper_2606_25082_b200 import binding as B
    from paper_2606_25082_b200 import workloads as W
    if args.impl == "reference":
        n = 512
        dt = [_dqn_oracle_sample(n) for _ in range(max(1, args.steps))]
        v = n * len(dt) / sum(dt)
        print(json.dumps({"impl": "reference", "metric": "dqn_transitions_per_s", "value": v, "unit": "transitions/s", "n_gpus": args.gpus, "steps": args.steps,
                          "warmup": args.warmup, "ms_per_step": 1e3 * sum(dt) / len(dt), "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
                          "data": "synthetic", "config": {"workload": "DQN", "batch": n}, "cpu_baseline": {"value": v, "unit": "transitions/s", "cores": 1, "kind": "oracle",
                          "sample": "one training step on %d transitions" % n}, "e2e": {"value": v, "unit": "transitions/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}))
        return 0
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    peaks, peak_src = _peaks()
    batch = args.envs if args.envs and args.envs % 128 == 0 else 32768
    cap = 24 * 8192
    net = W.make_qnet(1003, 12, 256)
    d = B.Dqn(net, cap, batch, 0.9, 1e-3, 1003)
    g = torch.Generator(device="cuda"); g.manual_seed(0)
    S, S2 = torch.randn((cap, 64), device="cuda", generator=g), torch.randn((cap, 64), device="cuda", generator=g)
    A = torch.randint(0, 12, (cap,), device="cuda", dtype=torch.uint8, generator=g); R = torch.randn(cap, device="cuda", generator=g)
    d.push(S, A, R, S2)
    loss = torch.zeros(1, dtype=torch.float32, device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream()
    for w in range(max(3, args.warmup)):
        d.train_step(w, loss_out=loss); flush.fill_(w & 0xFF)
    torch.cuda.synchronize()
    sampler = ClockSampler(0)
    pairs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    l0 = d.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for k in range(args.steps):
        pairs[k][0].record(stream)
        d.train_step(100 + k, loss_out=loss)
        pairs[k][1].record(stream)
        flush.fill_(k & 0xFF)                                                          # L2 flush between iterations
    e1.record(stream)
    torch.cuda.synchronize()
    clocks = sampler.stop()
    launches = d.launch_count() - l0
    step_ms = statistics.mean(a.elapsed_time(b) for a, b in pairs)
    wall_s = e0.elapsed_time(e1) / 1e3
    # end to end: the batch comes from pinned HOST buffers, the loss goes back to the host, every step
    hs, hs2 = torch.randn((batch, 64)).pin_memory(), torch.randn((batch, 64)).pin_memory()
    ha, hr = torch.randint(0, 12, (batch,), dtype=torch.uint8).pin_memory(), torch.randn(batch).pin_memory()
    ds, ds2, da, dr = (torch.empty_like(x, device="cuda") for x in (hs, hs2, ha, hr))
    n_e2e = max(1, min(args.steps, 5))
    torch.cuda.synchronize(); t0 = time.perf_counter()
    for k in range(n_e2e):
        ds.copy_(hs, non_blocking=True); ds2.copy_(hs2, non_blocking=True); da.copy_(ha, non_blocking=True); dr.copy_(hr, non_blocking=True)
        d.train_on(ds, da, dr, ds2, None, loss_out=loss)
        float(loss.item())
    e2e_s = time.perf_counter() - t0
    h2d = hs.numel() * 4 * 2 + ha.numel() + hr.numel() * 4
    tf32_peak = float(peaks.get("bf16_tflops", peaks.get("bf16_tflops_burst", 1685.8))) / 2.0      # the guide's nominal ratio TF32 : BF16 = 1 : 2
    achieved = DQN_FLOP_PER_TRANSITION * batch / (step_ms / 1e3) / 1e12
    from paper_2606_25082_b200 import ncu_summary                   # DRAM bytes of the eleven products of one step, from the committed capture
    try:
        with open(NCU_SUMMARY) as f:
            cap = json.load(f).get("gemm_tf32x3_kernel (the 11 products of one step)|DQN|%d" % batch)
    except Exception:
        cap = None
    traffic = cap.get("dram_bytes") if cap and cap.get("csrc_sha16") == ncu_summary.csrc_sha16() else None
    cpu = None
    if not args.no_cpu_baseline:
        n = 512
        dt = _dqn_oracle_sample(n)
        cpu = {"value": n / dt, "unit": "transitions/s", "cores": 1, "kind": "oracle", "sample": "one double-precision training step on %d transitions (%.2f s)" % (n, dt)}
    line = {"metric": "dqn_transitions_per_s", "value": batch * args.steps / wall_s, "unit": "transitions/s", "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * wall_s / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "tf32x3 (fp32 in, fp32 accumulate)",
            "data": "synthetic", "config": {"workload": "DQN", "batch": batch, "replay": cap, "net": "64-256-256-12", "l2": "flushed between iterations (256 MiB write)"},
            "train_steps_per_s": 1e3 / step_ms, "e2e": {"value": batch * n_e2e / e2e_s, "unit": "transitions/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": 4, "steps": n_e2e},
            "gpu_launches": launches, "clocks": clocks,
            "roofline": {"bound": "tensor", "achieved": achieved, "peak": tf32_peak, "unit": "TFLOP/s", "frac": achieved / tf32_peak, "traffic": traffic,
                         "traffic_scope": "DRAM bytes of the eleven tensor-core launches of one step (ncu --set full, profiles/r2_dqn.md); achieved is over all kernels of the step",
                         "kernel": "gemm_tf32x3_kernel<BN, MN> (the eleven products of a step: 128 x 256, 128 x 128, 128 x 16 tiles, K-major; 128 x 32 and 128 x 128 MN-major)", "step_ms": step_ms, "flop_per_transition_algorithmic": DQN_FLOP_PER_TRANSITION,
                         "issued_over_algorithmic": 3.0, "peak_source": "%s bf16 dense / 2 (TF32 : BF16 = 1 : 2, B200_PROFILING.md)" % peak_src},
            "cpu_baseline": cpu}
    print(json.dumps(line))
    d.close()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="C5", choices=["C1", "C2", "C3", "C4", "C5", "DQN"])
    ap.add_argument("--envs", type=int, default=0, help="environments per GPU (default: the workload's BASELINE size)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-step-api", action="store_true", help="skip the secondary mig_sim_step measurement")
    ap.add_argument("--algo", type=int, default=-1, choices=[-1, 0, 1, 2, 3, 4], help="override the workload's scheduling algorithm for every env (4 = EDF-SS with restricted preemption); -1 = the workload's own")
    ap.add_argument("--envs-per-warp", type=int, default=0, choices=[0, 1, 2, 4, 8, 16, 32],
                    help="thread-per-environment kernel: environments in each warp (0 = the library's choice: one resident wave); a study knob, see profiles/r2_thread.md")
    ap.add_argument("--prefetch", type=int, default=1, choices=[0, 1],
                    help="1 (default): mig_sim_set_prefetch -- the next step's arrival lists are drawn in the tail of this step's event loop (same results; "
                         "the line's `serial` object is the same measurement with it off); thread-per-environment kernel only")
    ap.add_argument("--tile", type=int, default=0, choices=[0, 1, 8, 16, 32], help="lanes per environment (0 = library default = 1: one thread per environment; 8, 16, 32: warp tiles)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    if args.workload == "DQN":
        return run_dqn(args)
    if not args.envs:
        args.envs = {"C1": 1, "C2": 1024, "C3": 4096, "C4": 8192, "C5": 65536}[args.workload]
    global _ALGO_OVERRIDE
    _ALGO_OVERRIDE = args.algo                            # (worker processes are forked after this)
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
