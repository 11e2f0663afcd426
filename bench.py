#!/usr/bin/env python
"""bench.py -- spin-flip attempts/ns of the whole PT hot path on BASELINE.json's config 4
(L=64, R=128, Gaussian field h=2.0, geometric T in [0.8, 6.0], exchange every 10, seed 4).

One "step" = one parallel-tempering move: exchange_every (=10) checkerboard Metropolis
sweeps of all 128 replicas + the per-replica energy reduction + one exchange step.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfg4]

N > 1 (torchrun, one rank per GPU): every rank runs its own disorder realisation of the same
workload (seed 4 + rank) -- independent problems, no data-path collective, "scaling": "weak".
Prints ONE JSON line on rank 0.
"""
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

METRIC = "spin-flip attempts/ns (all replicas) at L=64,R=128; % of sweep roofline"
UNIT = "attempts/ns"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg4")
    ap.add_argument("--variant", type=int, default=0, help="kernel variant (0 = automatic)")
    ap.add_argument("--packing", type=int, default=8)
    ap.add_argument("--multi", default="realisations", choices=["realisations", "replicas"],
                    help="N > 1: independent disorder realisations per rank (weak scaling, no collective; default) or the "
                         "replicas of ONE realisation dealt to the ranks (PAPER.md:123-137; strong scaling, one all-gather "
                         "of 24 B per replica per exchange step)")
    ap.add_argument("--window", default="contiguous", choices=["contiguous", "rr"],
                    help="replica split: contiguous windows of ceil(R/N) slots (PAPER.md:125, Eq. 6) or round-robin, slot i on rank i mod N (PAPER.md:153)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--e2e-handles", type=int, default=4,
                    help="end-to-end leg: handles (host threads, streams) whose steps overlap, copies against sweeps; 1 = one handle, serial")
    ap.add_argument("--stage-timing", action="store_true",
                    help="debug builds with -DRFIM_RES_TIMING only: print the resident kernel's per-stage globaltimer stamps of one step")
    ap.add_argument("--no-secondary", action="store_true", help="skip the secondary workloads (config 5 int8 / bit-packed, config 3, sustained config 4)")
    return ap.parse_args()


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "25"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
                for nm, val in zip(names, r[3:7]):
                    if val.lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                pass
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(wl, threads, r_sample, sweeps, steps, warmup, seed):
    """Time the oracle, as it stands, on a bounded sample of the workload: r_sample replicas spread over
    the ladder, `sweeps` sweeps + one exchange step per step.  Returns attempts/ns."""
    import numpy as np
    import oracle
    T = wl.temperatures()
    sel = np.unique(np.round(np.linspace(0, wl.R - 1, r_sample)).astype(int))
    o = oracle.Oracle(wl.L, len(sel), wl.J, wl.h, wl.field_kind, seed, threads=threads)
    o.set_temperatures(T[sel])
    for _ in range(warmup):
        o.sweep(sweeps, sweeps)
    t0 = time.perf_counter()
    for _ in range(steps):
        o.sweep(sweeps, sweeps)
    dt = time.perf_counter() - t0
    attempts = float(wl.N) * len(sel) * sweeps * steps
    return attempts / dt * 1e-9, dt / max(steps, 1) * 1e3, len(sel)


def workload_name(wl, seed):
    """config.workload: one spelling for both arms (ours and --impl reference)."""
    return (f"{wl.name}: L={wl.L} R={wl.R} D={wl.D} {'Gaussian' if wl.field_kind else 'bimodal'} h={wl.h} "
            f"T {wl.ladder} [{wl.t_min},{wl.t_max}] exchange_every={wl.exchange_every} seed={seed}")


def run_reference(args, wl, rank, world):
    if rank != 0:
        return
    cores = os.cpu_count() or 1
    # size the per-step sample so that (steps + warmup) steps end within ~2 minutes
    total_steps = args.steps + args.warmup
    rate_guess = 0.02e9 * max(1, min(cores, 16)) * 0.6            # attempts/s, from the oracle's measured single-core rate
    budget_attempts = 100.0 * rate_guess / max(total_steps, 1)
    sweeps = wl.exchange_every
    r_sample = int(budget_attempts / (wl.N * sweeps))
    if r_sample < 2:
        r_sample = 2
        sweeps = max(1, int(budget_attempts / (wl.N * 2)))
        sweeps = min(sweeps, wl.exchange_every)
    r_sample = min(r_sample, wl.R)
    threads = max(1, min(cores, r_sample))
    value, ms_per_step, r_used = oracle_sample(wl, threads, r_sample, sweeps, args.steps, args.warmup, wl.seeds[0])
    sample = f"{r_used} of {wl.R} replicas (evenly spread over the ladder) x {sweeps} sweeps + 1 exchange step per step, L={wl.L}"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "u8", "data": "synthetic",
            "config": {"workload": workload_name(wl, wl.seeds[0]),
                       "reference": "CPU oracle (oracle/rfim_oracle.cpp) as it stands, bounded sample per step"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    args = parse()
    from paper_1508_06268_b200 import workloads
    wl = workloads.CONFIGS[args.workload]
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, wl, rank, world)
        return

    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_1508_06268_b200 import binding, sharding

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    k = wl.exchange_every
    replicas = world > 1 and args.multi == "replicas" and wl.D == 1
    def make_replica_shard():
        """One realisation, its replica slots dealt to the ranks; the library issues the NCCL calls itself."""
        if args.window == "rr":
            hs = binding.RfimPT(wl.L, wl.R, wl.J, wl.h, wl.field_kind, seed=wl.seeds[0], shard_rr=(rank, world))
        else:
            hs = binding.RfimPT(wl.L, wl.R, wl.J, wl.h, wl.field_kind, seed=wl.seeds[0], shard=sharding.replica_window(wl.R, world, rank))
        try:
            hs.set_nccl(sharding.NcclComm(rank, world))
        except Exception:                           # no usable libnccl: fall back to the torch.distributed callbacks
            hs.set_gather(sharding.make_terms_gather(rank, world))
            hs.set_broadcast(sharding.make_lattice_broadcast())
        return hs

    if replicas:
        g = make_replica_shard()
    else:
        seeds = sharding.rank_seeds(wl.seeds, rank)    # each rank: its own disorder realisation(s)
        if wl.D == 1:
            g = binding.RfimPT(wl.L, wl.R, wl.J, wl.h, wl.field_kind, seed=seeds[0])
        else:
            g = binding.RfimPT(wl.L, wl.R, wl.J, wl.h, wl.field_kind, seeds=seeds)
    if args.packing != 8:
        g.set_packing(args.packing)
    if args.variant:
        g.set_kernel_variant(args.variant)
    g.set_temperatures(wl.temperatures())
    attempts_per_step = float(wl.N) * wl.R * wl.D * k            # per rank (realisations) ...
    if replicas:
        attempts_per_step /= world                                  # ... or this rank's share of the one realisation

    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2

    def timed_steps(n_steps, exchange_every):
        """n_steps steps, each bracketed by CUDA events on the launch stream, L2 flushed between steps."""
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n_steps)]
        for a, b in ev:
            flush.zero_()
            a.record()
            g.sweep(k, exchange_every)
            b.record()
        torch.cuda.synchronize()
        return [a.elapsed_time(b) for a, b in ev]

    for _ in range(max(args.warmup, 3)):
        g.sweep(k, k)
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    l0 = g.diagnostics()["launches"]
    barrier()
    t_wall = time.perf_counter()
    ms = timed_steps(args.steps, k)
    barrier()
    t_wall = time.perf_counter() - t_wall
    l1 = g.diagnostics()["launches"]
    # dominant kernel alone (sweeps only, no reduction / exchange), same launch configuration
    ms_sweep = timed_steps(args.steps, 0)
    clocks = sampler.stop()
    total_ms = float(sum(ms))
    total_ms_sweep = float(sum(ms_sweep))
    total_ms, total_ms_sweep = sharding.max_over_ranks([total_ms, total_ms_sweep], device="cuda")
    value = sharding.whole_job_rate(attempts_per_step * args.steps, world, total_ms)
    sweep_rate = attempts_per_step * args.steps / (total_ms_sweep * 1e6)      # per GPU

    # the two candidate bounds, measured in this run on this GPU (north_star)
    ph_ms, ph_att = binding.bench_philox(4000, stream=torch.cuda.current_stream().cuda_stream)
    philox_bound = ph_att / (ph_ms * 1e6)
    st_ms, st_bytes = binding.bench_stream(1 << 30, stream=torch.cuda.current_stream().cuda_stream)
    stream_gbs = st_bytes / (st_ms * 1e6)
    # what one more warp instruction costs a sub-partition that is running the Philox stream
    issue_probe = None
    if world == 1:
        cs = torch.cuda.current_stream().cuda_stream
        ms0, wr = binding.bench_issue(0, 0, stream=cs)
        mhz = 1965.0
        cyc0 = ms0 * 1e-3 * mhz * 1e6 / wr
        issue_probe = {"philox_only_cycles_per_warp_row": cyc0, "assumed_sm_mhz": mhz,
                       "cycles_per_extra_warp_instruction": {}}
        for name, kind in binding.PROBE_KINDS.items():
            ms1, _ = binding.bench_issue(kind, 8, stream=cs)
            issue_probe["cycles_per_extra_warp_instruction"][name] = (ms1 - ms0) * 1e-3 * mhz * 1e6 / wr / 2.0
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    bytes_per_attempt = 2.0 if args.packing == 8 else 0.25
    hbm_bound = hbm_peak / bytes_per_attempt                                  # attempts/ns if HBM were the limit
    bound = min(philox_bound, hbm_bound)
    # The issue-rate bound DESIGN.md section 6 derives for a Philox4x32-10 stream on one SM sub-partition: one call = 18.25
    # IMAD.WIDE (warp-uniform products hoisted) + 21 three-input XORs, each holding the integer issue port for 2 cycles
    # -> 4 attempts per (18.25 + 21) * 2 cycles per lane-slot ... expressed per SM: 32 lanes * 4 sub-partitions * 4 attempts
    clocks_mhz = clocks.get("sm_mhz") or float(peaks.get("sm_max_mhz", 1965.0))
    n_sm = torch.cuda.get_device_properties(local_rank).multi_processor_count
    philox_theory = 32.0 * 4 * 4 / ((18.25 + 21.0) * 2.0) * n_sm * clocks_mhz * 1e-3          # attempts/ns
    traffic, traffic_source = None, None
    try:
        cap = json.load(open(os.path.join(ROOT, "profiles", "r2_res_sweep_full.json")))
        if wl.name == cap.get("workload") and args.packing == cap.get("packing_bits", 8) and world == 1:
            traffic = float(cap["dram_bytes_read"]) + float(cap["dram_bytes_write"])
            traffic_source = f"profiles/r2_res_sweep_full.json (ncu --set full capture at commit {cap.get('commit')}; not measured in this run)"
    except Exception:
        pass
    roofline = {"bound": "alu" if philox_bound <= hbm_bound else "hbm", "achieved": sweep_rate, "peak": bound, "unit": UNIT,
                "frac": sweep_rate / bound,
                "traffic": traffic, "traffic_source": traffic_source,
                "traffic_unit": "bytes per launch (ncu dram__bytes_read.sum + dram__bytes_write.sum)",
                "algorithmic_bytes_per_launch": 2.0 * wl.N * wl.R * wl.D / (8 if args.packing == 1 else 1),
                "kernel": "k_sweep_res, sweeps only (exchange_every = 0), timed alone with CUDA events over the same steps",
                "philox_bound_measured": philox_bound, "philox_bound_issue_model": philox_theory,
                "frac_vs_issue_model": sweep_rate / min(philox_theory, hbm_bound), "hbm_bound": hbm_bound,
                "hbm_peak_gbs": hbm_peak, "hbm_peak_source": "MEASURED_PEAKS.json" if peaks else "fallback 6650 GB/s",
                "stream_rmw_gbs_this_run": stream_gbs,
                "algorithmic_bytes_per_attempt": bytes_per_attempt,
                "achieved_algorithmic_gbs": sweep_rate * bytes_per_attempt,
                "issue_cost_probe": issue_probe,
                "whole_step_frac": (value / world) / bound,
                "whole_step_frac_vs_issue_model": (value / world) / min(philox_theory, hbm_bound)}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "strong" if replicas else "weak", "vs_baseline": None,
            "dtype": "u8" if args.packing == 8 else "u1", "data": "synthetic",
            "config": {"workload": workload_name(wl, wl.seeds[0]),
                       "step": f"{k} sweeps + energy reduction + 1 exchange step", "l2": "flushed between steps (256 MiB memset)",
                       "packing_bits": args.packing, "kernel_variant": args.variant,
                       "parallelism": "1 GPU" if world == 1 else (f"replicas of one realisation over {world} GPUs, all-gather of energy terms per exchange step"
                                                                     if replicas else f"{world} independent realisations, one per GPU")},
            "clocks": clocks, "gpu_launches": int(l1 - l0), "wall_s_timed_region": t_wall, "roofline": roofline}

    if args.stage_timing and world == 1:
        import ctypes
        lib = binding.load()
        if hasattr(lib, "rfim_pt_debug_timing"):
            names = ["start", "setup_done", "run_loaded", "tasks_done_warp0", "after_barrier", "run_stored", "end"]
            rows = {}
            for kk, tag in ((0, "sweeps_only"), (k, "whole_step")):
                acc = []
                for _ in range(7):
                    flush.zero_(); torch.cuda.synchronize()
                    g.sweep(k, kk); torch.cuda.synchronize()
                    buf = np.zeros((256, 8), dtype=np.uint64)
                    lib.rfim_pt_debug_timing(buf.ctypes.data_as(ctypes.c_void_p))
                    t = buf[:torch.cuda.get_device_properties(local_rank).multi_processor_count].astype(np.int64)
                    acc.append((t - t[:, 0].min()) / 1e3)
                rel = np.median(np.stack(acc[2:]), axis=0)
                rows[tag] = {nm: {"median_over_ctas_us": float(np.median(rel[:, i])), "max_over_ctas_us": float(rel[:, i].max())} for i, nm in enumerate(names)}
            line["stage_timing_us"] = rows
        else:
            line["stage_timing_us"] = "library not built with -DRFIM_RES_TIMING"

    # N > 1: the paper's own multi-GPU mode next to the default (independent realisations): ONE realisation, replicas dealt to the
    # ranks, one all-gather of 24 B per replica per exchange step -- strong scaling, measured in the same run
    if world > 1 and not replicas and wl.D == 1:
        try:
            hs = make_replica_shard()
            hs.set_temperatures(wl.temperatures())
            for _ in range(3):
                hs.sweep(k, k)
            barrier()
            ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
            for a, b in ev:
                flush.zero_()
                a.record(); hs.sweep(k, k); b.record()
            torch.cuda.synchronize()
            barrier()
            ms_split = sharding.max_over_ranks([float(sum(a.elapsed_time(b) for a, b in ev))], device="cuda")[0]
            att_total = float(wl.N) * wl.R * k * args.steps
            line["replica_split"] = {"scaling": "strong", "value": att_total / (ms_split * 1e6), "unit": UNIT,
                                     "ms_per_step": ms_split / args.steps, "window": args.window,
                                     "collective": "ncclAllGather of 24 B per replica per exchange step, issued by the library"}
            hs.close()
        except Exception as e:                      # never lose the primary line to the secondary measurement
            line["replica_split"] = {"error": repr(e)[:300]}

    # secondary workloads ("also reported for config 5 int8 and bit-packed"), each with its own device timing
    if world == 1 and not args.no_secondary:
        def timed_other(h, kk, n_steps, do_flush=True):
            for _ in range(3):
                h.sweep(kk, kk)
            ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n_steps)]
            for a, b in ev:
                if do_flush:
                    flush.zero_()
                a.record(); h.sweep(kk, kk); b.record()
            torch.cuda.synchronize()
            return float(sum(a.elapsed_time(b) for a, b in ev)) / n_steps

        def entry(w2, ms_step, extra=None):
            att = float(w2.N) * w2.R * w2.D * w2.exchange_every
            e = {"workload": f"{w2.name}: L={w2.L} R={w2.R} D={w2.D} {'Gaussian' if w2.field_kind else 'bimodal'} h={w2.h} exchange_every={w2.exchange_every}",
                 "value": att / (ms_step * 1e6), "unit": UNIT, "ms_per_step": ms_step, "frac": att / (ms_step * 1e6) / bound,
                 "step": f"{w2.exchange_every} sweeps + energy reduction + 1 exchange step, L2 flushed between steps"}
            e.update(extra or {})
            return e

        secondary = {}
        n_sec = max(5, min(args.steps, 20))
        if wl.name == "cfg4" and args.packing == 8:
            # the production protocol: ONE call of rfim_pt_sweep(10^4, 10), no flush, CUDA events around it, clocks sampled
            s2 = ClockSampler(local_rank); s2.start()
            runs = []
            for _ in range(3):                      # three calls, the median: a call may grow the device time series (an allocation)
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(); g.sweep(wl.sweeps, k); b.record(); torch.cuda.synchronize()
                runs.append(a.elapsed_time(b))
            c2 = s2.stop()
            ms_run = sorted(runs)[1]
            att = float(wl.N) * wl.R * wl.sweeps
            secondary["cfg4_sustained"] = {"workload": f"cfg4: one rfim_pt_sweep({wl.sweeps}, {k}) call (12 parallel-tempering moves per launch), no L2 flush", "value": att / (ms_run * 1e6),
                                           "unit": UNIT, "ms_total": ms_run, "ms_all_calls": runs, "ms_per_step": ms_run / (wl.sweeps / k),
                                           "frac": att / (ms_run * 1e6) / bound, "clocks": c2}
            # temporal blocking: sweeps fused per resident pass, exact dynamics (halo rows
            # exchanged every phase), no measurement / exchange step; HBM bytes per attempt = 2 / sweeps_per_launch
            tb = []
            for spl in (1, 2, 5, 10, 20, 50, 100):
                reps = max(3, 60 // spl)
                g.sweep(spl, 0)
                ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
                for a, b in ev:
                    flush.zero_()
                    a.record(); g.sweep(spl, 0); b.record()
                torch.cuda.synchronize()
                t = sorted(a.elapsed_time(b) for a, b in ev)[reps // 2]
                tb.append({"sweeps_per_launch": spl, "value": float(wl.N) * wl.R * spl / (t * 1e6), "ms_per_launch": t,
                           "hbm_bytes_per_attempt": 2.0 / spl})
            secondary["temporal_blocking"] = {"workload": "cfg4, sweeps only, one launch = sweeps_per_launch sweeps of every replica, L2 flushed between launches",
                                              "unit": UNIT, "points": tb}
        w5 = workloads.CONFIGS["cfg5"]
        h5 = binding.RfimPT(w5.L, w5.R, w5.J, w5.h, w5.field_kind, seeds=list(w5.seeds))
        h5.set_temperatures(w5.temperatures())
        secondary["cfg5_u8"] = entry(w5, timed_other(h5, w5.exchange_every, n_sec), {"dtype": "u8"})
        h5.set_packing(1)
        secondary["cfg5_u1"] = entry(w5, timed_other(h5, w5.exchange_every, n_sec), {"dtype": "u1", "note": "spins bit-packed in HBM"})
        h5.close()
        w3 = workloads.CONFIGS["cfg3"]
        h3 = binding.RfimPT(w3.L, w3.R, w3.J, w3.h, w3.field_kind, seed=w3.seeds[0])
        h3.set_temperatures(w3.temperatures())
        secondary["cfg3"] = entry(w3, timed_other(h3, w3.exchange_every, n_sec), {"dtype": "u8"})
        # config 3's production run as ONE call (the library holds as many exchange periods per launch as fit in 127 sweeps)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); h3.sweep(w3.sweeps, w3.exchange_every); b.record(); torch.cuda.synchronize()
        att3 = float(w3.N) * w3.R * w3.sweeps
        secondary["cfg3_sustained"] = {"workload": f"cfg3: one rfim_pt_sweep({w3.sweeps}, {w3.exchange_every}) call, no L2 flush",
                                       "value": att3 / (a.elapsed_time(b) * 1e6), "unit": UNIT, "ms_total": a.elapsed_time(b),
                                       "ms_per_step": a.elapsed_time(b) / (w3.sweeps / w3.exchange_every),
                                       "frac": att3 / (a.elapsed_time(b) * 1e6) / bound}
        h3.close()
        w2 = workloads.CONFIGS["cfg2"]
        h2 = binding.RfimPT(w2.L, w2.R, w2.J, w2.h, w2.field_kind, seed=w2.seeds[0])
        h2.set_temperatures(w2.temperatures())
        secondary["cfg2"] = entry(w2, timed_other(h2, w2.exchange_every, n_sec), {"dtype": "u8"})
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); h2.sweep(w2.sweeps, w2.exchange_every); b.record(); torch.cuda.synchronize()
        att2 = float(w2.N) * w2.R * w2.sweeps
        secondary["cfg2_sustained"] = {"workload": f"cfg2: one rfim_pt_sweep({w2.sweeps}, {w2.exchange_every}) call, no L2 flush",
                                       "value": att2 / (a.elapsed_time(b) * 1e6), "unit": UNIT, "ms_total": a.elapsed_time(b),
                                       "ms_per_step": a.elapsed_time(b) / (w2.sweeps / w2.exchange_every),
                                       "frac": att2 / (a.elapsed_time(b) * 1e6) / bound}
        h2.close()
        line["secondary"] = secondary

    # end to end through the C ABI with HOST buffers, every step: H2D of every lattice (the step's input state) from pinned
    # memory, the step, D2H of every lattice and of the observables (the step's result).  Timed twice: with the bit-packed
    # host format (1 bit per spin, rfim_pt_*_spins_all_bits: the headline e2e) and with the int8 +-1 format (8x the bytes).
    if not args.no_e2e:
        n_e2e = max(3, min(args.steps, 20))
        obs_bytes = 2 * 8 * wl.D * wl.R

        def e2e_leg(host, put, get, what):
            get(host)
            for it in range(2 + n_e2e):
                if it == 2:
                    barrier()
                    t0 = time.perf_counter()
                put(host)
                g.sweep(k, k)
                get(host)
                g.observables()
            barrier()
            dt = sharding.max_over_ranks([time.perf_counter() - t0], device="cuda")[0]
            return {"value": attempts_per_step * n_e2e * world / (dt * 1e9), "unit": UNIT,
                    "h2d_bytes_per_step": int(host.nbytes), "d2h_bytes_per_step": int(host.nbytes + obs_bytes),
                    "steps": n_e2e, "what": what}

        def e2e_pipelined(n_pipe):
            """The same four calls per step, on n_pipe handles (independent realisations of the workload), each driven by its own
            host thread on its own stream: the copies of one handle's step overlap the sweep of another's (the sweeps themselves
            take the whole GPU in turn).  Every step still copies its inputs in from pinned host memory and its results out."""
            import threading
            hs, hosts = [g], []
            for i in range(1, n_pipe):
                sd = [int(s) + 7919 * i for s in seeds] if not replicas else None
                hi = binding.RfimPT(wl.L, wl.R, wl.J, wl.h, wl.field_kind, seed=sd[0]) if wl.D == 1 else \
                    binding.RfimPT(wl.L, wl.R, wl.J, wl.h, wl.field_kind, seeds=sd)
                if args.packing != 8:
                    hi.set_packing(args.packing)
                if args.variant:
                    hi.set_kernel_variant(args.variant)
                hi.set_temperatures(wl.temperatures())
                hs.append(hi)
            for hi in hs:
                hosts.append(torch.empty((wl.D, hi.stored_slots, wl.N // 8), dtype=torch.uint8).pin_memory().numpy())
            # distinct stream priorities: when a sweep ends, the copy-out kernel of the handle that just finished is picked before
            # the next handle's queued sweep, so the handles do not fall into lock-step (all copies, then all sweeps)
            streams = [torch.cuda.Stream(priority=-(i % 4)) for i in range(len(hs))]
            per = max(6, n_e2e)                   # steps per handle: long enough that filling and draining the pipeline do not count
            errs = []

            def one(i, n):
                try:
                    torch.cuda.set_device(local_rank)
                    with torch.cuda.stream(streams[i]):
                        hs[i].use_current_torch_stream()
                        for _ in range(n):
                            hs[i].set_spins_all_bits(hosts[i])
                            hs[i].sweep(k, k)
                            hs[i].get_spins_all_bits(out=hosts[i])
                            hs[i].observables()
                except Exception as e:            # surfaces after the join
                    errs.append(e)

            for i, hi in enumerate(hs):
                hi.get_spins_all_bits(out=hosts[i])
            for phase_n in (1, per):              # one warm-up round, then the timed one
                barrier()
                t0 = time.perf_counter()
                th = [threading.Thread(target=one, args=(i, phase_n)) for i in range(n_pipe)]
                for t in th:
                    t.start()
                for t in th:
                    t.join()
                barrier()
                dt = time.perf_counter() - t0
            g.use_current_torch_stream()
            for hi in hs[1:]:
                hi.close()
            if errs:
                raise errs[0]
            dt = sharding.max_over_ranks([dt], device="cuda")[0]
            return {"value": attempts_per_step * per * n_pipe * world / (dt * 1e9), "unit": UNIT,
                    "h2d_bytes_per_step": int(hosts[0].nbytes), "d2h_bytes_per_step": int(hosts[0].nbytes + obs_bytes),
                    "steps": per * n_pipe, "handles": n_pipe,
                    "what": f"per step: rfim_pt_set_spins_all_bits(host) + rfim_pt_sweep(k,k) + rfim_pt_get_spins_all_bits(host) + rfim_pt_observables; "
                            f"{n_pipe} handles (independent realisations) driven by {n_pipe} host threads on {n_pipe} streams of distinct priority, so one handle's copies "
                            f"overlap another's sweep; wall clock over all steps"}

        bits = torch.empty((wl.D, g.stored_slots, wl.N // 8), dtype=torch.uint8).pin_memory().numpy()
        serial = e2e_leg(bits, g.set_spins_all_bits, lambda h_: g.get_spins_all_bits(out=h_),
                         "rfim_pt_set_spins_all_bits(host) + rfim_pt_sweep(k,k) + rfim_pt_get_spins_all_bits(host) + rfim_pt_observables, one handle, "
                         "every call waited for before the next")
        line["e2e"] = serial
        if not replicas and args.e2e_handles > 1:
            try:
                piped = e2e_pipelined(args.e2e_handles)
                if piped["value"] > serial["value"]:
                    line["e2e"] = piped
                    line["e2e_one_handle"] = serial
                else:
                    line["e2e_pipelined"] = piped
            except Exception as e:                 # never lose the line to the overlapped leg
                line["e2e_pipelined"] = {"error": repr(e)}
        host = torch.empty((wl.D, g.stored_slots, wl.N), dtype=torch.int8).pin_memory().numpy()
        line["e2e_int8"] = e2e_leg(host, g.set_spins_all, lambda h_: g.get_spins_all(out=h_),
                                   "rfim_pt_set_spins_all(host) + rfim_pt_sweep(k,k) + rfim_pt_get_spins_all(host) + rfim_pt_observables")

    d = g.diagnostics()
    line["diagnostics"] = d
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cores = os.cpu_count() or 1
        threads = max(1, min(cores, 16))
        r_s = min(wl.R, 4 * threads)
        v0, ms0, r_used = oracle_sample(wl, threads, r_s, k, 1, 0, wl.seeds[0])      # one step, to size the sample
        n_b = int(max(2, min(200, 12e3 / max(ms0, 1.0))))                            # about 12 s of oracle work
        v, ms_b, r_used = oracle_sample(wl, threads, r_s, k, n_b, 0, wl.seeds[0])
        v1, ms1, r1 = oracle_sample(wl, 1, 4, k, 2, 0, wl.seeds[0])                   # and on ONE core
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle",
                                "single_core": {"value": v1, "unit": UNIT, "cores": 1,
                                                "sample": f"{r1} of {wl.R} replicas x 2 steps of ({k} sweeps + 1 exchange step), L={wl.L}"},
                                "sample": f"{r_used} of {wl.R} replicas x {n_b} steps of ({k} sweeps + 1 exchange step), L={wl.L} "
                                          f"({ms_b * n_b / 1e3:.1f} s wall, oracle as it stands, {threads} OpenMP threads over replicas)"}
    if rank == 0:
        print(json.dumps(line), flush=True)
    g.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
