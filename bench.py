#!/usr/bin/env python
"""bench.py -- whole-hot-path benchmark of necsim-b200 (contract: see DESIGN.md section 7).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config c1..c5] [--small]

A "step" is one pass of the whole hot path S0-S6 (necsim_simulate: sample mask -> lineage queue, epochs of
the simulate kernel with duplicate culling, sort/unique -> species) over the synthetic config. Default workload:
C5 (BASELINE.json configs[4], the largest; the one north_star quotes the roofline target on).
`value` = DISTINCT lineage events (loc, k, j) per second of the whole job (the oracle's count of the workload, scheduling
          independent), inputs resident in HBM (device time, CUDA events); raw executed events per second ride along as
          `raw_events_per_s` (redundancy = raw / distinct). Without a stored count (reduced configs) value = raw, `value_kind` says which.
`e2e`   = the same through necsim_simulate_host: pinned host mask in, events + labels back to the host each step.
`--impl reference` times the CPU oracle (as it stands, one core) on a bounded sample of the same workload.
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
sys.path.insert(0, ROOT)
from paper_2108_05815_b200 import inputs as I  # noqa: E402
from paper_2108_05815_b200 import dist as D    # noqa: E402

METRIC = "lineage_events_per_s"
UNIT = "events/s"
MAKERS = dict(c3t=lambda: I.c3_matrix(side=64, deme=1000), c1=I.c1_nonspatial, c2=I.c2_implicit, c3=I.c3_matrix, c4=I.c4_gaussian, c5=I.c5_stress, c6=I.c6_bigdeme, c7=I.c7_habitat_loss)
SMALL = dict(zip(("c1", "c2", "c3", "c4", "c5"), range(5)))
# Algorithmic integer instructions per executed event (minimal 32-bit instruction sequence of
# each primitive, weighted by the expected number of draws per event at mu = 2 and the measured attempts per event).
I_EVENT = dict(c3t=252, c1=230, c2=232, c3=252, c4=263, c5=272, c6=259, c7=272)   # c6: one attempt + 5 % resampling, index draw, deme32 gather; c7 = c5's landscape with eras
# The same count when the event-time search is decided by the binary32 filter (a time draw is then hash 12 +
# advance 2 + lg2 / scale 4 + accumulate and compare 5 = 23 instead of 68): what the kernels must issue at the least.
I_EVENT_FILTERED = dict(c3t=140, c1=118, c2=120, c3=140, c4=151, c5=160, c6=147, c7=160)
# issue-slot peak: 148 SMs x 4 schedulers x 32 lanes x 1 instr/clk x sm_max_mhz (B300_MICROARCH "Pipe rates")
def alu_peak(sm_count, sm_mhz):
    return sm_count * 4 * 32 * sm_mhz * 1e6


def profile_traffic(kernel, name, sampler):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch of the dominant kernel, read from the committed ncu summary
    (profiles/r2_ncu_<kernel>_<config>.md, line `traffic_bytes_per_launch=N`); None when there is no capture for this case."""
    if sampler != "exp":
        return None, None
    f = os.path.join(ROOT, "profiles", "r2_ncu_%s_%s.md" % (kernel, name))
    if not os.path.exists(f):
        return None, None
    for line in open(f):
        if line.startswith("traffic_bytes_per_launch="):
            return int(line.split("=")[1].split()[0]), os.path.relpath(f, ROOT)
    return None, None


def make_cfg(name, small):
    if name == "c6":                                     # SURVEY NEXT-4 shape; --small: demes of ~360
        return I.c6_bigdeme(deme_mean=360, sample=0.05) if small else I.c6_bigdeme()
    if name == "c3t":                                    # C3's shape with demes of 1000: 4.1e6 lineages on the 128 MiB alias table (throughput probe)
        return I.c3_matrix(side=13, deme=50) if small else I.c3_matrix(side=64, deme=1000)
    if name == "c7":                                     # temporally varying habitat
        return I.c7_habitat_loss(side=128, blur_radius=4.0, nu=1e-3, sample=0.3, switch_k=40) if small else I.c7_habitat_loss()
    return I.small_configs()[SMALL[name]] if small else MAKERS[name]()


def cpu_sample(cfg, name, budget_events=30_000_000):
    """Bounded sample of the workload for the oracle: a thinned sample mask and a per-lineage step cap."""
    n_ind = I.n_individuals(cfg)
    mask = np.ones(n_ind, np.uint8) if cfg["mask"] is None else np.asarray(cfg["mask"], np.uint8).copy()
    rng = np.random.Generator(np.random.PCG64(12345))
    n_lin, max_steps = 4000, 20_000
    idx = np.flatnonzero(mask)
    if len(idx) > n_lin:
        keep = rng.choice(idx, n_lin, replace=False)
        mask = np.zeros(n_ind, np.uint8); mask[keep] = 1
    desc = "%d of %d sampled lineages of %s, dedup on, at most %d events each" % (int(mask.sum()), len(idx), name, max_steps)
    return mask, max_steps, desc


def run_oracle_sample(cfg, name):
    from oracle import oracle as O            # cpu_baseline / --impl reference: the only bench legs that may use oracle/
    mask, max_steps, desc = cpu_sample(cfg, name)
    sc = O.Scenario(**I.scenario_kwargs(cfg))
    t0 = time.perf_counter()
    res = sc.simulate(cfg["seed"], cfg["nu"], mask, dedup=True, max_steps=max_steps)
    dt = time.perf_counter() - t0
    return res["stats"]["n_events"] / dt, dt, res["stats"]["n_events"], desc


class ClockSampler(threading.Thread):
    """Samples nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md clocks line)."""
    Q = "index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown," \
        "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, gpu_index=0):
        super().__init__(daemon=True)
        self.rows, self.proc, self.gpu_index = [], None, gpu_index

    def run(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu_index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            for line in self.proc.stdout:
                self.rows.append([c.strip() for c in line.split(",")])
        except Exception:
            pass

    def stop(self):
        if self.proc:
            self.proc.terminate()
        sm = [float(r[1]) for r in self.rows if len(r) >= 9 and r[1].replace(".", "").isdigit()]
        mx = [float(r[2]) for r in self.rows if len(r) >= 9 and r[2].replace(".", "").isdigit()]
        reasons = set()
        for r in self.rows:
            if len(r) >= 9:
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=max(mx) if mx else None, reasons=sorted(reasons), samples=len(sm))


def unique_events(cfg, args):
    """Distinct events (loc, k, j) of the workload, counted by the oracle's full-size run (tests/golden/, written by
    tests/golden/gen_golden.py from oracle/ only); raw events / this = redundant work left by the lossy dedup cache."""
    f = os.path.join(ROOT, "tests", "golden", "full_configs_poisson.json" if args.sampler == "poisson" else "full_configs.json")
    if args.small or not os.path.exists(f):
        return None
    records = json.load(open(f))
    for extra in ("full_config_c6.json", "full_config_c7.json"):
        e = os.path.join(ROOT, "tests", "golden", extra)
        if args.sampler == "exp" and os.path.exists(e):
            records += json.load(open(e))
    for g in records:
        if g["name"] == cfg["name"]:
            return g["unique_events"]
    return None


def reference_arm(args, cfg, name):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    for _ in range(args.warmup):
        pass                                   # the oracle has no warm-up state; W is accepted and ignored
    vals, secs, desc, ev = [], [], "", 0
    for _ in range(max(1, min(args.steps, 3))):
        v, dt, ev, desc = run_oracle_sample(cfg, name)
        vals.append(v); secs.append(dt)
    v = float(np.mean(vals))
    print(json.dumps({"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": len(vals), "warmup": args.warmup,
                      "ms_per_step": 1e3 * float(np.mean(secs)), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                      "dtype": "int64", "data": "synthetic", "config": {"workload": cfg["name"], "event_time_sampler": args.sampler, "sample": desc},
                      "cpu_baseline": {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc},
                      "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


def probe_arm(args, cfg, name, sc, ns, torch, d_mask, n_s):
    """Micro-workloads for profiling (one kernel launch of interest each)."""
    if args.probe == "mode_t":
        n_ev = args.probe_events or 200
        p = ns.make_params(dedup=False, max_steps=n_ev, tail_threshold=1)
        for _ in range(1 + max(args.steps, 1)):
            r = sc.simulate_raw(cfg["seed"], cfg["nu"], d_mask, n_s, p)
        v = r.n_events_raw / (r.ms_simulate * 1e-3)
        print(json.dumps({"probe": "mode_t", "workload": cfg["name"], "event_time_sampler": args.sampler, "lineages": int(r.n_lineages), "events_per_lineage": n_ev,
                          "ms": r.ms_simulate, "events": int(r.n_events_raw), "events_per_s": v, "roofline_frac": v * I_EVENT[name] / alu_peak(148, 1965.0)}))
    else:
        n_ev, n_lin = args.probe_events or 20000, 148
        rng = np.random.Generator(np.random.PCG64(5))
        mask = np.zeros(sc.n_individuals, np.uint8); mask[rng.choice(sc.n_individuals, n_lin, replace=False)] = 1
        dm = torch.from_numpy(mask).cuda()
        out = {"probe": "tail_latency", "workload": cfg["name"], "event_time_sampler": args.sampler, "lineages": n_lin, "events_per_lineage": n_ev}
        for dedup in (True, False):
            p = ns.make_params(tail_threshold=10**9, max_steps=n_ev, dedup=dedup, block_threads=32)
            for _ in range(1 + max(args.steps, 1)):
                r = sc.simulate_raw(cfg["seed"], 0.0, dm, n_lin, p)
            out["dedup_on" if dedup else "dedup_off"] = {"ms": r.ms_simulate_tail, "us_per_sequential_event": r.ms_simulate_tail * 1e3 / n_ev,
                                                          "exact_rounds_per_event": int(r.n_tail_rounds_exact) / max(int(r.n_events_tail), 1)}
        print(json.dumps(out))


def partitioned_arm(args, cfg, name, sc, ns, torch, dist, world, rank, local, flush, params):
    """The isolated-partitions path: rank r simulates its contiguous share of the sample with no communication,
    then one all-gather of the species tables and necsim_merge_species on every rank. value = distinct events of the WHOLE sample per
    second of the slowest rank (strong scaling); duplication = events executed by all ranks / distinct events (the paper's
    duplication factor, L1469)."""
    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def step():
        flush.fill_(1)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        out = D.simulate_partitioned(sc, cfg["seed"], cfg["nu"], cfg["mask"], rank=rank, world=world, params=params)
        e1.record(); e1.synchronize()
        return out, e0.elapsed_time(e1)

    for _ in range(args.warmup):
        step()
    sampler = ClockSampler(local)
    sampler.start()
    barrier()
    ms, ms_merge, ev, launches, out = 0.0, 0.0, 0, 0, None
    for _ in range(args.steps):
        out, dt = step()
        ms += dt; ms_merge += out["ms_merge"]
        if out["local"] is not None:
            ev += out["local"].n_events_raw; launches += out["local"].n_kernel_launches + 57     # + the merge's kernels (18 radix passes x 3, unpack, flag, write)
    barrier()
    clocks = sampler.stop()
    (ms, ms_merge), (ev_all,) = D.aggregate([ms, ms_merge], [float(ev)], device="cuda")
    if rank == 0:
        K = args.steps
        uniq = unique_events(cfg, args)
        value = (uniq * K if uniq else ev_all) / (ms * 1e-3)
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": args.warmup, "ms_per_step": ms / K,
                "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "int64", "data": "synthetic",
                "value_kind": "distinct events of the whole sample / device time of the slowest rank" if uniq else "raw executed events of all ranks / device time",
                "config": {"workload": cfg["name"], "event_time_sampler": args.sampler, "nu": cfg["nu"], "mode": "MODE-S, isolated partitions + merge",
                           "l2": "256 MiB flush write between steps", "parallelism": "partitions x%d" % world},
                "clocks": clocks, "gpu_launches": int(launches),
                "richness": int(out["richness"]), "raw_events_all_ranks_per_step": ev_all / K,
                "duplication_factor": (ev_all / K) / uniq if uniq else None,
                "merge": {"ms_per_step": ms_merge / K, "what": "all-gather of the species tables (32 B per species) + necsim_merge_species + label translation"},
                "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": int(0 if cfg["mask"] is None else len(cfg["mask"])), "d2h_bytes_per_step": 0,
                        "note": "the partition mask is built on the host and copied in inside the timed region; results stay on the device"}}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="c5", choices=sorted(MAKERS))
    ap.add_argument("--small", action="store_true", help="the reduced config of the same kind (for testing the harness)")
    ap.add_argument("--sampler", default="exp", choices=["exp", "poisson"],
                    help="event-time sampler of the scenario (DESIGN.md 2.4 / 2.7): same law, different realisation")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--probe", default=None, choices=["mode_t", "tail_latency"],
                    help="run ONE micro-workload instead of the bench step and print a small JSON line (the ncu captures of profiles/ use "
                         "these): mode_t = the saturated launch alone (dedup off, --probe-events events per lineage, per-lane kernel); "
                         "tail_latency = 148 lineages, --probe-events events each, one lineage per warp on its own SM: microseconds per sequential event")
    ap.add_argument("--probe-events", type=int, default=0, help="events per lineage of a --probe run (default 200 / 20000)")
    ap.add_argument("--mode", default="replicas", choices=["replicas", "partitioned"],
                    help="N > 1 (and N = 1): replicas = every rank an independent replicate (weak scaling, the default); partitioned = the "
                         "sample split over the ranks as isolated partitions, ONE all-gather of the species tables and a device-side merge "
                         "(PAPER.md L1082-1086; DESIGN.md section 8) -- strong scaling of one simulation")
    ap.add_argument("--event-stream", type=int, default=0, metavar="LOG2_CAP",
                    help="also time the path with the full event stream recorded (SURVEY NEXT-3; DESIGN.md 6.4): the stream holds up to "
                         "2^LOG2_CAP distinct events, the per-epoch ring 2^min(LOG2_CAP, 28) records")
    args = ap.parse_args()
    name = args.config
    cfg = make_cfg(name, args.small)
    cfg["sampler"] = 1 if args.sampler == "poisson" else 0
    if args.impl == "reference":
        return reference_arm(args, cfg, name)

    import torch
    import torch.distributed as dist
    from paper_2108_05815_b200 import necsim as ns
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    # weak scaling: every rank runs the same landscape with its own seed (independent replicate simulations,
    # the paper's repeated-runs use, L1240-1246); no data-path collective.
    seed = D.replica_seed(cfg["seed"], rank)
    sc = ns.Scenario(**I.scenario_kwargs(cfg))
    n_ind, n_s = sc.n_individuals, I.n_sampled(cfg)
    h_mask = None
    d_mask = None
    if cfg["mask"] is not None:
        h_mask_t = torch.from_numpy(np.ascontiguousarray(cfg["mask"], dtype=np.uint8)).pin_memory()
        h_mask = h_mask_t.numpy()
        d_mask = h_mask_t.cuda()
    h_events = torch.empty(n_s * 32, dtype=torch.uint8).pin_memory().numpy().view(ns.EVENT_DTYPE)
    h_labels = torch.empty(n_s, dtype=torch.int32).pin_memory().numpy().view(np.uint32)
    params = ns.make_params()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")      # > 126 MB L2
    if args.probe:
        return probe_arm(args, cfg, name, sc, ns, torch, d_mask, n_s)
    if args.mode == "partitioned":
        return partitioned_arm(args, cfg, name, sc, ns, torch, dist, world, rank, local, flush, params)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def step_device():
        flush.fill_(1)
        torch.cuda.synchronize()
        return sc.simulate_raw(seed, cfg["nu"], d_mask, n_s, params)

    def step_host():
        flush.fill_(1)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        r = sc.simulate_host_raw(seed, cfg["nu"], h_mask, n_s, params, h_events, h_labels)
        return r, time.perf_counter() - t0

    for _ in range(args.warmup):
        step_device()
    sampler = ClockSampler(local)
    sampler.start()
    barrier()
    ms, ev, sim_ms, tail_ms, ev_tail, launches, epochs, res = 0.0, 0, 0.0, 0.0, 0, 0, 0, None
    for _ in range(args.steps):
        res = step_device()
        ms += res.ms_total; sim_ms += res.ms_simulate; ev += res.n_events_raw; launches += res.n_kernel_launches; epochs += res.n_epochs
        tail_ms += res.ms_simulate_tail; ev_tail += res.n_events_tail
    barrier()
    clocks = sampler.stop()
    # end to end: host buffers in, host buffers out, copies inside the timed region
    step_host()
    e2e_s, e2e_ev, res_h = 0.0, 0, None
    barrier()
    for _ in range(args.steps):
        res_h, dt = step_host()
        e2e_s += dt; e2e_ev += res_h.n_events_raw
    barrier()
    (ms, e2e_ms, sim_ms), (ev_all, e2e_ev_all) = D.aggregate([ms, e2e_s * 1e3, sim_ms], [float(ev), float(e2e_ev)], device="cuda")
    if rank == 0:
        K = args.steps
        raw_value = D.throughput(ev_all, ms)
        uniq = unique_events(cfg, args) if world == 1 else None      # the stored count belongs to the config's own seed (rank 0)
        value, value_kind = (uniq * K / (ms * 1e-3), "distinct events (oracle's count of the workload) / device time") if uniq else \
                            (raw_value, "raw executed events / device time (no stored count of distinct events for this case)")
        prop = torch.cuda.get_device_properties(local)
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))) if os.path.exists(os.path.join(ROOT, "MEASURED_PEAKS.json")) else {}
        sm_max = float(peaks.get("sm_max_mhz", clocks.get("sm_max_mhz") or 1965.0))
        peak = alu_peak(prop.multi_processor_count, sm_max)
        # dominant kernel of a step = the one with the larger summed device time (CUDA events around every launch; the ncu launch
        # list profiles/r2_launches_c5.md agrees on its share): algorithmic instructions of its launches / that time
        dom_ms, dom_ev, dom_name = (tail_ms, ev_tail, "tail_kernel") if tail_ms >= sim_ms - tail_ms else (sim_ms - tail_ms, ev - ev_tail, "simulate_kernel")
        achieved = dom_ev * I_EVENT[name] / max(dom_ms * 1e-3, 1e-12)
        int_meas = {k: ns.int_peak(i, 2048)[0] for i, k in enumerate(("hash_round_mix", "imad_only", "alu_only"))}
        # the measured peak that binds for this instruction mix: the hash round (IMAD.WIDE on the FMA pipe + LOP3 on the ALU pipe,
        # about 40 % of the path's instructions are multiplies) -- below the issue-slot peak because IMAD.WIDE is not full rate
        peak_meas = int_meas["hash_round_mix"]
        traffic, traffic_src = profile_traffic(dom_name, name, args.sampler)
        # random 32-byte-sector gather peaks: the denominators for the table gathers (alias matrix, habitat, dedup cache)
        gather_meas = {"l2_32MiB_GBs": ns.gather_peak(32 << 20)[0] / 1e9, "hbm_4GiB_GBs": ns.gather_peak(4 << 30)[0] / 1e9}
        # MODE-T: the saturated workload (dedup off, every lineage advanced 200 events): where the ALU roofline is meaningful
        rt = sc.simulate_raw(seed, cfg["nu"], d_mask, n_s, ns.make_params(dedup=False, max_steps=200))
        mode_t = rt.n_events_raw / (rt.ms_simulate * 1e-3)
        sat_evs = (ev - ev_tail) / max((sim_ms - tail_ms) * 1e-3, 1e-9)
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": args.warmup, "ms_per_step": ms / K,
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int64", "data": "synthetic",
                "value_kind": value_kind, "raw_events_per_s": raw_value,
                "config": {"workload": cfg["name"], "event_time_sampler": args.sampler, "n_lineages": int(res.n_lineages), "nu": cfg["nu"], "mode": "MODE-S (dedup on, to completion)",
                           "l2": "256 MiB flush write between steps", "parallelism": "replicas x%d" % world},
                "clocks": clocks,
                "e2e": {"value": (uniq * K if uniq else e2e_ev_all) / (e2e_ms * 1e-3), "unit": UNIT, "ms_per_step": e2e_ms / K,
                        "h2d_bytes_per_step": int(0 if h_mask is None else h_mask.nbytes),
                        "d2h_bytes_per_step": int(res_h.richness * 32 + res_h.n_lineages * 4)},
                "gpu_launches": int(launches),
                "individuals_per_s": world * res.n_lineages / (ms / K * 1e-3),
                "richness": int(res.richness), "epochs_per_step": epochs / K, "raw_events_per_step": ev / K,
                "unique_events": uniq, "redundancy": (ev / K) / uniq if uniq else None,
                "phases": {"saturated": {"events_per_s": sat_evs, "ms_per_step": (sim_ms - tail_ms) / K,
                                         "events_per_step": (ev - ev_tail) / K, "kernel": "simulate_kernel (one lineage per lane)",
                                         "roofline_frac": sat_evs * I_EVENT[name] / peak},
                           "tail": {"events_per_s": ev_tail / max(tail_ms * 1e-3, 1e-9), "ms_per_step": tail_ms / K, "events_per_step": ev_tail / K,
                                    "exact_rounds_per_event": int(res.n_tail_rounds_exact) / max(int(res.n_events_tail), 1),
                                    "kernel": "tail_kernel (one lineage per warp; bound by event latency x chain length, DESIGN.md 6.3)"}},
                "roofline": {"bound": "alu", "kernel": dom_name + " (all its launches of the timed steps)", "achieved": achieved / 1e12, "peak": peak / 1e12,
                             "unit": "Tinstr/s", "frac": achieved / peak,
                             "peak_measured": peak_meas / 1e12, "frac_measured": achieved / peak_meas,
                             "binding_pipe": "FMA pipe for the multiplies (IMAD.WIDE.U32, not full rate) with the ALU pipe beside it: the measured "
                                             "hash-round mix is the ceiling of this instruction mix; `peak` is the issue-slot bound above it",
                             "traffic": traffic, "traffic_source": traffic_src,
                             "instr_per_event": I_EVENT[name], "instr_per_event_filtered": I_EVENT_FILTERED[name],
                             "frac_filtered_count": dom_ev * I_EVENT_FILTERED[name] / max(dom_ms * 1e-3, 1e-12) / peak,
                             "instr_per_event_check": "profiles/r2_sass_mix_simulate_kernel_c5.md (executed instructions per event by pipe, ncu source counters)",
                             "note": "latency-bound by construction: one lineage per warp walks a serial chain of ~ln(S)/nu events (DESIGN.md 6.3)",
                             "peak_source": "derived: SMs x 4 schedulers x 32 lanes x sm_max_mhz (DESIGN.md section 6); peak_measured: necsim_debug_int_peak in this run",
                             "measured_int_peaks_Tinstr_s": {k: v / 1e12 for k, v in int_meas.items()},
                             "measured_random_sector_gather_peaks": gather_meas},
                "mode_t": {"value": mode_t, "unit": UNIT, "what": "dedup off, 200 events per lineage, saturated machine",
                           "roofline_frac": mode_t * I_EVENT[name] / peak, "frac_measured": mode_t * I_EVENT[name] / peak_meas,
                           "frac_filtered_count": mode_t * I_EVENT_FILTERED[name] / peak,
                           "ncu": "profiles/r2_ncu_simulate_kernel_c5_modeT.md"}}
        if args.event_stream:
            # the same step with every executed event recorded, sorted by time and deduplicated per epoch on the device
            pr = ns.make_params(record_events=True, event_ring_capacity=1 << min(args.event_stream, 28), event_stream_capacity=1 << args.event_stream)
            rs, s_ms = None, 0.0
            for i in range(1 + K):
                flush.fill_(1)
                torch.cuda.synchronize()
                rs = sc.simulate_raw(seed, cfg["nu"], d_mask, n_s, pr)
                s_ms += rs.ms_total if i else 0.0
            line["event_stream"] = {"ms_per_step": s_ms / K, "distinct_events": int(rs.n_stream_events), "epochs": int(rs.n_epochs),
                                    "distinct_events_per_s": int(rs.n_stream_events) * K / (s_ms * 1e-3), "launches_per_step": int(rs.n_kernel_launches)}
        if not args.no_cpu_baseline and world == 1:
            v, dt, n_ev, desc = run_oracle_sample(cfg, name)
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc, "seconds": dt}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
