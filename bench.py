#!/usr/bin/env python
"""bench.py — accepted hops/s and proposals/s of the PR-KMC hot path (BASELINE.json metric).

A "step" is one cg_run(hops_per_step) of the whole hot path (propose, select, apply, update)
on the headline workload, config 5 of BASELINE.json (L=512, T=0.05, E=0.01, M=65536, seed 8).
N GPUs run N independent replicas (seeds 8, 9, ...),
no data-path collective; value = hops of all replicas / max-over-devices device time.  Under torchrun
(WORLD_SIZE set) every rank drives its own GPU; started plainly with --gpus N, ONE process drives N
devices (a replica needs nothing from the others, so no process group is needed).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
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

import workloads  # noqa: E402

METRIC, UNIT = "accepted_hops_per_s", "hops/s"


def rank_world():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def reduce_over_ranks(ms, units, dist=None):
    """(device ms of this rank, units it processed) -> (max ms over ranks, sum of units)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(ms), int(units)
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(ms)], dtype=torch.float64, device=dev)
    u = torch.tensor([int(units)], dtype=torch.int64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), int(u.item())


def replica_config(rank):
    """Rank r runs config 5 with seed 8 + r: independent samples, the paper's own
    recommendation for using more hardware."""
    cfg = dict(workloads.CONFIGS[workloads.HEADLINE][0])
    cfg["seed"] += rank
    return cfg


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=lambda: self.rows.extend(self.proc.stdout), daemon=True)
            self.t.start()
        except OSError:
            self.proc = None
        return self

    def __exit__(self, *a):
        if self.proc:
            time.sleep(0.15)
            self.proc.terminate()
            self.t.join(timeout=2)

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            reasons.update(n for n, v in zip(names, f[3:7]) if v.lower() == "active")
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


class OneCore:
    """The serial oracle pinned to one core for its timed loop (the paper's baseline is
    "a fair serial single CPU core").  Its one-time O(N^2) set-up may use every core."""

    def __enter__(self):
        self.old = None
        try:
            self.old = os.sched_getaffinity(0)
            os.sched_setaffinity(0, {sorted(self.old)[-1]})
        except (AttributeError, OSError):
            self.old = None
        return self

    def __exit__(self, *a):
        if self.old:
            os.sched_setaffinity(0, self.old)


def time_oracle(cfg, seconds, chunk):
    """The oracle as it stands, one core, on a bounded sample of the workload."""
    from oracle import cgo
    kw = workloads.init_args(cfg)
    t0 = time.perf_counter()
    o = cgo.Oracle(hop_log=False, **kw)
    t_init = time.perf_counter() - t0
    with OneCore():
        hops, t0 = 0, time.perf_counter()
        while True:
            o.run(chunk)
            hops += chunk
            el = time.perf_counter() - t0
            if el >= seconds:
                break
    c = o.counters()
    return {"hops": hops, "seconds": el, "init_seconds": t_init, "attempts": c["attempts"],
            "update_seconds": o.update_seconds(), "near_ties": o.near_ties()}


def run_reference(args):
    """--impl reference: the CPU oracle (serial mixed algorithm) on host cores."""
    rank, world = rank_world()
    if rank != 0:
        return
    from oracle import cgo
    cfg = replica_config(0)
    kw = workloads.init_args(cfg)
    hops_per_step = args.ref_hops_per_step
    o = cgo.Oracle(hop_log=False, **kw)
    with OneCore():
        for _ in range(args.warmup):
            o.run(hops_per_step)
        a0 = o.counters()["attempts"]
        t0 = time.perf_counter()
        for _ in range(args.steps):
            o.run(hops_per_step)
        el = time.perf_counter() - t0
    hops = args.steps * hops_per_step
    c = o.counters()
    value = hops / el
    sample = "%d steps x %d hops of config 5 after %d warm-up hops from the random start" % (
        args.steps, hops_per_step, args.warmup * hops_per_step)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * el / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": "cfg5_L512 (L=512, T=0.05, E=0.01, xi=1, W=1, seed=8); M only enters "
                               "the oracle's iteration bookkeeping", "hops_per_step": hops_per_step},
        "attempts_per_s": (c["attempts"] - a0) / el,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
                         "host_cores": os.cpu_count(), "pinned": "one core (sched_setaffinity)"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


CTL_BYTES = 176  # sizeof(CgCtl) in csrc/cg.cu: the control block cg_set_state / cg_get_state move


L2_PROBES = [  # the shapes that came out on top of the sweep (profiles/r2_l2_sweep.txt), re-measured live
    dict(mode="rmw", nbytes=16 << 20, ctas_per_sm=8, threads=128, vec_bytes=16),
    dict(mode="rmw", nbytes=4 << 20, ctas_per_sm=8, threads=128, vec_bytes=16),
    dict(mode="rmw", nbytes=16 << 20, ctas_per_sm=4, threads=256, vec_bytes=16),
    dict(mode="rmw", nbytes=16 << 20, ctas_per_sm=2, threads=512, vec_bytes=16),
]


def static_profile():
    """Counters that only ncu can give, from the committed capture of this kernel (profiles/r2_ncu_counters.csv:
    key,value lines; NOT re-measured here, and labelled static in the output)."""
    try:
        rows = [l.strip().split(",", 1) for l in open(os.path.join(ROOT, "profiles", "r2_ncu_counters.csv"))
                if l.strip() and not l.startswith("#")]
        d = dict(rows)
        return {"source": d["source"], "dram_bytes_per_hop": float(d["dram_bytes_per_hop"]),
                "l2_bytes_per_hop": float(d["l2_bytes_per_hop"])}
    except (OSError, ValueError, KeyError):
        return None


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    rank, world = rank_world()
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    # torchrun: one rank per GPU.  Plain start: this process drives --gpus devices itself.
    if world > 1:
        devices = [local]
        torch.cuda.set_device(local)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    else:
        devices = list(range(min(max(args.gpus, 1), torch.cuda.device_count())))
        torch.cuda.set_device(devices[0])
    import paper_1407_5026_b200 as pkg

    n_rep = len(devices) if world == 1 else world
    H, K, W = args.hops_per_step, args.steps, args.warmup
    reps = []
    for k, dev in enumerate(devices):
        torch.cuda.set_device(dev)
        sms = torch.cuda.get_device_properties(dev).multi_processor_count
        cfg = replica_config(rank + k)
        kw = workloads.init_args(cfg, sms * 2048)
        warm_kw = dict(kw, seed=kw["seed"] + 1000)
        reps.append(dict(
            dev=dev, cfg=cfg, kw=kw, warm_kw=warm_kw,
            warm=pkg.CoulombGlass(device=dev, **warm_kw),     # warm-up replica: same shape, other seed
            g=pkg.CoulombGlass(device=dev, **kw),             # the timed workload starts at hop 0
            flush=torch.zeros(512 << 20, dtype=torch.uint8, device="cuda:%d" % dev)))   # > 126 MB L2
        if args.cluster:
            reps[-1]["warm"].set_tuning(0, args.cluster)
            reps[-1]["g"].set_tuning(0, args.cluster)
        if args.ctas or args.threads:
            reps[-1]["warm"].set_launch(args.ctas, args.threads)
            reps[-1]["g"].set_launch(args.ctas, args.threads)
    torch.cuda.set_device(devices[0])
    N = reps[0]["kw"]["L"] ** 2

    def barrier():
        for r in reps:
            torch.cuda.synchronize(r["dev"])
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(W):
        for r in reps:
            r["warm"].run(H)
    barrier()
    for r in reps:
        with torch.cuda.device(r["dev"]):
            r["ev"] = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    with ClockSampler(devices[0]) as clk:
        for k in range(K):
            for r in reps:                    # the replicas' launches are asynchronous: the devices run side by side
                with torch.cuda.device(r["dev"]):
                    r["flush"].add_(1)        # L2 flush between timed steps (not timed)
                    e0, e1 = r["ev"][k]
                    e0.record()
                    r["g"].run(H)             # ONE persistent kernel launch = one step
                    e1.record()
        barrier()
    ms_dev = [sum(e0.elapsed_time(e1) for e0, e1 in r["ev"]) for r in reps]
    ms_rank = max(ms_dev)
    ms, hops_all = reduce_over_ranks(ms_rank, K * H * len(reps), dist if world > 1 else None)
    g, warm = reps[0]["g"], reps[0]["warm"]
    c = g.counters()
    assert all(r["g"].counters()["hops"] == K * H for r in reps)

    # ---- end to end through the C ABI with pinned HOST buffers (restore -> run -> read back), every replica: the SAME
    # workload as above (a fresh sim of the same seed, hops 1..K*H), its state living in host memory between the steps
    for r in reps:
        with torch.cuda.device(r["dev"]):
            r["e"] = pkg.CoulombGlass(device=r["dev"], **r["kw"])
            if args.cluster:
                r["e"].set_tuning(0, args.cluster)
            if args.ctas or args.threads:
                r["e"].set_launch(args.ctas, args.threads)
        r["n_host"] = torch.empty(N, dtype=torch.int8).pin_memory().numpy()
        r["eps_host"] = torch.empty(N, dtype=torch.float64).pin_memory().numpy()
        with torch.cuda.device(r["dev"]):
            _, r["dP"] = r["e"].state_into(r["n_host"], r["eps_host"])
            r["wc"] = r["e"].counters()
    barrier()
    t0 = time.perf_counter()
    for _ in range(K):
        for r in reps:
            with torch.cuda.device(r["dev"]):
                r["e"].set_state(r["n_host"], r["eps_host"], r["wc"]["attempts"], r["wc"]["hops"], r["dP"])    # H2D
                r["e"].run(H)
        for r in reps:
            with torch.cuda.device(r["dev"]):
                _, r["dP"] = r["e"].state_into(r["n_host"], r["eps_host"])                               # D2H, syncs
                r["wc"] = r["e"].counters()
    barrier()
    assert all(r["wc"]["hops"] == K * H and r["wc"]["attempts"] == r["g"].counters()["attempts"] for r in reps)   # the same chain
    e2e_ms, e2e_hops = reduce_over_ranks(1e3 * (time.perf_counter() - t0), K * H * len(reps),
                                         dist if world > 1 else None)
    bitmap = 4 * ((N + 31) // 32)
    e2e = {"value": e2e_hops / (e2e_ms * 1e-3), "unit": UNIT,
           "h2d_bytes_per_step": 8 * N + bitmap + CTL_BYTES,
           "d2h_bytes_per_step": 8 * N + bitmap + 3 * CTL_BYTES,
           "what": "the same workload (fresh sim, same seed, hops 1..steps*hops_per_step): cg_set_state(host n, eps) + cg_run + "
                   "cg_get_state(host n, eps) + cg_get_counters per step and replica; wall clock"}

    if rank != 0:
        return
    sec = ms * 1e-3
    tun = g.tuning()
    out = {
        "metric": METRIC, "value": hops_all / sec, "unit": UNIT, "n_gpus": n_rep, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "cfg5_L512: L=512 N=262144 T=0.05 E=0.01 xi=1 W=1 M=65536 seed=8(+replica), "
                               "hops 1..steps*hops_per_step from the random start",
                   "hops_per_step": H, "launch": g.launch(), "tuning": tun, "replicas": n_rep,
                   "processes": world, "devices_per_process": len(devices),
                   "l2": "flushed between timed steps (512 MiB write); within a step the state is "
                         "L2-resident by construction"},
        "proposals_per_s": c["proposals_evaluated"] / (ms_dev[0] * 1e-3) if n_rep == 1 else None,
        "attempts_per_s": c["attempts"] / (ms_dev[0] * 1e-3) if n_rep == 1 else None,
        "rank0": {"attempts": c["attempts"], "iterations": c["iterations"],
                  "proposals_evaluated": c["proposals_evaluated"],
                  "mean_p": c["iterations"] / c["hops"], "acceptance": c["hops"] / c["attempts"],
                  "proposals_per_s": c["proposals_evaluated"] / (ms_dev[0] * 1e-3),
                  "us_per_hop": 1e3 * ms_dev[0] / c["hops"]},
        "gpu_launches": K * len(reps),
        "e2e": e2e,
        "clocks": clk.summary(),
    }

    # ---- roofline of the eps update (16 N algorithmic bytes per hop, L2-resident)
    probes = [dict(pr, gbs=pkg.bench_l2(pr["nbytes"], reps=1000, trials=5, mode=pr["mode"],
                                        ctas_per_sm=pr["ctas_per_sm"], threads=pr["threads"],
                                        vec_bytes=pr["vec_bytes"])) for pr in L2_PROBES]
    l2_peak = max(pr["gbs"] for pr in probes)
    achieved = 16.0 * N * c["hops"] / (ms_dev[0] * 1e-3) / 1e9
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except OSError:
        pass
    prof = static_profile()
    out["roofline"] = {
        "bound": "l2", "kernel": "cg_pr_persistent (the whole hop: propose, select, apply, update; one launch per step)",
        "achieved": achieved, "peak": l2_peak, "unit": "GB/s", "frac": achieved / l2_peak,
        "traffic": prof["dram_bytes_per_hop"] * c["hops"] / K if prof else None,
        "traffic_static": {"static": True, "source": prof["source"], "dram_bytes_per_hop": prof["dram_bytes_per_hop"],
                           "l2_bytes_per_hop": prof["l2_bytes_per_hop"]} if prof else None,
        "peak_source": "measured live: cg_bench_l2, read-modify-write through L2 (ld.cg/st.cg), 1000 passes per launch, best of "
                       "5, maximum over the shapes that won the sweep of profiles/r2_l2_sweep.txt (MEASURED_PEAKS.json has "
                       "no L2 figure; read-only probes reach more, write-only less: see that file)",
        "peak_probes": probes,
        "algorithmic_bytes_per_hop": 16 * N,
        "hbm_peak_gbs": peaks.get("hbm_gbs"), "frac_of_hbm_peak": achieved / peaks["hbm_gbs"] if peaks.get("hbm_gbs") else None,
    }
    # the paper's split W_R / W_U from the kernel that runs: timed build, the next hops of the warm replica
    if warm.launch()["threads"] == 544:
        warm.set_phase_timers(True)
        warm.phase_cycles(reset=True)
        it0 = warm.counters()["iterations"]
        warm.run(20000)
        pc = warm.phase_cycles()
        xc = warm.exchange_cycles()
        warm.set_phase_timers(False)
        n_it = warm.counters()["iterations"] - it0
        w = max(pc["warps"], 1)
        out["in_loop_cycles_per_iteration"] = {
            "total": pc["total"] / n_it, "propose": pc["propose"] / w / n_it, "update_W_U": pc["update"] / w / n_it,
            "wait": pc["wait"] / w / n_it, "what": "CTA 0, mean over its worker warps; timed build of the same kernel, 20000 hops",
            "exchange_warp": {k: xc[k] / max(xc["warps"], 1) / n_it for k in ("recycle", "gate", "own_workers", "scan", "publish")},
            "exchange_warp_what": "mean over the exchange warps of all CTAs (cg_get_exchange_cycles)"}
    # the update kernel alone on scripted hops (forward log + its reversal = back to the start state)
    warm_kw = reps[0]["warm_kw"]
    u = pkg.CoulombGlass(device=devices[0], hop_log=2000, **warm_kw)
    u.run(2000)
    _, hi, hj = u.hops()
    v = pkg.CoulombGlass(device=devices[0], **warm_kw)
    si = np.concatenate([hi, hj[::-1]]); sj = np.concatenate([hj, hi[::-1]])
    best = min(v.apply_hops(si, sj) for _ in range(5))
    upd = 16.0 * N * si.size / (best * 1e-3) / 1e9
    out["roofline_update_kernel"] = {
        "bound": "l2", "kernel": "cg_update_scripted: STAND-ALONE DIAGNOSTIC kernel (step a6 alone, %d scripted hops per launch, eps "
                                 "register-resident across hops; algorithmic bytes, not measured traffic)" % si.size,
        "achieved": upd, "peak": l2_peak, "unit": "GB/s", "frac": upd / l2_peak, "us_per_hop": 1e3 * best / si.size}

    if n_rep == 1 and not args.no_cpu_baseline:
        r = time_oracle(reps[0]["cfg"], args.cpu_seconds, 250)
        out["cpu_baseline"] = {
            "value": r["hops"] / r["seconds"], "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": "first %d hops of config 5 from the random start (%.1f s; init %.1f s not timed), the plain oracle as it "
                      "stands, pinned to one core" % (r["hops"], r["seconds"], r["init_seconds"]),
            "attempts_per_s": r["attempts"] / r["seconds"], "host_cores": os.cpu_count(),
            "W_U_us_per_hop": 1e6 * r["update_seconds"] / r["hops"],
            "update_gbs": 16.0 * N * r["hops"] / r["update_seconds"] / 1e9, "near_ties": r["near_ties"]}
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--hops-per-step", type=int, default=100_000)
    ap.add_argument("--ref-hops-per-step", type=int, default=2_000)
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--ctas", type=int, default=0)
    ap.add_argument("--threads", type=int, default=0)
    ap.add_argument("--cluster", type=int, default=0,
                    help="thread-block cluster size (0: automatic; 1 for runs under ncu, which cannot replay cooperative cluster launches)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
