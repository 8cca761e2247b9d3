"""Per-config throughput report and replica packing (§8f-2), through the Python binding.

    python -m paper_1407_5026_b200.report --configs [--hops 200000] [--warm 2000]
    python -m paper_1407_5026_b200.report --replicas [--hops 100000]
    python -m paper_1407_5026_b200.report --observables [--hops 200000]
    python -m paper_1407_5026_b200.report --l2            # sweep of the L2 roofline probe (cg_bench_l2)
    python -m paper_1407_5026_b200.report --update        # step a6 alone: gather kernel against bulk-copy staged kernel
    python -m paper_1407_5026_b200.report --tuning        # snapshot interval H and cluster size at configs 3 and 5
    python -m paper_1407_5026_b200.report --cubic         # 3D cubic lattices (64^3 = the headline footprint)
    python -m paper_1407_5026_b200.report --soak          # 34 M hops: different shapes / kernels give the same chain
    python -m paper_1407_5026_b200.report --one cfg5_L512 [--hops 20000]    # one config, two launches (ncu target)
    python -m paper_1407_5026_b200.report --l2-one        # the best L2 probe shape alone (ncu target)

--configs: every workload of BASELINE.json (workloads.CONFIGS), a bounded prefix of its chain, one line each:
accepted hops/s, window proposals evaluated/s (M per PR iteration), attempts consumed/s
(m = (p-1)M + q per hop), mean p and mean q (0-based label of the executed proposal),
acceptance A = hops/attempts over the run and over its last 10 %, the paper's split of the time per hop
 measured inside the persistent kernel that runs (`cg_get_phase_cycles`, timed build of the same
kernel, a second pass over the same hops): per worker warp of CTA 0 and per iteration, cycles spent testing
proposals (propose), in its share of the eps update (update = W_U in the loop) and waiting for the outcome
(wait); W_R = propose + wait; next to it the update alone (`cg_apply_hops`) with its algorithmic GB/s (16 N bytes
per hop), and the drift of the incremental eps against a full-sum recomputation.

--replicas: independent sims side by side on one GPU: packed into ONE persistent launch (`cg_run_many`), and
as separate persistent kernels on separate CUDA streams.

--observables: the read-only device passes of include/cg.h "Observables" on a chain with its hop log: the
deterministic clock t = attempts/Gamma next to the stochastic one of step 3c ("does not produce any
appreciable difference"), sigma0 = dP/(N E t), the density of states around the
Coulomb gap, the length of the P(t) series, and what each call costs (wall time of the whole call,
device-to-host copy included).

Needs a CUDA device; nothing here computes on the host.
"""
import argparse
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np      # noqa: E402
import torch            # noqa: E402

import workloads        # noqa: E402
from . import binding   # noqa: E402


def _timed(fn):
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1)


def update_alone_us(kw, n_script=1000):
    """W_U: microseconds per hop of step a6 alone at this lattice, on hops of its own chain."""
    u = binding.CoulombGlass(hop_log=n_script, **kw)
    u.run(n_script)
    _, hi, hj = u.hops()
    v = binding.CoulombGlass(**kw)
    si = np.concatenate([hi, hj[::-1]])
    sj = np.concatenate([hj, hi[::-1]])
    best = min(v.apply_hops(si, sj) for _ in range(3))
    return 1e3 * best / si.size


def report_configs(hops, warm):
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    print("# %s, %d SMs; %d warm-up hops, then min(config's hops, %d) timed in 10 chunks" % (
        torch.cuda.get_device_name(0), sms, warm, hops))
    for name, cfgs in workloads.CONFIGS.items():
        for cfg in cfgs:
            kw = workloads.init_args(cfg, sms * 2048)
            N, M = kw["L"] ** 2, kw["M"]
            g = binding.CoulombGlass(**kw)
            H = min(cfg["hops"], hops)
            chunk = H // 10
            g.run(warm)
            torch.cuda.synchronize()
            c0 = g.counters()
            ms, cs = 0.0, [c0]
            for _ in range(10):
                ms += _timed(lambda: g.run(chunk))
                cs.append(g.counters())
            c, c9 = cs[-1], cs[-2]
            Hd = c["hops"] - c0["hops"]
            it = c["iterations"] - c0["iterations"]
            at = c["attempts"] - c0["attempts"]
            mean_q = (at - (it - Hd) * M) / Hd - 1.0
            A_all = Hd / at
            A_last = (c["hops"] - c9["hops"]) / (c["attempts"] - c9["attempts"])
            us_hop = 1e3 * ms / Hd
            w_u = update_alone_us(kw)
            ln = g.launch()
            # the paper's split, from the timed build of the same kernel on the next `chunk` hops
            split = ""
            if ln["threads"] == 544 and g.labels_per_thread() <= 1:
                g.set_phase_timers(True)
                g.phase_cycles(reset=True)
                it0 = g.counters()["iterations"]
                g.run(chunk)
                pc = g.phase_cycles()
                xc = g.exchange_cycles()
                g.set_phase_timers(False)
                n_it = g.counters()["iterations"] - it0
                w = max(pc["warps"], 1)
                xw = max(xc["warps"], 1)
                split = ("  in-loop cycles/iteration: total %.0f = propose %.0f + update %.0f + wait %.0f; exchange warps (mean of "
                         "%d CTAs): recycle %.0f gate %.0f own workers %.0f scan %.0f publish %.0f" % (
                             pc["total"] / n_it, pc["propose"] / w / n_it, pc["update"] / w / n_it, pc["wait"] / w / n_it, xw,
                             xc["recycle"] / xw / n_it, xc["gate"] / xw / n_it, xc["own_workers"] / xw / n_it,
                             xc["scan"] / xw / n_it, xc["publish"] / xw / n_it))
            print("%-9s T=%-5g M=%-6d %3d CTAs x %d, H=%d, %d label(s)/thread: %7.0f hops/s  %.2e proposals/s  %.2e attempts/s  "
                  "p=%.3f q=%8.1f  A=%.2e (last 10%%: %.2e)  %5.3f us/hop%s  "
                  "update alone %.3f us/hop = %6.0f GB/s  drift %.1e" % (
                      name, kw["T"], M, ln["n_ctas"], ln["threads"], g.tuning()["snapshot_interval"], g.labels_per_thread(),
                      Hd / ms * 1e3, M * it / ms * 1e3,
                      at / ms * 1e3, it / Hd, mean_q, A_all, A_last, us_hop, split, w_u,
                      16.0 * N / w_u / 1e3, g.recompute_eps()))
            sys.stdout.flush()


def report_3d(hops):
    """The cubic lattice at the headline footprint N = 64^3 = 2^18 and at 32^3."""
    print("# %s: 3D cubic lattices, %d hops after 2000 warm-up hops" % (torch.cuda.get_device_name(0), hops))
    for kw in (dict(L=64, T=0.05, E=0.01, seed=64, M=65536), dict(L=32, T=0.05, E=0.01, seed=32, M=8192),
               dict(L=16, T=0.1, E=0.01, seed=16, M=1024), dict(L=8, T=0.1, E=0.0, seed=8, M=256)):
        g = binding.CoulombGlass(dim=3, **kw)
        g.run(2000)
        torch.cuda.synchronize()
        c0 = g.counters()
        ms = _timed(lambda: g.run(hops))
        c = g.counters()
        ln = g.launch()
        print("3D L=%-3d N=%-7d T=%-5g M=%-6d %3d CTAs x %4d (%s kernel): %7.0f hops/s  %.3f us/hop  A=%.2e  q=%.1f  drift %.1e" % (
            kw["L"], g.N, kw["T"], kw["M"], ln["n_ctas"], ln["threads"], g.kernel(), hops / ms * 1e3, ms * 1e3 / hops,
            hops / (c["attempts"] - c0["attempts"]), (c["attempts"] - c0["attempts"]) / hops - 1.0, g.recompute_eps()))
        sys.stdout.flush()


def report_soak():
    """Long chains of every config in two or three different launch shapes / kernels / tunings: they must be the SAME
    chain (final occupations, eps bit for bit, clock, dP, attempts, the whole hop log) - a soak for rare races."""
    import time

    def run(kw, hops, shape=None, tuning=None, chunks=1):
        g = binding.CoulombGlass(hop_log=hops, **kw)
        if tuning:
            g.set_tuning(*tuning)
        if shape:
            g.set_launch(*shape)
        t0 = time.time()
        for _ in range(chunks):
            g.run(hops // chunks)
        if hops % chunks:
            g.run(hops % chunks)
        torch.cuda.synchronize()
        dt = time.time() - t0
        n, eps, t, dP = g.state()
        return dict(n=n, eps=eps, t=t, dP=dP, c=g.counters(), h=g.hops(0, hops), dt=dt, launch=g.launch(), kernel=g.kernel(),
                    tun=g.tuning(), drift=g.recompute_eps())

    def same(a, b):
        return (np.array_equal(a["n"], b["n"]) and np.array_equal(a["eps"], b["eps"]) and a["t"] == b["t"] and a["dP"] == b["dP"]
                and a["c"]["attempts"] == b["c"]["attempts"] and a["c"]["hops"] == b["c"]["hops"]
                and all(np.array_equal(x, y) for x, y in zip(a["h"], b["h"])))

    sms = torch.cuda.get_device_properties(0).multi_processor_count
    cases = [
        ("cfg5_L512", 0, 4_000_000, [dict(), dict(shape=(sms, 544), tuning=(2, 1)), dict(shape=(100, 608), tuning=(4, 2), chunks=7)]),
        ("cfg3_L128", 3, 6_000_000, [dict(), dict(shape=(19, 544), tuning=(1, 1)), dict(shape=(48, 544), tuning=(8, 16), chunks=5)]),
        ("cfg4_L256", 3, 400_000, [dict(), dict(shape=(sms, 544), tuning=(1, 1)), dict(shape=(74, 544), tuning=(4, 2))]),
        ("cfg4_L256", 0, 3_000_000, [dict(), dict(shape=(37, 1024), tuning=(2, 1))]),
        ("cfg2_L64", 0, 6_000_000, [dict(), dict(shape=(1, 1024)), dict(shape=(5, 544), tuning=(8, 1), chunks=3)]),
        ("cfg1_L16", 0, 10_000_000, [dict(), dict(shape=(1, 544), tuning=(2, 1)), dict(shape=(3, 256), chunks=4)]),
    ]
    # the single-CTA kernels (512 and 1024 threads, 2/4/8 labels per thread) against the dataflow kernel, 2D and 3D, hot and cold
    extra = [
        ("L=32 M=1024", dict(L=32, T=0.08, E=0.01, seed=5, M=1024), 4_000_000, [dict(), dict(shape=(3, 544), tuning=(2, 1))]),
        ("L=64 M=2000", dict(L=64, T=0.05, E=0.01, seed=2, M=2000), 2_000_000, [dict(shape=(1, 512)), dict(shape=(5, 544))]),
        ("L=128 M=4096", dict(L=128, T=0.05, E=0.01, seed=5, M=4096), 1_000_000, [dict(shape=(1, 512)), dict(), dict(shape=(19, 544), tuning=(4, 1))]),
        ("3D L=8 M=256", dict(L=8, dim=3, T=0.1, E=0.01, seed=8, M=256), 4_000_000, [dict(), dict(shape=(2, 544))]),
        ("3D L=16 M=3000", dict(L=16, dim=3, T=0.05, E=0.01, seed=13, M=3000), 1_000_000, [dict(shape=(1, 512)), dict()]),
        ("cold L=16 M=4096", dict(L=16, T=0.01, E=0.0, seed=6, M=4096), 20_000, [dict(shape=(1, 512)), dict(), dict(shape=(2, 544))]),
    ]
    print("# %s: soak - every line below the reference must say identical: True" % torch.cuda.get_device_name(0))
    for name, idx, hops, variants in cases + [(n, k, h, v) for n, k, h, v in extra]:
        kw = idx if isinstance(idx, dict) else workloads.init_args(workloads.CONFIGS[name][idx], sms * 2048)
        idx = 0 if isinstance(idx, dict) else idx
        ref = None
        for v in variants:
            r = run(kw, hops, **v)
            tag = "%s kernel %s, H=%d cluster=%d" % (
                r["kernel"], r["launch"], r["tun"]["snapshot_interval"], r["tun"]["cluster_size"])
            if ref is None:
                ref = r
                print("%s[%d] M=%d, %d hops: reference %s: %.1f s, %d attempts, drift %.1e" % (
                    name, idx, kw["M"], hops, tag, r["dt"], r["c"]["attempts"], r["drift"]))
            else:
                print("    %s: %.1f s, identical: %s, drift %.1e" % (tag, r["dt"], same(ref, r), r["drift"]))
            sys.stdout.flush()


def report_l2():
    """Sweep of the L2 roofline probe: buffer size, CTAs per SM, threads, access width, mode."""
    print("# %s: cg_bench_l2, GB/s (read-modify-write counts read + written bytes), best of 5 launches of 500 passes" % (
        torch.cuda.get_device_name(0)))
    best = {}
    for mode in ("rmw", "read", "write"):
        for mib in (0.5, 2, 4, 16):
            for cps, thr in ((1, 512), (2, 512), (4, 256), (2, 1024), (8, 128), (4, 512)):
                for vec in (16, 32):
                    gb = binding.bench_l2(int(mib * 2**20), reps=500, trials=5, mode=mode, ctas_per_sm=cps,
                                          threads=thr, vec_bytes=vec)
                    print("%-5s %4.1f MiB  %d CTAs/SM x %4d threads  %2d-byte accesses: %8.0f GB/s" % (
                        mode, mib, cps, thr, vec, gb))
                    if gb > best.get(mode, (0,))[0]:
                        best[mode] = (gb, mib, cps, thr, vec)
            sys.stdout.flush()
    for mode, (gb, mib, cps, thr, vec) in best.items():
        print("best %-5s: %8.0f GB/s at %.1f MiB, %d CTAs/SM x %d threads, %d-byte accesses" % (mode, gb, mib, cps, thr, vec))


def report_update():
    """Step a6 alone at the headline footprints: the gather kernel against the bulk-copy staged kernel."""
    print("# %s: cg_apply_hops, 4000 scripted hops (a chain's own hops and their reversal), best of 5" % (
        torch.cuda.get_device_name(0)))
    for label, dim, kw in (("2D L=512", 2, dict(L=512, T=0.05, E=0.01, seed=1008, M=65536)),
                           ("2D L=128", 2, dict(L=128, T=0.05, E=0.01, seed=1005, M=4096)),
                           ("3D L=64", 3, dict(L=64, T=0.05, E=0.01, seed=64, M=65536))):
        u = binding.CoulombGlass(hop_log=2000, dim=dim, **kw)
        u.run(2000)
        _, hi, hj = u.hops()
        si = np.concatenate([hi, hj[::-1]])
        sj = np.concatenate([hj, hi[::-1]])
        ref = None
        for kern in ("gathers", "staged"):
            v = binding.CoulombGlass(dim=dim, **kw)
            best = min(v.apply_hops(si, sj, kernel=kern) for _ in range(5))
            eps = v.state()[1]
            same = "" if ref is None else ("  eps bit-identical to the gather kernel: %s" % np.array_equal(eps, ref))
            ref = eps if ref is None else ref
            print("%-9s %-8s %.4f us/hop  %6.0f GB/s algorithmic (16 N bytes per hop)%s" % (
                label, kern, 1e3 * best / si.size, 16.0 * v.N * si.size / (best * 1e-3) / 1e9, same))
        sys.stdout.flush()


def report_tuning(hops):
    """cg_set_tuning A/B: snapshot interval H and thread-block clusters (DSMEM posts)."""
    print("# %s: %d hops after 150000 warm-up hops (relaxed system)" % (torch.cuda.get_device_name(0), hops))
    for name, idx in (("cfg3_L128", 2), ("cfg5_L512", 0)):
        kw = workloads.init_args(workloads.CONFIGS[name][idx])
        for H, cs in ((1, 1), (2, 1), (4, 1), (8, 1), (4, 2), (4, 4), (4, 8), (4, 16)):
            g = binding.CoulombGlass(**kw)
            try:
                g.set_tuning(H, cs)
            except binding.CgError as e:
                print("%s H=%d cluster=%d: %s" % (name, H, cs, e))
                continue
            g.run(150000)
            torch.cuda.synchronize()
            ms = _timed(lambda: g.run(hops))
            ln = g.launch()
            print("%-9s H=%d cluster=%-2d %3d CTAs x %4d threads (%s labels): %7.0f hops/s  %.3f us/hop" % (
                name, H, cs, ln["n_ctas"], ln["threads"],
                "cached" if kw["M"] <= ln["n_ctas"] * (ln["threads"] - 96) else "recomputed",
                hops / ms * 1e3, ms * 1e3 / hops))
            sys.stdout.flush()


def report_replicas(hops):
    def run(name, idxs, copies):
        sims = []
        for r in range(copies):
            for i in idxs:
                kw = workloads.init_args(workloads.CONFIGS[name][i])
                kw["seed"] += 100 * r
                sims.append(binding.CoulombGlass(stream=torch.cuda.Stream(), **kw))
        for g in sims:
            g.run(1000)
        torch.cuda.synchronize()

        def go():
            for g in sims:
                g.run(hops)
            for g in sims:
                torch.cuda.current_stream().wait_stream(g._stream)
        ms = _timed(go)
        print("%s x%d replicas (%d CTAs each): %.0f hops/s aggregate, %.0f per replica" % (
            name, len(sims), sims[0].launch()["n_ctas"], len(sims) * hops / ms * 1e3, hops / ms * 1e3))
        sys.stdout.flush()

    def packed(name, idxs, copies, n_ctas=0, threads=544):
        """The same replica sets through cg_run_many: one launch, every sim on its own CTAs."""
        sims = []
        for r in range(copies):
            for i in idxs:
                kw = workloads.init_args(workloads.CONFIGS[name][i])
                kw["seed"] += 100 * r
                g = binding.CoulombGlass(**kw)
                if n_ctas:
                    g.set_launch(n_ctas, threads)
                sims.append(g)
        binding.run_many(sims, 1000)
        torch.cuda.synchronize()
        ms = _timed(lambda: binding.run_many(sims, hops))
        print("%s x%d replicas packed into one launch (%d CTAs x %d threads each, %s kernel): %.0f hops/s aggregate, %.0f per replica" % (
            name, len(sims), sims[0].launch()["n_ctas"], sims[0].launch()["threads"], sims[0].kernel(),
            len(sims) * hops / ms * 1e3, hops / ms * 1e3))
        sys.stdout.flush()

    sms = torch.cuda.get_device_properties(0).multi_processor_count
    packed("cfg3_L128", [0, 1, 2, 3], 1)
    packed("cfg3_L128", [0, 1, 2, 3], 2, n_ctas=sms // 8)
    packed("cfg1_L16", [0], 32)
    packed("cfg1_L16", [0], sms)
    packed("cfg2_L64", [0], sms // 5, n_ctas=5)
    packed("cfg2_L64", [0], sms, n_ctas=1, threads=1024)        # config 2 on ONE SM each: the single-CTA kernel
    packed("cfg3_L128", [0, 1, 2, 3], sms // 4, n_ctas=1, threads=512)   # config 3 (its four temperatures) on ONE SM each: 8 labels per thread
    run("cfg3_L128", [0, 1, 2, 3], 1)     # the temperature sweep of config 3 as one replica set
    run("cfg3_L128", [0, 1, 2, 3], 2)
    run("cfg1_L16", [0], 1)
    run("cfg1_L16", [0], 32)
    run("cfg1_L16", [0], 148)
    run("cfg2_L64", [0], 29)


def report_observables(hops):
    import time
    print("# %s; %d hops from the random start, hop log on" % (torch.cuda.get_device_name(0), hops))

    def wall(fn):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        r = fn()
        return r, 1e3 * (time.perf_counter() - t0)

    for name, idx in (("cfg3_L128", 1), ("cfg5_L512", 0)):
        cfg = workloads.CONFIGS[name][idx]
        kw = workloads.init_args(cfg)
        g = binding.CoulombGlass(hop_log=hops, **kw)
        g.run(hops)
        t_det = g.state()[2]
        g.time_stochastic()                                  # first call: context warm-up
        t_st, ms_t = wall(g.time_stochastic)
        (hist, outside), ms_d = wall(lambda: g.dos(-4.0, 2.0**-4, 128))
        (t, P), ms_s = wall(g.series)
        sig, _ = wall(g.sigma0)
        gdos = hist / (g.N * 2.0**-4)
        mid = 64                                             # bin [0, 1/16)
        print("%s T=%-5g: t_det %.6e  t_stoch %.6e (rel. diff %+.2e)  sigma0 %.4e  dP %d" % (
            name, kw["T"], t_det, t_st, t_st / t_det - 1, sig, P[-1]))
        print("    g(eps) at eps = -2, -1, -0.5, -0.25, 0, 0.25, 0.5, 1, 2: %s  (outside [-4,4): %d)" % (
            " ".join("%.3f" % gdos[mid + int(e * 16)] for e in (-2, -1, -0.5, -0.25, 0, 0.25, 0.5, 1, 2)), outside))
        print("    cost: time_stochastic %.2f ms (%d logged hops), dos %.2f ms (N = %d), series %.2f ms (%d points)" % (
            ms_t, hops, ms_d, g.N, ms_s, t.size))
        sys.stdout.flush()


def report_one(name, idx, hops, warm, cluster=0):
    """One config, two launches of the persistent kernel (warm-up, then `hops` hops): the target of the ncu captures
    under profiles/ (`-k regex:cg_pr_persistent --launch-skip 1 --launch-count 1`)."""
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    kw = workloads.init_args(workloads.CONFIGS[name][idx], sms * 2048)
    g = binding.CoulombGlass(**kw)
    if cluster:
        g.set_tuning(0, cluster)          # ncu cannot replay cooperative launches with a cluster dimension: --cluster 1 there
    g.run(warm)
    torch.cuda.synchronize()
    ms = _timed(lambda: g.run(hops))
    c = g.counters()
    print("%s[%d] %s: %d hops after %d warm-up hops: %.0f hops/s, %d iterations in all, launch %s, H=%d, labels/thread %d" % (
        name, idx, kw, hops, warm, hops / ms * 1e3, c["iterations"], g.launch(), g.tuning()["snapshot_interval"],
        g.labels_per_thread()) + ", cluster %d" % g.tuning()["cluster_size"])


def report_l2_one():
    """The best read-modify-write shape of the L2 probe sweep, a few launches: the target of its ncu capture."""
    gb = binding.bench_l2(16 << 20, reps=500, trials=3, mode="rmw", ctas_per_sm=8, threads=128, vec_bytes=16)
    print("cg_bench_l2 rmw 16 MiB, 8 CTAs/SM x 128 threads, 16-byte accesses: %.0f GB/s" % gb)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", action="store_true")
    ap.add_argument("--replicas", action="store_true")
    ap.add_argument("--observables", action="store_true")
    ap.add_argument("--l2", action="store_true")
    ap.add_argument("--update", action="store_true")
    ap.add_argument("--tuning", action="store_true")
    ap.add_argument("--cubic", action="store_true", help="throughput on 3D cubic lattices")
    ap.add_argument("--soak", action="store_true", help="long chains in different shapes and kernels must be identical")
    ap.add_argument("--one", default="", help="CONFIG[:index], e.g. cfg5_L512 or cfg3_L128:3")
    ap.add_argument("--l2-one", action="store_true")
    ap.add_argument("--cluster", type=int, default=0, help="cluster size for --one (0: automatic)")
    ap.add_argument("--hops", type=int, default=0)
    ap.add_argument("--warm", type=int, default=2000)
    a = ap.parse_args()
    if not torch.cuda.is_available():
        raise SystemExit("report needs a CUDA device: the hot path has no CPU fallback")
    if a.one:
        name, _, idx = a.one.partition(":")
        report_one(name, int(idx or 0), a.hops or 20_000, a.warm, a.cluster)
    if a.l2_one:
        report_l2_one()
    if a.configs:
        report_configs(a.hops or 200_000, a.warm)
    if a.replicas:
        report_replicas(a.hops or 100_000)
    if a.observables:
        report_observables(a.hops or 200_000)
    if a.l2:
        report_l2()
    if a.update:
        report_update()
    if a.tuning:
        report_tuning(a.hops or 100_000)
    if a.cubic:
        report_3d(a.hops or 50_000)
    if a.soak:
        report_soak()


if __name__ == "__main__":
    main()
