"""GPU parity: libcg.so (through its C ABI) against the CPU oracle, element by element.

Bar (BASELINE.json north_star): hop log (attempt, i, j) and occupations bit-identical;
eps within 1e-12 relative (expected bit-identical); incremental eps within 1e-9 of the
from-scratch recomputation; counters (attempts, iterations, proposals) identical.
"""
import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def cg():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1407_5026_b200 import build
    build.build()
    import paper_1407_5026_b200 as pkg
    return pkg


def _compare(g, o, hops, check_eps_bits=True):
    ga, gi, gj = g.hops(0, hops)
    oa, oi, oj = o.hops(0, hops)
    bad = np.flatnonzero((ga != oa) | (gi != oi) | (gj != oj))
    assert bad.size == 0, "first divergence at hop %d: gpu %s oracle %s" % (
        bad[0], (ga[bad[0]], gi[bad[0]], gj[bad[0]]), (oa[bad[0]], oi[bad[0]], oj[bad[0]]))
    gn, ge, gt, gp = g.state()
    on, oe, ot, op = o.state()
    assert np.array_equal(gn, on) and gn.sum() == g.N // 2
    assert gt == ot and gp == op
    assert np.allclose(ge, oe, rtol=1e-12, atol=0)
    if check_eps_bits:
        assert np.array_equal(ge, oe)
    assert g.counters() == o.counters()
    assert o.near_ties() == 0          # O10 certificate: decisions did not depend on the libm


@pytest.mark.parametrize("L", [4, 8, 16, 64, 256])
def test_init_is_bit_identical(cg, oracle_lib, L):
    """Step a0: tables, disorder, occupations and the full-sum eps."""
    g = cg.CoulombGlass(L, W=1.0, xi=1.0, T=0.1, E=0.01, seed=40 + L, M=64)
    o = oracle_lib.Oracle(L, W=1.0, xi=1.0, T=0.1, E=0.01, seed=40 + L, M=64)
    tg, to = g.tables(), o.tables()
    kl = tg["K_live"]
    assert tg["K"] == to["K"] and tg["S"] == to["S"] and tg["Gamma"] == to["Gamma"]
    for key in ("dy", "dx", "cdf", "invr_k"):
        assert np.array_equal(tg[key], to[key][:kl]), key
    assert np.all(to["cdf"][kl - 1:] == 1.0)           # entries past the live prefix can never be drawn
    assert np.array_equal(g.phi(), o.phi())
    gn, ge, gt, gp = g.state()
    on, oe, _, _ = o.state()
    assert np.array_equal(gn, on) and np.array_equal(ge, oe) and gt == 0.0 and gp == 0
    assert g.recompute_eps() == 0.0


CASES = [  # (name, index, hops compared) — prefixes the oracle finishes in seconds
    ("cfg1_L16", 0, 100_000),
    ("cfg2_L64", 0, 60_000),
    ("cfg3_L128", 0, 20_000), ("cfg3_L128", 3, 20_000),
    ("cfg4_L256", 1, 6_000),
    ("cfg5_L512", 0, 3_000),
]


@pytest.mark.parametrize("name,idx,hops", CASES)
def test_hop_log_matches_oracle(cg, oracle_lib, name, idx, hops):
    kw = workloads.init_args(workloads.CONFIGS[name][idx])
    g = cg.CoulombGlass(hop_log=hops, **kw)
    o = oracle_lib.Oracle(**kw)
    g.run(hops)
    o.run(hops)
    _compare(g, o, hops)
    assert g.recompute_eps() < 1e-9


def test_split_runs_continue_the_same_chain(cg, oracle_lib):
    kw = workloads.init_args(workloads.CONFIGS["cfg2_L64"][0])
    g = cg.CoulombGlass(hop_log=5000, **kw)
    for part in (1, 7, 992, 4000):        # cg_run(a); cg_run(b) == cg_run(a+b)
        g.run(part)
    o = oracle_lib.Oracle(**kw)
    o.run(5000)
    _compare(g, o, 5000)


@pytest.mark.parametrize("n_ctas,threads", [(1, 256), (3, 256), (8, 544), (37, 1024), (148, 544), (131, 1024), (100, 608)])
def test_result_is_independent_of_launch_shape(cg, oracle_lib, n_ctas, threads):
    kw = dict(L=64, T=0.05, E=0.02, seed=77, M=1000)     # M not a multiple of anything: ragged label tail
    g = cg.CoulombGlass(hop_log=4000, **kw)
    g.set_launch(n_ctas, threads)
    assert g.launch()["n_ctas"] == n_ctas and g.launch()["threads"] == threads
    g.run(4000)
    o = oracle_lib.Oracle(**kw)
    o.run(4000)
    _compare(g, o, 4000)


@pytest.mark.parametrize("M", [1, 2, 31, 33, 4096, 303104])
def test_trajectory_is_independent_of_M(cg, oracle_lib, M):
    """Reading G8: only the iteration bookkeeping depends on M; M=1 is the serial algorithm,
    M = 148*2048 exceeds the resident threads."""
    hops = 300 if M == 1 else 3000
    kw = dict(L=32, T=0.08, E=0.01, seed=5, M=M)
    g = cg.CoulombGlass(hop_log=hops, **kw)
    g.run(hops)
    o = oracle_lib.Oracle(**kw)
    o.run(hops)
    _compare(g, o, hops)
    c = g.counters()
    assert c["proposals_evaluated"] == M * c["iterations"]


def test_smallest_lattice_and_hot_cold_limits(cg, oracle_lib):
    for kw, hops in ((dict(L=4, T=0.5, E=0.0, seed=3, M=12), 20000),
                     (dict(L=4, T=5.0, E=0.3, seed=4, M=5), 20000),      # hot: A ~ 1, q = 0 mostly
                     (dict(L=16, T=0.01, E=0.0, seed=6, M=4096), 300),   # cold: many empty windows
                     (dict(L=8, W=0.0, T=0.1, E=0.0, seed=9, M=64), 5000),   # no disorder
                     (dict(L=32, W=2.0, xi=2.0, T=0.2, E=-0.05, seed=10, M=256), 5000)):  # paper's width, xi=2
        g = cg.CoulombGlass(hop_log=hops, **kw)
        g.run(hops)
        o = oracle_lib.Oracle(**kw)
        o.run(hops)
        _compare(g, o, hops)


def test_update_kernel_alone_on_scripted_hops(cg, oracle_lib):
    """Step a6 by itself: eps bit-identical after scripted hops from an oracle log."""
    for L, hops in ((16, 2000), (128, 1500), (512, 300)):
        kw = dict(L=L, T=0.1, E=0.01, seed=90 + L, M=256)
        o = oracle_lib.Oracle(**kw)
        o.run(hops)
        _, i, j = o.hops()
        g = cg.CoulombGlass(**kw)
        ms = g.apply_hops(i, j)
        assert ms > 0
        gn, ge, _, gp = g.state()
        on, oe, _, op = o.state()
        assert np.array_equal(gn, on) and np.array_equal(ge, oe) and gp == op
        assert g.counters()["hops"] == hops
        with pytest.raises(cg.CgError):           # a hop from an empty site violates theta_ij
            empty = int(np.flatnonzero(gn == 0)[0]); occ = int(np.flatnonzero(gn == 1)[0])
            g.apply_hops([empty], [occ])


def test_checkpoint_restore(cg, oracle_lib):
    kw = workloads.init_args(workloads.CONFIGS["cfg2_L64"][0])
    g = cg.CoulombGlass(**kw)
    g.run(3000)
    n, eps, t, dP = g.state()
    c = g.counters()
    g2 = cg.CoulombGlass(hop_log=2000, **kw)
    g2.set_state(n, eps, c["attempts"], c["hops"], dP)
    g2.run(2000)
    o = oracle_lib.Oracle(**kw)
    o.run(5000)
    oa, oi, oj = o.hops(3000, 2000)
    ga, gi, gj = g2.hops(0, 2000)
    assert np.array_equal(ga, oa) and np.array_equal(gi, oi) and np.array_equal(gj, oj)
    assert np.array_equal(g2.state()[1], o.state()[1]) and g2.state()[3] == o.state()[3]


def test_long_run_properties_at_headline_size(cg):
    """Full-size config 5 in the launch shape bench.py times: properties that hold at any length."""
    kw = workloads.init_args(workloads.CONFIGS["cfg5_L512"][0])
    g = cg.CoulombGlass(hop_log=200_000, **kw)
    g.run(200_000)
    n, eps, t, dP = g.state()
    c = g.counters()
    assert n.sum() == g.N // 2 and c["hops"] == 200_000
    assert g.recompute_eps() < 1e-9
    assert abs(eps.sum() - g.phi().sum()) < 1e-6          # sum eps = sum phi at half filling
    a, i, j = g.hops()
    assert np.all(np.diff(a.astype(np.int64)) > 0) and a[-1] + 1 == c["attempts"]
    assert t == c["attempts"] / g.tables()["Gamma"]
    dx = (j.astype(np.int64) % 512 - i.astype(np.int64) % 512) % 512
    dx = np.where(dx > 256, dx - 512, dx)
    assert dP == dx.sum()
    assert c["proposals_evaluated"] == kw["M"] * c["iterations"] and c["iterations"] >= c["hops"]
    # replaying the log on the initial occupations gives the final occupations
    g0 = cg.CoulombGlass(**kw)
    n0 = g0.state()[0].astype(np.int64)
    np.subtract.at(n0, i, 1); np.add.at(n0, j, 1)
    assert np.array_equal(n0, n)


def test_launch_shape_may_change_between_runs(cg, oracle_lib):
    """The exchange slots, publication words and the eps ring carry over from one launch shape to the
    next: the chain must not notice (stale words of other shapes are never mistaken for arrivals)."""
    kw = dict(L=128, T=0.1, E=0.01, seed=21, M=4096)
    g = cg.CoulombGlass(hop_log=6000, **kw)
    for n_ctas, threads, hops in ((0, 0, 1500), (37, 256, 1000), (148, 1024, 1500), (5, 544, 500), (0, 0, 1500)):
        g.set_launch(n_ctas, threads)
        g.run(hops)
    o = oracle_lib.Oracle(**kw)
    o.run(6000)
    _compare(g, o, 6000)
    assert g.recompute_eps() < 1e-9


@pytest.mark.parametrize("n_ctas,threads,M", [(148, 544, 303104), (30, 544, 303104), (148, 256, 65536), (20, 1024, 65536), (148, 1024, 65536)])
def test_labels_recomputed_or_cached(cg, oracle_lib, n_ctas, threads, M):
    """M larger than the label-owning threads of the grid takes the path that decodes every label in
    every iteration; otherwise proposals are cached.  Both must give the serial chain."""
    kw = dict(L=256, T=0.05, E=0.01, seed=31, M=M)
    g = cg.CoulombGlass(hop_log=3000, **kw)
    g.set_launch(n_ctas, threads)
    g.run(3000)
    o = oracle_lib.Oracle(**kw)
    o.run(3000)
    _compare(g, o, 3000)


@pytest.mark.parametrize("kw,n_ctas,K,hops", [
    (dict(L=16, T=0.01, E=0.0, seed=6, M=3000), 2, 4, 300),      # cold: whole windows rejected, every slot of a thread consumed at once
    (dict(L=16, T=0.01, E=0.0, seed=6, M=897), 2, 2, 300),       # one single label in the second slot
    (dict(L=32, T=5.0, E=0.3, seed=4, M=7168), 2, 8, 20000),     # hot: q = 0 mostly; the most labels per thread, M = K P exactly
    (dict(L=64, T=0.05, E=0.01, seed=2, M=5000), 3, 4, 20000),   # ragged last slot, three CTAs
    (dict(L=64, T=0.03, E=0.01, seed=12, M=40000), 37, 3, 20000),
    (dict(L=16, dim=3, T=0.05, E=0.01, seed=13, M=9000), 8, 3, 6000),
    (dict(L=32, T=0.08, E=0.01, seed=5, M=4096), 1, 0, 2000),    # more than 8 labels per thread: recomputed
])
def test_several_cached_labels_per_thread(cg, oracle_lib, kw, n_ctas, K, hops):
    """M larger than the label-owning threads P of the grid (M up to the resident threads and beyond):
    every thread keeps K = ceil(M / P) <= 8 proposals decoded, slot 0 in registers, the others in shared memory;
    the lowest accepting label over all slots wins (labels of slot k rank after all labels of slot k - 1).  Split
    runs re-decode the slots; the chain must be the serial one whatever K."""
    g = cg.CoulombGlass(hop_log=hops, **kw)
    g.set_launch(n_ctas, 544)
    assert g.labels_per_thread() == K
    g.run(hops // 3)
    g.run(hops - hops // 3)
    o = oracle_lib.Oracle(**kw)
    o.run(hops)
    _compare(g, o, hops)
    c = g.counters()
    assert c["proposals_evaluated"] == kw["M"] * c["iterations"]
    assert g.recompute_eps() < 1e-9


@pytest.mark.parametrize("kw,explicit,hops", [
    (dict(L=16, T=0.1, E=0.0, seed=1, M=256), False, 30000),             # config 1: chosen automatically
    (dict(L=4, T=0.5, E=0.0, seed=3, M=12), False, 5000),
    (dict(L=16, T=0.01, E=0.0, seed=6, M=512), False, 300),              # cold: whole windows rejected
    (dict(L=8, T=5.0, E=0.3, seed=4, M=5), False, 20000),                # hot: q = 0 mostly
    (dict(L=32, T=0.08, E=0.01, seed=5, M=500), False, 6000),            # N/2 = 512 sites per thread pair, ragged M
    (dict(L=64, T=0.05, E=0.01, seed=2, M=512), True, 6000),             # 8 sites per thread, asked for
    (dict(L=8, dim=3, T=0.05, E=0.01, seed=13, M=384), False, 6000),     # cubic lattice
    (dict(L=16, dim=3, T=0.1, E=-0.02, seed=14, M=100), True, 4000),
])
def test_single_cta_kernel(cg, oracle_lib, kw, explicit, hops):
    """A sim whose labels and sites fit one CTA runs in cg_pr_single (512 threads, eps and occupations in shared
    memory, two CTA barriers per iteration); the chain must be the serial one, also across launches."""
    g = cg.CoulombGlass(hop_log=hops, **kw)
    if explicit:
        g.set_launch(1, 512)
    assert g.launch()["n_ctas"] == 1 and g.launch()["threads"] == 512 and g.labels_per_thread() == 1 and g.kernel() == "single"
    g.run(hops // 3)
    g.run(hops - hops // 3)
    o = oracle_lib.Oracle(**kw)
    o.run(hops)
    _compare(g, o, hops)
    assert g.recompute_eps() < 1e-9
    # the same chain goes on in the dataflow kernel and back
    g.set_launch(1, 544)
    g2 = cg.CoulombGlass(hop_log=hops + 600, **kw)
    g2.set_launch(3 if kw["L"] >= 8 else 1, 544)
    g2.run(hops)
    g2.set_launch(1, 512)
    g2.run(300)
    g2.set_launch(2 if kw["L"] >= 8 else 1, 544)
    g2.run(300)
    o.run(600)
    _compare(g2, o, hops + 600)


@pytest.mark.parametrize("kw,shape,hops", [
    (dict(L=32, T=0.08, E=0.01, seed=5, M=1024), None, 6000),            # automatic: M = the threads of the CTA, no idle lanes
    (dict(L=32, T=0.08, E=0.01, seed=5, M=700), None, 6000),
    (dict(L=64, T=0.05, E=0.0, seed=2, M=1024), (1, 1024), 6000),        # config 2 on one SM (replica packing)
    (dict(L=16, dim=3, T=0.05, E=0.01, seed=13, M=1000), (1, 1024), 4000),
    (dict(L=16, T=0.01, E=0.0, seed=6, M=1024), None, 300),              # cold: whole windows rejected
])
def test_single_cta_kernel_with_1024_threads(cg, oracle_lib, kw, shape, hops):
    g = cg.CoulombGlass(hop_log=hops, **kw)
    if shape:
        g.set_launch(*shape)
    assert g.kernel() == "single" and g.launch()["n_ctas"] == 1 and g.launch()["threads"] == 1024
    g.run(hops // 2)
    g.run(hops - hops // 2)
    o = oracle_lib.Oracle(**kw)
    o.run(hops)
    _compare(g, o, hops)
    assert g.recompute_eps() < 1e-9


@pytest.mark.parametrize("kw,K,hops", [
    (dict(L=128, T=0.2, E=0.01, seed=3, M=4096), 8, 4000),               # config 3 on ONE SM (replica packing)
    (dict(L=128, T=0.03, E=0.01, seed=6, M=4096), 8, 3000),
    (dict(L=64, T=0.05, E=0.0, seed=2, M=2000), 4, 6000),                # ragged M: labels beyond M are not tested
    (dict(L=64, T=0.05, E=0.0, seed=2, M=1024), 2, 6000),
    (dict(L=16, T=0.01, E=0.0, seed=6, M=4096), 8, 300),                 # cold: whole windows rejected, all 8 slots consumed at once
    (dict(L=16, dim=3, T=0.05, E=0.01, seed=13, M=3000), 8, 4000),
    (dict(L=128, T=0.1, E=0.01, seed=4, M=256), 2, 3000),                # few labels, eps beyond the 64 KiB of the one-label kernel
])
def test_single_cta_kernel_with_several_labels_per_thread(cg, oracle_lib, kw, K, hops):
    """(1 CTA, 512 threads) for M > 512 or N > 8192: cg_pr_singlek, K = 2, 4 or 8 labels per thread in registers, the lowest
    accepting label and its sites in one 64-bit shared atomicMin.  Must be the serial chain; split runs re-decode the slots."""
    g = cg.CoulombGlass(hop_log=hops, **kw)
    g.set_launch(1, 512)
    assert g.kernel() == "single" and g.launch()["threads"] == 512 and g.labels_per_thread() == K
    g.run(hops // 3)
    g.run(hops - hops // 3)
    o = oracle_lib.Oracle(**kw)
    o.run(hops)
    _compare(g, o, hops)
    c = g.counters()
    assert c["proposals_evaluated"] == kw["M"] * c["iterations"]
    assert g.recompute_eps() < 1e-9


def test_single_cta_kernel_refuses_what_does_not_fit(cg):
    g = cg.CoulombGlass(L=16, T=0.1, M=4096)
    assert g.launch()["threads"] == 544 and g.kernel() == "dataflow"      # M beyond 1024 labels: the dataflow kernel by default
    g = cg.CoulombGlass(L=16, T=0.1, M=4097)
    with pytest.raises(cg.CgError):
        g.set_launch(1, 512)                           # more than 8 labels per thread
    g = cg.CoulombGlass(L=256, T=0.1, M=256)
    with pytest.raises(cg.CgError):
        g.set_launch(1, 512)                           # eps does not fit shared memory


def test_config4_M_sweep_is_one_trajectory(cg):
    """Config 4 of BASELINE.json (L=256, T=0.02): the hop log must be the same for every M (reading G8),
    including M = resident threads of the chip; only iterations and proposals differ."""
    import torch
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    logs = []
    for cfg in workloads.CONFIGS["cfg4_L256"]:
        kw = workloads.init_args(cfg, sms * 2048)
        g = cg.CoulombGlass(hop_log=20000, **kw)
        g.run(20000)
        c = g.counters()
        assert c["proposals_evaluated"] == kw["M"] * c["iterations"]
        logs.append((g.hops(), g.state(), c["attempts"]))
    for (h, st, a) in logs[1:]:
        for x, y in zip(h, logs[0][0]):
            assert np.array_equal(x, y)
        assert np.array_equal(st[0], logs[0][1][0]) and np.array_equal(st[1], logs[0][1][1]) and a == logs[0][2]


def test_largest_supported_lattice(cg, oracle_lib):
    """L = 1024 (N = 2^20): init bit-identical, a short prefix of the chain, drift of the update."""
    kw = dict(L=1024, T=0.05, E=0.01, seed=12, M=65536)
    g = cg.CoulombGlass(hop_log=400, **kw)
    o = oracle_lib.Oracle(**kw)
    assert np.array_equal(g.state()[1], o.state()[1])
    g.run(400)
    o.run(400)
    _compare(g, o, 400)
    assert g.recompute_eps() < 1e-9


def test_replicas_on_separate_streams_run_concurrently_and_independently(cg, oracle_lib):
    """Independent samples (the paper's recommended use of more hardware): config 3's four
    temperatures as four sims on four streams, launched back to back; each must be its own serial chain."""
    import torch
    sims = []
    for cfg in workloads.CONFIGS["cfg3_L128"]:
        kw = workloads.init_args(cfg)
        sims.append((kw, cg.CoulombGlass(hop_log=5000, stream=torch.cuda.Stream(), **kw)))
    for _, g in sims:
        g.run(5000)                       # asynchronous: the four persistent kernels overlap
    for kw, g in sims:
        o = oracle_lib.Oracle(**kw)
        o.run(5000)
        _compare(g, o, 5000)


def test_replicas_packed_into_one_launch(cg, oracle_lib):
    """cg_run_many: config 3's four temperatures, 19 CTAs each, side by side
    in ONE persistent launch, in two calls (the chains continue); each is its own serial chain."""
    sims = []
    for cfg in workloads.CONFIGS["cfg3_L128"]:
        kw = workloads.init_args(cfg)
        sims.append((kw, cg.CoulombGlass(hop_log=5000, **kw)))
    cg.run_many([g for _, g in sims], 3000)
    cg.run_many([g for _, g in sims][::-1], 2000)      # order in the launch does not matter
    for kw, g in sims:
        o = oracle_lib.Oracle(**kw)
        o.run(5000)
        _compare(g, o, 5000)


def test_many_one_cta_replicas_and_mixed_calls(cg, oracle_lib):
    """One CTA per sim, one sim per SM, different seeds and temperatures; cg_run and cg_run_many mix freely."""
    import torch
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    kws = [dict(L=16, W=1.0, xi=1.0, T=0.05 + 0.001 * r, E=0.01, seed=900 + r, M=256) for r in range(sms)]
    sims = [cg.CoulombGlass(hop_log=4000, **kw) for kw in kws]
    sims[3].run(500)
    cg.run_many(sims[:3] + sims[4:], 500)
    cg.run_many(sims, 3500)
    for r in (0, 3, 77, sms - 1):
        o = oracle_lib.Oracle(**kws[r])
        o.run(4000)
        _compare(sims[r], o, 4000)
    for g in sims:
        assert g.counters()["hops"] == 4000 and g.recompute_eps() < 1e-9


def test_run_many_refuses_what_it_cannot_run(cg):
    kw = workloads.init_args(workloads.CONFIGS["cfg5_L512"][0])
    a, b = cg.CoulombGlass(**kw), cg.CoulombGlass(**dict(kw, seed=99))
    with pytest.raises(cg.CgError):          # 2 x 148 CTAs cannot be resident together
        cg.run_many([a, b], 10)
    with pytest.raises(cg.CgError):          # the same sim twice
        cg.run_many([a, a], 10)
    c = cg.CoulombGlass(16, T=0.1, seed=1, M=256)
    with pytest.raises(cg.CgError):          # different launch shapes (register tiling)
        cg.run_many([a, c], 10)
    cg.run_many([a], 10)                     # a single sim is fine
    assert a.counters()["hops"] == 10


def test_tuning_never_changes_results(cg, oracle_lib):
    """cg_set_tuning: snapshot interval H (deferred eps write-through) and thread-block clusters
    (posts through distributed shared memory) are performance knobs only: the chain is the oracle's for every
    setting, also when they change between runs of one chain, with several CTAs per cluster and ragged shapes."""
    kw = dict(L=128, T=0.1, E=0.01, seed=21, M=4096)
    o = oracle_lib.Oracle(**kw)
    o.run(6000)
    for H, cs in ((1, 1), (2, 2), (8, 1), (4, 4), (4, 8), (1, 16)):
        g = cg.CoulombGlass(hop_log=6000, **kw)
        g.set_tuning(H, cs)
        assert g.tuning() == {"snapshot_interval": H, "cluster_size": cs}
        assert g.launch()["n_ctas"] % cs == 0
        for hops in (1, 2, 3, 1994, 7, 3993):      # launches that end between snapshots
            g.run(hops)
        _compare(g, o, 6000)
        assert g.recompute_eps() < 1e-9
    g = cg.CoulombGlass(hop_log=6000, **kw)
    for H, cs, n_ctas, hops in ((4, 1, 0, 1000), (8, 2, 6, 1000), (1, 4, 16, 1000), (2, 8, 8, 1500), (4, 16, 32, 1500)):
        g.set_tuning(H, cs)
        g.set_launch(n_ctas, 544)
        g.run(hops)
    _compare(g, o, 6000)


def test_headline_config_in_clusters(cg, oracle_lib):
    """Config 5 (L=512, M=65536) launched in thread-block clusters: fewer, larger CTAs (the GPCs strand SMs)."""
    kw = workloads.init_args(workloads.CONFIGS["cfg5_L512"][0])
    o = oracle_lib.Oracle(**kw)
    o.run(3000)
    for cs in (2, 8, 16):
        g = cg.CoulombGlass(hop_log=3000, **kw)
        g.set_tuning(0, cs)
        g.run(3000)
        _compare(g, o, 3000)


@pytest.mark.parametrize("L,M,hops", [(4, 16, 5000), (8, 64, 5000), (16, 1024, 6000), (32, 8192, 3000)])
def test_cubic_lattice_matches_oracle(cg, oracle_lib, L, M, hops):
    """the L^3 lattice.  Tables, disorder, occupations and the full-sum eps
    bit-identical, then the chain."""
    kw = dict(L=L, W=1.0, xi=1.0, T=0.1, E=0.02, seed=300 + L, M=M)
    g = cg.CoulombGlass(hop_log=hops, dim=3, **kw)
    o = oracle_lib.Oracle(dim=3, **kw)
    tg, to = g.tables(), o.tables()
    kl = tg["K_live"]
    assert tg["K"] == to["K"] and tg["S"] == to["S"] and tg["Gamma"] == to["Gamma"]
    for key in ("dz", "dy", "dx", "cdf", "invr_k"):
        assert np.array_equal(tg[key], to[key][:kl]), key
    assert np.all(to["cdf"][kl - 1:] == 1.0)
    assert np.array_equal(g.phi(), o.phi())
    assert np.array_equal(g.state()[0], o.state()[0]) and np.array_equal(g.state()[1], o.state()[1])
    assert g.recompute_eps() == 0.0
    g.run(hops)
    o.run(hops)
    _compare(g, o, hops)
    assert g.recompute_eps() < 1e-9


def test_cubic_lattice_at_the_headline_footprint(cg, oracle_lib):
    """L = 64 cubed: N = 262144, the footprint of config 5, all SMs; the live tower (about 48 000 displacements)
    no longer fits shared memory, its tail is read from L2.  Launch shapes and tuning as in 2D."""
    kw = dict(L=64, W=1.0, xi=1.0, T=0.05, E=0.01, seed=64, M=65536)
    o = oracle_lib.Oracle(dim=3, **kw)
    g = cg.CoulombGlass(hop_log=2500, dim=3, **kw)
    assert g.tables()["K_live"] > 2048
    assert np.array_equal(g.state()[1], o.state()[1])
    g.run(1500)
    g.set_tuning(2, 4)
    g.run(1000)
    o.run(2500)
    _compare(g, o, 2500)
    assert g.recompute_eps() < 1e-9
    # the update alone on the oracle's hops
    u = cg.CoulombGlass(dim=3, **kw)
    _, i, j = o.hops()
    assert u.apply_hops(i, j) > 0
    assert np.array_equal(u.state()[1], o.state()[1]) and u.state()[3] == o.state()[3]


def test_scripted_hops_are_validated_before_anything_changes(cg):
    g = cg.CoulombGlass(16, T=0.1, seed=3, M=64, hop_log=10)
    n, eps, _, dP = g.state()
    occ, emp = np.flatnonzero(n == 1), np.flatnonzero(n == 0)
    with pytest.raises(cg.CgError):           # the third hop starts from a site the first one emptied
        g.apply_hops([occ[0], occ[1], occ[0]], [emp[0], emp[1], emp[2]])
    n2, eps2, _, dP2 = g.state()
    assert np.array_equal(n, n2) and np.array_equal(eps, eps2) and dP == dP2 and g.counters()["hops"] == 0
    g.apply_hops([occ[0], emp[0]], [emp[0], occ[0]])       # there and back: legal in this order
    assert np.array_equal(g.state()[0], n) and np.allclose(g.state()[1], eps, atol=1e-13)
    with pytest.raises(cg.CgError):           # scripted hops are not in the log
        g.hops(0, 1)
    with pytest.raises(cg.CgError):           # first + count must not wrap
        g._check(g._lib.cg_get_hops(g._h, 2**64 - 1, 2, None, None, None))


FULL = [("cfg1_L16", 0), ("cfg2_L64", 0), ("cfg3_L128", 0), ("cfg3_L128", 1), ("cfg3_L128", 2), ("cfg3_L128", 3),
        ("cfg4_L256", 2), ("cfg4_L256", 3), ("cfg5_L512", 0)]


@pytest.fixture(scope="module")
def full_oracles(oracle_lib):
    """The oracle's runs of BASELINE.json's configs at their FULL hop counts, all started at once on host
    threads (the C library runs without the interpreter lock; each run is single-threaded): about five
    minutes of wall time on the GPU box instead of ten.  Config 4's trajectory does not depend on M
    (reading G8), so its two M values share one run."""
    import threading
    runs = {}

    def start(name, idx):
        cfg = workloads.CONFIGS[name][idx]
        o = oracle_lib.Oracle(**workloads.init_args(cfg))
        th = threading.Thread(target=o.run, args=(cfg["hops"],))
        th.start()
        runs[(name, idx)] = (o, th)

    for name, idx in FULL:
        if (name, idx) != ("cfg4_L256", 3):
            start(name, idx)
    runs[("cfg4_L256", 3)] = runs[("cfg4_L256", 2)]
    return runs


@pytest.mark.slow
@pytest.mark.parametrize("name,idx", FULL)
def test_full_length_configs(cg, oracle_lib, full_oracles, name, idx):
    """BASELINE.json's configs at their FULL hop counts (1e5 / 1e6 hops), hop log, occupations, eps, clock,
    dP and counters element by element.  CG_SKIP_FULL_PARITY=1 skips (several minutes of oracle time)."""
    import os
    import torch
    if os.environ.get("CG_SKIP_FULL_PARITY") == "1":
        pytest.skip("CG_SKIP_FULL_PARITY=1")
    cfg = workloads.CONFIGS[name][idx]
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    kw = workloads.init_args(cfg, sms * 2048)
    hops = cfg["hops"]
    g = cg.CoulombGlass(hop_log=hops, **kw)
    g.run(hops)
    assert g.recompute_eps() < 1e-9
    o, th = full_oracles[(name, idx)]
    th.join()
    if kw["M"] == o.M:
        _compare(g, o, hops)
    else:       # config 4 at M = resident threads: the oracle ran with M = 65536; iterations follow from its log
        for x, y in zip(g.hops(0, hops), o.hops(0, hops)):
            assert np.array_equal(x, y)
        assert np.array_equal(g.state()[0], o.state()[0]) and np.array_equal(g.state()[1], o.state()[1])
        assert g.state()[2:] == o.state()[2:] and o.near_ties() == 0
        ends = o.hops(0, hops)[0].astype(np.int64) + 1
        m = np.diff(np.concatenate([[0], ends]))
        its = int(sum(oracle_lib.pr_split(int(v), kw["M"])[0] for v in m))     # p = ceil(m / M) per hop
        c = g.counters()
        assert c["attempts"] == ends[-1] and c["iterations"] == its and c["proposals_evaluated"] == its * kw["M"]
