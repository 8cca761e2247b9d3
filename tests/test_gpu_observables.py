"""GPU parity of the observables (include/cg.h "Observables") against the oracle.

Bar: integer results (DOS bin counts, polarisation series P) and the results of single IEEE
operations on identical operands (series t, sigma0) bit-exact; the normal deviates within
1e-14 relative (CUDA's log/cos and glibc's differ by <= 2 ulp each); the
stochastic time within 1e-11 relative for H <= 1e5 hops (H * 2^-53 summation-order bound plus
the deviates' error).
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


@pytest.mark.parametrize("first,count", [(0, 5000), (2**32 - 100, 200), (2**40 + 7, 1), (12345, 0)])
def test_normal_deviates_match_oracle(cg, oracle_lib, first, count):
    g = cg.CoulombGlass(16, T=0.1, seed=77, M=64)
    o = oracle_lib.Oracle(16, T=0.1, seed=77, M=64)
    z = g.normals(first, count)
    ref = np.array([o.normal_of_hop(first + k) for k in range(count)])
    assert z.shape == ref.shape
    assert np.allclose(z, ref, rtol=1e-14, atol=1e-16)


CASES = [("cfg1_L16", 0, 20_000), ("cfg2_L64", 0, 20_000), ("cfg3_L128", 2, 6_000), ("cfg5_L512", 0, 2_500)]


@pytest.mark.parametrize("name,idx,hops", CASES)
def test_observables_match_oracle(cg, oracle_lib, name, idx, hops):
    kw = workloads.init_args(workloads.CONFIGS[name][idx])
    g = cg.CoulombGlass(hop_log=hops, **kw)
    o = oracle_lib.Oracle(**kw)
    g.run(hops // 2); g.run(hops - hops // 2)            # two launches: the log carries over
    o.run(hops)
    assert g.counters() == o.counters()

    # step 3c
    tg, to = g.time_stochastic(), o.time_stochastic()
    assert abs(tg - to) <= 1e-11 * abs(to)
    assert tg == g.time_stochastic()                      # fixed summation tree: reproducible to the bit

    # shared-memory bins, one bin, a narrow window, and the global-atomics path (> 8192 bins)
    for lo, width, nbins in [(-4.0, 2.0**-4, 128), (-8.0, 16.0, 1), (-0.25, 2.0**-7, 64), (-3.0, 6.0 / 20000, 20000),
                             (0.1, 0.013, 37)]:
        hg, outg = g.dos(lo, width, nbins)
        ho, outo = o.dos(lo, width, nbins)
        assert np.array_equal(hg, ho) and outg == outo, (lo, width, nbins)
        assert int(hg.sum()) + outg == g.N

    # full series and windows that straddle the 2048-hop scan chunks
    tg_, Pg = g.series()
    to_, Po = o.series()
    assert np.array_equal(Pg, Po) and np.array_equal(tg_, to_)
    assert Pg[-1] == g.state()[3]
    for first, count in [(2047, 3), (hops - 1, 1), (1, 2048), (hops // 3, 0)]:
        t2, P2 = g.series(first, count)
        assert np.array_equal(P2, Po[first:first + count]) and np.array_equal(t2, to_[first:first + count])

    if kw["E"] != 0.0:
        assert g.sigma0() == o.sigma0()
    else:
        with pytest.raises(cg.binding.CgError):
            g.sigma0()


def test_log_enabled_in_the_middle_of_a_chain(cg, oracle_lib):
    """Time before the enabling point enters deterministically; hop indices of the deviates stay global."""
    kw = workloads.init_args(workloads.CONFIGS["cfg1_L16"][0])
    g = cg.CoulombGlass(**kw)
    o = oracle_lib.Oracle(**kw)
    g.run(1500); o.run(1500)
    t_det_1500, ts_1500 = o.state()[2], o.time_stochastic()
    g.enable_hop_log(4000)
    assert g.time_stochastic() == t_det_1500             # nothing logged yet
    g.run(4000); o.run(4000)
    expect = t_det_1500 + (o.time_stochastic() - ts_1500)
    assert abs(g.time_stochastic() - expect) <= 1e-11 * abs(expect)
    tg, Pg = g.series()
    to, Po = o.series(1500, 4000)
    assert np.array_equal(tg, to)
    assert np.array_equal(Pg, Po - o.series(1499, 1)[1][0])   # P counts from the enabling point


def test_observables_need_a_complete_log(cg):
    kw = workloads.init_args(workloads.CONFIGS["cfg1_L16"][0])
    g = cg.CoulombGlass(**kw)
    g.run(10)
    for call in (g.time_stochastic, lambda: g.series(0, 1)):
        with pytest.raises(cg.binding.CgError) as e:
            call()
        assert e.value.code == cg.binding.CG_EINVAL
    g.enable_hop_log(100)
    g.run(100)
    g.time_stochastic(); g.series(0, 100)
    with pytest.raises(cg.binding.CgError):
        g.series(50, 51)                                  # past the logged hops
    g.run(1)                                              # the log has overflowed: m of later hops is lost
    with pytest.raises(cg.binding.CgError):
        g.time_stochastic()
    # scripted hops are not logged: the log-based observables refuse until the log is enabled again
    g.enable_hop_log(100)
    g.run(5)
    _, hi, hj = g.hops(4, 1)
    g.apply_hops(hj, hi)                                  # a valid scripted hop: the last executed one, reversed
    with pytest.raises(cg.binding.CgError):
        g.series(0, 1)
    g.enable_hop_log(100)
    g.run(3)
    assert g.series()[0].size == 3
    # the density of states needs no log; bad arguments are refused
    h, out = g.dos(-4.0, 0.5, 16)
    assert int(h.sum()) + out == g.N
    for lo, width, nbins in [(0.0, 0.0, 4), (0.0, -1.0, 4), (0.0, 1.0, 0)]:
        with pytest.raises(cg.binding.CgError):
            g.dos(lo, width, nbins)
