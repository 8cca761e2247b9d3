"""Pins for the oracle's observables (O11-O14 in oracle/cg_oracle.h).

PAPER.md:78 (step 3c, Gaussian time increment), PAPER.md:92 (density of states),
PAPER.md:65-67, 94 (polarisation, conductivity).  Each test checks the oracle against
something other than itself: a library distribution, numpy's histogram on exact edges,
a hand-built hop script with known dx, the closed forms of the paper.
"""
import math

import numpy as np
import pytest
from scipy import stats


def _philox_words(oracle_lib, seed, h, domain):
    return oracle_lib.philox4x32_10((h & 0xFFFFFFFF, h >> 32, domain, 0), (seed & 0xFFFFFFFF, seed >> 32))


def test_normal_deviates_follow_the_standard_normal(oracle_lib):
    """z_h (Box-Muller, Philox domain 3) against scipy's normal CDF: KS, moments, tails."""
    o = oracle_lib.Oracle(16, T=0.1, seed=99, M=16)
    z = np.array([o.normal_of_hop(h) for h in range(200000)])
    assert stats.kstest(z, "norm").pvalue > 1e-3
    n = z.size
    assert abs(z.mean()) < 5 / math.sqrt(n)
    assert abs(z.var() - 1) < 5 * math.sqrt(2 / n)
    assert abs(stats.skew(z)) < 5 * math.sqrt(6 / n)
    assert abs(stats.kurtosis(z)) < 5 * math.sqrt(24 / n)
    # a dropped factor 2 under the root or cos <-> sin leaves the moments; the tails and
    # independence of consecutive hops would still have to hold
    assert abs((np.abs(z) > 1.959963984540054).mean() - 0.05) < 5 * math.sqrt(0.05 * 0.95 / n)
    assert abs(np.corrcoef(z[:-1], z[1:])[0, 1]) < 5 / math.sqrt(n)


def test_normal_deviate_is_box_muller_of_its_philox_block(oracle_lib):
    """Word use of reading G19, recomputed with Python's math module (independent libm call path)."""
    seed = 0x123456789ABCDEF
    o = oracle_lib.Oracle(16, T=0.1, seed=seed, M=16)
    for h in (0, 1, 77, 2**32 + 5, 2**40 + 123):
        w = _philox_words(oracle_lib, seed, h, 3)
        u1 = ((((w[0] << 32) | w[1]) >> 11) + 1) * 2.0**-53
        u2 = (((w[2] << 32) | w[3]) >> 11) * 2.0**-53
        z = math.sqrt(-2.0 * math.log(u1)) * math.cos(2.0 * math.pi * u2)
        assert o.normal_of_hop(h) == pytest.approx(z, rel=1e-14, abs=1e-15)
    # domain separation: the deviates do not reuse the attempt stream (domain 0)
    w0 = _philox_words(oracle_lib, seed, 0, 0)
    assert tuple(w0) != tuple(_philox_words(oracle_lib, seed, 0, 3))


@pytest.mark.parametrize("A,M", [(0.02, 64), (0.3, 4)])
def test_stochastic_time_has_the_papers_mean_and_variance(oracle_lib, A, M):
    """dt ~ Normal(m/Gamma, sqrt(m)/Gamma).  On the fixed-A chain (state untouched)
    Gamma*(t_stoch - t_det) = sum_h sqrt(m_h) z_h has variance sum_h m_h = attempts; over R
    independent seeds the standardised values must be standard normal."""
    R, hops = 200, 400
    vals = []
    for r in range(R):
        o = oracle_lib.Oracle(16, T=0.1, seed=5000 + r, M=M)
        o.set_fixed_A(A)
        o.run(hops)
        attempts = o.counters()["attempts"]
        t_det = o.state()[2]
        Gamma = o.tables()["Gamma"]
        assert t_det == attempts / Gamma
        vals.append((o.time_stochastic() - t_det) * Gamma / math.sqrt(attempts))
        o.close()
    vals = np.array(vals)
    assert stats.kstest(vals, "norm").pvalue > 1e-3
    assert abs(vals.mean()) < 4 / math.sqrt(R)
    assert abs(vals.var(ddof=1) - 1) < 4 * math.sqrt(2 / (R - 1))


def test_stochastic_time_is_the_hop_ordered_sum_of_gaussian_increments(oracle_lib):
    """t_stoch rebuilt from the hop log: m_h from consecutive attempt indices, z_h from the
    deviate of hop h; physical chain on config 1's lattice."""
    o = oracle_lib.Oracle(16, T=0.1, seed=1, M=256)
    o.run(3000)
    a, _, _ = o.hops()
    ends = a.astype(np.int64) + 1
    m = np.diff(np.concatenate([[0], ends])).astype(np.float64)
    t_det = o.state()[2]
    Gamma = o.counters()["attempts"] / t_det
    z = np.array([o.normal_of_hop(h) for h in range(m.size)])
    t = math.fsum(m / Gamma + np.sqrt(m) / Gamma * z)
    assert o.time_stochastic() == pytest.approx(t, rel=1e-12)
    # the stochastic clock stays within a few standard deviations of the deterministic one
    assert abs(o.time_stochastic() - t_det) * Gamma < 6 * math.sqrt(ends[-1])


def test_dos_matches_numpy_histogram_on_exact_edges(oracle_lib):
    """normalised histogram of eps_k.  With a power-of-two bin width the edges
    lo + b*width are exact, so numpy.histogram (half-open bins) is the same definition."""
    o = oracle_lib.Oracle(64, T=0.05, seed=2, M=1024)
    o.run(500)
    eps = o.state()[1]
    lo, width, nbins = -4.0, 2.0**-4, 128
    hist, outside = o.dos(lo, width, nbins)
    edges = lo + width * np.arange(nbins + 1)
    inside = eps[(eps >= edges[0]) & (eps < edges[-1])]
    ref, _ = np.histogram(inside, bins=edges)
    # numpy closes the last bin on the right; no eps sits exactly on that edge here
    assert not np.any(eps == edges[-1])
    assert np.array_equal(hist.astype(np.int64), ref)
    assert int(hist.sum()) + outside == o.N
    # a narrow window: everything else is reported as outside
    hist2, out2 = o.dos(-0.5, 2.0**-5, 32)
    assert int(hist2.sum()) == int(((eps >= -0.5) & (eps < 0.5)).sum())
    assert out2 == o.N - int(hist2.sum())
    # normalisation of g: sum_b g_b * width = fraction of sites inside
    g = hist / (o.N * width)
    assert g.sum() * width == pytest.approx(1 - outside / o.N, rel=1e-15)


def test_dos_places_edge_values_in_the_upper_bin(oracle_lib):
    """Half-open bins [lo + b*width, lo + (b+1)*width): a value on an edge belongs to the bin it opens."""
    o = oracle_lib.Oracle(16, T=0.1, seed=3, M=16)
    eps = o.state()[1]
    width, checked = 2.0**-3, 0
    for k in range(o.N):
        hist, outside = o.dos(eps[k], width, 1)           # eps_k opens bin 0
        assert int(hist[0]) == int(((eps >= eps[k]) & (eps < eps[k] + width)).sum()) >= 1
        lo = eps[k] - width
        if lo + width == eps[k] and (eps[k] - lo) / width == 1.0:   # eps_k sits exactly on the upper edge
            hist, outside = o.dos(lo, width, 1)
            assert int(hist[0]) == int(((eps >= lo) & (eps < eps[k])).sum())
            hist2, _ = o.dos(lo, width, 2)
            assert int(hist2[1]) >= 1                      # ... and opens bin 1
            checked += 1
    assert checked > 10


def test_polarisation_series_and_sigma0_on_a_scripted_chain(oracle_lib):
    """dP and the series from hops whose dx is known by construction:
    +1 steps along x, a wrap-around step (minimum image), a pure-y hop, a tie at L/2 (-> +L/2, G3)."""
    L = 8
    o = oracle_lib.Oracle(L, T=0.1, E=0.02, seed=4, M=8)
    n = np.zeros(L * L, np.int8)
    n[: L * L // 2] = 1                  # rows 0..3 occupied, rows 4..7 empty
    o.set_state(n, next_attempt=0)
    site = lambda y, x: y * L + x
    # scripted physical hops are only available through apply_hops (no hop log, no attempts),
    # so dP is pinned here and the series below on a physical chain with its hop log
    i = [site(3, 7), site(3, 0), site(2, 5), site(1, 1)]
    j = [site(4, 0), site(4, 1), site(5, 5), site(6, 5)]
    dx = [1, 1, 0, 4]                    # 7->0 wraps to +1; 1->5 is the tie L/2 -> +4
    o.apply_hops(i, j)
    assert o.state()[3] == sum(dx)
    o.close()

    o = oracle_lib.Oracle(16, T=0.1, E=0.01, seed=6, M=32)
    o.run(4000)
    a, hi, hj = o.hops()
    xi, xj = hi.astype(np.int64) % 16, hj.astype(np.int64) % 16
    d = (xj - xi) % 16
    d = np.where(d > 8, d - 16, d)
    t, P = o.series()
    assert np.array_equal(P, np.cumsum(d))
    n_, eps, t_end, dP = o.state()
    assert P[-1] == dP
    Gamma = o.counters()["attempts"] / t_end
    assert np.allclose(t, (a.astype(np.float64) + 1) / Gamma, rtol=1e-15)
    assert np.all(np.diff(t) > 0)
    # a window of the series is the same prefix sum
    t2, P2 = o.series(1000, 50)
    assert np.array_equal(P2, P[1000:1050]) and np.array_equal(t2, t[1000:1050])
    # Eq.(3) / PAPER.md:94: sigma0 = P / (N E t)
    assert o.sigma0() == pytest.approx(dP / (256 * 0.01 * t_end), rel=1e-15)


def test_sigma0_needs_a_field(oracle_lib):
    o = oracle_lib.Oracle(16, T=0.1, E=0.0, seed=1, M=16)
    o.run(10)
    with pytest.raises(Exception):
        o.sigma0()
