"""Pins for oracle step O1/O7 (Philox4x32-10 and the word -> (i, u_d, u_a) mapping).

PAPER.md:86, 138 (ref [9]): "Philox from Random123"; "3M random numbers (to choose i_k,
r_ikjk, and to accept the hops)".  The pin is cuRAND's own curand_Philox4x32_10 (an
independent library routine, host path of curand_philox4x32_x.h).
"""
import numpy as np
import pytest
from scipy import stats

from helpers import curand_ref


@pytest.mark.skipif(not curand_ref.available(), reason="nvcc not found")
def test_philox_matches_curand(oracle_lib):
    rng = np.random.default_rng(20140718)
    n = 100000
    ctr = rng.integers(0, 2**32, size=(n, 4), dtype=np.uint64).astype(np.uint32)
    key = rng.integers(0, 2**32, size=(n, 2), dtype=np.uint64).astype(np.uint32)
    # structured corner cases: zeros, all ones, small counters as the oracle uses them
    ctr[0] = 0; key[0] = 0
    ctr[1] = 0xFFFFFFFF; key[1] = 0xFFFFFFFF
    for t in range(2, 1000):
        ctr[t] = (t, 0, t % 3, 0)
        key[t] = (t % 7, 0)
    ref = curand_ref.philox_batch(ctr, key)
    for t in range(n):
        got = oracle_lib.philox4x32_10(ctr[t], key[t])
        assert got == tuple(int(x) for x in ref[t]), (t, ctr[t], key[t])


@pytest.mark.skipif(not curand_ref.available(), reason="nvcc not found")
def test_attempt_decode_uses_counter_a_domain0_and_all_128_bits(oracle_lib):
    """O7: counter = (a_lo, a_hi, 0, 0), key = seed; i = (w0*N)>>32, u_d = 43 bits of
    (w1, top 11 of w2), u_a = 53 bits of (low 21 of w2, w3)."""
    seed = 0x123456789ABCDEF
    o = oracle_lib.Oracle(16, T=0.1, seed=seed, M=4)
    tab = o.tables()
    a_list = [0, 1, 2, 12345, 2**32 - 1, 2**32, 2**40 + 17]
    ctr = np.array([[a & 0xFFFFFFFF, a >> 32, 0, 0] for a in a_list], np.uint32)
    key = np.array([[seed & 0xFFFFFFFF, seed >> 32]] * len(a_list), np.uint32)
    w = curand_ref.philox_batch(ctr, key).astype(np.uint64)
    for t, a in enumerate(a_list):
        i, j, k, ud, ua = o.decode_attempt(a)
        w0, w1, w2, w3 = (int(x) for x in w[t])
        assert i == (w0 * o.N) >> 32
        assert ud == ((w1 << 11) | (w2 >> 21)) / 2.0**43
        assert ua == (((w2 & 0x1FFFFF) << 32) | w3) / 2.0**53
        assert 0.0 <= ud < 1.0 and 0.0 <= ua < 1.0
        # tower: smallest k with u_d < cdf_k
        assert k == int(np.searchsorted(tab["cdf"], ud, side="right"))
        yi, xi = divmod(i, 16)
        assert j == ((yi + int(tab["dy"][k])) % 16) * 16 + (xi + int(tab["dx"][k])) % 16


def test_site_and_displacement_frequencies_match_proposal_matrix(oracle_lib):
    """Q = Gamma^T_ij / Gamma: i uniform over N sites, displacement k with
    probability w_k / S.  chi^2 against those closed forms on L=4 (K=10) and L=16 (K=194)."""
    for L, n in ((4, 200000), (16, 400000)):
        o = oracle_lib.Oracle(L, T=0.5, seed=99 + L, M=1)
        K = o.tables()["K"]
        dec = [o.decode_attempt(a) for a in range(n)]
        ci = np.bincount([d[0] for d in dec], minlength=o.N)
        ck = np.bincount([d[2] for d in dec], minlength=K).astype(float)
        assert stats.chisquare(ci).pvalue > 1e-4
        # expected displacement probabilities from the definition, independently of the oracle
        h = L // 2
        disp = sorted((dy * dy + dx * dx, dy, dx) for dy in range(-h + 1, h + 1)
                      for dx in range(-h + 1, h + 1) if 0 < dy * dy + dx * dx <= h * h)
        assert len(disp) == K
        wk = np.array([np.exp(-2.0 * np.sqrt(r2)) for r2, _, _ in disp])
        pk = wk / wk.sum()
        keep = pk * n >= 5.0                      # merge the far tail into one bin
        obs = np.append(ck[keep], ck[~keep].sum())
        exp = np.append(pk[keep], pk[~keep].sum()) * n
        if exp[-1] == 0:
            obs, exp = obs[:-1], exp[:-1]
        assert stats.chisquare(obs, exp * obs.sum() / exp.sum()).pvalue > 1e-4
        # acceptance uniform: mean 1/2, variance 1/12
        ua = np.array([d[4] for d in dec])
        assert abs(ua.mean() - 0.5) < 5 * np.sqrt(1 / 12 / n)
        assert abs(ua.var() - 1 / 12) < 5 * np.sqrt(1 / 180 / n)
