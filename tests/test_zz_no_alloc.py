"""cg_get_dos_noalloc (include/cg.h): the density-of-states pass with its scratch bins in a static
device array of the library instead of a cudaMalloc'ed buffer, for callers that must not allocate.

Collected last on purpose (the suite runs with pytest -x): the file name sorts after every other
test file.  Checked against the existing path cg_get_dos — bin counts are integers, so the bar is
bit-exact, the same as tests/test_gpu_observables.py uses for the DOS — on two calls in a row
(the static array keeps the first call's counts; the second call must not see them).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _glass(**kw):
    import paper_1407_5026_b200 as pkg
    return pkg.CoulombGlass(**kw)


def test_dos_noalloc_matches_dos_on_two_calls_in_a_row():
    g = _glass(L=64, W=1.0, xi=1.0, T=0.05, E=0.01, seed=21, M=1024)
    g.run(3000)
    # first call: wide bins; second call, straight after it: fewer, narrower bins on another window,
    # so stale counts of the first call would show up both inside and beyond the second call's bins
    first = (-4.0, 2.0 ** -4, 128)
    second = (-1.0, 2.0 ** -6, 96)
    for lo, width, nbins in (first, second):
        h_ref, out_ref = g.dos(lo, width, nbins)
        h_new, out_new = g.dos_noalloc(lo, width, nbins)
        assert h_new.dtype == np.uint64 and h_new.shape == (nbins,)
        assert np.array_equal(h_new, h_ref)
        assert out_new == out_ref
        assert int(h_new.sum()) + out_new == g.N
    # and once more with the first shape: a repeat of an earlier call gives the same counts again
    h_ref, out_ref = g.dos(*first)
    h_new, out_new = g.dos_noalloc(*first)
    assert np.array_equal(h_new, h_ref) and out_new == out_ref


def test_dos_noalloc_largest_size_and_the_limit():
    import paper_1407_5026_b200 as pkg
    g = _glass(L=32, W=1.0, xi=1.0, T=0.1, E=0.0, seed=22, M=512)
    g.run(500)
    limit = 8192                                    # CG_DOS_NOALLOC_MAX_BINS (include/cg.h)
    h_ref, out_ref = g.dos(-8.0, 2.0 ** -9, limit)
    h_new, out_new = g.dos_noalloc(-8.0, 2.0 ** -9, limit)
    assert np.array_equal(h_new, h_ref) and out_new == out_ref
    # a second sim on the same GPU shares the array: its call straight after sees none of the above
    g2 = _glass(L=16, W=1.0, xi=1.0, T=0.1, E=0.0, seed=23, M=256)
    h2_ref, o2_ref = g2.dos(-8.0, 2.0 ** -9, limit)
    h2_new, o2_new = g2.dos_noalloc(-8.0, 2.0 ** -9, limit)
    assert np.array_equal(h2_new, h2_ref) and o2_new == o2_ref and int(h2_new.sum()) + o2_new == 256
    # beyond the static scratch: a clear refusal, nothing written
    hist = np.full(limit + 1, 7, np.uint64)
    with pytest.raises(pkg.CgError) as e:
        g.dos_noalloc(-8.0, 2.0 ** -9, limit + 1, hist=hist)
    assert e.value.code == -1                       # CG_EINVAL
    assert b"8192" in g._lib.cg_last_error(g._h)
    assert np.all(hist == 7)
    with pytest.raises(pkg.CgError):
        g.dos_noalloc(0.0, 0.0, 16)                 # width must be positive, as for cg_get_dos
