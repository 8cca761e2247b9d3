"""CPU-side checks of the C-ABI boundary: the library builds for sm_100a, loads, exports every
symbol include/cg.h declares, validates arguments, and fails loudly without a GPU."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def cg():
    from paper_1407_5026_b200 import build
    build.build()
    import paper_1407_5026_b200 as pkg
    return pkg


def test_every_declared_symbol_is_exported(cg):
    hdr = open(os.path.join(ROOT, "include", "cg.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(cg_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(cg.EXPORTS)
    lib = cg.lib()
    for name in declared:
        assert hasattr(lib, name), name


def test_no_torch_or_cxx_types_in_the_header():
    hdr = open(os.path.join(ROOT, "include", "cg.h")).read()
    assert "torch" not in hdr.lower().replace("a torch uint8 tensor", "") and "std::" not in hdr
    assert 'extern "C"' in hdr


def test_argument_validation_and_loud_failure_without_gpu(cg):
    lib = cg.lib()
    h = C.c_void_p(1)
    assert lib.cg_init(C.byref(h), 15, 1.0, 1.0, 0.1, 0.0, 1, 4) == cg.binding.CG_EINVAL and not h.value
    assert lib.cg_init(C.byref(h), 16, 1.0, 0.0, 0.1, 0.0, 1, 4) == cg.binding.CG_EINVAL
    assert lib.cg_init(C.byref(h), 16, 1.0, 1.0, 0.0, 0.0, 1, 4) == cg.binding.CG_EINVAL
    assert lib.cg_init(C.byref(h), 16, 1.0, 1.0, 0.1, 0.0, 1, 0) == cg.binding.CG_EINVAL
    assert lib.cg_init(C.byref(h), 24, 1.0, 1.0, 0.1, 0.0, 1, 4) == cg.binding.CG_EUNSUPPORTED
    assert lib.cg_init(C.byref(h), 2048, 1.0, 1.0, 0.1, 0.0, 1, 4) == cg.binding.CG_EUNSUPPORTED
    assert lib.cg_init(C.byref(h), 16, 1.0, 1.0, 0.1, 0.0, 1, (1 << 27) + 1) == cg.binding.CG_EUNSUPPORTED
    assert lib.cg_init3(C.byref(h), 128, 1.0, 1.0, 0.1, 0.0, 1, 4) == cg.binding.CG_EUNSUPPORTED and not h.value
    assert lib.cg_init3(C.byref(h), 7, 1.0, 1.0, 0.1, 0.0, 1, 4) == cg.binding.CG_EINVAL
    assert lib.cg_workspace_bytes3(64, 65536) >= 12 * 8 * 64 ** 3 and lib.cg_workspace_bytes3(128, 4) == 0
    assert lib.cg_init(None, 16, 1.0, 1.0, 0.1, 0.0, 1, 4) == cg.binding.CG_EINVAL
    assert lib.cg_run(None, 1) == cg.binding.CG_EINVAL
    assert lib.cg_workspace_bytes(512, 65536) >= 4 * 8 * 512 * 512
    assert lib.cg_workspace_bytes(15, 4) == 0
    assert lib.cg_strerror(cg.binding.CG_EUNSUPPORTED).decode().startswith("problem not supported")
    import torch
    if not torch.cuda.is_available():
        assert lib.cg_init(C.byref(h), 16, 1.0, 1.0, 0.1, 0.0, 1, 4) == cg.binding.CG_ECUDA and not h.value
        with pytest.raises(RuntimeError):
            cg.CoulombGlass(16)


def test_product_path_never_touches_the_oracle():
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_1407_5026_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh")):
                text = open(os.path.join(dirpath, f)).read()
                assert "cgo_" not in text and "import oracle" not in text and "from oracle" not in text, f
    for f in ("cg_oracle.c", "cg_oracle.h", "cgo.py"):
        text = open(os.path.join(ROOT, "oracle", f)).read()
        assert "import paper_1407_5026_b200" not in text and "from paper_1407_5026_b200" not in text
        assert "libcg.so" not in text and '#include "cg.h"' not in text


def test_diagnostic_entry_points_validate_arguments(cg):
    lib = cg.lib()
    assert lib.cg_set_tuning(None, 0, 0) == cg.binding.CG_EINVAL
    assert lib.cg_get_tuning(None, None, None) == cg.binding.CG_EINVAL
    assert lib.cg_get_phase_cycles(None, None, None, None, None, None, 0) == cg.binding.CG_EINVAL
    assert lib.cg_set_launch(None, 0, 0) == cg.binding.CG_EINVAL
    assert lib.cg_get_counters(None, None, None, None, None) == cg.binding.CG_EINVAL
    assert lib.cg_get_exchange_cycles(None, None) == cg.binding.CG_EINVAL
    assert lib.cg_get_labels_per_thread(None, None) == cg.binding.CG_EINVAL
    out = C.c_double()
    assert lib.cg_bench_l2(100, 1, 1, 0, 2, 512, 16, C.byref(out)) == cg.binding.CG_EINVAL       # too small a buffer
    assert lib.cg_bench_l2(1 << 20, 1, 1, 3, 2, 512, 16, C.byref(out)) == cg.binding.CG_EINVAL   # no such mode
    assert lib.cg_bench_l2(1 << 20, 1, 1, 0, 2, 512, 24, C.byref(out)) == cg.binding.CG_EINVAL   # 16 or 32 bytes
    assert lib.cg_strerror(cg.binding.CG_EDEVICE).decode().startswith("the persistent kernel abandoned")


def test_observable_entry_points_validate_arguments(cg):
    """include/cg.h "Observables": a null sim or result pointer is CG_EINVAL, never a crash."""
    lib = cg.lib()
    E = cg.binding.CG_EINVAL
    d, u = C.c_double(), C.c_uint64()
    assert lib.cg_get_time_stochastic(None, C.byref(d)) == E
    assert lib.cg_get_normals(None, 0, 1, None) == E
    assert lib.cg_get_dos(None, 0.0, 1.0, 4, None, C.byref(u)) == E
    assert lib.cg_get_dos_noalloc(None, 0.0, 1.0, 4, None, C.byref(u)) == E
    assert lib.cg_get_series(None, 0, 0, None, None) == E
    assert lib.cg_get_sigma0(None, C.byref(d)) == E
