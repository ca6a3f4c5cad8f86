"""CPU-only checks of the boundary: the CUDA library builds for sm_100a, loads, exports every symbol
include/kf_b200.h declares, and fails loudly without a GPU (no compute calls here)."""
import ctypes as C
import os
import re
import shutil

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "kf_b200.h")


@pytest.fixture(scope="module")
def lib():
    from paper_1705_02876_b200 import build as kbuild
    if not os.path.exists(kbuild.LIB) or kbuild.needs_build():
        if shutil.which("nvcc") is None and not os.path.exists("/usr/local/cuda/bin/nvcc"):
            pytest.skip("no nvcc to build libkf_b200.so")
        kbuild.build()
    from paper_1705_02876_b200.binding import load_library
    return load_library()


def _declared():
    src = open(HEADER).read()
    return re.findall(r"KF_API\s+[\w\s\*]+?\b(kf_\w+)\s*\(", src)


def test_header_declares_the_north_star_calls():
    names = _declared()
    for must in ("kf_fit_tracks", "kf_score_candidates", "kf_bin_hits", "kf_create", "kf_destroy", "kf_strerror"):
        assert must in names
    assert len(names) == len(set(names)) >= 18


def test_library_exports_every_declared_symbol(lib):
    from paper_1705_02876_b200.binding import EXPORTS
    names = _declared()
    assert sorted(names) == sorted(EXPORTS)
    for n in names:
        assert getattr(lib, n) is not None


def test_abi_version_and_error_strings(lib):
    import paper_1705_02876_b200 as K
    assert K.abi_version() == 14
    assert K.binding.hit_record_floats() == 12
    seen = set()
    for code in (0, -1, -2, -3, -4, -5, -6, -7, -99):
        s = K.strerror(code)
        assert isinstance(s, str) and s
        seen.add(s)
    assert len(seen) == 9


def test_null_arguments_are_rejected_without_a_device(lib):
    assert lib.kf_create(None, 0, None) == -1
    assert lib.kf_destroy(None) == -1
    assert lib.kf_fit_tracks(None, None, None, None, None) == -1
    assert lib.kf_fit_tracks_host(None, None, None, None, None) == -1
    assert lib.kf_fit_tracks_host_diag(None, None, None, None, None) == -1
    assert lib.kf_fit_tracks_host_compact(None, None, None, None, None) == -1
    assert lib.kf_fit_tracks_indexed(None, None, None, None, 0, None, None, None) == -1
    assert lib.kf_fit_tracks_refit(None, None, None, None, 10.0, None, None) == -1
    assert lib.kf_fit_tracks_smooth(None, None, None, None, None, None) == -1
    assert lib.kf_bin_hits(None, 1.0, None, None) == -1
    assert lib.kf_score_candidates(None, None, 0, None, None, None, 2, 30.0, 1, None, None, None, None) == -1
    assert lib.kf_score_candidates_static(None, None, 0, None, None, None, 2, 30.0, 1, None, None, None, None) == -1
    assert lib.kf_bin_layers(None, 1, None, None, None) == -1
    assert lib.kf_build_combinatorial(None, None, 0, 1, None, None, None, 2, 30.0, 4, None, None, 0) == -1
    assert lib.kf_build_combinatorial_events(None, None, 0, 1, 1, None, None, None, None, 2, 30.0, 4, None, None, 0) == -1
    assert lib.kf_build_best_hit(None, None, 0, 1, None, None, None, 2, 30.0, 1, None, None, None, 0) == -1
    assert lib.kf_build_best_hit_events(None, None, 0, 1, 1, None, None, None, None, 2, 30.0, 1, None, None, 0) == -1
    assert lib.kf_build_best_hit_host(None, None, 0, 1, None, None, 40, 64, 1.2, 2, 30.0, 1, None, None, 0) == -1
    assert lib.kf_order_candidates(None, None, 0, None, 40, 64, 1.2, None) == -1
    assert lib.kf_measure_fp32_peak(None, 3, None) == -1
    assert lib.kf_last_cuda_error(None) == 0
    assert lib.kf_set_option(None, 1, 0) == -1
    assert lib.kf_graph_begin(None) == -1
    assert lib.kf_graph_end(None, None) == -1
    assert lib.kf_graph_launch(None, None) == -1
    assert lib.kf_graph_destroy(None) == -1


def test_no_cpu_fallback(lib):
    """Without a CUDA device the product path must fail loudly, not compute on the host."""
    import torch
    import paper_1705_02876_b200 as K
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(K.KFError) as e:
        K.KFContext(0)
    assert e.value.code == -5


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1705_02876_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("no CPU or PyTorch fallback", ""), f
    src = open(os.path.join(ROOT, "oracle", "kf_oracle.py")).read() + open(os.path.join(ROOT, "oracle", "kf_oracle.c")).read()
    assert "paper_1705_02876_b200 import" not in src and "kf_b200.h" not in src and "kf_math" not in src
