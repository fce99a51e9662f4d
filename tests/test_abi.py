"""CPU checks of the boundary: the C-ABI library builds for sm_100a, loads, exports every
symbol include/fredec.h declares, validates arguments and fails loudly without a GPU."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def fr():
    from paper_1309_0100_b200 import build
    build.build()
    import paper_1309_0100_b200 as fr
    fr.lib()
    return fr


def declared_symbols(header):
    """Every function a header under include/ declares."""
    text = re.sub(r"/\*.*?\*/", "", open(os.path.join(ROOT, "include", header)).read(), flags=re.S)
    return sorted(set(re.findall(r"\b(fredec_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_exported_and_bound(fr):
    """fredec.h <-> libfredec_b200.so <-> the binding, name for name; the measurement probes of
    fredec_bench.h live in libfredec_bench.so and the product library does not export them."""
    import subprocess
    from paper_1309_0100_b200 import _binding
    names = declared_symbols("fredec.h")
    assert len(names) >= 14
    L = ctypes.CDLL(_binding.LIB_PATH)
    for n in names:
        assert hasattr(L, n), f"{n} declared in fredec.h but not exported"
        assert n in _binding.SIGNATURES, f"{n} has no ctypes signature in the binding"
    assert sorted(_binding.SIGNATURES) == names
    exported = subprocess.run(["nm", "-D", "--defined-only", _binding.LIB_PATH], capture_output=True, text=True).stdout
    exported = sorted(set(re.findall(r"\b(fredec_[a-z0-9_]+)$", exported, flags=re.M)))
    assert exported == names, "the product library exports exactly what fredec.h declares"
    bench_names = declared_symbols("fredec_bench.h")
    assert sorted(_binding.BENCH_SIGNATURES) == bench_names and len(bench_names) == 2
    B = ctypes.CDLL(_binding.BENCH_LIB_PATH)
    for n in bench_names:
        assert hasattr(B, n) and not hasattr(L, n)
    assert fr.fredec_bench_fp64_name(0) and fr.fredec_bench_fp64_name(10_000) is None


def test_library_targets_sm_100a(fr):
    import subprocess
    from paper_1309_0100_b200 import _binding
    out = subprocess.run(["cuobjdump", "-lelf", _binding.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_no_oracle_or_cpu_fallback_in_product():
    """The product package must not import or call anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_1309_0100_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f
                assert "liboracle" not in text and "oracle_fredec" not in text, f


def test_strerror_and_version(fr):
    L = fr.lib()
    assert fr.fredec_version() >= 100
    for code in (0, -1, -2, -3, -4, -5):
        assert len(L.fredec_strerror(code)) > 0


def test_argument_validation_needs_no_gpu(fr):
    t = np.linspace(0, 10, 20); x = np.sin(t); w = np.ones(20); base = np.ones((1, 20))

    def code(fn):
        with pytest.raises(fr.FredecError) as e:
            fn()
        return e.value.code

    assert code(lambda: fr.fredec_scan(t, x, w, base, 0.1, 0.0, 5)) == fr.FREDEC_EINVAL
    assert code(lambda: fr.fredec_scan(t, x, w, base, -1.0, 0.1, 5)) == fr.FREDEC_EINVAL
    assert code(lambda: fr.fredec_scan(t, x, w, base, 0.1, float("nan"), 5)) == fr.FREDEC_EINVAL
    assert code(lambda: fr.fredec_scan(t, x, w, base, 0.1, 0.1, 0)) == fr.FREDEC_EINVAL
    assert code(lambda: fr.fredec_scan(t[:3], x[:3], w[:3], base[:, :3], 0.1, 0.1, 5)) == fr.FREDEC_EINVAL
    assert code(lambda: fr.fredec_scan(t, x, w, np.ones((65, 20)), 0.1, 0.1, 5)) == fr.FREDEC_EINVAL
    assert code(lambda: fr.fredec_topk(np.zeros(4), 5)) == fr.FREDEC_EINVAL
    assert code(lambda: fr.fredec_topk(np.zeros(4000), 1025)) == fr.FREDEC_EINVAL


def test_noalloc_entry_point_checks_sizes_before_touching_cuda(fr):
    """fredec_topk_noalloc: argument and capacity errors come back without a GPU (and without a CUDA call)."""
    L = fr.lib()
    z = np.zeros(4000); idx = np.zeros(200, dtype=np.int64); cnt = np.zeros(1, dtype=np.int32)
    pz, pi, pc = z.ctypes.data, idx.ctypes.data, cnt.ctypes.data
    assert L.fredec_topk_noalloc(pz, 4000, fr.FREDEC_TOPK_NOALLOC_K_MAX + 1, pi, pc, None) == fr.FREDEC_ELIMIT
    assert L.fredec_topk_noalloc(pz, 4000, 0, pi, pc, None) == fr.FREDEC_EINVAL
    assert L.fredec_topk_noalloc(pz, 4, 5, pi, pc, None) == fr.FREDEC_EINVAL
    assert L.fredec_topk_noalloc(None, 4000, 5, pi, pc, None) == fr.FREDEC_EINVAL
    assert L.fredec_topk_noalloc(pz, 4000, 5, pi, pc, None) in (fr.FREDEC_EINVAL, fr.FREDEC_ECUDA)  # host pointers
    assert b"capacity" in L.fredec_strerror(fr.FREDEC_ELIMIT)


def test_compute_fails_loudly_without_gpu(fr):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    t = np.linspace(0, 10, 20); x = np.sin(t); w = np.ones(20); base = np.ones((1, 20))
    with pytest.raises(fr.FredecError) as e:
        fr.fredec_scan(t, x, w, base, 0.1, 0.1, 5)
    assert e.value.code == fr.FREDEC_ECUDA


def test_missing_library_raises(monkeypatch, tmp_path):
    from paper_1309_0100_b200 import _binding
    monkeypatch.setattr(_binding, "_lib", None)
    monkeypatch.setattr(_binding, "LIB_PATH", str(tmp_path / "nope.so"))
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        _binding.lib()
