"""Host-side checks of the C-ABI library (no GPU): it builds for sm_100a, exports every symbol
include/glisse.h declares, and fails loudly — never falls back to a CPU path — without a device."""
import ctypes
import os
import re
import subprocess

import numpy as np
import pytest

from paper_2011_03484_b200 import build as cuda_build
from paper_2011_03484_b200 import inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    return cuda_build.build()


def _declared_symbols(header):
    src = open(os.path.join(ROOT, "include", header)).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(glisse_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(libpath):
    """include/glisse.h (the interface) and include/glisse_test.h (measurement / test hooks)."""
    from paper_2011_03484_b200 import binding
    declared = _declared_symbols("glisse.h")
    hooks = _declared_symbols("glisse_test.h")
    assert len(declared) >= 20 and len(hooks) >= 5 and not set(declared) & set(hooks)
    assert sorted(binding.EXPORTS) == declared       # the binding mirrors the headers, name for name
    assert sorted(binding.TEST_EXPORTS) == hooks
    L = ctypes.CDLL(libpath)
    for name in declared + hooks:
        assert hasattr(L, name), name


def test_library_is_sm100a_and_uses_bulk_async_copies(libpath):
    """cuobjdump: the particle kernel is compiled for sm_100a and stages the planet log with
    cp.async.bulk (SASS UBLKCP) on an mbarrier (SYNCS) — B200_PROFILING.md's evidence table."""
    out = subprocess.run(["cuobjdump", "-sass", libpath], capture_output=True, text=True, check=True).stdout
    assert "sm_100a" in out
    assert "UBLKCP" in out and "SYNCS" in out
    assert "DFMA" in out and "MUFU.RSQ64H" in out


def test_host_only_entry_points(libpath):
    L = ctypes.CDLL(libpath)
    L.glisse_log_stride.restype = ctypes.c_int
    assert [L.glisse_log_stride(k) for k in (0, 1, 4, 8, 32)] == [4, 6, 16, 28, 100]
    assert L.glisse_log_stride(-1) == 0 and L.glisse_log_stride(33) == 0
    L.glisse_strerror.restype = ctypes.c_char_p
    assert L.glisse_strerror(0) == b"ok" and b"planet" in L.glisse_strerror(-4)
    from paper_2011_03484_b200 import binding
    p = binding.GlisseParams()
    L.glisse_default_params(ctypes.byref(p))
    assert (p.kepler_iters, p.kepler_tol, p.chunk_steps, p.resync_chunks) == (5, 1e-14, 1024, 1)
    assert (p.snapshot_chunks, p.resonance_chunks, p.bin_iterations, p.scheme, p.guess_order, p.segment_steps) == (
        0, 0, 2, 0, 0, 128)
    assert p.r_min == 0.0 and p.r_max == float("inf")


def test_no_cpu_fallback_without_a_device():
    """Without a CUDA device the product path must fail loudly (GLISSE_ECUDA), not compute."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2011_03484_b200 import binding
    w = inputs.config(1).subset(4)
    with pytest.raises(binding.GlisseError) as ei:
        binding.GlisseSim.from_workload(w)
    assert ei.value.status == binding.ECUDA
    with pytest.raises(binding.GlisseError):
        binding.fp64_peak_probe()


def test_product_never_imports_the_oracle():
    """The oracle is test infrastructure: nothing under the package or bench's product arm imports it."""
    pkg = os.path.join(ROOT, "paper_2011_03484_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".inc")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt, f
                assert "glisse_oracle" not in txt, f
    cpp = open(os.path.join(ROOT, "oracle", "glisse_oracle.cpp")).read()
    assert not re.search(r'#include\s*"', cpp)          # system headers only: no shared header
    py = open(os.path.join(ROOT, "oracle", "__init__.py")).read()
    assert not re.search(r"^\s*(import|from)\s+paper_2011_03484_b200", py, flags=re.M)
