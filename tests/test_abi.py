"""CPU-side checks of the C-ABI library: it builds, loads and exports every symbol that
include/gtb.h declares; argument validation that needs no GPU; the product never touches oracle/."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from conftest import ROOT
from paper_2509_06525_b200 import binding as gtb
from paper_2509_06525_b200 import build as gtb_build


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "gtb.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gtb_[a-z0-9_]+)\s*\(", text)))


def test_library_builds_for_sm_100a_and_exports_every_declared_symbol():
    path = gtb_build.build()
    assert os.path.exists(path)
    lib = C.CDLL(path)
    declared = _declared_symbols()
    assert len(declared) >= 15
    for name in declared:
        assert hasattr(lib, name), name
    assert sorted(gtb.EXPORTS) == declared
    assert "arch=compute_100a,code=sm_100a" in gtb_build.NVCC_FLAGS
    assert "-lineinfo" in gtb_build.NVCC_FLAGS


def test_status_strings_and_version():
    assert gtb.status_string(0) == "ok"
    for st in range(-9, 0):
        assert gtb.status_string(st) not in ("ok", "unknown status")
    assert gtb.status_string(-99) == "unknown status"
    assert gtb.version() >= 100
    assert gtb.launch_count() >= 0


def test_workspace_queries_scale_linearly():
    n = 1_000_000
    assert gtb.build_workspace_bytes(n) >= 40 * n
    assert gtb.build_workspace_bytes(2 * n) < 2.2 * gtb.build_workspace_bytes(n)
    w = gtb.kpm_workspace_bytes(n, 3000, 8)
    assert w >= 2 * n * 8 * 16                      # two vector sets
    assert w < 2 * n * 8 * 16 + 64 * 2**20          # + partial sums only
    assert gtb.kpm_workspace_bytes(0, 10, 1) == 0


def test_argument_validation_needs_no_gpu():
    lib = gtb.lib()
    box = np.array([10.0, 10.0, 10.0])
    pbc = np.array([1, 1, 0], dtype=np.int32)
    width = C.c_int32(-1)
    fake = C.c_void_p(256)   # never dereferenced: validation fails first

    def nw(n, box, cutoff, pos=fake, wout=C.byref(width)):
        return lib.gtb_neighbor_width(pos, C.c_int64(n), C.c_void_p(box.ctypes.data),
                                      C.c_void_p(pbc.ctypes.data), C.c_double(cutoff), None, fake,
                                      C.c_size_t(0), None, wout)

    assert nw(10, box, -1.0) == gtb.ERR_INVALID_ARG
    assert nw(10, box, 6.0) == gtb.ERR_BOX_TOO_SMALL           # 10 < 2*6
    assert nw(2**31, box, 1.0) == gtb.ERR_INDEX_RANGE
    assert nw(10, box, 1.0) == gtb.ERR_WORKSPACE                # ws_bytes = 0
    assert nw(0, box, 1.0) == gtb.OK and width.value == 0       # empty input
    assert nw(10, box, 1.0, pos=None) == gtb.ERR_INVALID_ARG

    ell = gtb._Ell(100, 3, 256, 256, None)
    mu = C.c_void_p(256)
    def km(a=8.5, M=16, R=2, Rb=2, mode=0, ws_bytes=0, opt=None):
        return lib.gtb_kpm_moments(C.byref(ell), C.c_double(a), C.c_double(0.0), C.c_int32(M),
                                   C.c_int32(R), C.c_int32(Rb), C.c_uint64(1), C.c_int32(mode), mu,
                                   fake, C.c_size_t(ws_bytes), None, opt)
    assert km(a=0.0) == gtb.ERR_INVALID_ARG
    assert km(M=0) == gtb.ERR_INVALID_ARG
    assert km(R=0) == gtb.ERR_INVALID_ARG
    assert km(Rb=65) == gtb.ERR_INVALID_ARG
    assert km(mode=2) == gtb.ERR_INVALID_ARG
    assert km() == gtb.ERR_WORKSPACE
    assert km(mode=gtb.MODE_ORB4 | gtb.MODE_ORB9) == gtb.ERR_INVALID_ARG
    for bad in (gtb.options(kernel=9), gtb.options(tile_stages=9), gtb.options(flags=1 << 20)):
        assert km(opt=C.byref(bad)) == gtb.ERR_INVALID_ARG
    half = gtb.options()
    half.loop_begin = 256                                       # an event pair must be complete
    assert km(opt=C.byref(half)) == gtb.ERR_INVALID_ARG
    assert km(opt=C.byref(gtb.options(kernel=gtb.KERNEL_ROW))) == gtb.ERR_WORKSPACE
    assert lib.gtb_dos(None, 4, C.c_double(1.0), C.c_double(0.0), 1, None, 4, C.c_double(1.0),
                       None, None) == gtb.ERR_INVALID_ARG


def test_library_does_not_read_the_environment():
    """Kernel selection goes through gtb_kpm_options (include/gtb.h), never through getenv (the
    statically linked CUDA runtime imports getenv itself, so the sources are what is checked)."""
    csrc = os.path.join(ROOT, "paper_2509_06525_b200", "csrc")
    for f in os.listdir(csrc):
        if f.endswith((".cu", ".cuh")):
            text = open(os.path.join(csrc, f)).read()
            assert "getenv" not in text and "environ" not in text, f


def test_product_does_not_reach_the_oracle():
    # the oracle is test infrastructure: nothing under the package may import, load or name it
    pkg = os.path.join(ROOT, "paper_2509_06525_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "libgtbo" not in text and "gtbo_" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".h")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "libgtb_kpm" not in text and "paper_2509_06525_b200.binding" not in text, f


@pytest.mark.skipif(__import__("torch").cuda.is_available(), reason="only meaningful without a GPU")
def test_compute_calls_fail_loudly_without_a_gpu():
    import torch
    with pytest.raises((TypeError, RuntimeError, AssertionError)):
        gtb.random_phase_fill(1, 0, 2, 16, device="cuda")
    with pytest.raises(TypeError):
        gtb.dos(torch.zeros(4, dtype=torch.float64), 1.0, 0.0, torch.zeros(4, dtype=torch.float64))
