"""Host-side checks that need no GPU: the C-ABI library loads and exports every symbol that
include/floodped.h declares; argument validation; workspace sizing."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_1908_05232_b200 import binding, build, scenarios as S

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load_library()


def _declared():
    src = open(os.path.join(ROOT, "include", "floodped.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sim_[a-z_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(lib):
    names = _declared()
    assert len(names) >= 15
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(binding.EXPORTS) == names


def test_workspace_bytes_scales_with_problem(lib):
    small = binding.workspace_bytes(S.make(1))
    sc = S.make(1)
    assert small > 64 * 64 * 8 * 9
    sc2 = S.make(1, n=128)
    big = binding.workspace_bytes(sc2)
    assert 3.5 < big / small < 4.5


def test_validation_errors_do_not_need_a_gpu(lib):
    sc = S.make(1)
    m = binding._Marshalled(sc)
    out = C.c_size_t()
    m.grid.real_bits = 16
    assert lib.sim_workspace_bytes(C.byref(m.grid), 0, C.byref(m.params), C.byref(out)) == binding.SIM_EINVAL
    assert b"real_bits" in lib.sim_last_error(None)
    m.grid.real_bits = 64
    m.grid.nx = 0
    assert lib.sim_workspace_bytes(C.byref(m.grid), 0, C.byref(m.params), C.byref(out)) == binding.SIM_EINVAL
    m.grid.nx, m.grid.ny = 65536, 65536                  # nx * ny does not fit the int32 cell index
    assert lib.sim_workspace_bytes(C.byref(m.grid), 0, C.byref(m.params), C.byref(out)) == binding.SIM_EINVAL
    assert b"2^31" in lib.sim_last_error(None)
    m.grid.nx, m.grid.ny = 46340, 46340                  # the largest square that does: sizes only, no allocation
    assert lib.sim_workspace_bytes(C.byref(m.grid), 1000, C.byref(m.params), C.byref(out)) == binding.SIM_OK
    assert out.value > 46340 * 46340 * (6 * 8 + 2 * 8)
    m.grid.nx, m.grid.ny = 64, 64
    m.params.R_int = 0.0
    assert lib.sim_workspace_bytes(C.byref(m.grid), 0, C.byref(m.params), C.byref(out)) == binding.SIM_EINVAL
    # NULL handle is rejected, not dereferenced
    assert lib.sim_step(None, 1) == binding.SIM_EINVAL
    assert lib.sim_get_stats(None, None) == binding.SIM_EINVAL
    lib.sim_destroy(None)


def test_create_fails_loudly_without_a_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    sc = S.make(1)
    m = binding._Marshalled(sc)
    h = C.c_void_p()
    rc = lib.sim_create(C.byref(m.grid), C.byref(m.topo), C.c_void_p(m.manning.ctypes.data), C.byref(m.peds),
                        C.byref(m.params), None, None, C.byref(h))
    assert rc == binding.SIM_ECUDA and not h.value
    assert b"no CPU fallback" in lib.sim_last_error(None)
    with pytest.raises(RuntimeError):
        binding.Sim(sc)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1908_05232_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "floodped_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1908_05232_b200" not in txt and "from paper_1908_05232_b200" not in txt
            assert "floodped.h" not in txt and "csrc" not in txt.replace("(paper_1908_05232_b200/csrc)", "")
