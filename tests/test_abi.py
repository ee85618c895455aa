"""The C-ABI library loads on a CPU-only box and exports every symbol include/pinmpc.h declares.
No compute call is made here (no GPU)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2606_05687_b200 import build
    build.build()
    from paper_2606_05687_b200 import binding
    return binding.load()


def _declared():
    src = open(os.path.join(ROOT, "include", "pinmpc.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(pinmpc_[a-z_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    names = _declared()
    assert len(names) >= 15 and "pinmpc_solve" in names and "pinmpc_get" in names
    for n in names:
        assert hasattr(lib, n), n
    from paper_2606_05687_b200 import binding
    assert sorted(binding.EXPORTS) == names


def test_host_only_entry_points_without_a_gpu(lib):
    from paper_2606_05687_b200 import binding
    lay = binding.make_layout()
    base = binding.pinmpc_workspace_bytes(13, 12, 50, 4096, lay)
    dense = binding.pinmpc_workspace_bytes(13, 12, 50, 4096, lay, binding.METHOD_DENSE)
    st = 4096 * 50
    # outputs x,u,z,y (13 + 36 floats per stage) + the structured solver's factors (178 per stage + q_0) + the chunk
    # operators of the chunked iteration kernel (ceil(N / 5) - 2 = 8 matrices of 144 floats per env)
    per_stage = (13 + 36) + (72 + 12 + 6 + 2 + 24 + 28 + 32)
    lo = (st * per_stage + 4096 * 12 + 4096 * 8 * 144) * 4
    assert base >= lo and base < lo + 20 * 256 + 3 * 4096 * 4
    assert dense > base + st * (169 + 156 + 156 + 144) * 4
    assert binding.pinmpc_workspace_bytes(12, 12, 50, 64, lay) == 0          # nx must be 13
    assert binding.pinmpc_workspace_bytes(13, 14, 50, 64, lay) == 0          # nu must match the layout
    assert binding.pinmpc_workspace_bytes(13, 12, 513, 64, lay) == 0         # N_MAX
    assert binding.pinmpc_workspace_bytes(13, 12, 10, 0, lay) == 0           # empty batch
    assert binding.pinmpc_workspace_bytes(13, 12, 0, 4, lay) == 0            # empty horizon
    assert binding.pinmpc_workspace_bytes(13, 18, 30, 64, binding.make_layout(2, 2)) > 0
    # create must refuse bad arguments before touching the device
    h = ctypes.c_void_p()
    st_ = lib.pinmpc_create(ctypes.byref(h), 13, 12, 10, 4, ctypes.byref(lay), 1.0, 10, None, 0)
    assert st_ == binding.EINVAL and not h.value
    assert b"workspace" in lib.pinmpc_last_error(None)
    st_ = lib.pinmpc_create(ctypes.byref(h), 13, 12, 10, 4, ctypes.byref(lay), -1.0, 10, ctypes.c_void_p(256), 1 << 20)
    assert st_ == binding.EINVAL
    assert lib.pinmpc_solve(None, None) == binding.EINVAL
    lib.pinmpc_destroy(None)


def test_product_path_does_not_import_the_oracle():
    """The CUDA package must never route through oracle/ (no CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2606_05687_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "pinmpc_oracle" not in txt, f
    orc = open(os.path.join(ROOT, "oracle", "__init__.py")).read() + open(os.path.join(ROOT, "oracle", "pinmpc_oracle.c")).read()
    assert not re.search(r"^\s*(import|from)\s+paper_2606_05687_b200", orc, flags=re.M)
    assert "pinmpc_common" not in orc and '#include "pinmpc.h"' not in orc
