import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def oracle_lib():
    import oracle
    oracle.build()
    return oracle


def pytest_terminal_summary(terminalreporter):
    """Worst measured residual excess of the GPU parity tests (what the absolute floor of reading D15 has to cover)."""
    mod = sys.modules.get("test_gpu_parity")
    if mod is not None and max(mod.WORST_RES.values()) >= 0:
        terminalreporter.write_line("parity residuals: worst (|dr| - 1e-3 r) / (1 + |u|_inf): "
                                    + ", ".join(f"{k} {v:.2e}" for k, v in mod.WORST_RES.items()) + f" (floor {mod.RES_FLOOR:.1e})")
