"""pytest configuration: registers the `gpu` marker; makes the repo root importable."""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


# GPU runs use -x: the core parity file goes first, then the rest of the product's paths, the N1(a) experiment last,
# so that a failure in a NEXT-row path cannot hide the verdict on the hot path itself.
_GPU_ORDER = ["test_gpu_parity.py", "test_biased_table.py", "test_spectral.py", "test_tensor_wide.py"]


def pytest_collection_modifyitems(config, items):
    def key(item):
        name = os.path.basename(str(item.fspath))
        if item.get_closest_marker("gpu") is None or name not in _GPU_ORDER:
            return -1
        return _GPU_ORDER.index(name)
    items.sort(key=key)           # stable: CPU tests and the order inside a file are unchanged
