"""pytest configuration: marker registration and import paths.

`-m "not gpu"` tests run on a CPU-only box (oracle pins, host logic, C-ABI symbol table);
`-m gpu` tests are the CUDA-vs-oracle parity tests and need a B200.
"""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
for p in (ROOT, os.path.join(ROOT, "oracle")):
    if p not in sys.path:
        sys.path.insert(0, p)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")
