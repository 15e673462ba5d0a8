import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


# The plane lists of the clearance grid are made by the first run of >= 2e7 histories after a build; the GPU tests run
# fewer, so they ask for the lists from the first run on: every parity test then goes through them.
os.environ.setdefault("GADEP_LIST_MIN_HISTORIES", "0")


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on the B200 box)")
