import os, sys
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    # the multi-process oracle helpers fork after torch started its threads; the children only run the C oracle
    config.addinivalue_line("filterwarnings", "ignore:.*multi-threaded.*fork.*:DeprecationWarning")
