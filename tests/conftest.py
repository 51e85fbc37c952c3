import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    config.addinivalue_line("markers", "slow: long statistical run (still CPU-only)")


@pytest.fixture(scope="session")
def olib():
    import oracle
    return oracle.lib()


def build_mutant_oracle(tmp_path, name, old, new):
    """The oracle source with ONE textual substitution, compiled to a throw-away shared object (never the library the
    parity tests use) and given the oracle's ctypes signatures.  Pins use it to show that they catch a wrong reading:
    the mutation lives in the test, not as a "be wrong" switch inside the oracle."""
    import ctypes as C
    import subprocess
    import oracle
    from oracle import binding
    src = open(os.path.join(os.path.dirname(oracle.__file__), "hpmc_oracle.cpp")).read()
    assert src.count(old) == 1, (name, src.count(old))
    cpp, so = str(tmp_path / ("m_%s.cpp" % name)), str(tmp_path / ("m_%s.so" % name))
    with open(cpp, "w") as f:
        f.write(src.replace(old, new))
    subprocess.run(["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC",
                    "-o", so, cpp], check=True)
    return binding.apply_signatures(C.CDLL(so))
