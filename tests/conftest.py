import os
import sys

import pytest

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def tiny_phantom():
    import vmat_inputs

    return vmat_inputs.make_phantom("tiny", seed=0)


@pytest.fixture(scope="session")
def tiny_oracle(tiny_phantom):
    from oracle import Oracle

    return Oracle.from_phantom(tiny_phantom)


@pytest.fixture(scope="session")
def tiny_solution(tiny_oracle):
    """The oracle's free run on configs[0] (24 beams -> 24 iterations)."""
    return tiny_oracle.solve(40)
