import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on the B200 box)")


@pytest.fixture(scope="session")
def consts():
    from paper_2405_01491_b200 import inputs
    return inputs.ani2x_constants()


@pytest.fixture(scope="session")
def ani_model(consts):
    """Full ANI-2x widths, one random-init net, non-zero biases so CELU's negative branch is exercised."""
    from oracle import nnp_oracle as orc
    from paper_2405_01491_b200 import inputs
    p = inputs.make_weights(inputs.SEED0, 1, bias_std=0.1)
    return orc.OracleModel(consts, inputs.WIDTHS, p, 1)


@pytest.fixture(scope="session")
def small_widths():
    return np.array([[1008, 24, 16, 8, 1]] * 7, dtype=np.int32)


@pytest.fixture(scope="session")
def small_model(consts, small_widths):
    """Same AEV, narrow MLPs: cheap enough for dense finite differences."""
    from oracle import nnp_oracle as orc
    from paper_2405_01491_b200 import inputs
    p = inputs.make_weights(inputs.SEED0 + 1, 1, widths=small_widths, bias_std=0.2)
    return orc.OracleModel(consts, small_widths, p, 1)


@pytest.fixture(scope="session")
def water64():
    from paper_2405_01491_b200 import inputs
    return inputs.water_box(64, 12.42, seed=inputs.SEED0 + 1)
