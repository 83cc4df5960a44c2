import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def tiny_cfg():
    """A 6x4x8 grid in a skewed cell: small enough for brute force, anisotropic enough to catch
    transposed axes, with ragged sizes (5 unocc, 3+2 projectors are set by the tests)."""
    import numpy as np
    from paper_1307_8052_b200 import workload as W
    cell = np.array([[5.0, 0.3, 0.0], [-0.7, 4.2, 0.2], [0.1, -0.4, 6.1]])
    return W.custom_config(100, cell, (6, 4, 8), (0.25, -0.125, 0.5), n_occ=2, n_unocc=5, ng_target=20,
                           n_omega=3, n_atoms=2, n_proj_per_atom=3, orb_ecut_ha=3.0)
