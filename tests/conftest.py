import os
import sys
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


@pytest.fixture(scope="session")
def swift_mat():
    """Material of BASELINE.json configs: E=70 GPa, nu=0.33, Lankford (0.7,0.6,0.8), Swift (500,0.01,0.2)."""
    import oracle
    r = oracle.hill_from_lankford(0.7, 0.6, 0.8)
    return oracle.mat_record(70000.0, 0.33, r, 1, 500.0, 0.01, 0.2)


@pytest.fixture(scope="session")
def voce_mat3():
    """PAPER.md:493-495 Table 3 (nu=0.3 assumed, reading G6): E=219 GPa, Q=410, b=3.8, sigma0=138,
    r11..r23 = 1.5449,1.0666,1,1.0307,(r13=1),(r23=1)."""
    import oracle
    return oracle.mat_record(219000.0, 0.3, [1.5449, 1.0666, 1.0, 1.0307, 1.0, 1.0], 0, 138.0, 410.0, 3.8)
