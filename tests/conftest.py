"""pytest configuration: registers the `gpu` marker and provides shared fixtures.

`-m "not gpu"` tests pin the CPU oracle against what the paper and the
mathematics fix, check host logic, and check that the C-ABI library loads and
exports every symbol include/qlga.h declares.  `-m gpu` tests are the parity
tests proper (CUDA path vs oracle through the C-ABI)."""
import json
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
GOLDEN = os.path.join(ROOT, "tests", "golden")


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


@pytest.fixture(scope="session")
def oracle():
    from oracle.qlga_oracle import Oracle
    return Oracle("double")


@pytest.fixture(scope="session")
def oracle_ld():
    from oracle.qlga_oracle import Oracle
    return Oracle("longdouble")


def load_golden(name):
    with open(os.path.join(GOLDEN, name)) as f:
        return json.load(f)


def eval_expr(expr, **names):
    """Evaluate an arithmetic expression string from a golden fixture."""
    ns = {"sqrt": np.sqrt, "__builtins__": {}}
    ns.update(names)
    return float(eval(expr, ns))  # noqa: S307 - fixtures are repo files


def table1_coeffs(row, E, couplings, free=(0.03, 0.02)):
    g0, g1, g2 = couplings
    exprs = load_golden("table1.json")["rows"][str(row)]
    return np.array([eval_expr(e, E=E, g0=g0, g1=g1, g2=g2, c2f=free[0], c1f=free[1])
                     for e in exprs])


def rel_l2(a, b):
    a = np.asarray(a); b = np.asarray(b)
    return float(np.sqrt(np.sum(np.abs(a - b) ** 2) / np.sum(np.abs(b) ** 2)))


def norm2(q):
    return float(np.sum(np.abs(np.asarray(q, dtype=np.clongdouble)) ** 2))
