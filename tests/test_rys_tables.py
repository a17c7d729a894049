"""CPU checks of the Rys quadrature tables the f-class kernels read (csrc/gen/gen_rys.py -> generated/rys_tables.bin).

The defining property of the N-point rule is  sum_i w_i u_i^k = F_k(T), k = 0..2N-1  (Dupuis-Rys-King; header of
csrc/adft_rys.cuh).  The moments are checked against the oracle's Boys function, which shares nothing with the table
generator (mpmath) or the device code; the table is evaluated exactly the way the kernel does (Clenshaw in fp64)."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, os.path.join(ROOT, "paper_2406_11185_b200", "csrc", "gen"))


@pytest.fixture(scope="module")
def tab():
    from paper_2406_11185_b200 import build
    import gen_rys
    build.generate_rys_tables()
    return gen_rys.read_blob(os.path.join(build.GEN, "rys_tables.bin"))


@pytest.mark.parametrize("N", range(1, 10))
def test_moments_match_oracle_boys(tab, N):
    import gen_rys
    import oracle
    rng = np.random.default_rng(100 + N)
    Ts = np.concatenate([[0.0, 1e-9, 0.5, 1.0, 79.999, 80.0, 80.001, 150.0, 1e4], rng.uniform(0, 100, 60),
                         np.arange(0, 81, 1.0) + 1e-12])
    for T in Ts:
        u, w = gen_rys.eval_table(tab, N, float(T))
        assert all(0.0 < x < 1.0 for x in u) and all(x > 0 for x in w)
        assert all(u[i] < u[i + 1] for i in range(N - 1))
        F = oracle.boys_ld(2 * N - 1, float(T))
        for k in range(2 * N):
            m = sum(wi * ui ** k for ui, wi in zip(u, w))
            assert abs(m - F[k]) <= 2e-14 * F[0], (N, T, k, m, F[k])


def test_table_header(tab):
    assert tab["nmax"] == 9 and tab["tmax"] == 80.0 and tab["h"] == 1.0 and tab["ncoef"] == 16
