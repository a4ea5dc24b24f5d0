"""bench.py's CPU legs: the slab form of the oracle step computes what the whole-lattice oracle calls compute."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def test_oracle_step_on_a_slab_matches_the_whole_lattice_operators(orc):
    import bench
    L, m0 = (6, 4, 4, 4), -0.2
    w = bench.OracleStep(L, m0)
    want = orc.dirac_eo(L, 0, m0, w.U, w.psi)
    for npl in (1, 3, 5):
        w.run(npl, 2)                      # leaves Dhat on the slab in w.out
        n = npl * w.s0
        assert np.abs(w.out[:n] - want[:n]).max() <= 1e-13
    # byte model of the step: the sum of the four operators' compulsory bytes (fp64, compressed links)
    V = 6 * 4 * 4 * 4
    assert w.bytes(L[0]) == V / 2 * 512 + V / 2 * 512 + V * 384 + V / 2 * 1152
    assert bench.workload_config(L) == bench.workload_config(L) and "lattice" in bench.workload_config(L)
