"""The process-parallel oracle wrapper of tests/_parallel_oracle.py gives bit for bit the serial oracle's trajectory
(it only distributes the independent bead evaluations of OraclePIMD._forces)."""
import numpy as np

import workloads
from oracle.pimd import OraclePIMD
from _parallel_oracle import ParallelOraclePIMD


def test_parallel_oracle_equals_serial_oracle_bitwise():
    cfg, wb, desc, w = workloads.make_config(0)
    args = (wb["types"], wb["masses"], wb["box"], cfg["P"], cfg["T"], cfg["dt"], cfg["gamma"])
    a = OraclePIMD(*args, seed=3)
    a.set_state(wb["x"], wb["p"])
    a.set_model(desc, w)
    b = ParallelOraclePIMD(*args, seed=3, workers=2)
    b.set_state(wb["x"], wb["p"])
    b.set_model(desc, w)
    try:
        a.step(2)
        b.step(2)
        assert np.array_equal(a.positions(), b.positions()) and np.array_equal(a.momenta(), b.momenta())
        assert np.array_equal(a.forces(), b.forces()) and np.array_equal(a.virial(), b.virial())
        ea, eb = a.estimators(), b.estimators()
        assert all(np.array_equal(ea[key], eb[key]) for key in ea)
    finally:
        b.close()
