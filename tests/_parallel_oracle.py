"""Test harness only: OraclePIMD with the force loop over the (independent) beads spread over worker processes.

The oracle evaluates one bead of configs[1] in ~0.4 s; 100 steps x 32 beads would take 20 minutes in one process.
The arithmetic is untouched: every bead still goes through oracle.se_e2_a.energy_forces, in a process of its own
(spawned, so no CUDA state of the test process is inherited), and the results are put together exactly as
OraclePIMD._forces does.
"""
import multiprocessing as mp
import os

import numpy as np

from oracle import nm, se_e2_a
from oracle.pimd import OraclePIMD

_W = {}


def _init(desc, weights, types, compressed):
    try:
        import threadpoolctl
        threadpoolctl.threadpool_limits(1)
    except ImportError:
        pass
    model = se_e2_a.Model(desc, weights)
    if compressed:
        from oracle import compress
        compress.compress(model)
    _W["model"] = model
    _W["types"] = types


def _bead(args):
    xk, box = args
    E, F, Xi = se_e2_a.energy_forces(xk, _W["types"], box, _W["model"])
    return E.sum(), F, Xi


class ParallelOraclePIMD(OraclePIMD):
    def __init__(self, *a, workers=None, **kw):
        super().__init__(*a, **kw)
        self._pool = None
        self._workers = workers or min(16, os.cpu_count() or 1)

    def set_model(self, desc, weights, compressed=False):
        self.close()
        self._pool = mp.get_context("spawn").Pool(self._workers, initializer=_init,
                                                  initargs=(desc, np.asarray(weights), self.types, compressed))
        super().set_model(desc, weights, compressed=compressed)

    def _forces(self):
        if self._pool is None or self.k_spring is not None:
            return super()._forces()
        res = self._pool.map(_bead, [(self.x[k], self.box) for k in range(self.P)])
        f = np.zeros((self.P, self.N, 3))
        for k, (U, F, Xi) in enumerate(res):
            f[k] = F
            self.U[k] = U
            self.Xi[k] = Xi
        self.f = f
        self.ft = nm.to_nm(self.M, f)

    def close(self):
        if self._pool is not None:
            self._pool.terminate()
            self._pool = None
