"""oracle.parallel -- the oracle of nk_oracle.py run over element chunks in a process pool.

TEST INFRASTRUCTURE ONLY (same rules as nk_oracle.py: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this).  It adds NO arithmetic: every
chunk is handed, unchanged, to the function of nk_oracle.py that the caller names; elements are
independent, so cutting a block into chunks changes nothing but the wall-clock time.
Workers are spawned (no fork of a process that may hold a CUDA context), import numpy and
nk_oracle only, and keep numpy's own thread pools at one thread each, so that `cores` workers
use `cores` host cores.  Element tables are built once per worker and cached; callers that time
the pool run one warm-up pass first (table construction is not part of the timed work).
"""
import multiprocessing as mp
import os

import numpy as np

_ELS = {}


def cpu_model():
    """model string of the host CPU (for the cpu_baseline record of bench.py)"""
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.lower().startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def _init():
    # one numpy (BLAS / OpenMP) thread per worker
    for k in ("OMP_NUM_THREADS", "OPENBLAS_NUM_THREADS", "MKL_NUM_THREADS"):
        os.environ[k] = "1"
    try:
        from threadpoolctl import threadpool_limits
        threadpool_limits(1)
    except Exception:
        pass


def _element(shape, P, Q):
    from . import nk_oracle as o
    key = (shape, P, Q)
    if key not in _ELS:
        _ELS[key] = o.Element(shape, P, Q)
    return _ELS[key]


def _work(task):
    from . import nk_oracle as o
    op, shape, P, Q, A, J, lam, x, want = task
    el = _element(shape, P, Q)
    if op == "helmholtz":
        y = o.helmholtz(el, A, J, lam, x)
    elif op == "laplacian":
        y = o.laplacian(el, A, J, x)
    elif op == "mass":
        y = o.mass(el, J, x)
    elif op == "bwdtrans":
        y = o.bwdtrans(el, x)
    elif op == "iprod":
        y = o.iprod(el, J, x)
    else:
        raise KeyError(op)
    return y if want else y.shape[0]


class OraclePool:
    """with OraclePool(cores) as pool: y = pool.apply("helmholtz", shape, P, Q, A, J, lam, x)"""

    def __init__(self, cores=None):
        self.cores = cores or os.cpu_count() or 1
        self.pool = None

    def __enter__(self):
        self.pool = mp.get_context("spawn").Pool(self.cores, initializer=_init)
        return self

    def __exit__(self, *exc):
        self.pool.close()
        self.pool.join()
        self.pool = None

    def apply(self, op, shape, P, Q, A, J, lam, x, chunk=None, want_result=True):
        """A [ne][npt][3][3], J [ne][npt], x [ne][...] numpy arrays; returns the oracle's output for all
        elements (want_result) or the number of elements processed."""
        ne = x.shape[0]
        if chunk is None:
            chunk = max(1, -(-ne // (4 * self.cores)))
        tasks = [(op, shape, P, Q, A[s:s + chunk], J[s:s + chunk], lam, x[s:s + chunk], want_result)
                 for s in range(0, ne, chunk)]
        out = self.pool.map(_work, tasks)
        if want_result:
            return np.concatenate(out, axis=0) if out else np.zeros((0,) + x.shape[1:])
        return int(sum(out))
