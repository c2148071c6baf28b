import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

GOLDEN = os.path.join(ROOT, "tests", "golden")


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def read_golden(name):
    """Parse a tests/golden/*.txt fixture: '#' comments, 'key: value' lines -> dict of str."""
    out = {}
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if not line:
                continue
            k, val = line.split(":", 1)
            out[k.strip()] = val.strip()
    return out


@pytest.fixture(scope="session")
def golden():
    return read_golden


# ---------------------------------------------------------------------------------------------------
# Long oracle trajectories for the full-length GPU parity runs (C1-C3 3600 steps, C4 600).
# The oracle is single-threaded C called through ctypes (the GIL is released during a call), so
# independent trajectories -- different configs, different storage layouts -- are advanced by a small thread
# pool while the GPU side of another test runs.  This is orchestration only: each trajectory is the
# oracle as it stands, `[remove_zero; step]` in a loop, with snapshots at the requested steps.
# ---------------------------------------------------------------------------------------------------
class OracleTrajectory:
    """Future of one oracle run: snapshots[k] = state after `checkpoints[k]` steps (xi, v, cell_id, idx and
    cell_start of the LAST of those steps, events so far)."""

    def __init__(self, pool, w, checkpoints):
        self.w, self.checkpoints = w, list(checkpoints)
        self.future = pool.submit(self._run)

    def _run(self):
        import oracle
        w = self.w
        xi, v, cell = w.xi.copy(), w.v.copy(), w.cell_id.copy()
        events, out, step = 0, [], 0
        for cp in self.checkpoints:
            idx = cs = None
            while step < cp:
                xi, v, cell = oracle.remove_zero(xi, v, cell)
                last = step == cp - 1
                idx, cs, nev = oracle.step(xi, v, cell, w.n_cell, w.dt, w.dV, w.kernel, w.kparam, w.seed, step,
                                           want_perm=last)
                events += nev
                step += 1
            out.append((xi.copy(), v.copy(), cell.copy(), idx, cs, events))
        return out

    def result(self):
        return self.future.result()


@pytest.fixture(scope="session")
def oracle_pool():
    import concurrent.futures
    workers = max(1, min(8, (os.cpu_count() or 2) - 1))
    pool = concurrent.futures.ThreadPoolExecutor(max_workers=workers)
    jobs = {}

    def submit(name, make_workload, checkpoints):
        """Starts (once per session) the trajectory `name`; returns its OracleTrajectory."""
        if name not in jobs:
            jobs[name] = OracleTrajectory(pool, make_workload(), checkpoints)
        return jobs[name]

    yield submit
    pool.shutdown(wait=False, cancel_futures=True)
