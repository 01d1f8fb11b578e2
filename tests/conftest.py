import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
for p in (ROOT, os.path.join(ROOT, "oracle")):
    if p not in sys.path:
        sys.path.insert(0, p)


# The tests' lattices are small: use the two-step band wherever there are 28 free rows, not only
# where it pays (include/lbm.h lbm_set_band), so that every parity test below a suspension also
# exercises the banded schedule.  The full-size configs use their bands under either setting.
os.environ.setdefault("LBM_BAND", "2")


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def ob():
    """The CPU oracle's ctypes binding (test infrastructure)."""
    import oracle_binding
    oracle_binding.lib()
    return oracle_binding


@pytest.fixture(scope="session")
def wl():
    from paper_2308_16597_b200 import workloads
    return workloads


class OracleFarm:
    """Long oracle runs of the protocol-horizon tests (config 3: 100 steps, config 4: 20 steps;
    minutes of single-thread CPU work each), advanced in background threads from the start of a
    GPU session so that they overlap the rest of the suite.  ctypes releases the GIL during
    oracle_step; the threads are daemons, so an aborted session (-x) still exits.  Test
    infrastructure only: the product never sees it."""

    PLAN = {"config3": (3, 24.0), "config4": (4, 90.0)}   # config index, host GB needed

    def __init__(self, ob, wl):
        import threading
        self.jobs = {}
        for name, (k, need_gb) in self.PLAN.items():
            if self._host_gb_free() < need_gb:
                self.jobs[name] = None
                continue
            w = wl.config(k)
            job = {"w": w, "sim": None, "err": None, "seconds": None}

            def run(job=job, w=w):
                import time
                try:
                    t0 = time.perf_counter()
                    o = ob.OracleSim.from_workload(w)
                    job["links0"] = o.links()
                    o.step(w.parity_steps)
                    job["seconds"] = time.perf_counter() - t0
                    job["sim"] = o
                except BaseException as e:   # reported by join()
                    job["err"] = e

            job["thread"] = threading.Thread(target=run, daemon=True, name="oracle-" + name)
            job["thread"].start()
            self.jobs[name] = job

    @staticmethod
    def _host_gb_free():
        import psutil
        return psutil.virtual_memory().available / 2 ** 30

    def join(self, name):
        """-> (workload, OracleSim advanced parity_steps, links at step 0), or None if the host is
        too small."""
        job = self.jobs.get(name)
        if job is None:
            return None
        job["thread"].join()
        if job["err"] is not None:
            raise job["err"]
        return job["w"], job["sim"], job["links0"]

    def release(self, name):
        job = self.jobs.get(name)
        if job:
            job["sim"] = None


@pytest.fixture(scope="session")
def farm(ob, wl):
    return OracleFarm(ob, wl)


@pytest.fixture(scope="session", autouse=True)
def _start_farm_with_the_gpu_session(request):
    """Start the long oracle runs right away when this is a GPU session (-m gpu on a box with a
    CUDA device); a CPU session never builds the farm."""
    expr = request.config.getoption("-m") or ""
    if "gpu" in expr and "not gpu" not in expr:
        try:
            import torch
            if torch.cuda.is_available():
                request.getfixturevalue("farm")
        except ImportError:
            pass
    yield
