import os
import shutil
import subprocess
import sys
import tempfile
import time

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

FULLSIZE_CASES = ("c5", "c4", "c3", "c2")          # longest first
_workers = {"dir": None, "procs": {}}


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def pytest_collection_finish(session):
    """The full-size one-step parity tests (tests/test_gpu_zz_fullsize_oracle.py) need minutes of single-threaded
    oracle time per config: start one oracle process per config NOW, so they run while the rest of the GPU suite does."""
    want = [it for it in session.items if "test_gpu_zz_fullsize_oracle" in it.nodeid]
    if not want or _workers["dir"] is not None:
        return
    try:
        import torch
        if not torch.cuda.is_available():
            return
    except Exception:
        return
    from oracle.build import build
    build()                                            # once, before the workers race for it
    base = "/dev/shm" if os.path.isdir("/dev/shm") and os.access("/dev/shm", os.W_OK) else None
    d = tempfile.mkdtemp(prefix="fs_fullsize_", dir=base)
    _workers["dir"] = d
    import re
    cases = [c for c in FULLSIZE_CASES if any(re.search(r"[\[-]%s[\]-]" % c, it.nodeid) or ("_%s_" % c) in it.nodeid for it in want)]
    for c in cases:
        log = open(os.path.join(d, c + ".log"), "w")
        _workers["procs"][c] = subprocess.Popen([sys.executable, os.path.join(ROOT, "tests", "fullsize_oracle_worker.py"), c, d],
                                                stdout=log, stderr=subprocess.STDOUT, cwd=ROOT)


def pytest_sessionfinish(session, exitstatus):
    for p in _workers["procs"].values():
        if p.poll() is None:
            p.kill()
    if _workers["dir"]:
        shutil.rmtree(_workers["dir"], ignore_errors=True)


@pytest.fixture(scope="session")
def fullsize_oracle():
    """wait(case) -> directory holding that case's oracle result (blocks until the worker has finished)."""
    def wait(case, timeout=1500.0):
        d, p = _workers["dir"], _workers["procs"].get(case)
        assert d is not None and p is not None, "full-size oracle worker for %s was not started" % case
        done = os.path.join(d, case + "_info.json")
        t0 = time.time()
        while not os.path.exists(done):
            if p.poll() is not None and not os.path.exists(done):
                raise RuntimeError("oracle worker %s exited %s:\n%s" % (case, p.returncode, open(os.path.join(d, case + ".log")).read()[-2000:]))
            if time.time() - t0 > timeout:
                raise RuntimeError("oracle worker %s timed out" % case)
            time.sleep(1.0)
        return d
    return wait


@pytest.fixture(scope="session")
def oracle_mod():
    import oracle
    oracle.lib()
    return oracle
