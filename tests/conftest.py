"""pytest configuration: registers the markers, puts the repo root on sys.path, and runs the full-size oracle
cases of tests/_oracle_runs.py in background processes while the other -m gpu tests execute."""
import json
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

_BACKGROUND = {}          # case name -> {"proc": Popen, "dir": path, "skip": reason or None}


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    config.addinivalue_line("markers", "slow: CPU test that takes more than ~20 s")
    config.addinivalue_line("markers", "fullsize_oracle(case): joins a background oracle run of tests/_oracle_runs.py")


def _has_gpu() -> bool:
    try:
        import torch
        return torch.cuda.is_available()
    except Exception:  # pragma: no cover
        return False


def pytest_collection_modifyitems(config, items):
    if _has_gpu():
        return
    skip = pytest.mark.skip(reason="no CUDA device in this container")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)


def pytest_collection_finish(session):
    """Start the oracle workers for the selected full-size tests (after -m / -k deselection)."""
    if not _has_gpu():
        return
    from tests._oracle_runs import CASES, host_memory_gb
    wanted = []
    for item in session.items:
        for mark in item.iter_markers("fullsize_oracle"):
            if mark.args[0] not in wanted:
                wanted.append(mark.args[0])
    free_gb = host_memory_gb()
    for name in wanted:
        need = CASES[name]["host_gb"]
        if free_gb < need + 4.0:
            _BACKGROUND[name] = {"proc": None, "dir": None,
                                 "skip": f"oracle case {name} needs {need:.0f} GB of host memory, {free_gb:.0f} GB available"}
            continue
        disk = CASES[name].get("disk_gb", 0.0)
        if disk and shutil.disk_usage(tempfile.gettempdir()).free / 1e9 < disk + 2.0:
            _BACKGROUND[name] = {"proc": None, "dir": None,
                                 "skip": f"oracle case {name} writes {disk:.0f} GB of fields to {tempfile.gettempdir()}"}
            continue
        free_gb -= need
        d = tempfile.mkdtemp(prefix=f"rism3d_oracle_{name}_")
        log = open(os.path.join(d, "worker.log"), "w")
        proc = subprocess.Popen([sys.executable, "-m", "tests._oracle_runs", name, d], cwd=ROOT, stdout=log,
                                stderr=subprocess.STDOUT)
        _BACKGROUND[name] = {"proc": proc, "dir": d, "skip": None, "t0": time.time()}


def pytest_sessionfinish(session, exitstatus):
    for entry in _BACKGROUND.values():
        if entry["proc"] is not None and entry["proc"].poll() is None:
            entry["proc"].kill()
        if entry["dir"]:
            shutil.rmtree(entry["dir"], ignore_errors=True)
    _BACKGROUND.clear()


@pytest.fixture
def fullsize_oracle(request):
    """-> (directory with G.npy, TAU.npy, W.npy, PHI.npy; the worker's status dict) of the case named by the test's
    `fullsize_oracle` marker; waits for the background process (at most 25 minutes)."""
    name = request.node.get_closest_marker("fullsize_oracle").args[0]
    entry = _BACKGROUND.get(name)
    if entry is None:
        pytest.skip("background oracle run was not started (no CUDA device at collection time)")
    if entry["skip"]:
        pytest.skip(entry["skip"])
    done = os.path.join(entry["dir"], "done.json")
    deadline = entry["t0"] + 1500.0
    while not os.path.exists(done):
        if entry["proc"].poll() is not None and not os.path.exists(done):
            with open(os.path.join(entry["dir"], "worker.log")) as f:
                pytest.fail(f"oracle worker {name} died:\n{f.read()[-2000:]}")
        if time.time() > deadline:
            pytest.fail(f"oracle worker {name} still running after 25 minutes")
        time.sleep(1.0)
    with open(done) as f:
        status = json.load(f)
    if not status.get("ok"):
        pytest.fail(f"oracle worker {name} failed:\n{status.get('error')}")
    return entry["dir"], status
