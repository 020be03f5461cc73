"""-m "not gpu": the host-side logic of bench.py -- algorithmic byte counts, the replica plumbing of a multi-GPU
run (world_size-2 gloo on CPU: barrier, max / sum over ranks, whole-job throughput), per-rank workloads, and the
reference arm's rank handling.  No CUDA, no oracle arithmetic checks here."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402


def test_kernel_words_add_up_to_the_design_total():
    # 2M + 12 + 1/n_v words per grid-point*site and iteration
    for n_v, M in [(2, 5), (4, 8), (4, 10)]:
        w = bench.kernel_words(n_v, M)
        assert abs(sum(w.values()) - (2 * M + 12 + 1.0 / n_v)) < 1e-12
        assert w["zinv_gram_solve"] == M + 3 and w["closure_zfwd"] == M + 3
    names = list(bench.kernel_words(4, 10))
    assert names == ["closure_zfwd", "y_fwd", "kspace_x", "y_inv", "zinv_gram_solve"]


def test_loop_kernel_names_match_the_library():
    import paper_2403_01039_b200 as lib
    from paper_2403_01039_b200 import build as _build
    _build.build(force=False)
    names = [lib.rism3d_loop_kernel_name(k) for k in range(lib.N_LOOP_KERNELS)]
    assert names == list(bench.kernel_words(4, 10))


def test_workload_inputs_differ_per_replica_but_keep_the_shape():
    cfg0, sv0, sol0, chi0 = bench.workload_inputs("C2", rank=0)
    cfg1, sv1, sol1, chi1 = bench.workload_inputs("C2", rank=1)
    assert cfg0 == cfg1 and sol0.n_atoms == sol1.n_atoms == 20
    assert not np.allclose(sol0.xyz, sol1.xyz)
    assert abs(sol1.q.sum()) < 1e-12
    again = bench.workload_inputs("C2", rank=1)[2]
    assert np.array_equal(again.xyz, sol1.xyz)           # seeded: the same replica always gets the same solute


WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch
import bench
rank, world = bench.dist_init("gloo")
import torch.distributed as dist
dist.barrier()
dev = torch.device("cpu")
ms_local = 10.0 * (rank + 1)                    # rank 1 is the slow one
value, ms_max = bench.aggregate_throughput(50.0, ms_local, dev)
mx = bench.reduce_scalars([float(rank), 2.0 - rank], "max", dev)
sm = bench.reduce_scalars([1.0, float(rank)], "sum", dev)
print(json.dumps({{"rank": rank, "world": world, "value": value, "ms_max": ms_max, "mx": mx, "sm": sm}}), flush=True)
dist.barrier()
dist.destroy_process_group()
"""


def test_replica_aggregation_world_size_2_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    port = 29600 + (os.getpid() % 300)
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=180)
        assert p.returncode == 0, err[-2000:]
        outs.append(json.loads(out.strip().splitlines()[-1]))
    for o in outs:
        assert o["world"] == 2
        assert o["ms_max"] == 20.0                           # the slowest rank's time
        assert abs(o["value"] - 100.0 / 20e-3) < 1e-9        # units of ALL ranks / max time
        assert o["mx"] == [1.0, 2.0] and o["sm"] == [2.0, 1.0]


def test_single_process_reductions_are_identities():
    assert bench.reduce_scalars([1.5, 2.5], "max", None) == [1.5, 2.5]
    v, ms = bench.aggregate_throughput(10.0, 5.0, None)
    assert ms == 5.0 and abs(v - 2000.0) < 1e-9


def test_reference_arm_nonzero_rank_exits_without_work():
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


@pytest.mark.slow
def test_reference_arm_prints_the_contract_line():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "C1",
                        "--steps", "1", "--warmup", "1"], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "iterations/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert line["gpu_launches"] == 0 and line["dtype"] == "f64"
