"""-m gpu: the slab decomposition (include/rism3d.h "Slab decomposition") against the oracle.

One GPU is what the test box has, so the n_ranks contexts of a run live in ONE process on ONE device and are driven
phase by phase on one stream (`iterate_in_lockstep`): every kernel of every rank is the kernel a multi-GPU run launches,
with that rank's slab geometry, base-pointer tables and Gram exchange; no kernel ever waits for another rank.  Staged
mode moves the blocks with device copies that stand in for the all-to-all; peer mode hands every rank the addresses of
the other ranks' arrays (here: plain device pointers of the same GPU), so the y passes write into / read from the other
ranks' k-space slabs directly, as they do over NVLink."""
import numpy as np
import pytest

from oracle import rism3d as o3
from workloads import Solute, load_chi, make_solute, solvent_by_name

pytestmark = pytest.mark.gpu


def _solute(seed, n, spread):
    rng = np.random.default_rng(seed)
    xyz = rng.uniform(-spread, spread, (n, 3))
    q = rng.normal(0.0, 0.3, n)
    return Solute("slab", xyz, q, rng.uniform(2.6, 3.4, n), rng.uniform(0.05, 0.2, n))


def _make(shape, spacing, solvent, P, sol, rcut, peer, **kw):
    import torch
    import paper_2403_01039_b200 as lib
    sv = solvent_by_name(solvent)
    k0, dk, chi = load_chi(sv.name)
    orc = o3.Rism3dOracle(shape, spacing, sv.n_v, **kw)
    orc.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
    orc.set_solute(sol.xyz, sol.q, sol.sigma, sol.eps, rcut=rcut)
    stream = torch.cuda.Stream()
    ranks = [lib.SlabSolver(shape, spacing, sv.n_v, P, r, stream=stream, **kw) for r in range(P)]
    for r in ranks:
        r.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
        r.set_solute(sol.xyz, sol.q, sol.sigma, sol.eps, rcut=rcut)
    if peer:
        loc = [r.local for r in ranks]
        for r in ranks:
            r.connect_peers([l["K"] for l in loc], [l["gram"] for l in loc], [l["flags"] for l in loc])
    return orc, ranks, sv


def _gather(ranks, which):
    """whole-grid field [n_sites][nx][ny][nz] from the ranks' slabs"""
    return np.concatenate([r.get_field(which) for r in ranks], axis=1)


@pytest.mark.parametrize("P,shape,solvent,rcut,peer", [
    (2, (32, 32, 32), "water", 0.0, False),
    (2, (32, 32, 32), "water", 0.0, True),
    (4, (32, 64, 16), "water", 7.0, False),
    (4, (64, 32, 32), "water_nacl_0.1M", 0.0, True),
    (8, (64, 64, 16), "water", 0.0, True),
    (2, (128, 16, 8), "water", 0.0, True),             # 128-point x lines on 8 rows per rank
    (4, (32, 256, 8), "water", 0.0, False),            # 256-point y lines through the row map; the three-pass k-space kernel
    (2, (512, 16, 8), "water", 5.0, True),             # the 512-point k-space kernel on a slab
    (2, (16, 128, 16), "water_nacl_0.1M", 0.0, False),
])
def test_slab_ranks_match_oracle(P, shape, solvent, rcut, peer):
    import paper_2403_01039_b200 as lib
    sol = _solute(sum(shape) + P, 4, 1.5)
    kw = dict(closure="KH", mdiis_nvec=5, mdiis_b=0.5, mdiis_restart=10.0)
    orc, ranks, sv = _make(shape, 0.5, solvent, P, sol, rcut, peer, **kw)
    # S0 on every slab
    Wo = orc.get_field("W")
    W = _gather(ranks, "W")
    assert W.shape == Wo.shape
    finite = np.abs(Wo) < 600.0
    assert np.max(np.abs(W - Wo)[finite]) < 1e-10
    phi = np.concatenate([r.get_field("PHI", 0) for r in ranks], axis=0)
    assert np.max(np.abs(phi - orc.phi)) < 1e-11 * np.max(np.abs(orc.phi))
    # the loop
    iters = 30
    orc.iterate(iters, 0.0)
    nd, rms = lib.iterate_in_lockstep(ranks, iters, 0.0)
    assert nd == iters
    hist = ranks[0].rms_history()
    np.testing.assert_allclose(hist, orc.rms_history, rtol=1e-6, atol=1e-12)
    for r in ranks[1:]:
        assert np.array_equal(r.rms_history(), hist)         # every rank solved the same small system
    assert np.max(np.abs(_gather(ranks, "G") - orc.get_field("G"))) <= 1e-9
    assert np.max(np.abs(_gather(ranks, "TAU") - orc.get_field("TAU"))) <= 1e-9
    # grid sums: every rank returns its slab's share
    mu = sum(lib.rism3d_free_energy(r.ctx, sv.n_v)[0] for r in ranks)
    mu_o, _ = orc.free_energy()
    assert abs(mu - mu_o) <= 1e-7 * abs(mu_o)
    v = sum(lib.rism3d_pmv(r.ctx, 0.05, sv.n_v)[0] for r in ranks)
    v_o, _ = orc.pmv(0.05)
    assert abs(v - v_o) <= 1e-7 * abs(v_o)
    grad = sum(lib.rism3d_gradient(r.ctx, sol.n_atoms) for r in ranks)
    go = orc.solvation_gradient()
    assert np.max(np.abs(grad - go)) <= 1e-8 * max(1.0, np.max(np.abs(go)))
    for r in ranks:
        r.close()


def test_staged_and_peer_mode_agree_bit_for_bit_and_with_one_rank():
    """same kernels, same arithmetic: only where the rows travel differs.  Against a single rank the Gram sums are
    added in a different order (per slab, then over ranks), so that comparison is to rounding, not to the bit."""
    import paper_2403_01039_b200 as lib
    shape, P = (32, 32, 32), 2
    sol = _solute(5, 5, 2.0)
    kw = dict(closure="PSE", pse_order=2, mdiis_nvec=4)
    _, staged, sv = _make(shape, 0.5, "water", P, sol, 0.0, False, **kw)
    _, peers, _ = _make(shape, 0.5, "water", P, sol, 0.0, True, **kw)
    lib.iterate_in_lockstep(staged, 20, 0.0)
    lib.iterate_in_lockstep(peers, 20, 0.0)
    assert np.array_equal(_gather(staged, "TAU"), _gather(peers, "TAU"))
    assert np.array_equal(staged[0].rms_history(), peers[1].rms_history())
    k0, dk, chi = load_chi(sv.name)
    one = lib.Solver(shape, 0.5, sv.n_v, **kw)
    one.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
    one.set_solute(sol.xyz, sol.q, sol.sigma, sol.eps)
    one.iterate(20, 0.0)
    np.testing.assert_allclose(staged[0].rms_history(), one.rms_history(), rtol=1e-9)
    assert np.max(np.abs(_gather(staged, "TAU") - one.get_field("TAU"))) <= 1e-10


@pytest.mark.parametrize("variant", ["anderson", "dynamic_b", "pse3_m1"])
def test_slab_ranks_with_the_other_accelerators(variant):
    """the modified Anderson method (weighted Gram row + the unweighted one for the rms travel together), the dynamic
    damping (the update reads both histories) and damped Picard iteration (M = 1, PSE-3) under the slab decomposition"""
    import paper_2403_01039_b200 as lib
    sol = _solute(9, 3, 1.2)
    kw = {"anderson": dict(closure="KH", accelerator="ANDERSON", mdiis_b=0.6, anderson_s=(0.2, 0.0)),
          "dynamic_b": dict(closure="KH", mdiis_nvec=4, mdiis_dynamic_b=(0.1, 1.0)),
          "pse3_m1": dict(closure="PSE", pse_order=3, mdiis_nvec=1, mdiis_b=0.2)}[variant]
    orc, ranks, sv = _make((32, 32, 32), 0.5, "water", 4, sol, 0.0, True, **kw)
    orc.iterate(25, 0.0)
    lib.iterate_in_lockstep(ranks, 25, 0.0)
    np.testing.assert_allclose(ranks[0].rms_history(), orc.rms_history, rtol=1e-6, atol=1e-12)
    assert np.max(np.abs(_gather(ranks, "G") - orc.get_field("G"))) <= 1e-9
    assert np.max(np.abs(_gather(ranks, "TAU") - orc.get_field("TAU"))) <= 1e-9
    for r in ranks:
        r.close()


def test_slab_convergence_stops_all_ranks_together():
    import paper_2403_01039_b200 as lib
    sol = Solute("ion", np.array([[0.0, 0.0, 0.0]]), np.array([1.0]), np.array([2.35]), np.array([0.13]))
    orc, ranks, sv = _make((32, 32, 32), 0.5, "water", 2, sol, 0.0, False, closure="KH", mdiis_nvec=5)
    n_o, rms_o = orc.iterate(400, 1e-6)
    nd, rms = lib.iterate_in_lockstep(ranks, 400, 1e-6)
    assert nd == n_o and rms < 1e-6 and abs(rms - rms_o) <= 1e-6 * rms_o
    assert np.max(np.abs(_gather(ranks, "G") - orc.get_field("G"))) <= 1e-9


def test_slab_argument_checks():
    import paper_2403_01039_b200 as lib
    p = lib.Rism3dParams()
    p.nx = p.ny = p.nz = 32
    p.spacing, p.n_sites, p.closure, p.pse_order, p.temperature = 0.5, 2, 1, 1, 298.0
    p.mdiis_nvec, p.mdiis_b, p.mdiis_restart, p.kappa, p.r_min = 5, 0.5, 10.0, 1.0, 1e-3
    p.n_ranks, p.rank = 2, 0
    assert lib.rism3d_workspace_bytes(p) > 0
    for bad_ranks, bad_rank in [(3, 0), (2, 2), (8, 0), (16, 0), (2, -1)]:      # 32 / 8 = 4 planes: not whole bricks
        p.n_ranks, p.rank = bad_ranks, bad_rank
        assert lib.rism3d_workspace_bytes(p) == 0
    one = lib.Solver(32, 0.5, 2)
    with pytest.raises(lib.Rism3dError):
        lib.rism3d_slab_phase(one.ctx, 0)                    # not a slab run
    one.close()


# ---- the multi-process driver (SlabSolver.iterate under torch.distributed) ------------------------------------------
MP_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import numpy as np
import torch
import torch.distributed as dist
import paper_2403_01039_b200 as lib
from workloads import Solute, load_chi, solvent_by_name

rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=world)       # one GPU on this box: the blocks travel through the host
sv = solvent_by_name("water")
k0, dk, chi = load_chi(sv.name)
d = np.load({inputs!r})
peer = {peer!r}
s = lib.SlabSolver((32, 32, 32), 0.5, sv.n_v, world, rank, closure="KH", mdiis_nvec=5, exportable=peer)
s.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
s.set_solute(d["xyz"], d["q"], d["sigma"], d["eps"])
if peer:
    # the other process's arrays mapped through CUDA IPC: this rank's y pass stores into THAT process's memory; the
    # host keeps the ranks in step (both time-slice one GPU: no kernel may wait for the other)
    s.connect_peers_ipc()
    nd, rms = s.iterate_host_ordered(25, 0.0)
else:
    nd, rms = s.iterate(25, 0.0)
mu, _ = s.free_energy()
grad = s.gradient()
np.savez(os.path.join({out!r}, f"rank{{rank}}.npz"), G=s.get_field("G"), TAU=s.get_field("TAU"), hist=s.rms_history(),
         nd=nd, mu=mu, grad=grad)
dist.barrier()
dist.destroy_process_group()
"""


@pytest.mark.parametrize("peer", [False, True])
def test_two_processes_share_one_solve(tmp_path, peer):
    """SlabSolver as a multi-GPU job runs it: one process per rank.  Both processes use this box's one GPU and a gloo
    group (host-side waits only; no kernel waits for another process).  peer = False: staged blocks and collectives
    between the phase calls; peer = True: each process maps the other's workspace (CUDA IPC) and the transposes are
    stores into / loads from the other process's memory."""
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    sol = _solute(21, 4, 1.5)
    inputs = str(tmp_path / "solute.npz")
    np.savez(inputs, xyz=sol.xyz, q=sol.q, sigma=sol.sigma, eps=sol.eps)
    script = tmp_path / "mp_worker.py"
    script.write_text(MP_WORKER.format(root=root, inputs=inputs, out=str(tmp_path), peer=peer))
    port = 29700 + (os.getpid() % 200)
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    for p in procs:
        out, err = p.communicate(timeout=600)
        assert p.returncode == 0, err[-3000:]
    sv = solvent_by_name("water")
    k0, dk, chi = load_chi(sv.name)
    orc = o3.Rism3dOracle((32, 32, 32), 0.5, sv.n_v, closure="KH", mdiis_nvec=5)
    orc.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
    orc.set_solute(sol.xyz, sol.q, sol.sigma, sol.eps)
    orc.iterate(25, 0.0)
    r = [np.load(tmp_path / f"rank{k}.npz") for k in range(2)]
    assert int(r[0]["nd"]) == 25
    np.testing.assert_allclose(r[0]["hist"], orc.rms_history, rtol=1e-6, atol=1e-12)
    assert np.array_equal(r[0]["hist"], r[1]["hist"])
    assert np.max(np.abs(np.concatenate([r[0]["G"], r[1]["G"]], axis=1) - orc.get_field("G"))) <= 1e-9
    mu_o, _ = orc.free_energy()
    assert abs(float(r[0]["mu"]) - mu_o) <= 1e-7 * abs(mu_o) and float(r[0]["mu"]) == float(r[1]["mu"])
    go = orc.solvation_gradient()
    assert np.max(np.abs(r[1]["grad"] - go)) <= 1e-8 * max(1.0, np.max(np.abs(go)))


def test_bench_decompose_slab_two_processes(tmp_path):
    """bench.py --decompose slab end to end (one solve over two ranks, strong scaling line), both ranks on this box's one
    GPU with a gloo group"""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    port = 29400 + (os.getpid() % 200)
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--decompose", "slab",
                                       "--backend", "gloo", "--workload", "C2", "--steps", "4", "--warmup", "5",
                                       "--max-iter", "600"], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=900)
        assert p.returncode == 0, err[-3000:]
        outs.append(out)
    line = json.loads(outs[0].strip().splitlines()[-1])
    assert outs[1].strip() == ""
    assert line["scaling"] == "strong" and line["n_gpus"] == 2 and line["value"] > 0 and line["gpu_launches"] > 0
    assert line["e2e"]["converged"] and 300 < line["e2e"]["iterations_to_converge"] < 450      # a single rank needs 359


def test_slab_peer_table_checks():
    import torch
    import paper_2403_01039_b200 as lib
    stream = torch.cuda.Stream()
    a = lib.SlabSolver(32, 0.5, 2, 2, 0, stream=stream)
    b = lib.SlabSolver(32, 0.5, 2, 2, 1, stream=stream)
    la, lb = a.local, b.local
    with pytest.raises(lib.Rism3dError):                     # entry `rank` must be the rank's own arrays
        a.connect_peers([lb["K"], la["K"]], [lb["gram"], la["gram"]], [lb["flags"], la["flags"]])
    with pytest.raises(lib.Rism3dError):
        a.connect_peers([la["K"], 0], [la["gram"], lb["gram"]], [la["flags"], lb["flags"]])
    with pytest.raises(lib.Rism3dError):
        a.phase(4)
    with pytest.raises(lib.Rism3dError):
        a.phase(0)                                           # no solute yet
    with pytest.raises(RuntimeError):
        a.iterate_host_ordered(1)                            # not in peer mode
    a.connect_peers([la["K"], lb["K"]], [la["gram"], lb["gram"]], [la["flags"], lb["flags"]])
    assert a.peer_mode
    a.close()
    b.close()


# ---- the in-stream barrier of peer mode ---------------------------------------------------------------------------
# Kernels that wait on one another must not be run as separate launches on one GPU (nothing guarantees that they are
# resident together), so the barrier is exercised as ONE cooperative launch whose blocks are the ranks and run the
# production barrier function (rism3d_debug_peer_barrier_selftest); the wait is bounded either way.
@pytest.mark.parametrize("P", [1, 2, 4, 8])
def test_peer_barrier_orders_the_ranks(P):
    import torch
    import paper_2403_01039_b200 as lib
    scratch = torch.empty(4096, dtype=torch.uint8, device="cuda")
    stream = torch.cuda.Stream()
    stream.wait_stream(torch.cuda.current_stream())
    errors, timeouts = lib.rism3d_debug_peer_barrier_selftest(0, scratch.data_ptr(), scratch.numel(), stream.cuda_stream,
                                                              P, 500, -1, 5.0)
    assert (errors, timeouts) == (0, 0)


def test_peer_barrier_gives_up_on_an_absent_rank():
    import time
    import torch
    import paper_2403_01039_b200 as lib
    scratch = torch.empty(4096, dtype=torch.uint8, device="cuda")
    stream = torch.cuda.Stream()
    stream.wait_stream(torch.cuda.current_stream())
    t0 = time.time()
    errors, timeouts = lib.rism3d_debug_peer_barrier_selftest(0, scratch.data_ptr(), scratch.numel(), stream.cuda_stream,
                                                              4, 10, 2, 0.05)
    assert (errors, timeouts) == (0, 3)                      # the three ranks that did arrive all report the missing one
    assert time.time() - t0 < 5.0                            # ... after the 50 ms limit, not never
    with pytest.raises(lib.Rism3dError):
        lib.rism3d_debug_peer_barrier_selftest(0, scratch.data_ptr(), 1024, stream.cuda_stream, 2, 1)     # scratch too small
    with pytest.raises(lib.Rism3dError):
        lib.rism3d_debug_peer_barrier_selftest(0, scratch.data_ptr(), 4096, stream.cuda_stream, 9, 1)     # > 8 ranks


def test_peer_timeout_setting_and_status():
    import torch
    import paper_2403_01039_b200 as lib
    assert "barrier" in lib.rism3d_status_string(-9)
    a = lib.SlabSolver(32, 0.5, 2, 2, 0, stream=torch.cuda.Stream())
    a.set_peer_timeout(2.0)
    for bad in (0.0, -1.0, 1e5, float("nan")):
        with pytest.raises(lib.Rism3dError) as e:
            a.set_peer_timeout(bad)
        assert e.value.status == -1
    a.close()
    one = lib.Solver(32, 0.5, 2)
    with pytest.raises(lib.Rism3dError) as e:
        lib.rism3d_slab_set_peer_timeout(one.ctx, 1.0)       # not a slab run
    assert e.value.status == -3
    one.close()
