"""-m "not gpu": host side of the slab decomposition (include/rism3d.h "Slab decomposition").

rism3d_slab_plan (host-only C) gives every rank its planes, its rows of the spectrum and the block size of the
transposes.  The world_size-2 gloo test below does the 3D shifted transform the way the CUDA ranks do it -- z and y
transforms on the rank's planes, rows laid out per destination ([d][ix_l][jy_l][row]), ONE all_to_all_single of equal
contiguous blocks, x transform on the rank's rows -- with numpy line transforms in place of the kernels, and compares
with the oracle's transform of the whole field; then the way back.  What it pins is the index map of the two
transposes and the plan arithmetic, which is all the multi-process path adds to the kernels tested on the GPU."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _params(lib, shape, n_sites, n_ranks, rank):
    p = lib.Rism3dParams()
    p.nx, p.ny, p.nz = shape
    p.spacing, p.n_sites, p.closure, p.pse_order, p.temperature = 0.5, n_sites, 1, 1, 298.0
    p.mdiis_nvec, p.mdiis_b, p.mdiis_restart, p.kappa, p.r_min = 5, 0.5, 10.0, 1.0, 1e-3
    p.n_ranks, p.rank = n_ranks, rank
    return p


def test_slab_plan_partitions_the_grid():
    import paper_2403_01039_b200 as lib
    from paper_2403_01039_b200 import build as _build
    _build.build(force=False)
    for shape, nv, P in [((32, 32, 32), 2, 2), ((64, 32, 16), 3, 4), ((256, 256, 256), 4, 8), ((64, 128, 32), 1, 8)]:
        planes, rows = [], []
        for r in range(P):
            info = lib.rism3d_slab_plan(_params(lib, shape, nv, P, r))
            planes += list(range(info.ix0, info.ix0 + info.nxl))
            rows += list(range(info.jy0, info.jy0 + info.nyl))
            padded = 1 if nv <= 1 else (2 if nv <= 2 else (4 if nv <= 4 else 8))
            assert info.n_sites_padded == padded
            assert info.row_elems == shape[2] // 2 * padded
            assert info.block_elems == info.nxl * info.nyl * info.row_elems
            # P blocks = this rank's share of the half spectrum = its share of the real field, in complex numbers
            assert P * info.block_elems * 2 == padded * shape[0] * shape[1] * shape[2] // P
        assert planes == list(range(shape[0])) and rows == list(range(shape[1]))
    one = lib.rism3d_slab_plan(_params(lib, (32, 64, 16), 2, 1, 0))
    assert (one.nxl, one.ix0, one.nyl, one.jy0) == (32, 0, 64, 0)
    for shape, P, r in [((32, 32, 32), 8, 0), ((32, 32, 32), 3, 0), ((32, 32, 32), 2, 2), ((64, 8, 32), 2, 0)]:
        with pytest.raises(lib.Rism3dError):
            lib.rism3d_slab_plan(_params(lib, shape, 2, P, r))


WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import numpy as np
import torch
import torch.distributed as dist
import paper_2403_01039_b200 as lib
from oracle import rism3d as o3

rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=world)
shape, nv, h = (16, 32, 16), 2, 0.5
nx, ny, nz = shape
p = lib.Rism3dParams()
p.nx, p.ny, p.nz = shape
p.spacing, p.n_sites, p.closure, p.pse_order, p.temperature = h, nv, 1, 1, 298.0
p.mdiis_nvec, p.mdiis_b, p.mdiis_restart, p.kappa, p.r_min = 5, 0.5, 10.0, 1.0, 1e-3
p.n_ranks, p.rank = world, rank
info = lib.rism3d_slab_plan(p)
nxl, ix0, nyl, jy0, Q = info.nxl, info.ix0, info.nyl, info.jy0, info.row_elems

f = np.random.default_rng(11).standard_normal((nv,) + shape)          # every rank draws the same whole field
# the whole-grid spectrum in the library's layout [jx][jy][p][site] (origin at index 0, no dV)
ref = np.ascontiguousarray(np.moveaxis((o3.shifted_dft_forward(f, h, (0.0, 0.0, 0.0)) / h ** 3)[:, :, :, 0::2], 0, -1))

def line(a, axis, sign):
    n = a.shape[axis]
    sh = [1] * a.ndim
    sh[axis] = n
    m = np.arange(n).reshape(sh)
    if sign < 0:
        return np.fft.fft(a * np.exp(-1j * np.pi * m / n), axis=axis)
    return np.fft.ifft(a, axis=axis) * np.exp(+1j * np.pi * m / n)

# phase 0 on this rank's planes: z (even j_z kept), y
mine = np.moveaxis(f[:, ix0:ix0 + nxl], 0, -1).astype(complex)          # [ix_l][iy][iz][site]
mine = line(mine, 2, -1)[:, :, 0::2, :]
mine = line(mine, 1, -1).reshape(nxl, ny, Q)
# the y pass writes row jy of plane ix_l to block d = jy // nyl at (ix_l * nyl + jy_l) * Q
stage = np.empty((world, nxl, nyl, Q), complex)
for d in range(world):
    stage[d] = mine[:, d * nyl:(d + 1) * nyl]
K = np.empty_like(stage)
dist.all_to_all_single(torch.from_numpy(K.view(np.float64).reshape(-1)), torch.from_numpy(stage.view(np.float64).reshape(-1)))
# block s of K holds planes s*nxl .. of this rank's rows: K is [jx -> ix][jy_l][Q]
Kx = line(K.reshape(nx, nyl, Q), 0, -1)
err_fwd = float(np.max(np.abs(Kx - ref[:, jy0:jy0 + nyl].reshape(nx, nyl, Q))))

# the way back: inverse x in place, blocks of planes return to their owners, inverse y reads row jy from block jy // nyl
Kb = line(Kx, 0, +1).reshape(world, nxl, nyl, Q)
back = np.empty_like(Kb)
dist.all_to_all_single(torch.from_numpy(back.view(np.float64).reshape(-1)), torch.from_numpy(np.ascontiguousarray(Kb).view(np.float64).reshape(-1)))
rows = np.concatenate([back[s] for s in range(world)], axis=1)            # [ix_l][jy][Q]
rows = line(rows, 1, +1).reshape(nxl, ny, nz // 2, nv)
# half spectrum -> real line: F_(n-1-j) = conj F_j on the half-integer grid
full = np.zeros((nxl, ny, nz, nv), complex)
full[:, :, 0::2] = rows
full[:, :, 1::2] = np.conj(rows[:, :, ::-1])
real = line(full, 2, +1)
err_bwd = float(np.max(np.abs(real - np.moveaxis(f[:, ix0:ix0 + nxl], 0, -1))))

# the Gram rows: all_gather of one row per rank into [world][row], in place
row = 2 * 18
g = torch.zeros(world * row, dtype=torch.float64)
g[rank * row:(rank + 1) * row] = float(rank + 1)
dist.all_gather_into_tensor(g, g[rank * row:(rank + 1) * row].clone())
gram_ok = bool(all(float(g[s * row]) == s + 1 for s in range(world)))
print(json.dumps(dict(rank=rank, err_fwd=err_fwd, err_bwd=err_bwd, gram_ok=gram_ok, scale=float(np.max(np.abs(ref))))), flush=True)
dist.barrier()
dist.destroy_process_group()
"""


def test_transposes_world_size_2_gloo(tmp_path):
    from paper_2403_01039_b200 import build as _build
    _build.build(force=False)
    script = tmp_path / "slab_worker.py"
    script.write_text(WORKER.format(root=ROOT))
    port = 29900 + (os.getpid() % 90)
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    for pr in procs:
        out, err = pr.communicate(timeout=240)
        assert pr.returncode == 0, err[-3000:]
        o = json.loads(out.strip().splitlines()[-1])
        assert o["err_fwd"] < 1e-12 * o["scale"] and o["err_bwd"] < 1e-12 and o["gram_ok"]
