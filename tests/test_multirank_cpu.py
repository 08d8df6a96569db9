"""world_size-2 gloo test (CPU) of the N > 1 bench logic: columns shard over ranks with no data-path
collective (band partitioning with n_r = 1); only the timing max-reduce crosses ranks.
The per-rank work here is the oracle on each rank's column block; the union must equal the full block."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import fe_oracle as fo
    from paper_2605_30128_b200 import inputs as inp
    cfg = inp.tiny_config(ncell=2, p=2, L=4.0, natoms=1, nproj=4, nvec=8, degree=5)
    mesh = fo.Mesh(cfg.ncell, cfg.L, cfg.p, cfg.kfrac)
    hi = inp.make_hamiltonian(cfg, mesh.node_coords())
    ham = fo.Hamiltonian(mesh, hi.V, hi.Bx, hi.By, hi.Bz, hi.supp_off, hi.supp_node, hi.nproj, hi.P, hi.D)
    per = cfg.nvec // world
    cols = list(range(rank * per, (rank + 1) * per))          # this rank's band block
    X = inp.make_vectors(cfg.nnodes, cols)
    Y = fo.cheb_filter_residual(ham, X, np.zeros(per), cfg.degree, 2.0, 40.0, -3.0)
    t = torch.tensor([float(rank + 1)], dtype=torch.float64)    # stand-in for the per-rank time
    dist.all_reduce(t, op=dist.ReduceOp.MAX)                     # the only cross-rank step
    np.save(os.path.join(out, f"y{rank}.npy"), Y)
    if rank == 0:
        np.save(os.path.join(out, "tmax.npy"), t.numpy())
    dist.barrier()
    dist.destroy_process_group()


def test_column_sharding_two_ranks_gloo(tmp_path):
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    sys.path.insert(0, ROOT)
    from oracle import fe_oracle as fo
    from paper_2605_30128_b200 import inputs as inp
    cfg = inp.tiny_config(ncell=2, p=2, L=4.0, natoms=1, nproj=4, nvec=8, degree=5)
    mesh = fo.Mesh(cfg.ncell, cfg.L, cfg.p, cfg.kfrac)
    hi = inp.make_hamiltonian(cfg, mesh.node_coords())
    ham = fo.Hamiltonian(mesh, hi.V, hi.Bx, hi.By, hi.Bz, hi.supp_off, hi.supp_node, hi.nproj, hi.P, hi.D)
    X = inp.make_vectors(cfg.nnodes, 8)
    full = fo.cheb_filter_residual(ham, X, np.zeros(8), cfg.degree, 2.0, 40.0, -3.0)
    got = np.concatenate([np.load(tmp_path / "y0.npy"), np.load(tmp_path / "y1.npy")], axis=2)
    assert np.linalg.norm(got - full) < 1e-13 * np.linalg.norm(full)
    assert np.load(tmp_path / "tmax.npy")[0] == 2.0
