"""The N > 1 path on CPU: units are sharded over ranks, each rank accumulates its own partial S (here with the
oracle standing in for the per-rank accumulation), the partial S are summed with a world_size-2 gloo all-reduce
through the same helper bench.py uses with NCCL, and the result equals the single-rank chi0."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1307_8052_b200 import sharding
from paper_1307_8052_b200 import workload as W


def test_shard_units_partition():
    for n_k, n_occ, world in [(1, 12, 2), (4, 64, 8), (64, 8, 8), (3, 5, 4), (1, 1, 4), (8, 120, 3), (2, 3, 16)]:
        seen = {}
        for r in range(world):
            for (k, lo, hi) in sharding.shard_units(n_k, n_occ, r, world):
                assert 0 <= lo < hi <= n_occ
                for b in range(lo, hi):
                    assert (k, b) not in seen, "a (k, band) was assigned twice"
                    seen[(k, b)] = r
        assert len(seen) == n_k * n_occ, "a (k, band) was dropped"
        loads = [sum(hi - lo for (_, lo, hi) in sharding.shard_units(n_k, n_occ, r, world)) for r in range(world)]
        if n_k * n_occ >= world and (n_k >= world or n_occ >= world):
            assert max(loads) - min(loads) <= max(n_occ, 1) * (1 if n_k >= world else 1)
    with pytest.raises(ValueError):
        sharding.shard_units(2, 2, 3, 2)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_path):
    import oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cell = np.array([[5.0, 0.3, 0.0], [-0.7, 4.2, 0.2], [0.1, -0.4, 6.1]])
    cfg = W.custom_config(300, cell, (6, 4, 8), (0.25, -0.125, 0.5), n_occ=3, n_unocc=5, ng_target=20, n_omega=3,
                          n_atoms=2, n_proj_per_atom=3, n_k=1, orb_ecut_ha=3.0)
    om, wt = W.omega_grid(cfg.n_omega)
    orc = oracle.Chi0Oracle(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt)
    Q, R = W.paw_Q(cfg, orc.K2), W.atom_positions(cfg)
    for (k, lo, hi) in sharding.shard_units(cfg.n_k, cfg.n_occ, rank, world):
        orc.add_kpoint(W.kpoint(cfg, k, occ=range(lo, hi)), cfg.n_proj, Q, R)
    S = torch.from_numpy(orc.S)
    sharding.allreduce_accumulators(S)
    if rank == 0:
        np.save(out_path, orc.get())
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_gloo_allreduce_matches_single_rank(tmp_path):
    import oracle
    out = str(tmp_path / "chi_sharded.npy")
    mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    got = np.load(out)
    cell = np.array([[5.0, 0.3, 0.0], [-0.7, 4.2, 0.2], [0.1, -0.4, 6.1]])
    cfg = W.custom_config(300, cell, (6, 4, 8), (0.25, -0.125, 0.5), n_occ=3, n_unocc=5, ng_target=20, n_omega=3,
                          n_atoms=2, n_proj_per_atom=3, n_k=1, orb_ecut_ha=3.0)
    om, wt = W.omega_grid(cfg.n_omega)
    orc = oracle.Chi0Oracle(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt)
    orc.add_kpoint(W.kpoint(cfg, 0), cfg.n_proj, W.paw_Q(cfg, orc.K2), W.atom_positions(cfg))
    want = orc.get()
    assert np.linalg.norm(got - want) <= 1e-13 * np.linalg.norm(want)
