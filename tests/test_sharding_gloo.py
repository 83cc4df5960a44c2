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


def test_omega_range_partition():
    for n_omega, world in [(16, 1), (16, 2), (16, 8), (16, 3), (8, 5), (3, 8), (0, 2)]:
        ranges = [sharding.omega_range(n_omega, r, world) for r in range(world)]
        assert ranges[0][0] == 0 and ranges[-1][1] == n_omega
        for (a, b), (c, d) in zip(ranges[:-1], ranges[1:]):
            assert a <= b == c <= d
        sizes = [b - a for a, b in ranges]
        assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        sharding.omega_range(4, 2, 2)


def _worker_rs(rank, world, port, out_dir):
    import oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cell = np.array([[5.0, 0.3, 0.0], [-0.7, 4.2, 0.2], [0.1, -0.4, 6.1]])
    cfg = W.custom_config(300, cell, (6, 4, 8), (0.25, -0.125, 0.5), n_occ=3, n_unocc=5, ng_target=20, n_omega=5,
                          n_atoms=2, n_proj_per_atom=3, n_k=1, orb_ecut_ha=3.0)
    om, wt = W.omega_grid(cfg.n_omega)
    orc = oracle.Chi0Oracle(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt)
    Q, R = W.paw_Q(cfg, orc.K2), W.atom_positions(cfg)
    for (k, lo, hi) in sharding.shard_units(cfg.n_k, cfg.n_occ, rank, world):
        orc.add_kpoint(W.kpoint(cfg, k, occ=range(lo, hi)), cfg.n_proj, Q, R)
    S = torch.from_numpy(orc.S)
    lo, hi = sharding.reduce_scatter_accumulators(S, cfg.n_omega)
    assert (lo, hi) == sharding.omega_range(cfg.n_omega, rank, world)
    # this rank's frequencies only (the oracle stands in for rpa_ec_q_range), then the scalar all-reduce
    chi_own = orc.get()[lo:hi]
    ec_part, e_part = oracle.ec_q(chi_own, W.coulomb(orc.K2), wt[lo:hi])
    ec = sharding.allreduce_scalar(ec_part)
    np.save(os.path.join(out_dir, f"chi_{rank}.npy"), chi_own)
    np.save(os.path.join(out_dir, f"ec_{rank}.npy"), np.array([ec, lo, hi]))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_gloo_reduce_scatter_by_frequency(tmp_path):
    """The alternative exchange of SURVEY 8(e): every rank ends up with the summed accumulators of its own frequencies,
    factorises those, and a scalar all-reduce gives E_c(q) on every rank."""
    import oracle
    mp.spawn(_worker_rs, args=(2, _free_port(), str(tmp_path)), nprocs=2, join=True)
    cell = np.array([[5.0, 0.3, 0.0], [-0.7, 4.2, 0.2], [0.1, -0.4, 6.1]])
    cfg = W.custom_config(300, cell, (6, 4, 8), (0.25, -0.125, 0.5), n_occ=3, n_unocc=5, ng_target=20, n_omega=5,
                          n_atoms=2, n_proj_per_atom=3, n_k=1, orb_ecut_ha=3.0)
    om, wt = W.omega_grid(cfg.n_omega)
    orc = oracle.Chi0Oracle(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt)
    orc.add_kpoint(W.kpoint(cfg, 0), cfg.n_proj, W.paw_Q(cfg, orc.K2), W.atom_positions(cfg))
    want = orc.get()
    ec_want, _ = orc.ec_q(W.coulomb(orc.K2))
    covered = 0
    for r in range(2):
        ec, lo, hi = np.load(tmp_path / f"ec_{r}.npy")
        lo, hi = int(lo), int(hi)
        got = np.load(tmp_path / f"chi_{r}.npy")
        assert np.linalg.norm(got - want[lo:hi]) <= 1e-13 * np.linalg.norm(want[lo:hi])
        assert abs(ec - ec_want) <= 1e-12 * abs(ec_want)
        covered += hi - lo
    assert covered == cfg.n_omega
