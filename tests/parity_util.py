"""Helpers shared by the GPU parity tests, smoke() and bench.py: run the same seeded k-points through the
CUDA library (via the C ABI binding) and through the CPU oracle, and compare."""
import numpy as np


def rel_fro(a, b):
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


def gpu_run(cfg, kds, use_paw=True, max_batch_pairs=0, want_ec=True, device="cuda:0", rank_k_mode=None, info=None):
    """chi0[nw][ng][ng] (numpy), (ec, e_omega) or None, g, K2 -- everything computed by librpa_chi0.so.
    rank_k_mode: None (the library's default, FP64 tensor cores) or (mode, digits) for rpa_chi0_set_rank_k_mode.
    info: a dict that receives "rank_k_batches" = (FP64 batches, int8 batches) the handle ran."""
    import torch
    from paper_1307_8052_b200 import binding as B
    from paper_1307_8052_b200 import workload as W
    om, wt = W.omega_grid(cfg.n_omega)
    ptot = int(cfg.n_proj.sum()) if use_paw else 0
    h = B.rpa_chi0_create(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt, max_batch_pairs, ptot, device)
    try:
        if rank_k_mode is not None:
            B.rpa_chi0_set_rank_k_mode(h, *rank_k_mode)
        g, K2 = B.rpa_chi0_gvectors(h)
        Qd = R = npj = None
        if use_paw and ptot:
            Qd = torch.from_numpy(W.paw_Q(cfg, K2)).to(device)
            R, npj = W.atom_positions(cfg), cfg.n_proj
        for kd in kds:
            B.add_kpoint_host(h, kd, npj, Qd, R)
        chi = np.stack([B.rpa_chi0_get(h, i).cpu().numpy() for i in range(cfg.n_omega)])
        ec = B.rpa_ec_q(h, W.coulomb(K2)) if want_ec else None
        # get after ec_q must return the same chi0 (accumulators untouched)
        if want_ec:
            again = B.rpa_chi0_get(h, 0).cpu().numpy()
            assert np.array_equal(again, chi[0])
        B.rpa_chi0_sync(h)
        if info is not None:
            info["rank_k_batches"] = B.rpa_chi0_rank_k_batches(h)
    finally:
        h.close()
    return chi, ec, g, K2


def oracle_run(cfg, kds, use_paw=True, want_ec=True, g=None, omega=None, eta=None):
    """omega / eta given: the real-axis route of the oracle (chi0 at omega + i eta, NEXT-4), no E_c."""
    import oracle
    from paper_1307_8052_b200 import workload as W
    om, wt = W.omega_grid(cfg.n_omega)
    if eta is not None:
        om, wt, want_ec = np.asarray(omega, dtype=np.float64), None, False
    orc = oracle.Chi0Oracle(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt, g=g, eta=eta)
    Q = R = npj = None
    if use_paw and int(cfg.n_proj.sum()):
        if g is None:
            Q = W.paw_Q(cfg, orc.K2)
        else:  # Q is generated on the full sphere, then restricted to the sampled rows
            gf, K2f = oracle.sphere(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg))
            lut = {tuple(v): i for i, v in enumerate(gf.tolist())}
            sel = np.array([lut[tuple(v)] for v in np.asarray(g).tolist()])
            Qf = W.paw_Q(cfg, K2f)
            parts, off = [], 0
            for ni in cfg.n_proj:
                blk = Qf[off:off + ni * ni * len(gf)].reshape(ni, ni, len(gf))
                parts.append(np.ascontiguousarray(blk[:, :, sel]).reshape(-1))
                off += ni * ni * len(gf)
            Q = np.concatenate(parts)
        R, npj = W.atom_positions(cfg), cfg.n_proj
    for kd in kds:
        orc.add_kpoint(kd, npj, Q, R)
    chi = orc.get()
    ec = orc.ec_q(W.coulomb(orc.K2)) if (want_ec and g is None) else None
    return chi, ec, orc.g, orc.K2
