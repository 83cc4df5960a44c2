"""Writes tests/golden/toy_oracle.txt.  Calls ONLY oracle/ (plus the seeded input generator): a few chi0
entries and E_c(q) of a slice of config 0 (BASELINE.json configs[0]; 4 occ x 7 unocc bands, all 155 G, 8 omega).
The paper prints no numeric chi0 / E_c, so these are oracle-written regression values,
not paper values.  Run: python -m tests.golden.make_golden"""
import os

import numpy as np

import oracle
from paper_1307_8052_b200 import workload as W


def compute():
    cfg = W.CONFIGS[0]
    om, wt = W.omega_grid(cfg.n_omega)
    orc = oracle.Chi0Oracle(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt)
    Q, R = W.paw_Q(cfg, orc.K2), W.atom_positions(cfg)
    orc.add_kpoint(W.kpoint(cfg, 0, unocc=range(0, 28, 4)), cfg.n_proj, Q, R)
    chi = orc.get()
    ec, e = orc.ec_q(W.coulomb(orc.K2))
    out = {"ng": complex(orc.ng, 0), "ec_q": complex(ec, 0)}
    for i in (0, 3, 7):
        out[f"e_omega[{i}]"] = complex(e[i], 0)
        for (a, b) in ((0, 0), (5, 2), (2, 5), (154, 77), (100, 100)):
            out[f"chi0[{i}][{a}][{b}]"] = complex(chi[i, a, b])
    return out


if __name__ == "__main__":
    vals = compute()
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "toy_oracle.txt")
    with open(path, "w") as fh:
        fh.write("# written by tests/golden/make_golden.py (oracle only); key re im\n")
        for k, v in vals.items():
            fh.write(f"{k} {v.real!r} {v.imag!r}\n")
    print("wrote", path)
