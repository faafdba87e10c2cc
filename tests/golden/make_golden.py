"""Writes tests/golden/c1_oracle_samples.txt.  Calls ONLY oracle/ and the seeded input recipe (no CUDA path).

    python tests/golden/make_golden.py

The paper prints no force or trajectory values for this path, so there is no
paper-printed fixture; this file pins the ORACLE's output on config C1 (BASELINE.json configs[0]) so that a later
change to the oracle's arithmetic shows up as a diff here and has to be justified in its commit message.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import tild_oracle as orc  # noqa: E402
from paper_2302_02474_b200 import inputs  # noqa: E402  (seeded inputs only: holds none of the method's arithmetic)

IDS = [0, 1, 9, 10, 19, 20, 777, 1234, 1999]
NSTEPS = 5


def compute():
    cfg = inputs.C1
    st = inputs.make_state(cfg)
    p = orc.OracleParams(cfg.n, cfg.n_species, cfg.box, cfg.grid, cfg.order, np.array(cfg.chi), cfg.kappa, cfg.sigma2,
                         k_bond=cfg.k_bond, r0_bond=cfg.r0_bond, dt=cfg.dt, gamma=cfg.gamma, kT=cfg.kT, mass=cfg.mass,
                         seed=cfg.philox_seed)
    x0, v0 = st.x.astype(np.float64), st.v.astype(np.float64)
    f0 = orc.force(p, x0, st.type, st.bond_partner)
    x5, v5, _ = orc.run(p, x0, v0, st.type, st.bond_partner, 0, NSTEPS)
    return f0[IDS], x5[IDS], v5[IDS]


def main():
    f0, x5, v5 = compute()
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "c1_oracle_samples.txt")
    with open(path, "w") as fh:
        fh.write("# written by tests/golden/make_golden.py from oracle/ only; config C1 (BASELINE.json configs[0])\n")
        fh.write("# columns: id  F0x F0y F0z  (total force at t=0)  x5 y5 z5  vx5 vy5 vz5  (state after 5 GJF steps)\n")
        for k, i in enumerate(IDS):
            fh.write(f"{i} " + " ".join(f"{v:.12e}" for v in (*f0[k], *x5[k], *v5[k])) + "\n")
    print(path)


if __name__ == "__main__":
    main()
