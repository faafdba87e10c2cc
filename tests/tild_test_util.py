"""Shared helpers for the parity tests: build oracle parameters and library parameters from one Config."""
import numpy as np

from oracle import tild_oracle as orc
from paper_2302_02474_b200 import inputs


def oracle_params(cfg, **over):
    kw = dict(n=cfg.n, S=cfg.n_species, L=cfg.box, N=cfg.grid, P=cfg.order, chi=np.array(cfg.chi), kappa=cfg.kappa,
              sigma2=cfg.sigma2, k_bond=cfg.k_bond, r0_bond=cfg.r0_bond, max_bonds=2, dt=cfg.dt, gamma=cfg.gamma,
              kT=cfg.kT, mass=cfg.mass, seed=cfg.philox_seed, charge=cfg.charge, bjerrum=cfg.bjerrum, a_charge=cfg.a_charge)
    kw.update(over)
    return orc.OracleParams(**kw)


def small_cfg(order=3, grid=(24, 20, 16), box=(12.0, 10.0, 8.0), n_chains=150, nb=8, S=2, number=11, **kw):
    """A small non-cubic melt: several tiles per axis and a ragged particle count."""
    from dataclasses import replace
    if S == 2:
        chains = (inputs.ChainSpec(n_chains, ((0, nb // 2), (1, nb - nb // 2))), inputs.ChainSpec(37, ((1, 1),)))
        chi = ((0.0, 0.8), (0.8, 0.0))
    else:
        chains = (inputs.ChainSpec(n_chains, ((0, nb),)), inputs.ChainSpec(n_chains // 2, ((1, nb),)),
                  inputs.ChainSpec(101, ((2, 1),)))
        chi = ((0.0, 0.4, 0.1), (0.4, 0.0, 0.9), (0.1, 0.9, 0.0))
    n = sum(c.count * c.length for c in chains)
    cfg = inputs.Config(f"small_P{order}", number, n, S, tuple(box), tuple(grid), order, chi, 20.0, chains=chains)
    return replace(cfg, **kw) if kw else cfg


def min_image(d, L):
    L = np.asarray(L, dtype=np.float64)
    return d - L * np.round(d / L)
