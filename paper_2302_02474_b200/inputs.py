"""Seeded synthetic inputs for the five BASELINE.json configs.

This module is shared by the CPU oracle's tests and the CUDA path and therefore holds NONE of the
method's arithmetic (no weights, no index map, no forces, no integrator): only the model parameters of
each config and the recipe for the initial particle state:

* chains are discrete Gaussian random walks: a uniform start in [0, L)^3, then each next bead =
  previous + N(0, 1/3) per axis (so <|dr|^2> = b^2 = 1, consistent with PAPER.md Eq. 2),
  wrapped into the box; solvent beads are uniform;
* block copolymer A_k B_k: first k beads of a chain are type 0, the rest type 1;
* v0 ~ N(0, kT/m) per axis; particle id = chain * N + s, solvent after the chains;
* bond_partner[i] = (i-1, i+1) inside a chain, -1 at chain ends and for solvent;
* numpy Generator(PCG64(seed)), float64 then cast to fp32; input seed = 1000 + config number,
  Philox seed = 2000 + config number.

The paper's own workloads (its "examples" folder) are not available; these inputs
take their structure (bead density ~2 Gaussian-chain melts in a periodic box, L54, L108-117).
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import List, Optional, Tuple

import numpy as np


@dataclass(frozen=True)
class ChainSpec:
    """`count` chains, each of sum(blocks) beads; blocks = ((type, length), ...)."""
    count: int
    blocks: Tuple[Tuple[int, int], ...]

    @property
    def length(self) -> int:
        return sum(b[1] for b in self.blocks)


@dataclass(frozen=True)
class Config:
    name: str
    number: int
    n: int
    n_species: int
    box: Tuple[float, float, float]
    grid: Tuple[int, int, int]
    order: int                       # P = nodes per dimension (reading A1)
    chi: Tuple[Tuple[float, ...], ...]
    kappa: float
    a: float = 0.5                   # smearing length; sigma^2 = 2 a^2
    k_bond: float = 1.5
    r0_bond: float = 0.0
    dt: float = 0.005
    gamma: float = 1.0
    kT: float = 1.0
    mass: float = 1.0
    steps: int = 100
    chains: Tuple[ChainSpec, ...] = ()
    memory_order: str = "chain"      # "chain" | "random" | "sorted" (C5 sweep)
    charge: Tuple[float, ...] = ()   # valence per species (A22); bjerrum = 0: no electrostatics
    bjerrum: float = 0.0
    a_charge: float = 0.5

    @property
    def input_seed(self) -> int:
        return 1000 + self.number

    @property
    def philox_seed(self) -> int:
        return 2000 + self.number

    @property
    def sigma2(self) -> float:
        return 2.0 * self.a * self.a

    @property
    def M(self) -> int:
        return self.grid[0] * self.grid[1] * self.grid[2]


def _chi2(c):
    return ((0.0, c), (c, 0.0))


C1 = Config("C1_diblock_2k", 1, 2000, 2, (10.0,) * 3, (16,) * 3, 2, _chi2(1.0), 50.0, steps=100,
            chains=(ChainSpec(100, ((0, 10), (1, 10))),))
C2 = Config("C2_diblock_64k", 2, 65536, 2, (32.0,) * 3, (64,) * 3, 3, _chi2(0.5), 25.0, steps=1000,
            chains=(ChainSpec(2048, ((0, 16), (1, 16))),))
# A20 reading: 8,388 A chains + 8,388 B chains of N=50 (419,400 beads each) + 209,776 solvent beads.
C3 = Config("C3_ternary_1m", 3, 1048576, 3, (80.0,) * 3, (128,) * 3, 3,
            ((0.0, 0.1, 0.0), (0.1, 0.0, 0.5), (0.0, 0.5, 0.0)), 25.0, steps=200,
            chains=(ChainSpec(8388, ((0, 50),)), ChainSpec(8388, ((1, 50),)), ChainSpec(209776, ((2, 1),))))
C4 = Config("C4_diblock_8m", 4, 8388608, 2, (160.0,) * 3, (256,) * 3, 4, _chi2(0.3), 25.0, steps=100,
            chains=(ChainSpec(131072, ((0, 32), (1, 32))),))


def c5(grid: int = 256, order: int = 4, memory_order: str = "random") -> Config:
    """Roofline sweep point: A20B20 melt, 4,194,304 particles, box 128^3 (A20: 104,857 chains + one A12B12).

    BASELINE.json gives no chi/kappa for C5; it reuses C4's (chi_AB = 0.3, kappa = 25)."""
    return Config(f"C5_sweep_g{grid}_p{order}_{memory_order}", 5, 4194304, 2, (128.0,) * 3, (grid,) * 3, order,
                  _chi2(0.3), 25.0, steps=50,
                  chains=(ChainSpec(104857, ((0, 20), (1, 20))), ChainSpec(1, ((0, 12), (1, 12)))),
                  memory_order=memory_order)


# Coacervate-like charged melt with the SIZE of the paper's example VII.A (434 chains x N = 82, half
# polycations, half polyanions, no solvent).  Its box, grid, spline order and parameters are not stated in the paper and
# its input files are not available: density 2, 48^3 grid, P = 2, kappa = 5, l_B = 1, a_q = 0.5 are this repo's choices.
# Context for the paper's 1429.6 time steps/s on a Quadro RTX 5000, not a parity case.
COAC = Config("COAC_434x82", 6, 35588, 2, (26.1,) * 3, (48,) * 3, 2, _chi2(0.0), 5.0, steps=1000,
              chains=(ChainSpec(217, ((0, 82),)), ChainSpec(217, ((1, 82),))), charge=(1.0, -1.0), bjerrum=1.0, a_charge=0.5)

CONFIGS = {"C1": C1, "C2": C2, "C3": C3, "C4": C4, "C5": c5(), "COAC": COAC}


def scaled(cfg: Config, chains_scale: float, box: float, grid: int, name: Optional[str] = None) -> Config:
    """A smaller instance of the same recipe (tests / CPU-baseline samples): same densities when the
    caller scales chain count and box volume together."""
    chains = tuple(ChainSpec(max(1, int(round(c.count * chains_scale))), c.blocks) for c in cfg.chains)
    n = sum(c.count * c.length for c in chains)
    return replace(cfg, name=name or f"{cfg.name}_scaled", n=n, box=(float(box),) * 3, grid=(grid,) * 3,
                   chains=chains)


@dataclass
class State:
    x: np.ndarray          # [n][3] float32, in [0, L)
    v: np.ndarray          # [n][3] float32
    type: np.ndarray       # [n] int32
    bond_partner: np.ndarray  # [n][2] int32, -1 = none


def make_state(cfg: Config, seed: Optional[int] = None) -> State:
    rng = np.random.Generator(np.random.PCG64(cfg.input_seed if seed is None else seed))
    L = np.asarray(cfg.box, dtype=np.float64)
    xs: List[np.ndarray] = []
    types: List[np.ndarray] = []
    partners: List[np.ndarray] = []
    offset = 0
    for spec in cfg.chains:
        nb, cnt = spec.length, spec.count
        start = rng.random((cnt, 1, 3)) * L
        steps = rng.normal(0.0, np.sqrt(1.0 / 3.0), size=(cnt, nb, 3))
        steps[:, 0, :] = 0.0
        pos = start + np.cumsum(steps, axis=1)
        xs.append(pos.reshape(-1, 3))
        t = np.concatenate([np.full(l, ty, dtype=np.int32) for ty, l in spec.blocks])
        types.append(np.tile(t, cnt))
        ids = offset + np.arange(cnt * nb, dtype=np.int64).reshape(cnt, nb)
        prev = ids - 1
        nxt = ids + 1
        prev[:, 0] = -1
        nxt[:, -1] = -1
        partners.append(np.stack([prev.reshape(-1), nxt.reshape(-1)], axis=1).astype(np.int32))
        offset += cnt * nb
    x = np.concatenate(xs, axis=0)
    assert x.shape[0] == cfg.n, (x.shape, cfg.n)
    x = x - L * np.floor(x / L)
    x32 = x.astype(np.float32)
    L32 = L.astype(np.float32)
    x32 = np.where(x32 >= L32, np.float32(0.0), x32)   # fp32 rounding may land exactly on L
    v = rng.normal(0.0, np.sqrt(cfg.kT / cfg.mass), size=(cfg.n, 3)).astype(np.float32)
    st = State(np.ascontiguousarray(x32), np.ascontiguousarray(v), np.concatenate(types),
               np.ascontiguousarray(np.concatenate(partners, axis=0)))
    if cfg.memory_order == "random":
        st = permute_state(st, rng.permutation(cfg.n))
    elif cfg.memory_order == "sorted":
        # spatially pre-sorted memory order (C5 sweep): by mesh cell, z fastest.  A plain spatial binning of the
        # inputs, not the method's index map: the library re-derives its own cells from the positions.
        N = np.asarray(cfg.grid, dtype=np.int64)
        c = np.minimum((st.x.astype(np.float64) / L * N).astype(np.int64), N - 1)
        st = permute_state(st, np.argsort((c[:, 0] * N[1] + c[:, 1]) * N[2] + c[:, 2], kind="stable"))
    return st


def permute_state(st: State, order: np.ndarray) -> State:
    """Re-label particles: new particle j is old particle order[j]; bond partners are remapped."""
    n = st.x.shape[0]
    inv = np.empty(n, dtype=np.int64)
    inv[order] = np.arange(n)
    bp = st.bond_partner[order]
    bp = np.where(bp >= 0, inv[np.maximum(bp, 0)], -1).astype(np.int32)
    return State(np.ascontiguousarray(st.x[order]), np.ascontiguousarray(st.v[order]),
                 np.ascontiguousarray(st.type[order]), np.ascontiguousarray(bp))
