"""ctypes front end of the CPU oracle (oracle/tild_oracle.c).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It imports nothing from paper_2302_02474_b200 and shares no code with the CUDA path.
It only marshals numpy arrays into the C functions; every step of the arithmetic is in the C file,
whose comments cite the PAPER.md passages.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tild_oracle.c")
_LIB = os.path.join(_HERE, "libtild_oracle.so")
MAX_SPECIES = 8


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no CUDA, no shared headers with the product)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
               _SRC, "-o", _LIB, "-lm"]
        subprocess.run(cmd, check=True, cwd=_HERE)
    return _LIB


class _Params(C.Structure):
    _fields_ = [
        ("n", C.c_int32), ("S", C.c_int32),
        ("L", C.c_double * 3),
        ("N", C.c_int32 * 3),
        ("P", C.c_int32),
        ("chi", C.c_double * (MAX_SPECIES * MAX_SPECIES)),
        ("kappa", C.c_double), ("sigma2", C.c_double), ("rho0", C.c_double),
        ("k_bond", C.c_double), ("r0_bond", C.c_double),
        ("max_bonds", C.c_int32),
        ("dt", C.c_double), ("gamma", C.c_double), ("kT", C.c_double), ("mass", C.c_double),
        ("seed", C.c_uint64),
        ("lambda_wlc", C.c_double), ("k_theta", C.c_double), ("theta0", C.c_double),
        ("charge", C.c_double * MAX_SPECIES), ("bjerrum", C.c_double), ("a_charge", C.c_double),
        ("integrator", C.c_int32),
        ("sampled_kernel", C.c_int32),
        ("deconvolve", C.c_int32),
        ("dim2", C.c_int32),
        ("mu_ms", C.c_double),
        ("q_pp", C.c_void_p),
        ("ms_partner", C.c_void_p),
    ]


@dataclass
class OracleParams:
    """The model statement (Eq. 1-4, Listing 1) as the oracle reads it."""
    n: int
    S: int
    L: tuple
    N: tuple
    P: int
    chi: np.ndarray            # [S][S] symmetric, diagonal ignored
    kappa: float
    sigma2: float
    rho0: float = 0.0          # <= 0 -> n / V
    k_bond: float = 1.5
    r0_bond: float = 0.0
    max_bonds: int = 2
    dt: float = 0.005
    gamma: float = 1.0
    kT: float = 1.0
    mass: float = 1.0
    seed: int = 0
    lambda_wlc: float = 0.0    # cosine angle potential lambda (1 + cos theta), Eq. 16; linear chains (A23)
    k_theta: float = 0.0       # harmonic angle potential k_theta (theta - theta0)^2, Eq. 17
    theta0: float = 0.0
    charge: tuple = ()         # valence per species (reading A22); bjerrum = 0 switches electrostatics off
    bjerrum: float = 0.0
    a_charge: float = 0.5
    integrator: int = 0        # 0 GJF (A11), 1 Euler-Maruyama (A11b), 2 velocity Verlet + Langevin ExtraForce (A24)
    sampled_kernel: bool = False  # u^ from the FFT of u_G sampled on the mesh (A5b) instead of analytic (A5)
    deconvolve: bool = False   # divide the pair kernel by W^(k)^2; default: plain u^(k) (A13)
    dim2: bool = False         # two-dimensional system: N[2] = 1, no motion along z (A27)
    mu_ms: float = 0.0         # Maier-Saupe mu (Eq. 20); needs ms_partner (A26)
    q_pp: np.ndarray = None    # per-particle charges [n] (A25); None = charges per species
    ms_partner: np.ndarray = None  # [n] orientation partner of every LC centre, -1 = not a centre
    _c: _Params = field(default=None, repr=False)

    def c(self) -> _Params:
        p = _Params()
        p.n, p.S = int(self.n), int(self.S)
        for a in range(3):
            p.L[a] = float(self.L[a])
            p.N[a] = int(self.N[a])
        p.P = int(self.P)
        chi = np.asarray(self.chi, dtype=np.float64)
        for i in range(self.S):
            for j in range(self.S):
                p.chi[i * MAX_SPECIES + j] = float(chi[i, j])
        V = float(self.L[0]) * float(self.L[1]) * float(self.L[2])
        p.kappa, p.sigma2 = float(self.kappa), float(self.sigma2)
        p.rho0 = float(self.rho0) if self.rho0 > 0 else self.n / V
        p.k_bond, p.r0_bond, p.max_bonds = float(self.k_bond), float(self.r0_bond), int(self.max_bonds)
        p.dt, p.gamma, p.kT, p.mass = float(self.dt), float(self.gamma), float(self.kT), float(self.mass)
        p.seed = int(self.seed)
        p.lambda_wlc = float(self.lambda_wlc)
        p.k_theta, p.theta0 = float(self.k_theta), float(self.theta0)
        for i, z in enumerate(self.charge):
            p.charge[i] = float(z)
        p.bjerrum, p.a_charge = float(self.bjerrum), float(self.a_charge)
        p.integrator = int(self.integrator)
        p.sampled_kernel = 1 if self.sampled_kernel else 0
        p.deconvolve = 1 if self.deconvolve else 0
        p.dim2 = 1 if self.dim2 else 0
        p.mu_ms = float(self.mu_ms)
        # the arrays must outlive the C call: keep contiguous copies on the dataclass
        if self.q_pp is not None:
            self._q = np.ascontiguousarray(self.q_pp, dtype=np.float64)
            p.q_pp = self._q.ctypes.data
        if self.ms_partner is not None:
            self._msp = np.ascontiguousarray(self.ms_partner, dtype=np.int32)
            p.ms_partner = self._msp.ctypes.data
        return p

    @property
    def M(self) -> int:
        return int(self.N[0]) * int(self.N[1]) * int(self.N[2])


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        assert _lib.orc_struct_size() == C.sizeof(_Params), "orc_params layout mismatch"
    return _lib


def _ptr(a, ct):
    return a.ctypes.data_as(C.POINTER(ct))


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def set_threads(t: int) -> None:
    lib().orc_set_threads(int(t))


def get_threads() -> int:
    return int(lib().orc_get_threads())


def weights(P: int, t: float) -> np.ndarray:
    w = np.zeros(P, dtype=np.float64)
    lib().orc_weights(C.c_int(P), C.c_double(t), _ptr(w, C.c_double))
    return w


def index_map(p: OracleParams, x):
    x = _f32(x)
    base = np.zeros((p.n, 3), dtype=np.int32)
    toff = np.zeros((p.n, 3), dtype=np.float32)
    key = np.zeros(p.n, dtype=np.uint32)
    cp = p.c()
    lib().orc_index_map(C.byref(cp), _ptr(x, C.c_float), _ptr(base, C.c_int32), _ptr(toff, C.c_float),
                        _ptr(key, C.c_uint32))
    return base, toff, key


def cell_sort(n: int, M: int, key):
    key = np.ascontiguousarray(key, dtype=np.uint32)
    perm = np.zeros(n, dtype=np.uint32)
    start = np.zeros(M + 1, dtype=np.uint32)
    lib().orc_cell_sort(C.c_int32(n), C.c_int32(M), _ptr(key, C.c_uint32), _ptr(perm, C.c_uint32),
                        _ptr(start, C.c_uint32))
    return perm, start


def spread(p: OracleParams, x, type_):
    x, type_ = _f32(x), _i32(type_)
    grid = np.zeros((p.S, p.N[0], p.N[1], p.N[2]), dtype=np.float64)
    cp = p.c()
    lib().orc_spread(C.byref(cp), _ptr(x, C.c_float), _ptr(type_, C.c_int32), _ptr(grid, C.c_double))
    return grid


def dft3d(a, sign: int) -> np.ndarray:
    """Unnormalised 3-D DFT with kernel exp(sign 2 pi i m.g/N) of a complex array [Nx][Ny][Nz]."""
    a = np.ascontiguousarray(a, dtype=np.complex128).copy()
    N = (C.c_int32 * 3)(*a.shape)
    lib().orc_dft3d(N, _ptr(a.view(np.float64), C.c_double), C.c_int(sign))
    return a


def dft1d(a, sign: int) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.complex128)
    out = np.zeros_like(a)
    lib().orc_dft1d(C.c_int(a.shape[0]), C.c_int(1), _ptr(a.view(np.float64), C.c_double),
                    _ptr(out.view(np.float64), C.c_double), C.c_int(sign))
    return out


def uhat_table(p: OracleParams) -> np.ndarray:
    """The pair kernel u^(m) of the k-space stage on the full spectrum [Nx][Ny][Nz] (analytic or sampled, deconvolved or not)."""
    out = np.zeros(tuple(int(v) for v in p.N), dtype=np.float64)
    cp = p.c()
    lib().orc_uhat_table(C.byref(cp), _ptr(out, C.c_double))
    return out


def kspace_force(p: OracleParams, grid):
    grid = _f64(grid)
    ff = np.zeros((p.S, 3, p.N[0], p.N[1], p.N[2]), dtype=np.float64)
    cp = p.c()
    lib().orc_kspace_force(C.byref(cp), _ptr(grid, C.c_double), _ptr(ff, C.c_double))
    return ff


def interp(p: OracleParams, ffield, x, type_):
    ffield, x, type_ = _f64(ffield), _f32(x), _i32(type_)
    f = np.zeros((p.n, 3), dtype=np.float64)
    cp = p.c()
    lib().orc_interp(C.byref(cp), _ptr(ffield, C.c_double), _ptr(x, C.c_float), _ptr(type_, C.c_int32),
                     _ptr(f, C.c_double))
    return f


def bond_force(p: OracleParams, x, partner):
    x, partner = _f64(x), _i32(partner)
    f = np.zeros((p.n, 3), dtype=np.float64)
    cp = p.c()
    lib().orc_bond_force(C.byref(cp), _ptr(x, C.c_double), _ptr(partner, C.c_int32), _ptr(f, C.c_double))
    return f


def force(p: OracleParams, x, type_, partner):
    """Total force (PM non-bonded + bonds) at positions x (double; PM part sees fl32(x))."""
    x, type_, partner = _f64(x), _i32(type_), _i32(partner)
    f = np.zeros((p.n, 3), dtype=np.float64)
    cp = p.c()
    lib().orc_force(C.byref(cp), _ptr(x, C.c_double), _ptr(type_, C.c_int32), _ptr(partner, C.c_int32),
                    _ptr(f, C.c_double))
    return f


def nonbonded_force(p: OracleParams, x, type_):
    x32 = _f32(x)
    return interp(p, kspace_force(p, spread(p, x32, type_)), x32, type_)


def philox4x32_10(ctr, key) -> np.ndarray:
    ctr = np.ascontiguousarray(ctr, dtype=np.uint32)
    key = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32_10(_ptr(ctr, C.c_uint32), _ptr(key, C.c_uint32), _ptr(out, C.c_uint32))
    return out


def noise(p: OracleParams, pid: int, step: int) -> np.ndarray:
    b = np.zeros(3, dtype=np.float64)
    cp = p.c()
    lib().orc_noise(C.byref(cp), C.c_uint32(pid), C.c_uint64(step), _ptr(b, C.c_double))
    return b


def normals(seed: int, pid: int, step: int) -> np.ndarray:
    z = np.zeros(3, dtype=np.float64)
    lib().orc_normals(C.c_uint64(seed), C.c_uint32(pid), C.c_uint64(step), _ptr(z, C.c_double))
    return z


def run(p: OracleParams, x, v, type_, partner, step0: int, nsteps: int, f=None):
    """Advance (x, v) by nsteps GJF steps.  Returns new (x, v, f) as float64 arrays."""
    x, v = _f64(x).copy(), _f64(v).copy()
    type_, partner = _i32(type_), _i32(partner)
    f = force(p, x, type_, partner) if f is None else _f64(f).copy()
    cp = p.c()
    lib().orc_run(C.byref(cp), _ptr(x, C.c_double), _ptr(v, C.c_double), _ptr(f, C.c_double),
                  _ptr(type_, C.c_int32), _ptr(partner, C.c_int32), C.c_uint64(step0), C.c_int32(nsteps))
    return x, v, f


def energy(p: OracleParams, x, v, type_, partner) -> np.ndarray:
    x, v, type_, partner = _f64(x), _f64(v), _i32(type_), _i32(partner)
    e = np.zeros(3, dtype=np.float64)
    cp = p.c()
    lib().orc_energy(C.byref(cp), _ptr(x, C.c_double), _ptr(v, C.c_double), _ptr(type_, C.c_int32),
                     _ptr(partner, C.c_int32), _ptr(e, C.c_double))
    return e


def virial(p: OracleParams, x, type_, partner) -> np.ndarray:
    """(bonded, non-bonded) pressure virial W = -dU/d ln(lambda) of the affine scaling; excess pressure = W / 3V."""
    x, type_, partner = _f64(x), _i32(type_), _i32(partner)
    w = np.zeros(2, dtype=np.float64)
    cp = p.c()
    lib().orc_virial(C.byref(cp), _ptr(x, C.c_double), _ptr(type_, C.c_int32), _ptr(partner, C.c_int32), _ptr(w, C.c_double))
    return w


def structure_factor(p: OracleParams, x, type_, species=None) -> np.ndarray:
    """S(m) = |rho^(m)|^2 / N of the mesh density of the chosen species (all when None), Eq. 23 L334 with
    rho^ taken from the spread density (the mesh the force path works on): rho^(m) = sum_g n(g) exp(-2 pi i m.g/N).
    Returned on the half spectrum [Nx][Ny][Nz/2+1] (the other half is its mirror image)."""
    g = spread(p, x, type_)
    sel = range(p.S) if species is None else list(species)
    n = sum(g[J] for J in sel)
    count = float(n.sum())
    rho = dft3d(n.astype(np.complex128), -1)
    return (np.abs(rho) ** 2 / count)[:, :, : int(p.N[2]) // 2 + 1]
