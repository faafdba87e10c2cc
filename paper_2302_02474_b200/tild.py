"""Thin ctypes binding over the C-ABI library (include/tild.h): same names, argument marshalling only.

PyTorch is used for device memory and the stream, nothing else: every step of the path runs in the
library's CUDA kernels.  There is no CPU fallback: `load()` raises if libtild.so is missing, and every
compute call needs CUDA tensors.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtild.so")
MAX_SPECIES = 8
MAX_BONDS = 4

OK, EINVAL, ENOMEM, ECUDA, ECUFFT, ESTATE = 0, -1, -2, -3, -4, -5
INTEGRATOR_GJF, INTEGRATOR_EM, INTEGRATOR_VV = 0, 1, 2
FLAG_TIMING, FLAG_NAIVE_SPREAD, FLAG_NAIVE_INTERP, FLAG_GRAPH, FLAG_DECONVOLVE, FLAG_SAMPLED_KERNEL = 1, 2, 4, 8, 16, 32
FLAG_PLAIN_FFT = 64
FLAG_GEN1_TILES = 128
FLAG_EAGER = 256
FLAG_2D = 512
FLAG_EXTRAS = 1024
FLAG_NO_TMA = 2048
FLAG_HOST_PIPELINE = 8192
FLAG_ARRIVAL_SORT = 16384
FLAG_NO_DEFRAG = 32768
FLAG_DEFRAG_SMALL = 65536
TIMING_NAMES = ("sort", "spread", "fft_fwd", "kspace", "fft_inv", "interp", "other", "total")

EXPORTS = (
    "tild_workspace_bytes", "tild_init", "tild_set_state", "tild_spread", "tild_kspace_force", "tild_interp",
    "tild_bond_force", "tild_step", "tild_get_state", "tild_energy", "tild_virial", "tild_set_charges", "tild_set_ms_partners", "tild_structure_factor", "tild_index_map", "tild_get_timings", "tild_run_host", "tild_run_host_submit", "tild_run_host_wait",
    "tild_philox_test", "tild_cell_start_noalloc", "tild_layout_info", "tild_segment_layout", "tild_launch_count", "tild_last_error", "tild_destroy", "tild_version",
)


class Params(C.Structure):
    """Mirror of `tild_params` (include/tild.h)."""
    _fields_ = [
        ("struct_size", C.c_uint32), ("n", C.c_int32), ("n_species", C.c_int32), ("order", C.c_int32),
        ("box", C.c_double * 3),
        ("grid", C.c_int32 * 3), ("max_bonds", C.c_int32),
        ("chi", C.c_double * (MAX_SPECIES * MAX_SPECIES)),
        ("kappa", C.c_double), ("a", C.c_double), ("sigma2", C.c_double), ("rho0", C.c_double),
        ("k_bond", C.c_double), ("r0_bond", C.c_double),
        ("dt", C.c_double), ("gamma", C.c_double), ("kT", C.c_double), ("mass", C.c_double),
        ("seed", C.c_uint64),
        ("resort_every", C.c_int32), ("flags", C.c_uint32),
        ("integrator", C.c_int32), ("tile_shape", C.c_int32),
        ("charge", C.c_double * MAX_SPECIES), ("bjerrum", C.c_double), ("a_charge", C.c_double),
        ("lambda_wlc", C.c_double),
        ("k_theta", C.c_double),
        ("theta0", C.c_double),
        ("mu_ms", C.c_double),
    ]


def make_params(n: int, n_species: int, box: Sequence[float], grid: Sequence[int], order: int, chi, kappa: float,
                a: float = 0.5, sigma2: float = 0.0, rho0: float = 0.0, k_bond: float = 1.5, r0_bond: float = 0.0,
                max_bonds: int = 2, dt: float = 0.005, gamma: float = 1.0, kT: float = 1.0, mass: float = 1.0,
                seed: int = 0, resort_every: int = 0, flags: int = 0, integrator: int = 0,
                charge: Sequence[float] = (), bjerrum: float = 0.0, a_charge: float = 0.5,
                lambda_wlc: float = 0.0, k_theta: float = 0.0, theta0: float = 0.0, tile_shape: int = 0, mu_ms: float = 0.0) -> Params:
    p = Params()
    p.struct_size = C.sizeof(Params)
    p.n, p.n_species, p.order = int(n), int(n_species), int(order)
    for k in range(3):
        p.box[k] = float(box[k])
        p.grid[k] = int(grid[k])
    p.max_bonds = int(max_bonds)
    chi = np.asarray(chi, dtype=np.float64)
    for i in range(n_species):
        for j in range(n_species):
            p.chi[i * MAX_SPECIES + j] = float(chi[i][j])
    p.kappa, p.a, p.sigma2, p.rho0 = float(kappa), float(a), float(sigma2), float(rho0)
    p.k_bond, p.r0_bond = float(k_bond), float(r0_bond)
    p.dt, p.gamma, p.kT, p.mass = float(dt), float(gamma), float(kT), float(mass)
    p.seed = int(seed)
    p.resort_every, p.flags = int(resort_every), int(flags)
    p.integrator, p.tile_shape = int(integrator), int(tile_shape)
    for i, z in enumerate(charge):
        p.charge[i] = float(z)
    p.bjerrum, p.a_charge = float(bjerrum), float(a_charge)
    p.lambda_wlc = float(lambda_wlc)
    p.k_theta, p.theta0 = float(k_theta), float(theta0)
    p.mu_ms = float(mu_ms)
    return p


def params_from_config(cfg, flags: int = 0, resort_every: int = 0, **overrides) -> Params:
    """`cfg` is a paper_2302_02474_b200.inputs.Config."""
    kw = dict(n=cfg.n, n_species=cfg.n_species, box=cfg.box, grid=cfg.grid, order=cfg.order, chi=cfg.chi,
              kappa=cfg.kappa, a=cfg.a, sigma2=cfg.sigma2, k_bond=cfg.k_bond, r0_bond=cfg.r0_bond, max_bonds=2,
              dt=cfg.dt, gamma=cfg.gamma, kT=cfg.kT, mass=cfg.mass, seed=cfg.philox_seed,
              resort_every=resort_every, flags=flags, charge=getattr(cfg, "charge", ()),
              bjerrum=getattr(cfg, "bjerrum", 0.0), a_charge=getattr(cfg, "a_charge", 0.5))
    kw.update(overrides)
    return make_params(**kw)


_lib = None


def load():
    """dlopen libtild.so and declare the prototypes.  Raises if the library has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2302_02474_b200.build` "
                           "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, i32, u64, sz = C.c_void_p, C.c_int32, C.c_uint64, C.c_size_t
    PP = C.POINTER(Params)
    lib.tild_workspace_bytes.argtypes = [PP, C.POINTER(sz)]
    lib.tild_init.argtypes = [C.POINTER(vp), PP, vp, sz, vp]
    lib.tild_set_state.argtypes = [vp, vp, vp, vp, vp, u64]
    lib.tild_spread.argtypes = [vp, vp, vp, vp]
    lib.tild_kspace_force.argtypes = [vp, vp, vp]
    lib.tild_interp.argtypes = [vp, vp, vp, vp, vp]
    lib.tild_bond_force.argtypes = [vp, vp, vp, vp]
    lib.tild_step.argtypes = [vp, i32]
    lib.tild_get_state.argtypes = [vp, vp, vp, vp, C.POINTER(u64)]
    lib.tild_energy.argtypes = [vp, C.POINTER(C.c_double * 3)]
    lib.tild_virial.argtypes = [vp, C.POINTER(C.c_double * 2)]
    lib.tild_set_charges.argtypes = [vp, vp]
    lib.tild_set_ms_partners.argtypes = [vp, vp]
    lib.tild_structure_factor.argtypes = [vp, C.c_uint32, vp, i32]
    lib.tild_index_map.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.tild_segment_layout.argtypes = [vp, vp, vp]
    lib.tild_get_timings.argtypes = [vp, C.POINTER(C.c_float * 8), C.POINTER(i32)]
    lib.tild_run_host.argtypes = [vp, vp, vp, vp, vp, u64, i32]
    lib.tild_run_host_submit.argtypes = [vp, vp, vp, vp, vp, u64, i32, vp, vp]
    lib.tild_run_host_wait.argtypes = [vp]
    lib.tild_philox_test.argtypes = [vp, vp, vp, vp, vp, i32]
    lib.tild_cell_start_noalloc.argtypes = [vp, i32, C.c_uint32, vp, vp, vp, C.c_char_p, sz]
    lib.tild_layout_info.argtypes = [vp, C.POINTER(C.c_uint64 * 8)]
    lib.tild_launch_count.argtypes = [vp]
    lib.tild_launch_count.restype = C.c_int64
    lib.tild_last_error.argtypes = [vp]
    lib.tild_last_error.restype = C.c_char_p
    lib.tild_destroy.argtypes = [vp]
    lib.tild_destroy.restype = None
    lib.tild_version.restype = C.c_char_p
    for name in EXPORTS:
        if name not in ("tild_launch_count", "tild_last_error", "tild_destroy", "tild_version"):
            getattr(lib, name).restype = C.c_int
    _lib = lib
    return lib


class TildError(RuntimeError):
    pass


NOALLOC_MAX_CELLS = 16777216


def tild_cell_start_noalloc(cell_key, n_cells: int, cell_start, n_bad=None, stream=None):
    """include/tild.h: cell offsets of the a1 index map with no context and no allocation (static device scratch).
    cell_key [n] and cell_start [n_cells + 1] (and n_bad [1]) are the caller's CUDA tensors (int32 holding uint32);
    asynchronous on `stream` (a torch stream; default: the current one).  Returns cell_start."""
    import torch
    lib = load()
    if stream is None:
        stream = torch.cuda.current_stream(cell_start.device)
    assert cell_start.numel() >= n_cells + 1 or n_cells > NOALLOC_MAX_CELLS
    msg = C.create_string_buffer(512)
    with torch.cuda.device(cell_start.device):
        rc = lib.tild_cell_start_noalloc(_dp(cell_key) if cell_key.numel() else None, int(cell_key.numel()), int(n_cells),
                                         _dp(cell_start), _dp(n_bad), C.c_void_p(stream.cuda_stream), msg, len(msg))
    if rc != OK:
        raise TildError(f"tild_cell_start_noalloc failed ({rc}): {msg.value.decode()}")
    return cell_start


def _dp(t) -> Optional[int]:
    """Device (or pinned host) pointer of a torch tensor; None passes NULL."""
    if t is None:
        return None
    assert t.is_contiguous(), "tensors passed to libtild must be contiguous"
    return t.data_ptr()


class Tild:
    """One TILD context: owns the torch workspace tensor and the opaque `tild_ctx*`."""

    def __init__(self, params: Params, device="cuda:0", stream=None):
        import torch
        self.torch = torch
        self.lib = load()
        if not torch.cuda.is_available():
            raise RuntimeError("libtild needs a CUDA device (there is no CPU fallback)")
        self.params = params
        self.device = torch.device(device)
        self.n, self.S = params.n, params.n_species
        self.N = tuple(params.grid)
        self.M = self.N[0] * self.N[1] * self.N[2]
        nbytes = C.c_size_t(0)
        rc = self.lib.tild_workspace_bytes(C.byref(params), C.byref(nbytes))
        if rc != OK:
            raise TildError(f"tild_workspace_bytes failed: {rc}")
        self.workspace_bytes = nbytes.value
        torch.cuda.set_device(self.device)
        self.workspace = torch.empty(nbytes.value + 256, dtype=torch.uint8, device=self.device)
        base = (self.workspace.data_ptr() + 255) // 256 * 256
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self.ctx = C.c_void_p()
        rc = self.lib.tild_init(C.byref(self.ctx), C.byref(params), base, nbytes.value, self.stream.cuda_stream)
        if rc != OK:
            raise TildError(f"tild_init failed: {rc}")

    def close(self):
        if getattr(self, "ctx", None) is not None and self.ctx.value:
            self.torch.cuda.synchronize(self.device)
            self.lib.tild_destroy(self.ctx)
            self.ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc: int, what: str):
        if rc != OK:
            msg = self.lib.tild_last_error(self.ctx)
            raise TildError(f"{what} failed ({rc}): {msg.decode() if msg else ''}")

    def _empty(self, shape, dtype):
        return self.torch.empty(shape, dtype=dtype, device=self.device)

    # ---- stage calls (pure functions of their arguments) ----
    def tild_spread(self, x, type_):
        grid = self._empty((self.S,) + self.N, self.torch.float32)
        self._check(self.lib.tild_spread(self.ctx, _dp(x), _dp(type_), _dp(grid)), "tild_spread")
        return grid

    def tild_kspace_force(self, grid):
        ff = self._empty((self.S, 3) + self.N, self.torch.float32)
        self._check(self.lib.tild_kspace_force(self.ctx, _dp(grid), _dp(ff)), "tild_kspace_force")
        return ff

    def tild_interp(self, ffield, x, type_):
        f = self._empty((self.n, 3), self.torch.float32)
        self._check(self.lib.tild_interp(self.ctx, _dp(ffield), _dp(x), _dp(type_), _dp(f)), "tild_interp")
        return f

    def tild_bond_force(self, x, bond_partner):
        f = self._empty((self.n, 3), self.torch.float32)
        self._check(self.lib.tild_bond_force(self.ctx, _dp(x), _dp(bond_partner), _dp(f)), "tild_bond_force")
        return f

    def tild_index_map(self, x, want_sort: bool = True):
        t = self.torch
        base = self._empty((self.n, 3), t.int32)
        key = self._empty((self.n,), t.int32)          # uint32 payload
        perm = self._empty((self.n,), t.int32) if want_sort else None
        start = self._empty((self.M + 1,), t.int32) if want_sort else None
        self._check(self.lib.tild_index_map(self.ctx, _dp(x), _dp(base), _dp(key), _dp(perm), _dp(start)), "tild_index_map")
        return base, key, perm, start

    # ---- the timed path ----
    def tild_set_state(self, x, v, type_, bond_partner, step0: int = 0):
        self._check(self.lib.tild_set_state(self.ctx, _dp(x), _dp(v), _dp(type_), _dp(bond_partner), step0), "tild_set_state")

    def tild_step(self, nsteps: int):
        self._check(self.lib.tild_step(self.ctx, int(nsteps)), "tild_step")

    def tild_get_state(self, want_v: bool = True, want_f: bool = False):
        t = self.torch
        x = self._empty((self.n, 3), t.float32)
        v = self._empty((self.n, 3), t.float32) if want_v else None
        f = self._empty((self.n, 3), t.float32) if want_f else None
        step = C.c_uint64(0)
        self._check(self.lib.tild_get_state(self.ctx, _dp(x), _dp(v), _dp(f), C.byref(step)), "tild_get_state")
        return x, v, f, step.value

    def tild_energy(self):
        """(kinetic, bond, non-bonded mesh) energies of the current state as a numpy array."""
        e = (C.c_double * 3)()
        self._check(self.lib.tild_energy(self.ctx, C.byref(e)), "tild_energy")
        return np.array([e[0], e[1], e[2]])

    def tild_set_charges(self, q=None):
        """Per-particle charges (float32 [n], original numbering) or None to go back to the charges per species."""
        self._check(self.lib.tild_set_charges(self.ctx, _dp(q) if q is not None else None), "tild_set_charges")

    def tild_set_ms_partners(self, partner=None):
        """Maier-Saupe orientation partners (int32 [n], -1 = not an LC centre) or None to switch the interaction off."""
        self._check(self.lib.tild_set_ms_partners(self.ctx, _dp(partner) if partner is not None else None), "tild_set_ms_partners")

    def tild_virial(self):
        """(bonded, non-bonded mesh) pressure virial of the current state as a numpy array; excess pressure = sum / 3V."""
        w = (C.c_double * 2)()
        self._check(self.lib.tild_virial(self.ctx, C.byref(w)), "tild_virial")
        return np.array([w[0], w[1]])

    def tild_structure_factor(self, species_mask: int, sk=None):
        """S(m) of the masked species on the half spectrum; pass a previous result as `sk` to accumulate into it."""
        acc = sk is not None
        if sk is None:
            sk = self._empty(self.N[:2] + (self.N[2] // 2 + 1,), self.torch.float32)
        self._check(self.lib.tild_structure_factor(self.ctx, int(species_mask), _dp(sk), 1 if acc else 0), "tild_structure_factor")
        return sk

    def tild_get_timings(self):
        ms = (C.c_float * 8)()
        nst = C.c_int32(0)
        self._check(self.lib.tild_get_timings(self.ctx, C.byref(ms), C.byref(nst)), "tild_get_timings")
        return dict(zip(TIMING_NAMES, [float(v) for v in ms])), nst.value

    def tild_run_host(self, x_host, v_host, type_host, bond_host, step0: int, nsteps: int):
        """x_host, v_host (updated in place), type_host, bond_host: CPU tensors (pinned for speed)."""
        for t in (x_host, v_host, type_host, bond_host):
            assert t is None or t.device.type == "cpu"
        self._check(self.lib.tild_run_host(self.ctx, _dp(x_host), _dp(v_host), _dp(type_host), _dp(bond_host),
                                           step0, int(nsteps)), "tild_run_host")

    def tild_run_host_submit(self, x_host, v_host, type_host, bond_host, step0: int, nsteps: int, x_out_host, v_out_host):
        """Pipelined tild_run_host for independent batches (FLAG_HOST_PIPELINE): returns when the inputs are consumed;
        the outputs are valid after the matching tild_run_host_wait()."""
        for t in (x_host, v_host, type_host, bond_host, x_out_host, v_out_host):
            assert t is None or t.device.type == "cpu"
        self._check(self.lib.tild_run_host_submit(self.ctx, _dp(x_host), _dp(v_host), _dp(type_host), _dp(bond_host), step0, int(nsteps),
                                                  _dp(x_out_host), _dp(v_out_host)), "tild_run_host_submit")

    def tild_run_host_wait(self):
        self._check(self.lib.tild_run_host_wait(self.ctx), "tild_run_host_wait")

    def tild_philox_test(self, ctr, key, want_gauss: bool = True):
        t = self.torch
        m = ctr.shape[0]
        out = self._empty((m, 4), t.int32)
        g = self._empty((m, 3), t.float32) if want_gauss else None
        self._check(self.lib.tild_philox_test(self.ctx, _dp(ctr), _dp(key), _dp(out), _dp(g), m), "tild_philox_test")
        return out, g

    def tild_layout_info(self) -> dict:
        info = (C.c_uint64 * 8)()
        self._check(self.lib.tild_layout_info(self.ctx, C.byref(info)), "tild_layout_info")
        names = ("tiles", "segments", "image_z", "smem_spread", "smem_interp", "tile_x", "tile_y", "tile_z")
        return dict(zip(names, [int(v) for v in info]))

    def tild_segment_layout(self):
        """(seg_base [tiles*S + 1], slot_id [n]) as int32 tensors holding the uint32 values."""
        torch = self.torch
        nseg = self.tild_layout_info()["segments"]
        seg = torch.empty(nseg + 1, dtype=torch.int32, device=self.device)
        ids = torch.empty(max(self.n, 1), dtype=torch.int32, device=self.device)
        self._check(self.lib.tild_segment_layout(self.ctx, _dp(seg), _dp(ids)), "tild_segment_layout")
        return seg, ids[: self.n]

    def tild_launch_count(self) -> int:
        return int(self.lib.tild_launch_count(self.ctx))
