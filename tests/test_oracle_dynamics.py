"""Pins for the oracle's bonds (O7b), GJF integrator (O8), noise (O9) and energy (O10).

Bonds: PAPER.md Eq. 2 L114, L209.  GJF: named at L352 (equations from Gronbech-Jensen & Farago 2013,
DESIGN.md reading A11): gamma = 0 must reduce to velocity Verlet step for step; the energy error must
scale as dt^2; a free particle must diffuse with D = kT/gamma; a harmonic dimer must sample
<r^2> = 3 kT / (2 k) (GJF is exact for configurational sampling of a harmonic well).
Philox: bit-equality with cuRAND's own Philox4x32-10 header compiled for the host (library routine).
"""
import ctypes as C
import os
import shutil
import subprocess

import numpy as np
import pytest
from scipy import stats

from oracle import tild_oracle as orc

HERE = os.path.dirname(os.path.abspath(__file__))


def _p(n, L=(8.0, 8.0, 8.0), N=(8, 8, 8), P=2, S=2, chi=1.0, kappa=5.0, **kw):
    chim = np.array([[0.0, chi], [chi, 0.0]])
    return orc.OracleParams(n, S, L, N, P, chim, kappa, 0.5, **kw)


def test_bond_force_closed_form_and_minimum_image():
    L = (8.0, 8.0, 8.0)
    x = np.array([[0.2, 4.0, 4.0], [7.9, 4.5, 3.0], [1.0, 1.0, 1.0]])
    bp = np.array([[-1, 1], [0, -1], [-1, -1]], dtype=np.int32)
    p = _p(3, k_bond=1.5, r0_bond=0.0)
    f = orc.bond_force(p, x, bp)
    d = np.array([0.2 - 7.9 + 8.0, -0.5, 1.0])                  # minimum image across the x boundary
    assert np.allclose(f[0], -2 * 1.5 * d, atol=1e-13)
    assert np.allclose(f[1], +2 * 1.5 * d, atol=1e-13)
    assert np.allclose(f[2], 0.0)
    # rest length r0: F = -2k (1 - r0/|d|) d
    p2 = _p(3, k_bond=2.0, r0_bond=0.7)
    f2 = orc.bond_force(p2, x, bp)
    r = np.linalg.norm(d)
    assert np.allclose(f2[0], -2 * 2.0 * (1 - 0.7 / r) * d, atol=1e-13)


def test_bond_forces_sum_to_zero_on_chains():
    from paper_2302_02474_b200 import inputs
    st = inputs.make_state(inputs.C1)
    p = _p(inputs.C1.n, L=inputs.C1.box, N=(4, 4, 4))
    f = orc.bond_force(p, st.x.astype(np.float64), st.bond_partner)
    assert np.abs(f.sum(0)).max() < 1e-10
    # energy derivative: U = k sum_bonds |d|^2  ->  F = -dU/dx by central differences
    x = st.x.astype(np.float64)
    v = np.zeros_like(x)
    p0 = _p(inputs.C1.n, L=inputs.C1.box, N=(4, 4, 4), chi=0.0, kappa=0.0)
    eps = 1e-5
    xp, xm = x.copy(), x.copy()
    xp[37, 2] += eps
    xm[37, 2] -= eps
    dU = (orc.energy(p0, xp, v, st.type, st.bond_partner)[1] - orc.energy(p0, xm, v, st.type, st.bond_partner)[1]) / (2 * eps)
    assert abs(-dU - f[37, 2]) < 1e-6


def _small_melt(seed=3, n_chains=20, nb=6, L=6.0):
    rng = np.random.default_rng(seed)
    start = rng.random((n_chains, 1, 3)) * L
    steps = rng.normal(0, np.sqrt(1 / 3), size=(n_chains, nb, 3))
    steps[:, 0] = 0
    x = (start + np.cumsum(steps, axis=1)).reshape(-1, 3) % L
    n = n_chains * nb
    ty = np.tile(np.repeat([0, 1], nb // 2), n_chains).astype(np.int32)
    ids = np.arange(n).reshape(n_chains, nb)
    prev, nxt = ids - 1, ids + 1
    prev[:, 0] = -1
    nxt[:, -1] = -1
    bp = np.stack([prev.ravel(), nxt.ravel()], 1).astype(np.int32)
    v = rng.normal(size=(n, 3))
    return x.astype(np.float32).astype(np.float64), v, ty, bp


def test_gjf_gamma0_is_velocity_verlet():
    x, v, ty, bp = _small_melt()
    n = x.shape[0]
    L = 6.0
    p = _p(n, L=(L,) * 3, N=(12,) * 3, P=3, gamma=0.0, dt=0.01)
    xo, vo, fo = orc.run(p, x, v, ty, bp, 0, 5)
    # velocity Verlet written out (Swope et al. 1982), force from the oracle's force routine
    xv, vv = x.copy(), v.copy()
    f = orc.force(p, xv, ty, bp)
    dt = 0.01
    for _ in range(5):
        vv = vv + 0.5 * dt * f
        xv = xv + dt * vv
        xv = xv - L * np.floor(xv / L)
        f = orc.force(p, xv, ty, bp)
        vv = vv + 0.5 * dt * f
    assert np.abs(xo - xv).max() < 1e-12
    assert np.abs(vo - vv).max() < 1e-11


def test_energy_error_scales_as_dt_squared():
    x, v, ty, bp = _small_melt(seed=5)
    n = x.shape[0]
    L = 6.0
    T = 0.32
    devs = []
    for dt in (0.02, 0.01):
        p = _p(n, L=(L,) * 3, N=(16,) * 3, P=4, gamma=0.0, dt=dt, kappa=5.0, chi=1.0)
        e0 = orc.energy(p, x, v, ty, bp).sum()
        es = []
        xc, vc, fc = x, v, None
        nst = int(round(T / dt))
        chunk = max(1, nst // 8)
        for s in range(0, nst, chunk):
            xc, vc, fc = orc.run(p, xc, vc, ty, bp, s, chunk, f=fc)
            es.append(orc.energy(p, xc, vc, ty, bp).sum())
        devs.append(np.abs(np.array(es) - e0).max())
    ratio = devs[0] / devs[1]
    assert 2.5 < ratio < 6.5, (devs, ratio)
    assert devs[1] < 1e-2 * abs(e0) + 1.0


def test_noise_is_keyed_by_id_and_step_and_has_gjf_variance():
    p = _p(4, gamma=2.0, kT=1.5, dt=0.01, seed=123456789012345)
    a = orc.noise(p, 7, 3)
    assert np.array_equal(a, orc.noise(p, 7, 3))
    assert not np.array_equal(a, orc.noise(p, 8, 3))
    assert not np.array_equal(a, orc.noise(p, 7, 4))
    z = np.array([orc.normals(42, i, 1) for i in range(20000)])
    assert abs(z.mean()) < 0.02
    assert np.abs(z.var(axis=0) - 1.0).max() < 0.04
    assert np.abs(np.corrcoef(z.T) - np.eye(3)).max() < 0.03
    for c in range(3):
        assert stats.kstest(z[:, c], "norm").pvalue > 1e-3
    b = np.array([orc.noise(p, i, 9) for i in range(20000)])
    assert abs(b.var() / (2 * 2.0 * 1.5 * 0.01) - 1) < 0.03


def test_normals_invert_to_the_philox_words_they_were_drawn_from():
    """Reading A12 / SURVEY O9, pinned through the INVERSE of the map (no forward Box-Muller is retyped here): from the
    oracle's normals (z0, z1, z2) of (seed, id, step) the radius gives back u0 = exp(-(z0^2 + z1^2)/2), the polar angle gives
    u1 = atan2(z1, z0) / 2 pi (mod 1), and z2 / sqrt(-2 ln u2) = cos 2 pi u3 gives u3 up to the reflection u -> 1 - u that
    the cosine cannot see.  Every u must be ((x >> 9) + 0.5) 2^-23 of the matching word x of Philox4x32-10 (itself pinned
    bit for bit against cuRAND's header) with counter (id, step lo, step hi, 0) and key (seed lo, seed hi): the top 23 bits
    of the words come back EXACTLY.  A swapped sine / cosine, another word order, a 24-bit or unshifted uniform, a missing
    half, a wrong counter layout: each fails."""
    rng = np.random.default_rng(2302)
    two23 = float(1 << 23)
    for _ in range(400):
        seed = int(rng.integers(0, 2 ** 63))
        pid = int(rng.integers(0, 2 ** 32))
        step = int(rng.integers(0, 2 ** 40))
        z = orc.normals(seed, pid, step)
        x = orc.philox4x32_10([pid, step & 0xFFFFFFFF, step >> 32, 0], [seed & 0xFFFFFFFF, seed >> 32]).astype(np.int64)
        k = x >> 9                                                      # the 23 bits the reading keeps
        u0 = np.exp(-0.5 * (z[0] ** 2 + z[1] ** 2))
        u1 = (np.arctan2(z[1], z[0]) / (2 * np.pi)) % 1.0
        assert abs(u0 * two23 - (k[0] + 0.5)) < 1e-3, (seed, pid, step)
        assert abs(u1 * two23 - (k[1] + 0.5)) < 1e-3, (seed, pid, step)
        u2 = (k[2] + 0.5) / two23
        c = z[2] / np.sqrt(-2.0 * np.log(u2))
        assert abs(c) <= 1.0 + 1e-12
        u3 = np.arccos(min(1.0, max(-1.0, c))) / (2 * np.pi)            # in [0, 1/2]
        want = (k[3] + 0.5) / two23
        want = min(want, 1.0 - want)
        assert abs(u3 - want) * two23 < 0.05, (seed, pid, step)
    # the amplitude of the thermostat noise: beta = sqrt(2 gamma kT dt) z, component by component
    p = _p(4, gamma=2.0, kT=1.5, dt=0.01, seed=987654321987)
    assert np.allclose(orc.noise(p, 11, 5), np.sqrt(2 * 2.0 * 1.5 * 0.01) * orc.normals(987654321987, 11, 5), rtol=1e-14, atol=0)


def test_free_particle_diffusion():
    """No forces (kappa = chi = k_bond = 0): <dr^2> = 6 (kT/gamma) [t - (1 - e^{-gamma t})/gamma] for thermal v0."""
    n = 3000
    rng = np.random.default_rng(2)
    L = 1000.0
    x = np.full((n, 3), 500.0) + rng.random((n, 3))
    v = rng.normal(size=(n, 3))
    ty = np.zeros(n, np.int32)
    bp = -np.ones((n, 2), np.int32)
    gamma, dt, nst = 5.0, 0.02, 200
    p = orc.OracleParams(n, 1, (L,) * 3, (4,) * 3, 1, np.zeros((1, 1)), 0.0, 0.5, k_bond=0.0, gamma=gamma, dt=dt, seed=99)
    x1, v1, _ = orc.run(p, x, v, ty, bp, 0, nst)
    t = dt * nst
    msd = ((x1 - x) ** 2).sum(1).mean()
    exact = 6 * (1.0 / gamma) * (t - (1 - np.exp(-gamma * t)) / gamma)
    assert abs(msd / exact - 1) < 0.06, (msd, exact)
    assert abs((v1 ** 2).mean() - 1.0) < 0.05        # kinetic temperature kT/m = 1 (dt-dependent bias is O(dt^2))


def test_harmonic_dimer_samples_boltzmann():
    """U = k r^2 -> <r^2> = 3 kT/(2k) = 1 for k = 1.5 (Eq. 2: b = 1)."""
    nd = 1500
    rng = np.random.default_rng(6)
    L = 1000.0
    c = rng.random((nd, 1, 3)) * 900 + 50
    x = (c + rng.normal(0, 0.4, size=(nd, 2, 3))).reshape(-1, 3)
    n = 2 * nd
    v = rng.normal(size=(n, 3))
    ty = np.zeros(n, np.int32)
    ids = np.arange(n).reshape(nd, 2)
    bp = -np.ones((n, 2), np.int32)
    bp[ids[:, 0], 1] = ids[:, 1]
    bp[ids[:, 1], 0] = ids[:, 0]
    p = orc.OracleParams(n, 1, (L,) * 3, (4,) * 3, 1, np.zeros((1, 1)), 0.0, 0.5, k_bond=1.5, gamma=2.0, dt=0.1, seed=5)
    xc, vc, fc = orc.run(p, x, v, ty, bp, 0, 100)
    r2 = []
    for k in range(6):
        xc, vc, fc = orc.run(p, xc, vc, ty, bp, 100 + 20 * k, 20, f=fc)
        d = xc[ids[:, 0]] - xc[ids[:, 1]]
        r2.append((d ** 2).sum(1).mean())
    assert abs(np.mean(r2) - 1.0) < 0.05, r2


@pytest.fixture(scope="module")
def curand_host(tmp_path_factory):
    if shutil.which("nvcc") is None:
        pytest.skip("nvcc not available to host-compile cuRAND's Philox header")
    out = str(tmp_path_factory.mktemp("philox") / "libphilox_curand_host.so")
    src = os.path.join(HERE, "helpers", "philox_curand_host.cu")
    subprocess.run(["nvcc", "-O1", "-Wno-deprecated-gpu-targets", "-shared", "-Xcompiler", "-fPIC", src, "-o", out],
                   check=True, capture_output=True)
    return C.CDLL(out)


def test_philox_matches_curand_header(curand_host):
    rng = np.random.default_rng(77)
    U = C.POINTER(C.c_uint32)
    cases = [(np.zeros(4, np.uint32), np.zeros(2, np.uint32)),
             (np.full(4, 0xFFFFFFFF, np.uint32), np.full(2, 0xFFFFFFFF, np.uint32))]
    for _ in range(500):
        cases.append((rng.integers(0, 2 ** 32, size=4, dtype=np.uint64).astype(np.uint32),
                      rng.integers(0, 2 ** 32, size=2, dtype=np.uint64).astype(np.uint32)))
    for ctr, key in cases:
        ref = np.zeros(4, np.uint32)
        curand_host.curand_philox_host(ctr.ctypes.data_as(U), key.ctypes.data_as(U), ref.ctypes.data_as(U))
        assert np.array_equal(orc.philox4x32_10(ctr, key), ref)


# ---- Euler-Maruyama (reading A11b) --------------------------------------------------------------------
def test_em_one_step_is_the_explicit_formula_with_the_gjf_noise():
    """r' = r + (dt/gamma) F + beta/gamma with beta the SAME noise GJF would draw for (id, step + 1); v untouched."""
    rng = np.random.default_rng(4)
    n, L = 40, (6.0, 5.0, 7.0)
    x = rng.random((n, 3)) * np.array(L)
    v = rng.normal(size=(n, 3))
    ty = rng.integers(0, 2, size=n).astype(np.int32)
    bp = -np.ones((n, 2), np.int32)
    bp[1:, 0] = np.arange(n - 1)
    bp[:-1, 1] = np.arange(1, n)
    p = orc.OracleParams(n, 2, L, (12, 10, 14), 3, np.array([[0, 1.0], [1.0, 0]]), 5.0, 0.5, gamma=2.0, dt=0.01, seed=7,
                         integrator=1)
    f0 = orc.force(p, x.astype(np.float32).astype(np.float64), ty, bp)
    x0 = x.astype(np.float32).astype(np.float64)
    x1, v1, f1 = orc.run(p, x0, v, ty, bp, 11, 1)
    beta = np.array([orc.noise(p, i, 12) for i in range(n)])
    want = x0 + (p.dt / p.gamma) * f0 + beta / p.gamma
    want -= np.array(L) * np.floor(want / np.array(L))
    assert np.abs(x1 - want).max() < 1e-12
    assert np.array_equal(v1, v)
    assert np.abs(f1 - orc.force(p, x1, ty, bp)).max() < 1e-12


def test_em_free_diffusion_and_dimer_stationary_variance():
    """No forces: every step adds N(0, 2 kT dt/gamma) per component, so <dr^2> = 6 (kT/gamma) t exactly in expectation.
    Harmonic dimer U = k d^2: the relative coordinate obeys d' = (1 - 4 k dt/gamma) d + noise of variance 4 kT dt/gamma,
    whose stationary variance per component is (4 kT dt/gamma) / (1 - (1 - 4 k dt/gamma)^2) (the finite-dt EM bias)."""
    n = 4000
    rng = np.random.default_rng(12)
    L = 1000.0
    x = np.full((n, 3), 500.0) + rng.random((n, 3))
    ty = np.zeros(n, np.int32)
    gamma, dt, nst = 2.0, 0.01, 100
    p = orc.OracleParams(n, 1, (L,) * 3, (4,) * 3, 1, np.zeros((1, 1)), 0.0, 0.5, k_bond=0.0, gamma=gamma, dt=dt, seed=3,
                         integrator=1)
    x1, _, _ = orc.run(p, x, np.zeros_like(x), ty, -np.ones((n, 2), np.int32), 0, nst)
    msd = ((x1 - x) ** 2).sum(1).mean()
    assert abs(msd / (6 * dt * nst / gamma) - 1) < 0.04, msd
    nd, k = 2000, 1.5
    c = rng.random((nd, 1, 3)) * 900 + 50
    xd = (c + rng.normal(0, 0.4, size=(nd, 2, 3))).reshape(-1, 3)
    bp = np.stack([np.arange(2 * nd) ^ 1, -np.ones(2 * nd, int)], axis=1).astype(np.int32)
    dt = 0.02
    q = orc.OracleParams(2 * nd, 1, (L,) * 3, (4,) * 3, 1, np.zeros((1, 1)), 0.0, 0.5, k_bond=k, gamma=gamma, dt=dt, seed=8,
                         integrator=1)
    xe, _, _ = orc.run(q, xd, np.zeros_like(xd), np.zeros(2 * nd, np.int32), bp, 0, 400)
    d = (xe[0::2] - xe[1::2])
    a = 1 - 4 * k * dt / gamma
    var = (4 * dt / gamma) / (1 - a * a)
    assert abs((d ** 2).mean() / var - 1) < 0.05, ((d ** 2).mean(), var)


# ---- cosine (wormlike-chain) angle potential, Eq. 16 L213 (reading A23) ----------------------
def _chain_partners(n_chains, nb):
    ids = np.arange(n_chains * nb).reshape(n_chains, nb)
    prev, nxt = ids - 1, ids + 1
    prev[:, 0] = -1
    nxt[:, -1] = -1
    return np.stack([prev.reshape(-1), nxt.reshape(-1)], axis=1).astype(np.int32)


def test_wlc_angle_force_is_minus_the_energy_gradient_and_conserves_momentum_and_torque():
    rng = np.random.default_rng(14)
    n_chains, nb, L = 3, 6, (7.0, 8.0, 9.0)
    n = n_chains * nb
    x = (rng.random((n_chains, 1, 3)) * np.array(L) + np.cumsum(rng.normal(0, 0.6, (n_chains, nb, 3)), axis=1)).reshape(-1, 3)
    x -= np.array(L) * np.floor(x / np.array(L))                       # some chains cross the periodic boundary
    bp = _chain_partners(n_chains, nb)
    p = orc.OracleParams(n, 1, L, (8, 8, 8), 2, np.zeros((1, 1)), 0.0, 0.5, k_bond=0.0, lambda_wlc=2.3)
    F = orc.bond_force(p, x, bp)
    ty, v = np.zeros(n, np.int32), np.zeros((n, 3))
    eps = 1e-6
    for i in (0, 1, 5, 7, 9, 17):
        for a in range(3):
            xp, xm = x.copy(), x.copy()
            xp[i, a] += eps
            xm[i, a] -= eps
            dE = (orc.energy(p, xp, v, ty, bp)[1] - orc.energy(p, xm, v, ty, bp)[1]) / (2 * eps)
            assert abs(F[i, a] + dE) < 1e-6 * max(1.0, np.abs(F).max()), (i, a, F[i, a], -dE)
    assert np.abs(F.sum(0)).max() < 1e-12 * max(1.0, np.abs(F).max())
    # torque about the chain's first bead (minimum-image unwrapped chain) vanishes chain by chain
    for c in range(n_chains):
        sl = slice(c * nb, (c + 1) * nb)
        r = x[sl] - x[c * nb]
        r -= np.array(L) * np.round(r / np.array(L))
        assert np.abs(np.cross(r, F[sl]).sum(0)).max() < 1e-9


def test_wlc_angle_special_cases():
    """Straight trimer: cos = -1, u = 0, no force.  Right angle with unit bonds: u = lambda; the end beads are pushed
    so as to open the angle with |F| = lambda / |d| (d cos/d r_i = d2_hat / |d1| at cos = 0)."""
    L = (20.0,) * 3
    bp = _chain_partners(1, 3)
    ty, v = np.zeros(3, np.int32), np.zeros((3, 3))
    p = orc.OracleParams(3, 1, L, (8, 8, 8), 2, np.zeros((1, 1)), 0.0, 0.5, k_bond=0.0, lambda_wlc=1.7)
    straight = np.array([[4.0, 5, 5], [5.0, 5, 5], [6.5, 5, 5]])
    assert np.abs(orc.bond_force(p, straight, bp)).max() < 1e-12 and abs(orc.energy(p, straight, v, ty, bp)[1]) < 1e-12
    right = np.array([[5.0, 6, 5], [5.0, 5, 5], [6.0, 5, 5]])
    F = orc.bond_force(p, right, bp)
    assert abs(orc.energy(p, right, v, ty, bp)[1] - 1.7) < 1e-12
    assert np.allclose(F[0], [-1.7, 0, 0]) and np.allclose(F[2], [0, -1.7, 0]) and np.allclose(F[1], [1.7, 1.7, 0])


def test_harmonic_angle_force_is_minus_the_energy_gradient_and_special_cases():
    """PAPER.md Eq. 17: u_h = k_theta (theta - theta0)^2.  Gradient check, conservation laws, and a right-angle
    trimer with theta0 = pi/3: U = k (pi/2 - pi/3)^2, end-bead force magnitude 2 k (theta - theta0) / |d|, closing the angle (theta > theta0: each end bead is pushed towards the other arm)."""
    rng = np.random.default_rng(15)
    n_chains, nb, L = 3, 6, (7.0, 8.0, 9.0)
    n = n_chains * nb
    x = (rng.random((n_chains, 1, 3)) * np.array(L) + np.cumsum(rng.normal(0, 0.6, (n_chains, nb, 3)), axis=1)).reshape(-1, 3)
    x -= np.array(L) * np.floor(x / np.array(L))
    bp = _chain_partners(n_chains, nb)
    p = orc.OracleParams(n, 1, L, (8, 8, 8), 2, np.zeros((1, 1)), 0.0, 0.5, k_bond=0.0, k_theta=1.3, theta0=2.0, lambda_wlc=0.4)
    F = orc.bond_force(p, x, bp)
    ty, v = np.zeros(n, np.int32), np.zeros((n, 3))
    eps = 1e-6
    for i in (0, 2, 6, 8, 11, 16):
        for a in range(3):
            xp, xm = x.copy(), x.copy()
            xp[i, a] += eps
            xm[i, a] -= eps
            dE = (orc.energy(p, xp, v, ty, bp)[1] - orc.energy(p, xm, v, ty, bp)[1]) / (2 * eps)
            assert abs(F[i, a] + dE) < 2e-6 * max(1.0, np.abs(F).max()), (i, a, F[i, a], -dE)
    assert np.abs(F.sum(0)).max() < 1e-12 * max(1.0, np.abs(F).max())
    q = orc.OracleParams(3, 1, (20.0,) * 3, (8, 8, 8), 2, np.zeros((1, 1)), 0.0, 0.5, k_bond=0.0, k_theta=1.5, theta0=np.pi / 3)
    right = np.array([[5.0, 6, 5], [5.0, 5, 5], [6.0, 5, 5]])
    b3 = _chain_partners(1, 3)
    assert abs(orc.energy(q, right, np.zeros((3, 3)), np.zeros(3, np.int32), b3)[1] - 1.5 * (np.pi / 6) ** 2) < 1e-12
    Fr = orc.bond_force(q, right, b3)
    mag = 2 * 1.5 * (np.pi / 2 - np.pi / 3)
    assert np.allclose(Fr[0], [mag, 0, 0]) and np.allclose(Fr[2], [0, mag, 0]) and np.allclose(Fr[1], [-mag, -mag, 0])
    at_rest = orc.OracleParams(3, 1, (20.0,) * 3, (8, 8, 8), 2, np.zeros((1, 1)), 0.0, 0.5, k_bond=0.0, k_theta=1.5, theta0=np.pi / 2)
    assert np.abs(orc.bond_force(at_rest, right, b3)).max() < 1e-12
