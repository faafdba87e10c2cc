"""Pins for the SURVEY 8(f) remainder in the oracle (round 2): velocity Verlet + Langevin ExtraForce (reading A24), the
pressure virial, per-particle charges (A25), the Maier-Saupe interaction (A26, Eq. 19-20) and 2-D mode (A27).
Everything the oracle is compared with here is written out independently: closed forms, finite differences of the
(separately pinned) energies, brute-force sums."""
import numpy as np
import pytest

from oracle import tild_oracle as orc
from test_oracle_force import CHI3, discrete_transfer, ewald_smeared_force, ksum_force
from test_oracle_force import ewald_smeared_energy

NOBOND = lambda n: -np.ones((n, 2), dtype=np.int32)


# ---- velocity Verlet + Langevin ExtraForce (A24) ---------------------------------------------------------------------
def free_params(n, integrator, gamma, dt=0.01, kT=1.3, mass=0.7, seed=5):
    return orc.OracleParams(n, 1, (9.0, 9.0, 9.0), (8, 8, 8), 2, np.zeros((1, 1)), kappa=0.0, sigma2=0.5, rho0=1.0, k_bond=0.0,
                            dt=dt, gamma=gamma, kT=kT, mass=mass, seed=seed, integrator=integrator)


def test_vv_without_friction_is_the_gjf_limit_velocity_verlet():
    rng = np.random.default_rng(1)
    n = 60
    L, N = (6.0, 4.5, 7.0), (12, 8, 10)
    x = rng.random((n, 3)) * np.array(L)
    v = rng.normal(size=(n, 3))
    ty = rng.integers(0, 3, size=n).astype(np.int32)
    bp = NOBOND(n)
    bp[1:, 0] = np.arange(n - 1)
    bp[:-1, 1] = np.arange(1, n)
    kw = dict(kappa=5.0, sigma2=0.5, rho0=2.0, gamma=0.0, dt=0.01)
    a = orc.run(orc.OracleParams(n, 3, L, N, 3, CHI3, integrator=0, **kw), x, v, ty, bp, 0, 7)
    b = orc.run(orc.OracleParams(n, 3, L, N, 3, CHI3, integrator=2, **kw), x, v, ty, bp, 0, 7)
    assert np.abs(a[0] - b[0]).max() < 1e-12 and np.abs(a[1] - b[1]).max() < 1e-12


def test_vv_langevin_one_step_is_the_formula_with_the_gjf_noise():
    """Free particles: v' = (1 - g)^2 v + (2 - g) beta / 2m,  x' = x + dt [(1 - g) v + beta / 2m],  g = gamma dt / 2m."""
    n = 40
    p = free_params(n, 2, gamma=2.0)
    rng = np.random.default_rng(2)
    x = rng.random((n, 3)) * 9.0
    v = rng.normal(size=(n, 3))
    ty = np.zeros(n, np.int32)
    x1, v1, _ = orc.run(p, x, v, ty, NOBOND(n), 11, 1)
    g = p.gamma * p.dt / (2 * p.mass)
    beta = np.array([orc.noise(p, i, 12) for i in range(n)])
    assert np.abs(v1 - ((1 - g) ** 2 * v + (2 - g) * beta / (2 * p.mass))).max() < 1e-13
    xe = (x + p.dt * ((1 - g) * v + beta / (2 * p.mass))) % 9.0
    assert np.abs(x1 - xe).max() < 1e-12


def test_vv_langevin_fluctuation_dissipation_and_free_diffusion():
    """Stationary velocity variance of the scheme in closed form, sigma^2 = (2 - g)^2 g (kT/m) / (1 - (1 - g)^4) -> kT/m, and
    the long-time mean squared displacement 6 (kT/gamma) t."""
    n, steps = 4000, 400
    p = free_params(n, 2, gamma=4.0, dt=0.02, kT=1.3, mass=0.7)
    x = np.full((n, 3), 4.5)
    v = np.zeros((n, 3))
    ty = np.zeros(n, np.int32)
    bp = NOBOND(n)
    x1, v1, _ = orc.run(p, x, v, ty, bp, 0, steps)
    g = p.gamma * p.dt / (2 * p.mass)
    var = (2 - g) ** 2 * g * (p.kT / p.mass) / (1 - (1 - g) ** 4)
    assert abs(var / (p.kT / p.mass) - 1) < 0.6 * g                     # the scheme's own bias is O(gamma dt): g / 2 to first order
    assert abs(v1.var() / var - 1) < 0.03, (v1.var(), var)
    # unwrapped displacement: run again in a huge box so that nothing wraps
    big = orc.OracleParams(n, 1, (1e4,) * 3, (8, 8, 8), 2, np.zeros((1, 1)), kappa=0.0, sigma2=0.5, rho0=1.0, k_bond=0.0,
                           dt=p.dt, gamma=p.gamma, kT=p.kT, mass=p.mass, seed=5, integrator=2)
    x0 = np.full((n, 3), 5e3)
    xa, va, _ = orc.run(big, x0, v, ty, bp, 0, 200)
    xb, _, _ = orc.run(big, xa, va, ty, bp, 200, steps)
    msd = ((xb - xa) ** 2).sum(1).mean()
    assert abs(msd / (6 * p.kT / p.gamma * steps * p.dt) - 1) < 0.06, msd


# ---- pressure virial ---------------------------------------------------------------------------------------------
def scaled(p, lam, **kw):
    from dataclasses import replace
    return replace(p, L=tuple(lam * l for l in p.L), **kw)


@pytest.mark.parametrize("variant", ["plain", "electrostatics", "ms_and_pp_charges"])
def test_virial_is_minus_the_derivative_of_the_energy_under_affine_scaling(variant):
    rng = np.random.default_rng(31)
    n = 90
    L, N = (6.0, 4.5, 7.0), (12, 10, 14)
    x = rng.random((n, 3)) * np.array(L)
    v = np.zeros((n, 3))
    ty = rng.integers(0, 3, size=n).astype(np.int32)
    bp = NOBOND(n)
    for c in range(0, n - 3, 3):
        bp[c, 1], bp[c + 1, 0], bp[c + 1, 1], bp[c + 2, 0] = c + 1, c, c + 2, c + 1
    kw = dict(kappa=5.0, sigma2=0.5, rho0=2.0, k_bond=1.7, r0_bond=0.4, lambda_wlc=0.6)
    if variant == "electrostatics":
        kw.update(charge=(1.0, -1.0, 0.0), bjerrum=1.5, a_charge=0.45, deconvolve=True)
    if variant == "ms_and_pp_charges":
        msp = -np.ones(n, dtype=np.int32)
        msp[0:n - 3:3] = np.arange(1, n - 2, 3)
        kw.update(q_pp=rng.normal(size=n), bjerrum=0.8, a_charge=0.5, mu_ms=1.3, ms_partner=msp)
    p = orc.OracleParams(n, 3, L, N, 4, CHI3, **kw)
    w = orc.virial(p, x, ty, bp)
    eps = 2e-4
    ep = orc.energy(scaled(p, 1 + eps), x * (1 + eps), v, ty, bp)
    em = orc.energy(scaled(p, 1 - eps), x * (1 - eps), v, ty, bp)
    d = (ep - em) / (2 * eps)
    assert abs(w[0] + d[1]) < 2e-5 * max(1.0, abs(d[1])), (w[0], -d[1])       # rho0 is a parameter, not n/V: kept fixed
    assert abs(w[1] + d[2]) < 2e-4 * max(1.0, abs(d[2])), (w[1], -d[2])       # positions pass through fp32 in the mesh part


# ---- per-particle charges (A25) ----------------------------------------------------------------------------------
def test_per_particle_charges_reduce_to_species_charges_and_match_ewald():
    rng = np.random.default_rng(11)
    L = (6.0, 6.0, 6.0)
    n, lB, aq = 8, 2.5, 0.5
    x = (rng.random((n, 3)) * 6.0).astype(np.float32)
    ty = np.array([0, 1] * (n // 2), dtype=np.int32)
    zsp = (1.0, -1.0)
    base = dict(kappa=3.0, sigma2=0.5, rho0=1.0, bjerrum=lB, a_charge=aq, k_bond=0.0)
    chi = np.array([[0.0, 0.8], [0.8, 0.0]])
    a = orc.force(orc.OracleParams(n, 2, L, (16,) * 3, 4, chi, charge=zsp, **base), x, ty, NOBOND(n))
    b = orc.force(orc.OracleParams(n, 2, L, (16,) * 3, 4, chi, q_pp=np.array([zsp[t] for t in ty]), **base), x, ty, NOBOND(n))
    assert np.abs(a - b).max() < 1e-11 * np.abs(a).max()
    # arbitrary charges (net charge allowed: the k = 0 mode is dropped) against the Ewald sum written in test_oracle_force
    q = rng.normal(size=n)
    ref = ewald_smeared_force(x, q, L, lB, aq, alpha=0.7 / (2 * aq))
    eref = ewald_smeared_energy(x, q, L, lB, aq, alpha=0.7 / (2 * aq))
    assert abs(eref - ewald_smeared_energy(x, q, L, lB, aq, alpha=1.0 / (2 * aq))) < 1e-9 * abs(eref)   # net charge included
    errs, eerrs = [], []
    for Ng in (24, 48):
        p = orc.OracleParams(n, 2, L, (Ng,) * 3, 4, np.zeros((2, 2)), kappa=0.0, sigma2=0.5, rho0=1.0, q_pp=q, bjerrum=lB,
                             a_charge=aq, deconvolve=True, k_bond=0.0)
        F = orc.force(p, x, ty, NOBOND(n))
        errs.append(np.abs(F - ref).max() / np.abs(ref).max())
        e = orc.energy(p, x.astype(np.float64), np.zeros((n, 3)), ty, NOBOND(n))
        eerrs.append(abs(e[2] - eref) / abs(eref))
    assert errs[0] < 2e-3 and errs[1] < 1e-4, errs
    assert eerrs[0] < 2e-3 and eerrs[1] < 1e-4, eerrs


# ---- Maier-Saupe (A26; Eq. 19-20) -----------------------------------------------------------------------
def ms_system(rng, n_c=14, L=(6.0, 5.0, 7.0)):
    """n_c LC centres, each with its own partner bead 0.6-1.0 away: particles 2i (centre) and 2i + 1 (partner)."""
    n = 2 * n_c
    x = np.zeros((n, 3))
    x[0::2] = rng.random((n_c, 3)) * np.array(L)
    d = rng.normal(size=(n_c, 3))
    d *= (0.6 + 0.4 * rng.random((n_c, 1))) / np.linalg.norm(d, axis=1, keepdims=True)
    x[1::2] = (x[0::2] + d) % np.array(L)
    msp = -np.ones(n, dtype=np.int32)
    msp[0::2] = np.arange(1, n, 2)
    return x, msp


def ms_params(n, L, N, msp, mu=1.4, P=4, **kw):
    return orc.OracleParams(n, 1, L, N, P, np.zeros((1, 1)), kappa=0.0, sigma2=0.5, rho0=2.0, k_bond=0.0, mu_ms=mu,
                            ms_partner=msp, **kw)


def test_ms_orientation_force_is_the_exact_gradient_and_momentum_is_conserved():
    """Moving only the partner bead j changes nothing but u_i: the mesh energy depends on it through S_i alone, and the
    gather is the adjoint of the spread, so F_j = -dU/dr_j holds to finite-difference accuracy on ANY mesh."""
    rng = np.random.default_rng(3)
    L, N = (6.0, 5.0, 7.0), (12, 10, 14)
    x, msp = ms_system(rng)
    n = len(x)
    p = ms_params(n, L, N, msp)
    ty = np.zeros(n, np.int32)
    x32 = x.astype(np.float32).astype(np.float64)
    F = orc.force(p, x32, ty, NOBOND(n))
    assert np.abs(F.sum(0)).max() < 1e-11 * np.abs(F).max() * n
    assert np.abs(F).max() > 1e-3
    eps = 1e-5
    for j in (1, 7, 13):
        for a in range(3):
            xp, xm = x32.copy(), x32.copy()
            xp[j, a] += eps
            xm[j, a] -= eps
            # the mesh part reads fl32(x): keep the partner's move out of it by moving a bead that carries no S
            dE = (orc.energy(p, xp, np.zeros((n, 3)), ty, NOBOND(n))[2] - orc.energy(p, xm, np.zeros((n, 3)), ty, NOBOND(n))[2]) / (2 * eps)
            assert abs(-dE - F[j, a]) < 1e-6 * np.abs(F).max(), (j, a, -dE, F[j, a])


def test_ms_position_force_converges_to_the_energy_gradient_under_refinement():
    rng = np.random.default_rng(4)
    L = (6.0, 6.0, 6.0)
    x, msp = ms_system(rng, n_c=10, L=L)
    n = len(x)
    ty = np.zeros(n, np.int32)
    rel = []
    for Ng in (12, 24):
        p = ms_params(n, L, (Ng,) * 3, msp)
        F = orc.force(p, x, ty, NOBOND(n))
        eps = 1e-3
        i = 4                                                      # a centre: move it together with its partner (u fixed)
        xp, xm = x.copy(), x.copy()
        for k in (i, i + 1):
            xp[k, 1] += eps
            xm[k, 1] -= eps
        dE = (orc.energy(p, xp, np.zeros((n, 3)), ty, NOBOND(n))[2] - orc.energy(p, xm, np.zeros((n, 3)), ty, NOBOND(n))[2]) / (2 * eps)
        rel.append(abs(-dE - (F[i, 1] + F[i + 1, 1])) / np.abs(F).max())
    assert rel[1] < 0.02 and rel[1] < rel[0], rel


def test_ms_pair_energy_matches_the_continuum_expression():
    """Two centres: U = -(mu/rho0) [ 2 (S_1 : S_2) u_G(r_12) + (S_1 : S_1 + S_2 : S_2) u_G(0) ] with S : S' = (u.u')^2 - 1/3
    (Eq. 20 with Eq. 19 inserted), approached by the mesh energy with the deconvolved kernel as the mesh is refined."""
    L = (8.0, 8.0, 8.0)
    x = np.array([[3.1, 4.2, 3.9], [3.1 + 0.8, 4.2, 3.9], [4.0, 3.6, 4.4], [4.0, 3.6 + 0.48, 4.4 + 0.64]])
    msp = np.array([1, -1, 3, -1], dtype=np.int32)
    u1, u2 = np.array([-1.0, 0, 0]), np.array([0, -0.6, -0.8])
    r12 = np.linalg.norm(x[0] - x[2])
    sigma2, mu, rho0 = 0.5, 1.4, 2.0
    uG = lambda r: (2 * np.pi * sigma2) ** -1.5 * np.exp(-r * r / (2 * sigma2))
    U = -(mu / rho0) * (2 * ((u1 @ u2) ** 2 - 1 / 3) * uG(r12) + 2 * (2 / 3) * uG(0.0))
    errs = []
    for Ng in (16, 32):
        p = ms_params(4, L, (Ng,) * 3, msp, mu=mu, deconvolve=True)
        e = orc.energy(p, x, np.zeros((4, 3)), np.zeros(4, np.int32), NOBOND(4))[2]
        errs.append(abs(e - U) / abs(U))
    assert errs[1] < 2e-3 and errs[1] < errs[0], (errs, U)


# ---- 2-D mode (A27) ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("P", [2, 3, 4])
def test_two_dimensional_lattice_particles_equal_the_2d_ksum(P):
    """N_z = 1: every z node is node 0 and the z weights sum to one, so the mesh sums are those of a two-dimensional
    system of area density n / (Lx Ly) in a slab of thickness Lz.  Particles at stencil centres in x and y: exact."""
    rng = np.random.default_rng(200 + P)
    L, N = (6.0, 4.5, 1.0), (12, 8, 1)
    h = np.array(L[:2]) / np.array(N[:2])
    n = 12
    cells = np.stack([rng.integers(0, N[a], size=n) for a in range(2)], axis=1)
    off = 0.0 if P % 2 == 1 else 0.5
    x = np.zeros((n, 3))
    x[:, :2] = (cells + off) * h
    x[:, 2] = rng.random(n)                                         # z is irrelevant
    x = x.astype(np.float32).astype(np.float64)
    ty = rng.integers(0, 3, size=n).astype(np.int32)
    p = orc.OracleParams(n, 3, L, N, P, CHI3, kappa=5.0, sigma2=0.5, rho0=2.0, k_bond=0.0, dim2=True)
    F = orc.force(p, x, ty, NOBOND(n))
    d1 = discrete_transfer(P)
    T2 = lambda KX, KY, KZ, hh: d1(KX, KY, np.zeros_like(KZ), hh)   # no smoothing along z (k_z = 0 only)
    ref = ksum_force(x, ty, L, N, CHI3, 5.0, 2.0, 0.5, T2)
    scale = np.sqrt((ref ** 2).sum(1).mean())
    assert scale > 1e-3 and np.abs(F[:, 2]).max() == 0.0
    assert np.abs(F[:, :2] - ref[:, :2]).max() < 2e-6 * scale


def test_two_dimensional_dynamics_stay_in_the_plane():
    rng = np.random.default_rng(9)
    n = 50
    L, N = (6.0, 4.5, 1.0), (12, 8, 1)
    x = rng.random((n, 3)) * np.array(L)
    v = rng.normal(size=(n, 3))
    v[:, 2] = 0.0
    ty = rng.integers(0, 3, size=n).astype(np.int32)
    for integ in (0, 1, 2):
        p = orc.OracleParams(n, 3, L, N, 3, CHI3, kappa=5.0, sigma2=0.5, rho0=2.0, k_bond=0.0, dim2=True, integrator=integ)
        x1, v1, _ = orc.run(p, x, v, ty, NOBOND(n), 0, 5)
        assert np.array_equal(x1[:, 2], x[:, 2]) and np.abs(v1[:, 2]).max() == 0.0
        assert np.abs(x1[:, :2] - x[:, :2]).max() > 1e-3
