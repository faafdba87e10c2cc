"""Pins for the oracle's particle-mesh non-bonded force (O3-O7): normalisation, signs, pair
coefficients c_IJ, axis order, Nyquist handling.

What fixes the result (Eq. 3-4, u_G L121, Eq. 18):
  the exact force of the model is  F_i = sum_j c_{I J} (d / sigma^2) u_G(|d|),  d = r_i - r_j (all
  periodic images), which in Fourier space is  F_i = -(1/V) sum_k i k u^(k) sum_J c_IJ S_J(k) e^{ik.r_i}.
  The particle-mesh result differs from it only through the assignment function W:
  (a) for particles sitting exactly at stencil centres the mesh sums are closed forms, so PM must equal
      a mesh-free k-sum with the discrete transfer factor D(k)^2 to round-off, for every P;
  (b) for general positions PM equals the k-sum with W^(k)^2 = prod sinc(k h/2)^(2P) up to aliasing,
      which falls quickly with P and under grid refinement;
  (c) PM converges to the bare analytic pair force as O(h^2);
  (d) the net non-bonded force is zero.
The k-sums and pair sums below are brute force written from those formulas, independent of the oracle.
"""
import numpy as np
import pytest

from oracle import tild_oracle as orc


def c_matrix(chi, kappa, rho0):
    S = chi.shape[0]
    c = np.full((S, S), kappa / rho0)
    for i in range(S):
        for j in range(S):
            if i != j:
                c[i, j] += chi[i, j] / rho0
    return c


def ksum_force(x, ty, L, N, chi, kappa, rho0, sigma2, transfer):
    """F_i = -(1/V) sum_m i k_grad u^(k) T(k) sum_J c_IJ S_J(k) exp(i k.r_i) over the grid's mode set.
    transfer(kx, ky, kz, h) -> T(k).  Nyquist modes: +pi N/L in u^, 0 in the gradient factor (A6)."""
    x = np.asarray(x, dtype=np.float64)
    L = np.asarray(L, dtype=np.float64)
    V = L.prod()
    S = chi.shape[0]
    c = c_matrix(chi, kappa, rho0)
    ks, kg = [], []
    for a in range(3):
        m = np.arange(N[a])
        mt = np.where(m <= N[a] // 2, m, m - N[a])
        k = 2 * np.pi * mt / L[a]
        g = k.copy()
        if N[a] % 2 == 0:
            g[N[a] // 2] = 0.0
        ks.append(k)
        kg.append(g)
    KX, KY, KZ = np.meshgrid(*ks, indexing="ij")
    GX, GY, GZ = np.meshgrid(*kg, indexing="ij")
    uhat = np.exp(-0.5 * sigma2 * (KX ** 2 + KY ** 2 + KZ ** 2))
    T = transfer(KX, KY, KZ, L / np.asarray(N))
    # structure factors S_J(k) = sum_{j in J} exp(-i k.r_j)
    phase = lambda r: np.exp(-1j * (KX * r[0] + KY * r[1] + KZ * r[2]))
    SJ = np.zeros((S,) + KX.shape, dtype=np.complex128)
    for j in range(x.shape[0]):
        SJ[ty[j]] += phase(x[j])
    F = np.zeros((x.shape[0], 3))
    for i in range(x.shape[0]):
        gI = sum(c[ty[i], J] * SJ[J] for J in range(S))
        common = uhat * T * gI * np.conj(phase(x[i]))
        for a, G in enumerate((GX, GY, GZ)):
            F[i, a] = (-(1j * G) * common).sum().real / V
    return F


def direct_pair_force(x, ty, L, chi, kappa, rho0, sigma2, images=2):
    """F_i = sum_j sum_images c_IJ (d/sigma^2) u_G(|d|); self-image terms cancel pairwise."""
    x = np.asarray(x, dtype=np.float64)
    L = np.asarray(L, dtype=np.float64)
    c = c_matrix(chi, kappa, rho0)
    n = x.shape[0]
    F = np.zeros((n, 3))
    rng = range(-images, images + 1)
    norm = (2 * np.pi * sigma2) ** -1.5
    for i in range(n):
        for j in range(n):
            for ax in rng:
                for ay in rng:
                    for az in rng:
                        d = x[i] - x[j] + np.array([ax, ay, az]) * L
                        r2 = (d ** 2).sum()
                        F[i] += c[ty[i], ty[j]] * d / sigma2 * norm * np.exp(-r2 / (2 * sigma2))
    return F


def discrete_transfer(P):
    """Mesh transfer of a particle at its stencil centre (t = 0): sum_j w_j exp(-i k node_j)."""
    def d1(kh):
        if P == 1:
            return np.ones_like(kh)
        if P == 2:
            return np.cos(kh / 2)
        if P == 3:
            return 0.75 + 0.25 * np.cos(kh)
        if P == 4:
            return (23.0 / 24.0) * np.cos(kh / 2) + (1.0 / 24.0) * np.cos(1.5 * kh)
        if P == 5:     # weights at t = 0: {1, 76, 230, 76, 1} / 384 on nodes -2..2
            return 115.0 / 192.0 + (19.0 / 48.0) * np.cos(kh) + (1.0 / 192.0) * np.cos(2 * kh)
        raise ValueError
    return lambda KX, KY, KZ, h: (d1(KX * h[0]) * d1(KY * h[1]) * d1(KZ * h[2])) ** 2


def sinc_transfer(P):
    s = lambda kh: np.sinc(kh / (2 * np.pi))                     # numpy sinc(x) = sin(pi x)/(pi x)
    return lambda KX, KY, KZ, h: (s(KX * h[0]) * s(KY * h[1]) * s(KZ * h[2])) ** (2 * P)


CHI3 = np.array([[0.0, 1.0, 0.3], [1.0, 0.0, 2.0], [0.3, 2.0, 0.0]])


@pytest.mark.parametrize("P", [1, 2, 3, 4, 5])
def test_lattice_particles_equal_closed_form_ksum(P):
    """(a) exact to round-off; non-cubic box and grid so a transposed axis fails."""
    rng = np.random.default_rng(100 + P)
    L, N = (6.0, 4.5, 7.0), (12, 8, 10)
    h = np.array(L) / np.array(N)
    n = 14
    cells = np.stack([rng.integers(0, N[a], size=n) for a in range(3)], axis=1)
    off = 0.0 if P % 2 == 1 else 0.5
    x = ((cells + off) * h).astype(np.float32).astype(np.float64)
    # positions must be exactly representable so that fl32(x * inv_h) gives t = 0: use h-friendly box
    ty = rng.integers(0, 3, size=n).astype(np.int32)
    p = orc.OracleParams(n, 3, L, N, P, CHI3, kappa=5.0, sigma2=0.5, rho0=2.0)
    base, toff, _ = orc.index_map(p, x)
    assert np.abs(toff).max() < 1e-6
    F = orc.nonbonded_force(p, x, ty)
    ref = ksum_force(x, ty, L, N, CHI3, 5.0, 2.0, 0.5, discrete_transfer(P))
    scale = np.sqrt((ref ** 2).sum(1).mean())
    assert scale > 1e-3
    assert np.abs(F - ref).max() < 2e-6 * scale      # fp32 positions: |t| <= 1e-6 instead of exactly 0


@pytest.mark.parametrize("P,bound_coarse,bound_fine", [(2, 0.4, 0.08), (3, 0.08, 0.01), (4, 0.03, 0.0015), (5, 0.02, 0.0005)])
def test_general_positions_vs_sinc_smeared_ksum(P, bound_coarse, bound_fine):
    """(b) PM = k-sum with W^(k)^2 up to aliasing; the error falls by > 2^P when h is halved."""
    rng = np.random.default_rng(7)
    L = (5.0, 5.0, 5.0)
    n = 10
    x = (rng.random((n, 3)) * 5.0).astype(np.float32)
    ty = rng.integers(0, 2, size=n).astype(np.int32)
    chi = np.array([[0.0, 1.0], [1.0, 0.0]])
    errs = []
    for Ng in (8, 16):
        N = (Ng,) * 3
        p = orc.OracleParams(n, 2, L, N, P, chi, kappa=3.0, sigma2=0.5, rho0=2.0)
        F = orc.nonbonded_force(p, x, ty)
        ref = ksum_force(x, ty, L, N, chi, 3.0, 2.0, 0.5, sinc_transfer(P))
        errs.append(np.abs(F - ref).max() / np.sqrt((ref ** 2).sum(1).mean()))
    assert errs[0] < bound_coarse and errs[1] < bound_fine, errs
    assert errs[0] / errs[1] > 2 ** P, errs


def test_single_gaussian_pair_converges_to_analytic_force():
    """(c) one A-B pair, chi = 1, kappa = 0 (SURVEY pins): PM -> (chi/rho0) (d/sigma^2) u_G(d) as O(h^2)."""
    L = (10.0, 10.0, 10.0)
    x = np.array([[4.1, 5.2, 4.9], [4.9, 4.7, 5.3]], dtype=np.float32)
    ty = np.array([0, 1], dtype=np.int32)
    chi = np.array([[0.0, 1.0], [1.0, 0.0]])
    ref = direct_pair_force(x, ty, L, chi, 0.0, 2.0, 0.5, images=1)
    assert np.allclose(ref[0], -ref[1])
    errs = []
    for Ng in (16, 32, 64):
        p = orc.OracleParams(2, 2, L, (Ng,) * 3, 4, chi, kappa=0.0, sigma2=0.5, rho0=2.0)
        F = orc.nonbonded_force(p, x, ty)
        errs.append(np.abs(F - ref).max() / np.abs(ref).max())
    # h = 0.625, 0.3125, 0.156: relative error O(P h^2 / (6 sigma^2)) -> 4x per halving
    assert errs[2] < 0.06, errs
    assert 2.5 < errs[0] / errs[1] < 5.5 and 3.3 < errs[1] / errs[2] < 4.7, errs   # asymptotically 4
    # direction and sign: repulsive along d
    d = (x[0] - x[1]).astype(np.float64)
    assert np.dot(F[0], d) > 0 and np.dot(F[1], d) < 0


def test_direct_pair_sum_equals_full_ksum():
    """The brute-force references agree with each other (periodic Gaussian pair sum == k-sum with T = 1 on a
    mode set large enough that u^ has decayed): ties the k-space convention to real space."""
    rng = np.random.default_rng(1)
    L = (4.0, 4.0, 4.0)
    n = 5
    x = rng.random((n, 3)) * 4.0
    ty = rng.integers(0, 2, size=n).astype(np.int32)
    chi = np.array([[0.0, 0.7], [0.7, 0.0]])
    one = lambda KX, KY, KZ, h: np.ones_like(KX)
    a = ksum_force(x, ty, L, (21, 21, 21), chi, 2.0, 1.5, 0.5, one)     # odd N: no Nyquist special case
    b = direct_pair_force(x, ty, L, chi, 2.0, 1.5, 0.5, images=3)
    assert np.abs(a - b).max() < 1e-9 * np.abs(b).max()


@pytest.mark.parametrize("P", [1, 2, 3, 4, 5])
def test_zero_net_force_and_self_force(P):
    """(d) momentum conservation to round-off (needs A6), and a lone particle feels no force."""
    rng = np.random.default_rng(21)
    L, N = (6.0, 4.5, 7.0), (12, 8, 10)
    n = 200
    x = (rng.random((n, 3)) * np.array(L)).astype(np.float32)
    ty = rng.integers(0, 3, size=n).astype(np.int32)
    p = orc.OracleParams(n, 3, L, N, P, CHI3, kappa=5.0, sigma2=0.5, rho0=2.0)
    F = orc.nonbonded_force(p, x, ty)
    rms = np.sqrt((F ** 2).sum(1).mean())
    assert np.abs(F.sum(0)).max() < 1e-12 * rms * n
    p1 = orc.OracleParams(1, 3, L, N, P, CHI3, kappa=5.0, sigma2=0.5, rho0=2.0)
    F1 = orc.nonbonded_force(p1, x[:1], ty[:1])
    assert np.abs(F1).max() < 1e-13


def test_kappa_only_force_is_species_blind_and_chi_is_antisymmetric_for_pair():
    rng = np.random.default_rng(4)
    L, N = (5.0,) * 3, (10,) * 3
    x = (rng.random((30, 3)) * 5.0).astype(np.float32)
    ty = rng.integers(0, 2, size=30).astype(np.int32)
    zero = np.zeros((2, 2))
    p = orc.OracleParams(30, 2, L, N, 3, zero, kappa=4.0, sigma2=0.5, rho0=2.0)
    Fa = orc.nonbonded_force(p, x, ty)
    Fb = orc.nonbonded_force(p, x, 1 - ty)
    assert np.allclose(Fa, Fb, atol=1e-12)
    # force is linear in the coefficients: F(kappa, chi) = F(kappa, 0) + F(0, chi)
    chi = np.array([[0.0, 1.3], [1.3, 0.0]])
    pc = orc.OracleParams(30, 2, L, N, 3, chi, kappa=0.0, sigma2=0.5, rho0=2.0)
    pkc = orc.OracleParams(30, 2, L, N, 3, chi, kappa=4.0, sigma2=0.5, rho0=2.0)
    assert np.allclose(orc.nonbonded_force(pkc, x, ty), Fa + orc.nonbonded_force(pc, x, ty), atol=1e-11)


def test_force_is_minus_gradient_of_mesh_energy_up_to_discretisation():
    """O10 vs O5-O7: central difference of the mesh energy along a particle coordinate approaches the
    ik-differentiated force as the grid is refined (they are not identical on a mesh)."""
    rng = np.random.default_rng(8)
    L = (5.0,) * 3
    n = 12
    x = (rng.random((n, 3)) * 5.0)
    ty = rng.integers(0, 2, size=n).astype(np.int32)
    chi = np.array([[0.0, 1.0], [1.0, 0.0]])
    bp = -np.ones((n, 2), dtype=np.int32)
    v = np.zeros((n, 3))
    rel = []
    for Ng in (10, 20):
        p = orc.OracleParams(n, 2, L, (Ng,) * 3, 4, chi, kappa=3.0, sigma2=0.5, rho0=2.0, k_bond=0.0)
        F = orc.nonbonded_force(p, x.astype(np.float32), ty)
        eps = 1e-3
        xp, xm = x.copy(), x.copy()
        xp[3, 1] += eps
        xm[3, 1] -= eps
        dE = (orc.energy(p, xp, v, ty, bp)[2] - orc.energy(p, xm, v, ty, bp)[2]) / (2 * eps)
        rel.append(abs(-dE - F[3, 1]) / np.abs(F[3]).max())
    assert rel[1] < 0.02 and rel[1] < rel[0], rel


# ---- assignment-function deconvolution (kernel u^(k) / W^(k)^2) --------------------------------------
def test_deconvolved_kernel_removes_the_assignment_smoothing():
    """Plain PM smears the pair kernel by W^2 (error vs the bare analytic force: tens of percent at h = 0.625,
    growing with P).  Dividing the kernel by W^(k)^2 leaves only aliasing: the error against the BARE analytic
    Gaussian pair force must drop well below the plain error and shrink with the order."""
    L = (10.0, 10.0, 10.0)
    x = np.array([[4.1, 5.2, 4.9], [4.9, 4.7, 5.3]], dtype=np.float32)
    ty = np.array([0, 1], dtype=np.int32)
    chi = np.array([[0.0, 1.0], [1.0, 0.0]])
    ref = direct_pair_force(x, ty, L, chi, 0.0, 2.0, 0.5, images=1)
    plain, dec = {}, {}
    for P in (2, 3, 4):
        for store, flag in ((plain, False), (dec, True)):
            p = orc.OracleParams(2, 2, L, (16,) * 3, P, chi, kappa=0.0, sigma2=0.5, rho0=2.0, deconvolve=flag)
            F = orc.nonbonded_force(p, x, ty)
            store[P] = np.abs(F - ref).max() / np.abs(ref).max()
    assert plain[2] > 0.2 and plain[4] > plain[2]                 # the smoothing error grows with P (A13)
    assert dec[2] < 0.15 and dec[3] < 0.06 and dec[4] < 0.02      # aliasing only
    assert dec[4] < dec[3] < dec[2]
    for P in (2, 3, 4):
        assert dec[P] < 0.35 * plain[P], (P, plain, dec)


def test_deconvolved_kernel_keeps_momentum_and_reduces_to_plain_at_k0():
    rng = np.random.default_rng(5)
    L, N = (6.0, 4.5, 7.0), (12, 8, 10)
    n = 150
    x = (rng.random((n, 3)) * np.array(L)).astype(np.float32)
    ty = rng.integers(0, 3, size=n).astype(np.int32)
    p = orc.OracleParams(n, 3, L, N, 3, CHI3, kappa=5.0, sigma2=0.5, rho0=2.0, deconvolve=True)
    F = orc.nonbonded_force(p, x, ty)
    assert np.abs(F.sum(0)).max() < 1e-10 * np.abs(F).max() * n   # the modified kernel is still real and even
    # a uniform density (only k = 0 populated) feels no force under either kernel
    q = orc.OracleParams(n, 3, L, N, 3, CHI3, kappa=5.0, sigma2=0.5, rho0=2.0)
    grid = np.ones((3,) + N)
    for params in (p, q):
        assert np.abs(orc.kspace_force(params, grid)).max() < 1e-12


# ---- structure factor of the mesh density (Eq. 23) ---------------------------------------------
def test_structure_factor_matches_particle_sum_times_assignment_transform():
    """S_mesh(k) = |sum_g n(g) e^{-ik.g h}|^2 / N.  For |k| well below the mesh Nyquist the mesh density is the particle
    density convolved with W, so S_mesh(k) = W^(k)^2 |sum_i e^{-ik.r_i}|^2 / N up to aliasing; S(0) = N."""
    rng = np.random.default_rng(9)
    L, N, P = (8.0, 6.0, 10.0), (16, 12, 20), 4
    n = 300
    x = (rng.random((n, 3)) * np.array(L)).astype(np.float32)
    ty = rng.integers(0, 2, size=n).astype(np.int32)
    p = orc.OracleParams(n, 2, L, N, P, np.zeros((2, 2)), kappa=1.0, sigma2=0.5)
    S = orc.structure_factor(p, x, ty)
    assert S.shape == (16, 12, 11)
    assert abs(S[0, 0, 0] - n) < 1e-9 * n
    xs = x.astype(np.float64)
    for m in [(1, 0, 0), (0, 2, 0), (1, 1, 1), (2, 0, 3), (15, 11, 1)]:          # (15, 11, .) = (-1, -1, .)
        mt = [mi if mi <= Ni // 2 else mi - Ni for mi, Ni in zip(m, N)]
        k = 2 * np.pi * np.array(mt) / np.array(L)
        direct = np.abs(np.exp(-1j * xs @ k).sum()) ** 2 / n
        w2 = np.prod([np.sinc(mi / Ni) ** (2 * P) for mi, Ni in zip(mt, N)])    # np.sinc(x) = sin(pi x)/(pi x)
        assert abs(S[m] - w2 * direct) < 2e-3 * max(1.0, direct), (m, S[m], w2 * direct)
    A = orc.structure_factor(p, x, ty, species=[0])
    assert abs(A[0, 0, 0] - (ty == 0).sum()) < 1e-9 * n


# ---- pair kernel from the FFT of the sampled real-space potential (reading A5b) -------
def test_sampled_kernel_is_the_aliased_sum_of_the_analytic_one():
    """Sampling u_G on the mesh and transforming gives, by Poisson summation, u^_s(m) = sum_G u^(k_m + G) over the mesh's
    reciprocal vectors G = 2 pi N_a j_a / L_a (box >> sigma, so periodic images of u_G are negligible); it tends to the
    analytic u^ where that has decayed at the mesh Nyquist, and u^_s(0) -> 1 (u_G is a unit Gaussian, L121)."""
    L, N, sigma2 = (10.0, 8.0, 12.0), (16, 12, 20), 0.5
    p = orc.OracleParams(1, 1, L, N, 2, np.zeros((1, 1)), 1.0, sigma2, sampled_kernel=True)
    t = orc.uhat_table(p)
    ana = orc.uhat_table(orc.OracleParams(1, 1, L, N, 2, np.zeros((1, 1)), 1.0, sigma2))
    for m in [(0, 0, 0), (1, 0, 0), (3, 2, 5), (8, 6, 10), (15, 11, 19), (7, 0, 1)]:
        mt = [mi if mi <= Ni // 2 else mi - Ni for mi, Ni in zip(m, N)]
        tot = 0.0
        for jx in range(-3, 4):
            for jy in range(-3, 4):
                for jz in range(-3, 4):
                    k = 2 * np.pi * (np.array(mt) + np.array(N) * np.array([jx, jy, jz])) / np.array(L)
                    tot += np.exp(-0.5 * sigma2 * (k ** 2).sum())
        assert abs(t[m] - tot) < 2e-7, (m, t[m], tot)      # the truncated tails of u_G beyond L/2 (5.7 sigma) are ~4e-8
    assert abs(t[0, 0, 0] - 1.0) < 1e-6
    assert 1e-6 < np.abs(t - ana).max() < 1e-2                               # h ~ 0.6 = 0.9 sigma: visible aliasing (4e-3)
    fine = orc.uhat_table(orc.OracleParams(1, 1, L, (40, 32, 48), 2, np.zeros((1, 1)), 1.0, sigma2, sampled_kernel=True))
    fana = orc.uhat_table(orc.OracleParams(1, 1, L, (40, 32, 48), 2, np.zeros((1, 1)), 1.0, sigma2))
    assert np.abs(fine - fana).max() < 1e-7                                  # h = 0.25: they coincide up to the truncated tails


def test_sampled_kernel_force_is_consistent():
    rng = np.random.default_rng(3)
    L, N = (6.0, 4.5, 7.0), (12, 8, 10)
    n = 120
    x = (rng.random((n, 3)) * np.array(L)).astype(np.float32)
    ty = rng.integers(0, 3, size=n).astype(np.int32)
    p = orc.OracleParams(n, 3, L, N, 3, CHI3, kappa=5.0, sigma2=0.5, rho0=2.0, sampled_kernel=True)
    q = orc.OracleParams(n, 3, L, N, 3, CHI3, kappa=5.0, sigma2=0.5, rho0=2.0)
    F, G = orc.nonbonded_force(p, x, ty), orc.nonbonded_force(q, x, ty)
    assert np.abs(F.sum(0)).max() < 1e-10 * np.abs(F).max() * n               # still momentum conserving
    rel = np.abs(F - G).max() / np.abs(G).max()
    assert 1e-5 < rel < 0.1, rel                                              # close to, but not, the analytic kernel


# ---- electrostatics on the same path (reading A22) ----------------------------------------------------
def ewald_smeared_force(x, z, L, lB, aq, alpha, kmax=10, images=2):
    """Textbook Ewald evaluation of the force between Gaussian-smeared charges, written independently of the oracle.
    Pair potential phi(r) = lB erf(r / 2 aq) / r, split as lB [erf(r/2aq) - erf(alpha r)] / r (short-ranged, summed over
    images in real space) + lB erf(alpha r) / r (smooth: k-space, 4 pi / k^2 exp(-k^2 / 4 alpha^2), k != 0).
    The result must not depend on alpha (alpha = 1 / 2 aq makes the real-space part vanish)."""
    from scipy.special import erf
    x = np.asarray(x, dtype=np.float64)
    L = np.asarray(L, dtype=np.float64)
    n = len(x)
    F = np.zeros((n, 3))
    rng_img = range(-images, images + 1)
    for i in range(n):
        for j in range(n):
            for a in rng_img:
                for b in rng_img:
                    for c in rng_img:
                        if i == j and a == b == c == 0:
                            continue
                        d = x[i] - x[j] + L * np.array([a, b, c])
                        r = np.linalg.norm(d)
                        # -d/dr {[erf(r/2aq) - erf(alpha r)] / r}
                        dphi = (erf(r / (2 * aq)) - erf(alpha * r)) / r ** 2 - (
                            np.exp(-r ** 2 / (4 * aq ** 2)) / (aq * np.sqrt(np.pi)) - 2 * alpha * np.exp(-(alpha * r) ** 2) / np.sqrt(np.pi)) / r
                        F[i] += lB * z[i] * z[j] * dphi * d / r
    V = L.prod()
    ms = np.arange(-kmax, kmax + 1)
    MX, MY, MZ = np.meshgrid(ms, ms, ms, indexing="ij")
    KX, KY, KZ = 2 * np.pi * MX / L[0], 2 * np.pi * MY / L[1], 2 * np.pi * MZ / L[2]
    K2 = KX ** 2 + KY ** 2 + KZ ** 2
    K2[kmax, kmax, kmax] = 1.0
    G = 4 * np.pi * lB * np.exp(-K2 / (4 * alpha ** 2)) / K2
    G[kmax, kmax, kmax] = 0.0
    S = sum(z[j] * np.exp(-1j * (KX * x[j, 0] + KY * x[j, 1] + KZ * x[j, 2])) for j in range(n))
    for i in range(n):
        ph = np.exp(1j * (KX * x[i, 0] + KY * x[i, 1] + KZ * x[i, 2]))
        for a, K in enumerate((KX, KY, KZ)):
            F[i, a] += (z[i] * (-1j * K) * G * S * ph).sum().real / V
    return F


def test_electrostatic_force_matches_ewald_of_smeared_charges():
    """PM electrostatics (charges per species, Coulomb kernel 4 pi lB exp(-k^2 aq^2)/k^2) with the deconvolved kernel on a
    fine mesh against the Ewald sum with a DIFFERENT splitting parameter (real-space erf differences + k-space)."""
    rng = np.random.default_rng(11)
    L = (6.0, 6.0, 6.0)
    n, lB, aq = 8, 2.5, 0.5
    x = (rng.random((n, 3)) * 6.0).astype(np.float32)
    ty = np.array([0, 1] * (n // 2), dtype=np.int32)
    zsp = (1.0, -1.0)
    z = np.array([zsp[t] for t in ty])
    a1 = ewald_smeared_force(x, z, L, lB, aq, alpha=1.0 / (2 * aq))          # real-space part vanishes identically
    a2 = ewald_smeared_force(x, z, L, lB, aq, alpha=0.7 / (2 * aq))          # genuinely split
    assert np.abs(a1 - a2).max() < 1e-9 * np.abs(a1).max()
    assert np.abs(a1.sum(0)).max() < 1e-9 * np.abs(a1).max()
    errs = []
    for Ng in (24, 48):
        p = orc.OracleParams(n, 2, L, (Ng,) * 3, 4, np.zeros((2, 2)), kappa=0.0, sigma2=0.5, rho0=1.0,
                             charge=zsp, bjerrum=lB, a_charge=aq, deconvolve=True)
        F = orc.nonbonded_force(p, x, ty)
        errs.append(np.abs(F - a2).max() / np.abs(a2).max())
    assert errs[0] < 2e-3 and errs[1] < 1e-4, errs                           # aliasing only; falls fast with h
    # opposite charges attract, equal charges repel (sign convention)
    q = orc.OracleParams(2, 2, L, (32,) * 3, 4, np.zeros((2, 2)), kappa=0.0, sigma2=0.5, rho0=1.0, charge=zsp, bjerrum=lB, a_charge=aq)
    xp = np.array([[2.0, 3.0, 3.0], [3.5, 3.0, 3.0]], dtype=np.float32)
    Fp = orc.nonbonded_force(q, xp, np.array([0, 1], np.int32))
    assert Fp[0, 0] > 0 and Fp[1, 0] < 0
    Fs = orc.nonbonded_force(q, xp, np.array([0, 0], np.int32))
    assert Fs[0, 0] < 0 and Fs[1, 0] > 0


def test_electrostatics_off_and_neutral_species_feel_nothing():
    rng = np.random.default_rng(2)
    L, N = (6.0, 4.5, 7.0), (12, 8, 10)
    n = 90
    x = (rng.random((n, 3)) * np.array(L)).astype(np.float32)
    ty = rng.integers(0, 3, size=n).astype(np.int32)
    base = orc.OracleParams(n, 3, L, N, 3, CHI3, kappa=5.0, sigma2=0.5, rho0=2.0)
    el = orc.OracleParams(n, 3, L, N, 3, CHI3, kappa=5.0, sigma2=0.5, rho0=2.0, charge=(1.0, -1.0, 0.0), bjerrum=1.7, a_charge=0.4)
    F0, F1 = orc.nonbonded_force(base, x, ty), orc.nonbonded_force(el, x, ty)
    assert np.abs(F1 - F0)[ty == 2].max() < 1e-12                             # the neutral species gains no force
    assert np.abs(F1 - F0)[ty != 2].max() > 1e-3
    assert np.abs(F1.sum(0)).max() < 1e-10 * np.abs(F1).max() * n            # momentum conservation survives


# ---- energies of the kernel variants (O10 with the sampled kernel / with electrostatics) ------------------------------
def test_sampled_kernel_mesh_energy_is_the_pair_sum_of_the_sampled_potential():
    """With P = 1 every particle is one unit of density on its nearest node, and the kernel obtained by transforming
    u_G sampled on the mesh (reading A5b) turns the mesh energy (1/2V) sum_m u^_s(m) sum_IJ c_IJ Re[n^_I n^_J*]
    into the plain double sum  1/2 sum_{a, b} c_{I(a) J(b)} u_G(minimum image of node_a - node_b)  (a = b included):
    the identity sum_m exp(2 pi i m (g - g') / N) = M delta_{g g'} makes it exact.  Written out by brute force here."""
    rng = np.random.default_rng(12)
    L, N, sigma2 = (6.0, 4.5, 7.0), (12, 8, 10), 0.5
    h = np.array(L) / np.array(N)
    n = 40
    cells = np.stack([rng.integers(0, N[a], size=n) for a in range(3)], axis=1)
    jitter = (rng.random((n, 3)) - 0.5) * 0.6                        # anywhere in the cell of the nearest node
    x = (((cells + jitter) % np.array(N)) * h).astype(np.float32)
    ty = rng.integers(0, 3, size=n).astype(np.int32)
    kappa, rho0 = 5.0, 2.0
    p = orc.OracleParams(n, 3, L, N, 1, CHI3, kappa=kappa, sigma2=sigma2, rho0=rho0, sampled_kernel=True, k_bond=0.0)
    base, _, _ = orc.index_map(p, x)
    node = base % np.array(N)
    c = c_matrix(CHI3, kappa, rho0)
    E = 0.0
    norm = (2 * np.pi * sigma2) ** -1.5
    for a in range(n):
        for b in range(n):
            d = (node[a] - node[b]) * h
            d -= np.array(L) * np.round(d / np.array(L))
            E += 0.5 * c[ty[a], ty[b]] * norm * np.exp(-(d ** 2).sum() / (2 * sigma2))
    bp = -np.ones((n, 2), dtype=np.int32)
    e = orc.energy(p, x.astype(np.float64), np.zeros((n, 3)), ty, bp)
    assert abs(e[2] - E) < 1e-10 * abs(E), (e[2], E)


def ewald_smeared_energy(x, z, L, lB, aq, alpha, kmax=12, images=2):
    """Energy of Gaussian-smeared point charges in a neutralising background (k = 0 dropped), self terms included:
    E = 1/2 sum_{i, j, images} z_i z_j phi(r),  phi(r) = lB erf(r / 2 aq) / r,  phi(0) = lB / (aq sqrt(pi)).
    Ewald split with parameter alpha: [erf(r/2aq) - erf(alpha r)] / r in real space (limit (2/sqrt(pi)) (1/2aq - alpha) at
    r = 0) + 4 pi exp(-k^2 / 4 alpha^2) / k^2 in k-space.  Independent of alpha; written independently of the oracle."""
    from scipy.special import erf
    x = np.asarray(x, dtype=np.float64)
    L = np.asarray(L, dtype=np.float64)
    n = len(x)
    E = 0.0
    rng_img = range(-images, images + 1)
    for i in range(n):
        for j in range(n):
            for a in rng_img:
                for b in rng_img:
                    for c in rng_img:
                        d = x[i] - x[j] + L * np.array([a, b, c])
                        r = np.linalg.norm(d)
                        if r == 0.0:
                            E += 0.5 * lB * z[i] * z[j] * (2 / np.sqrt(np.pi)) * (1 / (2 * aq) - alpha)
                        else:
                            E += 0.5 * lB * z[i] * z[j] * (erf(r / (2 * aq)) - erf(alpha * r)) / r
    V = L.prod()
    ms = np.arange(-kmax, kmax + 1)
    MX, MY, MZ = np.meshgrid(ms, ms, ms, indexing="ij")
    KX, KY, KZ = 2 * np.pi * MX / L[0], 2 * np.pi * MY / L[1], 2 * np.pi * MZ / L[2]
    K2 = KX ** 2 + KY ** 2 + KZ ** 2
    K2[kmax, kmax, kmax] = 1.0
    G = 4 * np.pi * lB * np.exp(-K2 / (4 * alpha ** 2)) / K2
    G[kmax, kmax, kmax] = 0.0
    S = sum(z[j] * np.exp(-1j * (KX * x[j, 0] + KY * x[j, 1] + KZ * x[j, 2])) for j in range(n))
    # net charge Q: the definition drops the k = 0 mode of the WHOLE pair potential (neutralising background), but the
    # real-space sum above contains the k = 0 component of its short-ranged part,
    # int d^3r lB [erf(r/2aq) - erf(alpha r)] / r = pi lB (1/alpha^2 - 4 aq^2): take it out again (zero for Q = 0)
    Q = float(np.sum(z))
    E -= 0.5 * Q * Q * np.pi * lB * (1.0 / alpha ** 2 - 4.0 * aq ** 2) / V
    return E + 0.5 * (G * np.abs(S) ** 2).sum() / V


def test_electrostatic_mesh_energy_matches_ewald_energy_of_smeared_charges():
    """O10 with a Bjerrum length: the mesh energy (1/2V) sum_{k != 0} u^_el(k) |rho^_c(k)|^2 (self terms included) with
    the deconvolved kernel against the Ewald ENERGY evaluated with two different splitting parameters."""
    rng = np.random.default_rng(11)
    L = (6.0, 6.0, 6.0)
    n, lB, aq = 8, 2.5, 0.5
    x = (rng.random((n, 3)) * 6.0).astype(np.float32)
    ty = np.array([0, 1] * (n // 2), dtype=np.int32)
    zsp = (1.0, -1.0)
    z = np.array([zsp[t] for t in ty])
    e1 = ewald_smeared_energy(x, z, L, lB, aq, alpha=1.0 / (2 * aq))         # real-space part vanishes identically
    e2 = ewald_smeared_energy(x, z, L, lB, aq, alpha=0.7 / (2 * aq))
    assert abs(e1 - e2) < 1e-9 * abs(e1), (e1, e2)
    bp = -np.ones((n, 2), dtype=np.int32)
    errs = []
    for Ng in (24, 48):
        p = orc.OracleParams(n, 2, L, (Ng,) * 3, 4, np.zeros((2, 2)), kappa=0.0, sigma2=0.5, rho0=1.0,
                             charge=zsp, bjerrum=lB, a_charge=aq, deconvolve=True, k_bond=0.0)
        e = orc.energy(p, x.astype(np.float64), np.zeros((n, 3)), ty, bp)
        errs.append(abs(e[2] - e2) / abs(e2))
    assert errs[0] < 2e-3 and errs[1] < 1e-4, (errs, e2)
