"""Pins for the oracle's assignment weights (O2), index map (O1) and cell sort (A16).

Weights: PAPER.md L223 cites the appendix of Deserno & Holm (ref. [40]) without reproducing it; the
pins are what that definition fixes: W^(P) is the P-fold convolution of the unit top-hat (checked
against a numerically convolved top-hat and against the textbook cardinal B-spline closed form),
partition of unity, exact first moment, mirror symmetry, and P=2 = linear interpolation (Fig. 1).
"""
import math

import numpy as np
import pytest

from oracle import tild_oracle as orc


def bspline_closed_form(P, x):
    """Centred cardinal B-spline of order P (support [-P/2, P/2]): textbook truncated-power formula."""
    s = 0.0
    for k in range(P + 1):
        y = x + P / 2.0 - k
        if y > 0:
            s += (-1) ** k * math.comb(P, k) * y ** (P - 1)
    if P == 1:
        return 1.0 if -0.5 <= x < 0.5 else 0.0
    return s / math.factorial(P - 1)


def node_offsets(P):
    """Stencil node coordinates relative to the stencil centre (centre = nearest node for odd P,
    midpoint of the two nearest nodes for even P)."""
    return np.arange(P) - (P - 1) / 2.0


@pytest.mark.parametrize("P", [1, 2, 3, 4, 5])
def test_partition_of_unity_first_moment_symmetry(P):
    for t in np.linspace(-0.5, 0.5, 101):
        w = orc.weights(P, float(t))
        assert abs(w.sum() - 1.0) < 1e-14
        assert (w >= -1e-16).all()
        if P >= 2:
            # sum_j node_j w_j = particle position (relative to the stencil centre)
            assert abs((node_offsets(P) * w).sum() - t) < 1e-14
        wm = orc.weights(P, float(-t))
        assert np.allclose(w, wm[::-1], atol=1e-15)


@pytest.mark.parametrize("P", [1, 2, 3, 4, 5])
def test_against_closed_form_bspline(P):
    for t in np.linspace(-0.499, 0.499, 37):
        w = orc.weights(P, float(t))
        ref = np.array([bspline_closed_form(P, float(o - t)) for o in node_offsets(P)])
        assert np.allclose(w, ref, atol=2e-14), (P, t, w, ref)


@pytest.mark.parametrize("P", [2, 3, 4, 5])
def test_against_numerically_convolved_top_hat(P):
    dx = 1.0 / 1000
    box = np.ones(1000)
    f = box.copy()
    for _ in range(P - 1):
        f = np.convolve(f, box) * dx
    xs = (np.arange(f.size) - (f.size - 1) / 2.0) * dx          # centred support [-P/2, P/2]
    for t in [-0.4, -0.123, 0.0, 0.25, 0.45]:
        w = orc.weights(P, t)
        ref = np.interp(node_offsets(P) - t, xs, f)
        assert np.allclose(w, ref, atol=3e-3), (P, t, w, ref)


def test_order2_is_linear_interpolation():
    # Fig. 1: first-order spline maps to the two nearest grid points: weights 1-d and d.
    for d in np.linspace(0, 1, 11):           # d = distance from the lower node in units of h
        w = orc.weights(2, float(d - 0.5))
        assert np.allclose(w, [1 - d, d], atol=1e-15)


def _params(n, L, N, P, S=1):
    return orc.OracleParams(n, S, L, N, P, np.zeros((S, S)), 1.0, 0.5)


@pytest.mark.parametrize("P", [1, 2, 3, 4, 5])
def test_index_map_definition(P):
    rng = np.random.default_rng(5)
    L, N = (10.0, 7.0, 12.5), (16, 12, 20)
    n = 5000
    x = (rng.random((n, 3)) * np.array(L)).astype(np.float32)
    p = _params(n, L, N, P)
    base, toff, key = orc.index_map(p, x)
    h = np.array(L) / np.array(N)
    s = x.astype(np.float64) / h                                  # double-precision position in grid units
    # the particle sits inside its stencil: node centre + t = s (to fp32 rounding of s)
    centre = base + (P - 1) / 2.0
    assert np.abs(centre + toff - s).max() < 4e-6 * max(N)
    assert (np.abs(toff) <= 0.5 + 1e-6).all()
    cell = np.floor(s).astype(np.int64) % np.array(N)
    key64 = (cell[:, 0] * N[1] + cell[:, 1]) * N[2] + cell[:, 2]
    # identical except possibly for particles within fp32 rounding of a cell boundary
    mism = key64 != key
    frac = s - np.floor(s)
    near = (np.minimum(frac, 1 - frac) < 1e-5).any(axis=1)
    assert (~mism | near).all()
    assert mism.mean() < 1e-3


def test_index_map_box_edges():
    # x = 0 and x just below L must land in cells 0 and N-1 (or wrap to 0) with nodes taken mod N
    L, N = (10.0, 10.0, 10.0), (16, 16, 16)
    x = np.array([[0.0, 0.0, 0.0], [np.nextafter(np.float32(10.0), np.float32(0.0))] * 3], dtype=np.float32)
    for P in (1, 2, 3, 4):
        p = _params(2, L, N, P)
        base, toff, key = orc.index_map(p, x)
        assert key[0] == 0
        cz = int(key[1]) % 16
        assert cz in (15, 0)
        assert (base[0] <= 0).all() and (base[0] > -P).all()


def test_cell_sort_properties():
    rng = np.random.default_rng(7)
    n, M = 20000, 4096
    key = rng.integers(0, M, size=n).astype(np.uint32)
    key[:100] = 17                                # a crowded cell
    perm, start = orc.cell_sort(n, M, key)
    assert np.array_equal(np.sort(perm), np.arange(n, dtype=np.uint32))
    assert (np.diff(key[perm].astype(np.int64)) >= 0).all()
    hist = np.bincount(key, minlength=M)
    assert np.array_equal(start, np.concatenate([[0], np.cumsum(hist)]).astype(np.uint32))
    # stable: ids ascend inside each cell  ==  numpy's stable argsort (library routine)
    assert np.array_equal(perm, np.argsort(key, kind="stable").astype(np.uint32))


def test_spread_mass_equals_particle_count():
    rng = np.random.default_rng(11)
    L, N = (10.0, 7.0, 12.5), (16, 12, 20)
    n = 3000
    x = (rng.random((n, 3)) * np.array(L)).astype(np.float32)
    ty = rng.integers(0, 3, size=n).astype(np.int32)
    for P in (1, 2, 3, 4):
        p = _params(n, L, N, P, S=3)
        g = orc.spread(p, x, ty)
        counts = np.bincount(ty, minlength=3)
        assert np.allclose(g.sum(axis=(1, 2, 3)), counts, rtol=0, atol=1e-9)
        assert (g >= 0).all()


def test_spread_single_particle_hits_expected_nodes():
    # one particle at (2.3 h, 5 h, 7.5 h), P = 2: brute-force CIC by hand
    L, N = (8.0, 8.0, 8.0), (8, 8, 8)
    x = np.array([[2.3, 5.0, 7.5]], dtype=np.float32)
    p = _params(1, L, N, 2)
    g = orc.spread(p, x, np.zeros(1, np.int32))[0]
    exp = np.zeros((8, 8, 8))
    for ix, wx in ((2, 0.7), (3, 0.3)):
        for iy, wy in ((5, 1.0), (6, 0.0)):
            for iz, wz in ((7, 0.5), (0, 0.5)):      # periodic wrap in z
                exp[ix, iy, iz] += wx * wy * wz
    assert np.allclose(g, exp, atol=1e-6)             # fp32 input position
