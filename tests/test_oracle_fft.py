"""Pins for the oracle's own mixed-radix DFT (O4/O6): a naive O(n^2) DFT written out from the
definition on small sizes (radix 2, 3, 5, 7 and a prime length), and numpy.fft (library routine)
on the grid sizes the configs use."""
import numpy as np
import pytest

from oracle import tild_oracle as orc


def naive_dft3(a, sign):
    out = a.astype(np.complex128)
    for ax, n in enumerate(a.shape):
        j = np.arange(n)
        W = np.exp(sign * 2j * np.pi * np.outer(j, j) / n)
        out = np.moveaxis(np.tensordot(W, np.moveaxis(out, ax, 0), axes=(1, 0)), 0, ax)
    return out


@pytest.mark.parametrize("shape", [(4, 4, 4), (6, 4, 12), (5, 7, 9), (12, 12, 12), (11, 2, 3)])
@pytest.mark.parametrize("sign", [-1, 1])
def test_against_naive_dft(shape, sign):
    rng = np.random.default_rng(3)
    a = rng.normal(size=shape) + 1j * rng.normal(size=shape)
    ref = naive_dft3(a, sign)
    got = orc.dft3d(a, sign)
    assert np.abs(got - ref).max() < 1e-11 * np.abs(ref).max()


@pytest.mark.parametrize("n", [16, 64, 128, 192, 256, 360])
def test_1d_against_numpy(n):
    rng = np.random.default_rng(n)
    a = rng.normal(size=n) + 1j * rng.normal(size=n)
    assert np.abs(orc.dft1d(a, -1) - np.fft.fft(a)).max() < 1e-11 * n
    assert np.abs(orc.dft1d(a, +1) - np.fft.ifft(a) * n).max() < 1e-11 * n


@pytest.mark.parametrize("shape", [(16, 16, 16), (64, 64, 64), (48, 32, 20)])
def test_3d_against_numpy(shape):
    rng = np.random.default_rng(9)
    a = rng.normal(size=shape) + 1j * rng.normal(size=shape)
    ref = np.fft.fftn(a)
    assert np.abs(orc.dft3d(a, -1) - ref).max() < 1e-12 * np.abs(ref).max() * 10
    assert np.abs(orc.dft3d(orc.dft3d(a, -1), +1) / a.size - a).max() < 1e-12


def test_delta_and_plane_wave():
    # closed forms: DFT of a delta at g0 is exp(-2 pi i m.g0/N); DFT of a plane wave is M at one mode
    N = (6, 8, 10)
    a = np.zeros(N, dtype=np.complex128)
    g0 = (2, 5, 7)
    a[g0] = 1.0
    m = np.meshgrid(*[np.arange(k) for k in N], indexing="ij")
    ref = np.exp(-2j * np.pi * sum(m[i] * g0[i] / N[i] for i in range(3)))
    assert np.abs(orc.dft3d(a, -1) - ref).max() < 1e-13
    m0 = (1, 3, 9)
    wave = np.exp(2j * np.pi * sum(m[i] * m0[i] / N[i] for i in range(3)))
    out = orc.dft3d(wave, -1)
    exp = np.zeros(N, dtype=np.complex128)
    exp[m0] = np.prod(N)
    assert np.abs(out - exp).max() < 1e-10
