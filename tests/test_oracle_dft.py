"""Pins for the oracle's DFT routines (P1) and the Appendix-A packed layout.

None of these retype the oracle's formula: they use closed forms, Parseval, the shift
theorem and the library routine numpy.fft.
"""
import numpy as np
import pytest

import oracle
from oracle import algorithms as alg


@pytest.mark.parametrize("n", [4, 8, 12, 30, 64, 256])
@pytest.mark.parametrize("sign", [-1, 1])
def test_naive_dft_matches_numpy_fft(n, sign):
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    ref = np.fft.fft(x) if sign < 0 else np.fft.ifft(x) * n
    got = oracle.dft_naive(x, sign)
    assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max()


@pytest.mark.parametrize("n", [2, 4, 8, 64, 256, 1024])
@pytest.mark.parametrize("sign", [-1, 1])
def test_radix2_fft_matches_definition_and_numpy(n, sign):
    rng = np.random.default_rng(100 + n)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    got = oracle.fft_radix2(x, sign)
    ref = np.fft.fft(x) if sign < 0 else np.fft.ifft(x) * n
    assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max()
    if n <= 256:
        assert np.abs(got - oracle.dft_naive(x, sign)).max() <= 1e-13 * np.abs(ref).max()


@pytest.mark.parametrize("n,q", [(16, 3), (64, 1), (64, 31), (30, 7)])
def test_single_cosine_closed_form(n, q):
    """DFT of cos(2 pi q i / n) is n/2 at +-q and zero elsewhere."""
    i = np.arange(n)
    X = oracle.dft_naive(np.cos(2 * np.pi * q * i / n))
    expect = np.zeros(n)
    expect[q] = n / 2
    expect[n - q] = n / 2
    assert np.abs(X - expect).max() <= 1e-13 * n


@pytest.mark.parametrize("n", [8, 64, 512])
def test_parseval_and_shift_theorem(n):
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n)
    fft = oracle.fft_radix2 if n > 64 else oracle.dft_naive
    X = fft(x)
    assert abs(np.sum(np.abs(X) ** 2) / n - np.sum(x ** 2)) <= 1e-12 * np.sum(x ** 2)
    # circular shift by s multiplies mode q by exp(-2 pi i q s / n)
    s = 3
    Xs = fft(np.roll(x, s))
    q = np.arange(n)
    assert np.abs(Xs - X * np.exp(-2j * np.pi * q * s / n)).max() <= 1e-12 * np.abs(X).max()
    # real input: Hermitian symmetry, zero imaginary part at modes 0 and n/2
    assert abs(X[0].imag) <= 1e-13 * np.abs(X).max()
    assert abs(X[n // 2].imag) <= 1e-13 * np.abs(X).max()
    assert np.abs(X[1:] - np.conj(X[1:][::-1])).max() <= 1e-12 * np.abs(X).max()


def test_inverse_roundtrip():
    rng = np.random.default_rng(5)
    x = rng.standard_normal(128) + 1j * rng.standard_normal(128)
    back = oracle.fft_radix2(oracle.fft_radix2(x, -1), +1) / 128
    assert np.abs(back - x).max() <= 1e-14 * np.abs(x).max() * 10


def test_dft_xy_matches_numpy_fft2_per_plane():
    rng = np.random.default_rng(6)
    f = rng.standard_normal((3, 8, 16))
    ref = np.fft.fft2(f, axes=(1, 2))
    for variant in (0, 1):
        got = oracle.dft_xy(f, -1, variant)
        assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max()
    back = oracle.dft_xy(ref, +1, 1) / (8 * 16)
    assert np.abs(back.real - f).max() <= 1e-13
    assert np.abs(back.imag).max() <= 1e-13


@pytest.mark.parametrize("n", [4, 8, 64])
def test_packed_halfcomplex_is_n_reals_and_invertible(n):
    """Appendix A: n reals in, n reals out, O(1) re-arrangement."""
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n)
    X = np.fft.rfft(x)
    packed = alg.pack_halfcomplex(X)
    assert packed.shape == (n,)
    assert packed[0] == X[0].real and packed[1] == X[n // 2].real
    Y = alg.unpack_halfcomplex(packed)
    # the only information dropped are the two always-zero imaginary parts
    assert abs(X[0].imag) < 1e-14 and abs(X[-1].imag) < 1e-13
    assert np.abs(Y[1:-1] - X[1:-1]).max() == 0.0
    assert np.abs(np.fft.irfft(Y, n) - x).max() <= 1e-14 * 10


def test_modified_wavenumbers_are_eigenvalues_of_periodic_stencil():
    """lambda_q: apply the 3-point periodic stencil to cos/sin(2 pi q i/n) (reading R1)."""
    n, L = 32, 4 * np.pi
    lam = oracle.modified_wavenumbers(n, L)
    dx = L / n
    i = np.arange(n)
    for q in range(n):
        for fn in (np.cos, np.sin):
            v = fn(2 * np.pi * q * i / n)
            lap = (np.roll(v, -1) - 2 * v + np.roll(v, 1)) / dx ** 2
            assert np.abs(lap - lam[q] * v).max() <= 1e-12 * max(1.0, abs(lam[q]))
    assert lam[0] == 0.0 and np.all(lam[1:] < 0)
    # high-accuracy reference for small q at large n: -4 sin^2(pi q/n)/dx^2 in long double
    n = 2048
    lam = oracle.modified_wavenumbers(n, 8 * np.pi)
    q = np.arange(n, dtype=np.longdouble)
    pil = 4 * np.arctan(np.longdouble(1))
    dxl = np.longdouble(8 * np.pi) / n          # the domain length is the double 8*pi
    ref = -4 * np.sin(pil * q / n) ** 2 / dxl ** 2
    rel = np.abs((lam - ref)[1:] / ref[1:]).astype(np.float64)
    assert rel.max() <= 1e-15 * 8
