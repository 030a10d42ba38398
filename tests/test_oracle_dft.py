"""Pins for oracle/dft.py: the radix FFT against the definition and against what Fourier analysis fixes."""
import numpy as np
import pytest

from oracle.dft import dft3_naive, fft3, fft_axis


@pytest.mark.parametrize("shape", [(6, 5, 4), (12, 10, 9), (8, 9, 15), (2, 3, 5), (10, 6, 7)])
@pytest.mark.parametrize("sign", [-1, +1])
def test_radix_fft_equals_definition(shape, sign):
    rng = np.random.default_rng(1)
    x = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
    ref = dft3_naive(x, sign)
    assert np.max(np.abs(fft3(x, sign) - ref)) < 1e-12 * np.max(np.abs(ref))
    assert np.max(np.abs(fft3(x, sign, backend="numpy") - ref)) < 1e-12 * np.max(np.abs(ref))


@pytest.mark.parametrize("shape,k", [((24, 24, 24), (3, 20, 1)), ((12, 10, 9), (11, 0, 4)), ((72, 4, 4), (5, 3, 1))])
def test_single_plane_wave_lands_on_its_index(shape, k):
    # x_j = exp(+2 pi i k.j/n): the forward (sign = -1) transform is N_r at index k and 0 elsewhere;
    # fixes the sign convention and the axis order
    j = np.meshgrid(*[np.arange(n) for n in shape], indexing="ij")
    ph = sum(k[i] * j[i] / shape[i] for i in range(3))
    x = np.exp(2j * np.pi * ph)
    X = fft3(x, -1)
    expect = np.zeros(shape, complex)
    expect[k] = np.prod(shape)
    assert np.max(np.abs(X - expect)) < 1e-9
    # and the sign = +1 transform puts it at -k
    X = fft3(x, +1)
    expect = np.zeros(shape, complex)
    expect[tuple((-np.array(k)) % np.array(shape))] = np.prod(shape)
    assert np.max(np.abs(X - expect)) < 1e-9


@pytest.mark.parametrize("n", [24, 48, 72, 96, 100, 128, 45, 50])
def test_1d_lengths_against_library(n):
    rng = np.random.default_rng(n)
    x = rng.standard_normal((n, 7)) + 1j * rng.standard_normal((n, 7))
    ref = np.fft.fft(x, axis=0)
    assert np.max(np.abs(fft_axis(x, 0, -1) - ref)) < 1e-12 * np.max(np.abs(ref))
    ref = np.fft.ifft(x, axis=0) * n
    assert np.max(np.abs(fft_axis(x, 0, +1) - ref)) < 1e-12 * np.max(np.abs(ref))


def test_round_trip_and_parseval():
    rng = np.random.default_rng(2)
    x = rng.standard_normal((24, 20, 18))
    X = fft3(x, -1)
    assert np.max(np.abs(fft3(X, +1) / x.size - x)) < 1e-13
    assert np.sum(np.abs(X) ** 2) / x.size == pytest.approx(np.sum(x * x), rel=1e-13)
    # real input: Hermitian spectrum X(-k) = conj X(k)
    Xm = np.roll(X[::-1, ::-1, ::-1], 1, axis=(0, 1, 2))
    assert np.max(np.abs(Xm - np.conj(X))) < 1e-10


def test_backends_agree_on_config_grids():
    rng = np.random.default_rng(3)
    # every grid the sampled-column parity checks use the library backend on, both signs, complex input
    for shape in [(24, 24, 24), (48, 48, 48), (72, 72, 72), (96, 96, 100)]:
        x = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
        for sign in (-1, +1):
            a = fft3(x, sign)
            b = fft3(x, sign, backend="numpy")
            assert np.max(np.abs(a - b)) < 1e-12 * np.max(np.abs(b))
