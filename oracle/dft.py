"""Discrete Fourier transforms for the oracle: the definition and a simple radix FFT.

Test infrastructure only (see oracle/__init__.py).

`dft3_naive` is the textbook definition written out as a dense
(N_r x N_r) matrix product, usable on tiny grids only.  `fft3` is a simple
recursive decimation-in-time mixed-radix FFT: a length n = p*m (p the smallest
prime factor) is split into its p residue classes, each transformed
recursively, twiddled and combined with a p-point DFT; lengths <= LEAF and
prime lengths use the definition (a dense DFT matrix).  Sign convention:
sign=-1 is exp(-i G.r) ("forward", r -> G), sign=+1 is exp(+i G.r); neither
normalises.  The paper only says "fast Fourier transforms (FFTs) between the
direct and reciprocal spaces" (section 4).

`fft3(..., backend="numpy")` calls numpy.fft (pocketfft) instead: a library
primitive serving as the same step, ~4x faster, used for the sampled-column
checks on the 48^3 / 72^3 configurations; the two backends are pinned equal.

Pins: tests/test_oracle_dft.py (definition vs fft3 on every radix mix, a single
plane wave, Parseval, round trip, numpy.fft as a library cross-check).
"""
import numpy as np

LEAF = 9  # lengths up to this use the dense definition


def dft3_naive(x, sign):
    """X[k1,k2,k3] = sum_j x[j] exp(sign * 2 pi i (k1 j1/n1 + k2 j2/n2 + k3 j3/n3))."""
    x = np.asarray(x)
    n1, n2, n3 = x.shape
    j1, j2, j3 = np.meshgrid(np.arange(n1), np.arange(n2), np.arange(n3), indexing="ij")
    j1 = j1.ravel(); j2 = j2.ravel(); j3 = j3.ravel()
    # phase[k, j] with k and j both flattened in C order
    ph = (np.outer(j1, j1) / n1 + np.outer(j2, j2) / n2 + np.outer(j3, j3) / n3)
    W = np.exp(sign * 2j * np.pi * ph)
    return (W @ x.ravel().astype(np.complex128)).reshape(n1, n2, n3)


def _smallest_prime_factor(n):
    p = 2
    while p * p <= n:
        if n % p == 0:
            return p
        p += 1
    return n


def _dft_matrix(n, sign):
    k = np.arange(n)
    return np.exp(sign * 2j * np.pi * np.outer(k, k) / n)


def _fft_first(x, sign):
    """1-D transform along axis 0 of a contiguous [n, R] array (decimation in time)."""
    n, R = x.shape
    p = _smallest_prime_factor(n)
    if p == n or n <= LEAF:
        return _dft_matrix(n, sign) @ x                 # the definition
    m = n // p
    xs = x.reshape(m, p, R)                              # x[q*p + r] -> xs[q, r]
    subs = np.empty((p, m, R), dtype=np.complex128)
    k2 = np.arange(m)[:, None]
    for r in range(p):
        sub = _fft_first(np.ascontiguousarray(xs[:, r, :]), sign)   # length-m transform of class r
        subs[r] = sub * np.exp(sign * 2j * np.pi * r * k2 / n)       # twiddle w_n^{r k2}
    # X[k1*m + k2] = sum_r w_p^{r k1} subs[r, k2]
    return (_dft_matrix(p, sign) @ subs.reshape(p, m * R)).reshape(n, R)


def fft_axis(x, axis, sign):
    y = np.ascontiguousarray(np.moveaxis(np.asarray(x, dtype=np.complex128), axis, 0))
    sh = y.shape
    y = _fft_first(y.reshape(sh[0], -1), sign).reshape(sh)
    return np.moveaxis(y, 0, axis)


def fft3(x, sign, backend="radix"):
    """3-D transform = three 1-D transforms, one per axis."""
    if backend == "numpy":
        x = np.asarray(x, dtype=np.complex128)
        if sign < 0:
            return np.fft.fftn(x)
        return np.fft.ifftn(x) * x.size
    if backend != "radix":
        raise ValueError(backend)
    y = np.asarray(x, dtype=np.complex128)
    for axis in range(3):
        y = fft_axis(y, axis, sign)
    return y
