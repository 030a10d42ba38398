"""Near-sightedness truncation of K1d (section 3.2): overlap function and pair mask.

Test infrastructure only (see oracle/__init__.py).

Eq. 32:  S_mn = int |phi~_m|^2 |phi~_n|^2 dr / sqrt( int |phi~_m|^4 dr  int |phi~_n|^4 dr ),
evaluated as sums over the FFT grid (the volume element cancels).  Pairs with S_mn < S_thr are dropped: tau~_mn = 0.
The localisation itself (maximally localised Wannier functions, ref. 84) is not described in the paper and is out of
scope; the orbitals handed in are taken as already localised.
Pins: tests/test_oracle_extensions.py (S_mm = 1, symmetry, Cauchy-Schwarz bound, disjoint supports give 0, value for
two plane-wave densities typed in closed form).
"""
import numpy as np


def overlap_matrix(phi):
    """phi [n, n1, n2, n3] real -> S [n, n] of Eq. 32."""
    d = np.asarray(phi, dtype=np.float64).reshape(len(phi), -1) ** 2         # |phi_m(r)|^2
    num = d @ d.T
    q = np.sqrt(np.sum(d * d, axis=1))
    return num / np.outer(q, q)


def pair_mask(S, s_thr):
    """True where the pair is kept: S_mn >= S_thr."""
    return np.asarray(S) >= s_thr
