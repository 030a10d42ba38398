"""Exact exchange operator and its adaptively compressed form (section 3.1, Eqs. 28-30).

Test infrastructure only (see oracle/__init__.py).

Eq. 28:  (V_X psi)(r) = - sum_v phi_v(r) C[phi_v psi](r)          (Gamma, real orbitals; C of oracle/liouville.py,
                                                                   G = 0 term zero, reading A10)
          brought back to the plane-wave sphere with the O7 convention.
Eq. 30:  W_i = V_X phi_i for i = 1..N_ACE (occupied orbitals first, then the extra ones the caller supplies),
          M_ij = <phi_i|W_j>,  M = -L L^T (Cholesky),  xi_k = sum_i W_i (L^-T)_ik.
Eq. 29:  V_X^ACE = - sum_k |xi_k><xi_k|.
The paper does not say where W lives; here everything after V_X is in the half-sphere storage with the Gamma inner
product (reading A20 of DESIGN.md): V_X^ACE reproduces the sphere projection of V_X phi_i on the N_ACE orbitals.
Pins: tests/test_oracle_extensions.py (brute-force V_X without FFT on a 6x5x4 cell, V_X^ACE phi_i = V_X phi_i,
symmetry and negative semi-definiteness, idempotent rebuild).
"""
import numpy as np


def exchange_apply(P, s, c):
    """Eq. 28 on one function given by its half-sphere coefficients c, orbitals of spin s of Problem P."""
    f = P.to_real(c)
    y = np.zeros(P.grid)
    for v in range(P.nocc[s]):
        y -= P.phi[s][v] * P.coulomb(P.phi[s][v] * f)
    return P.to_sphere(y)


def gamma_dot(a, b):
    """<a|b> of two half-sphere functions (real functions: c(-G) = conj c(G))."""
    return float(2.0 * np.real(np.vdot(a, b)) - a[0].real * b[0].real)


def build(P, s, extra=None):
    """xi [N_ACE, npwh] of spin s; extra = further (unoccupied) orbitals [n_extra, npwh] or None (Eq. 30)."""
    orbs = list(P.psi[s]) + ([] if extra is None else list(np.asarray(extra, dtype=np.complex128)))
    W = np.stack([exchange_apply(P, s, c) for c in orbs])
    n = len(orbs)
    M = np.array([[gamma_dot(orbs[i], W[j]) for j in range(n)] for i in range(n)])
    M = 0.5 * (M + M.T)
    L = np.linalg.cholesky(-M)                     # M = -L L^T
    Linv = np.linalg.inv(L)
    return np.tensordot(Linv, W, axes=1)           # xi_k = sum_i (L^-1)_ki W_i = sum_i W_i (L^-T)_ik


def ace_apply(xi, c):
    """Eq. 29: V_X^ACE c = - sum_k xi_k <xi_k|c>."""
    out = np.zeros_like(c)
    for x in xi:
        out = out - x * gamma_dot(x, c)
    return out
