"""Pins for oracle/davidson.py: a closed-form spectrum and dense diagonalisation on a tiny cell."""
import numpy as np
import pytest

from oracle import lattice as lat
from oracle import liouville as lv
from oracle.davidson import davidson
import synthetic_inputs as inputs


def test_d_only_closed_form():
    # Orbitals = the lowest real plane waves (1/sqrt(Omega), sqrt(2/Omega) cos(G.r)), eps_v = |G_v|^2/2,
    # alpha = 0, Hxc off  =>  A = P_c (T - eps_v): the spectrum is |G_c|^2/2 - eps_v over unoccupied plane waves.
    L, ecut = 8.0, 5.0
    lattice = np.eye(3) * L
    miller, g2 = lat.enumerate_half_sphere(lattice, ecut)
    npwh = len(miller)
    # occupy G = 0 and the cos-combination of the first shell member (1 of the 6 degenerate |m|=1 waves)
    psi = np.zeros((2, npwh), complex)
    psi[0, 0] = 1.0
    psi[1, 1] = 1 / np.sqrt(2)
    eig = np.array([0.0, 0.5 * g2[1]])
    P = lv.Problem(lattice, (12, 12, 12), ecut, 1, [psi], [eig], 0.0, use_hartree_fxc=False)
    # lowest excitations: from v=1 (eps = g2[1]/2) into the other |m| = 1 plane waves: omega = 0 (5 of them:
    # sin of the same G, and cos/sin of the two other axes), then from v=0 into |m|=1: omega = g2[1]/2
    rng = np.random.default_rng(0)
    x0 = inputs.trial_vectors(rng, [(2, psi)], 8)
    theta, X, it, res = davidson(P, 6, x0, tol=1e-9)
    assert np.allclose(theta[:5], 0.0, atol=1e-9)
    assert theta[5] == pytest.approx(0.5 * g2[1], abs=1e-9)


def dense_matrix(P, mode):
    """Matrix of A in an orthonormal real basis of the conduction space (tiny problems only)."""
    L = P.vector_len(mode)
    basis = []
    # real coordinates of the half-sphere storage: Re c(0), sqrt2 Re c(g), sqrt2 Im c(g)
    for i in range(L):
        for part in (1.0, 1j):
            if i % P.npwh == 0 and part == 1j:
                continue
            e = np.zeros(L, complex)
            e[i] = part if i % P.npwh == 0 else part / np.sqrt(2)
            basis.append(e)
    Bm = np.array([P.project_vector(e, mode) for e in basis])
    # orthonormalise the projected basis (rank = dim of conduction space)
    S = np.array([[P.vdot(a, b) for b in Bm] for a in Bm])
    w, U = np.linalg.eigh(S)
    keep = w > 1e-8
    Q = (U[:, keep] / np.sqrt(w[keep])).T @ Bm
    AQ = P.apply(Q, mode)
    H = np.array([[P.vdot(a, b) for b in AQ] for a in Q])
    return H


@pytest.mark.parametrize("mode", [lv.SPIN_CONSERVING, lv.SPIN_FLIP])
def test_davidson_finds_the_lowest_roots_of_the_dense_matrix(mode):
    lattice = [[4.0, 0, 0], [0.5, 4.2, 0], [0.3, -0.2, 4.5]]
    grid, ecut = (6, 5, 4), 6.0
    miller, g2 = lat.enumerate_half_sphere(lattice, ecut)
    rng = np.random.default_rng(21)
    psi = [inputs.orbitals(rng, n, g2, ecut) for n in (2, 2)]
    eig = [inputs.eigenvalues(rng, 2) for _ in range(2)]
    P = lv.Problem(lattice, grid, ecut, 2, psi, eig, 0.3)
    H = dense_matrix(P, mode)
    assert np.max(np.abs(H - H.T)) < 1e-11 * np.max(np.abs(H))
    exact = np.linalg.eigvalsh(0.5 * (H + H.T))
    if mode == lv.SPIN_CONSERVING:
        blocks = [(2, psi[0]), (2, psi[1])]
    else:
        blocks = [(2, psi[1])]
    x0 = inputs.trial_vectors(rng, blocks, 6)
    theta, X, it, res = davidson(P, 3, x0, mode=mode, tol=1e-8, max_subspace=30)
    assert np.max(np.abs(theta - exact[:3])) < 1e-10
    assert np.all(res <= 1e-8)


@pytest.mark.parametrize("mode", [lv.SPIN_CONSERVING, lv.SPIN_FLIP])
def test_projector_aware_correction_and_d_start_vectors(mode):
    """Readings A11b / A11c: the projector-aware correction solves P_c (T - eps_v - theta) P_c t = r on range(P_c) exactly, the
    start vectors are exact eigenvectors of D alone, and neither changes the converged roots (dense diagonalisation)."""
    from oracle.davidson import d_start_vectors, precond_projector
    lattice = [[4.0, 0, 0], [0.5, 4.2, 0], [0.3, -0.2, 4.5]]
    grid, ecut = (6, 5, 4), 6.0
    miller, g2 = lat.enumerate_half_sphere(lattice, ecut)
    rng = np.random.default_rng(22)
    psi = [inputs.orbitals(rng, n, g2, ecut) for n in (2, 2)]
    eig = [inputs.eigenvalues(rng, 2) for _ in range(2)]
    P = lv.Problem(lattice, grid, ecut, 2, psi, eig, 0.3)
    # (i) the correction: apply P_c (T - lam) P_c to t block by block and recover r (r taken in range(P_c))
    blocks = [(2, psi[0]), (2, psi[1])] if mode == lv.SPIN_CONSERVING else [(2, psi[1])]
    r = inputs.trial_vectors(rng, blocks, 1)[0]
    theta = 0.37
    t = precond_projector(P, r, theta, mode)
    assert np.linalg.norm(P.project_vector(t, mode) - t) < 1e-12 * np.linalg.norm(t)          # t lives in range(P_c)
    so = [0, 1] if mode == lv.SPIN_CONSERVING else [0]
    back, o = [], 0
    for b, s_occ in enumerate(so):
        s_tgt = s_occ if mode == lv.SPIN_CONSERVING else 1
        for v in range(2):
            tv = t[o:o + P.npwh]
            back.append(P.project_c((0.5 * P.g2 - P.eig[s_occ][v] - theta) * tv, s_tgt))
            o += P.npwh
    assert np.linalg.norm(np.concatenate(back) - r) < 1e-10 * np.linalg.norm(r)
    # (ii) D-only eigenvectors: with alpha = 0 and no Hxc the operator is D and x0 are exact eigenvectors, ascending
    P0 = lv.Problem(lattice, grid, ecut, 2, psi, eig, 0.0, use_hartree_fxc=False)
    x0 = d_start_vectors(P0, 5, mode)
    AX = P0.apply(x0, mode)
    ev = [P0.vdot(x0[i], AX[i]) for i in range(5)]
    for i in range(5):
        assert np.linalg.norm(AX[i] - ev[i] * x0[i]) < 1e-10
        assert P0.vdot(x0[i], x0[i]) == pytest.approx(1.0, abs=1e-12)
    assert np.all(np.diff(ev) >= -1e-12)
    exact0 = np.linalg.eigvalsh(dense_matrix(P0, mode))
    assert np.allclose(ev, exact0[:5], atol=1e-10)
    # (iii) the full solver with both readings finds the lowest roots of the dense matrix
    H = dense_matrix(P, mode)
    exact = np.linalg.eigvalsh(0.5 * (H + H.T))
    th, X, it, res = davidson(P, 3, d_start_vectors(P, 6, mode), mode=mode, tol=1e-8, max_subspace=30, precond="projector")
    assert np.max(np.abs(th - exact[:3])) < 1e-10 and np.all(res <= 1e-8)
