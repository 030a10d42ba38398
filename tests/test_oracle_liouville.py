"""Pins for oracle/liouville.py: closed forms, brute force on a tiny cell and the invariants the paper states."""
import math

import numpy as np
import pytest

from oracle import lattice as lat
from oracle import liouville as lv
from oracle import lda
import synthetic_inputs as inputs

HEX = [[9.0, 0, 0], [-4.5, 9.0 * math.sqrt(3) / 2, 0], [0, 0, 7.0]]
TRI = [[4.0, 0, 0], [0.5, 4.2, 0], [0.3, -0.2, 4.5]]


def small_problem(lattice=TRI, grid=(6, 5, 4), ecut=6.0, nspin=2, nocc=(3, 2), alpha=0.3, seed=7, vloc=False, **kw):
    miller, g2 = lat.enumerate_half_sphere(lattice, ecut)
    rng = np.random.default_rng(seed)
    psi = [inputs.orbitals(rng, nocc[s], g2, ecut, envelope=True) for s in range(nspin)]
    eig = [inputs.eigenvalues(rng, nocc[s]) for s in range(nspin)]
    vl = None
    if vloc:
        vl = [rng.standard_normal(grid) for _ in range(2)]
    P = lv.Problem(lattice, grid, ecut, nspin, psi, eig, alpha, vloc=vl, **kw)
    return P, rng


def trial(P, rng, nvec, mode=lv.SPIN_CONSERVING):
    if mode == lv.SPIN_CONSERVING:
        blocks = [(P.nocc[s], P.psi[s]) for s in range(P.nspin)]
    else:
        src = 0 if mode == lv.SPIN_FLIP else 1
        blocks = [(P.nocc[src], P.psi[1 - src])]
    return inputs.trial_vectors(rng, blocks, nvec)


def grid_points(P):
    j = np.meshgrid(*[np.arange(n) / n for n in P.grid], indexing="ij")
    return sum(j[i][..., None] * P.A[i] for i in range(3))          # [n1,n2,n3,3] cartesian


# ---------------------------------------------------------------------------------------------
def test_pair_densities_integrate_to_delta():
    P, _ = small_problem(lattice=np.eye(3) * 7.0, grid=(12, 10, 9), ecut=8.0, nocc=(4, 3))
    for s in range(2):
        S = np.einsum("iabc,jabc->ij", P.phi[s], P.phi[s]) * P.omega / P.nr
        assert np.max(np.abs(S - np.eye(P.nocc[s]))) < 1e-13


@pytest.mark.parametrize("lattice,grid", [(TRI, (6, 5, 4)), (HEX, (12, 12, 10))])
def test_to_real_is_the_plane_wave_sum(lattice, grid):
    # phi(r_j) = Omega^-1/2 sum_G c(G) exp(i G.r_j) evaluated with explicit cartesian G.r
    P, rng = small_problem(lattice=lattice, grid=grid, ecut=6.0 if lattice is TRI else 3.0)
    r = grid_points(P)
    G = P.miller @ P.B
    c = P.psi[0][1]
    ph = np.exp(1j * np.einsum("abcx,gx->abcg", r, G))
    direct = (ph @ c + np.conj(ph) @ np.conj(c) - c[0]).real / np.sqrt(P.omega)
    assert np.max(np.abs(direct - P.phi[0][1])) < 1e-12
    # and back
    back = P.to_sphere(P.phi[0][1])
    assert np.max(np.abs(back - c)) < 1e-13


@pytest.mark.parametrize("lattice,grid,m1,m2", [
    (np.eye(3) * 10.0, (12, 12, 12), (1, 0, 2), (0, 2, -1)),
    (HEX, (12, 12, 10), (1, 1, 0), (2, -1, 1)),
    (TRI, (10, 9, 8), (1, -1, 1), (1, -1, 1)),          # G1 = G2: exercises the zeroed G = 0 term
])
def test_plane_wave_pair_potential_closed_form(lattice, grid, m1, m2):
    # phi_1 = sqrt(2/Omega) cos(G1.r), phi_2 = sqrt(2/Omega) cos(G2.r)  =>
    # C[phi_1 phi_2] = (4 pi/Omega) [cos((G1+G2).r)/|G1+G2|^2 + cos((G1-G2).r)/|G1-G2|^2]   (G = 0 term dropped)
    P, _ = small_problem(lattice=lattice, grid=grid, ecut=1.0, nocc=(1, 1))
    r = grid_points(P)
    G1 = np.array(m1) @ P.B; G2 = np.array(m2) @ P.B
    p1 = np.sqrt(2 / P.omega) * np.cos(r @ G1)
    p2 = np.sqrt(2 / P.omega) * np.cos(r @ G2)
    expect = np.zeros(P.grid)
    for Gs in (G1 + G2, G1 - G2):
        if np.dot(Gs, Gs) > 1e-12:
            expect += 4 * np.pi / P.omega * np.cos(r @ Gs) / np.dot(Gs, Gs)
    assert np.max(np.abs(P.coulomb(p1 * p2) - expect)) < 1e-13 * max(1.0, np.max(np.abs(expect)))
    # Hartree potential of a single cosine
    assert np.max(np.abs(P.coulomb(np.cos(r @ G1)) - 4 * np.pi / np.dot(G1, G1) * np.cos(r @ G1))) < 1e-12


def brute_force_apply(P, x, mode):
    """A x from explicit cartesian sums: no FFT, no index maps (uses only P's inputs and the G list)."""
    r = grid_points(P).reshape(-1, 3)
    nr = len(r)
    G = P.miller @ P.B
    E = np.exp(1j * r @ G.T)                                            # [nr, npwh]

    def real(c):
        return ((E @ c) + (np.conj(E) @ np.conj(c)) - c[0]).real / np.sqrt(P.omega)

    def sphere(y):
        return (np.conj(E).T @ y) * np.sqrt(P.omega) / nr

    # all grid G vectors, from the signed Miller indices
    ms = np.array(np.meshgrid(*lat.grid_miller(P.grid), indexing="ij")).reshape(3, -1).T
    Gg = ms @ P.B
    g2 = (Gg * Gg).sum(1)
    Eg = np.exp(1j * r @ Gg.T)                                          # [nr, nr]

    def coulomb(rho):
        rt = (np.conj(Eg).T @ rho) / nr
        k = np.where(g2 > 1e-12, 4 * np.pi / np.where(g2 > 1e-12, g2, 1.0), 0.0)
        return (Eg @ (k * rt)).real

    phi = [np.array([real(c) for c in p]) for p in P.psi]
    xs = P.split(x, mode)
    a = [np.array([real(c) for c in blk]) for blk in xs]
    out = []
    if mode == lv.SPIN_CONSERVING:
        V = None
        if P.use_hartree_fxc:
            rho0 = [np.sum(p * p, 0) for p in phi]
            fuu, fud, fdd = lda.fxc(rho0[0], rho0[1])
            d = [np.sum(phi[s] * a[s], 0) for s in range(2)]
            vh = coulomb(d[0] + d[1])
            V = [vh + fuu * d[0] + fud * d[1], vh + fud * d[0] + fdd * d[1]]
        for s in range(2):
            for v in range(P.nocc[s]):
                y = np.zeros(nr)
                if V is not None:
                    y += phi[s][v] * V[s]
                for vp in range(P.nocc[s]):
                    y -= P.alpha * a[s][vp] * coulomb(phi[s][vp] * phi[s][v])
                if P.vloc is not None:
                    y += P.vloc[s].reshape(-1) * a[s][v]
                yg = sphere(y) + (0.5 * (G * G).sum(1) - P.eig[s][v]) * xs[s][v]
                for c in P.psi[s]:
                    yg = yg - c * (2 * np.real(np.vdot(c, yg)) - c[0].real * yg[0].real)
                out.append(yg)
    else:
        so = 0 if mode == lv.SPIN_FLIP else 1
        st = 1 - so
        for v in range(P.nocc[so]):
            y = np.zeros(nr)
            for vp in range(P.nocc[so]):
                y -= P.alpha * a[0][vp] * coulomb(phi[so][vp] * phi[so][v])
            if P.vloc is not None:
                y += P.vloc[st].reshape(-1) * a[0][v]
            yg = sphere(y) + (0.5 * (G * G).sum(1) - P.eig[so][v]) * xs[0][v]
            for c in P.psi[st]:
                yg = yg - c * (2 * np.real(np.vdot(c, yg)) - c[0].real * yg[0].real)
            out.append(yg)
    return np.concatenate(out)


@pytest.mark.parametrize("mode", [lv.SPIN_CONSERVING, lv.SPIN_FLIP, lv.SPIN_FLIP_DOWN_UP])
@pytest.mark.parametrize("vloc", [False, True])
def test_apply_equals_brute_force_on_tiny_cell(mode, vloc):
    P, rng = small_problem(vloc=vloc)
    X = trial(P, rng, 2, mode)
    AX = P.apply(X, mode)
    for k in range(2):
        ref = brute_force_apply(P, X[k], mode)
        assert np.linalg.norm(AX[k] - ref) < 1e-12 * np.linalg.norm(ref)


def test_eq31_unitary_invariance_of_k1d():
    # PAPER.md:230-237 (Eq. 31): K1d is invariant under a unitary rotation of the occupied orbitals.
    # With degenerate eigenvalues the whole operator is covariant: out_v = sum_m U_vm out~_m.
    P, rng = small_problem(lattice=np.eye(3) * 6.0, grid=(9, 8, 10), ecut=7.0, nocc=(4, 3))
    for s in range(2):
        P.eig[s][:] = -0.2
    X = trial(P, rng, 1)[0]
    AX = P.split(P.apply(X[None])[0], 0)
    U = [np.linalg.qr(rng.standard_normal((n, n)))[0] for n in P.nocc]
    psi_t = [U[s].T @ P.psi[s] for s in range(2)]                     # phi~_n = sum_v U_vn phi_v
    Pt = lv.Problem(P.A, P.grid, P.ecut, 2, psi_t, P.eig, P.alpha)
    xs = P.split(X, 0)
    Xt = np.concatenate([(U[s].T @ xs[s]).reshape(-1) for s in range(2)])
    AXt = Pt.split(Pt.apply(Xt[None])[0], 0)
    for s in range(2):
        assert np.linalg.norm(U[s] @ AXt[s] - AX[s]) < 1e-12 * np.linalg.norm(AX[s])


@pytest.mark.parametrize("mode", [lv.SPIN_CONSERVING, lv.SPIN_FLIP])
def test_operator_is_symmetric_on_the_conduction_space(mode):
    P, rng = small_problem(lattice=HEX, grid=(12, 12, 10), ecut=3.0, nocc=(4, 3), vloc=True)
    X = trial(P, rng, 3, mode)
    AX = P.apply(X, mode)
    M = np.array([[P.vdot(X[i], AX[j]) for j in range(3)] for i in range(3)])
    assert np.max(np.abs(M - M.T)) < 1e-12 * np.max(np.abs(M))
    # range of A is inside the conduction space: projecting again changes nothing
    for k in range(3):
        assert np.linalg.norm(P.project_vector(AX[k], mode) - AX[k]) < 1e-12 * np.linalg.norm(AX[k])


def test_linear_in_alpha_and_alpha_zero_limit():
    # alpha = 0 => K1d = 0
    kw = dict(lattice=TRI, grid=(6, 5, 4), ecut=6.0, nocc=(3, 2), seed=11)
    P0, rng = small_problem(alpha=0.0, **kw)
    P1, _ = small_problem(alpha=0.2, **kw)
    P2, _ = small_problem(alpha=0.4, **kw)
    X = trial(P0, rng, 1)
    y0, y1, y2 = P0.apply(X), P1.apply(X), P2.apply(X)
    assert np.linalg.norm((y2 - y0) - 2 * (y1 - y0)) < 1e-12 * np.linalg.norm(y2 - y0)
    assert np.linalg.norm(y1 - y0) > 1e-3 * np.linalg.norm(y0)
    # alpha = 0 and no Hxc: A = P_c (T - eps)
    Pn, _ = small_problem(alpha=0.0, use_hartree_fxc=False, **kw)
    y = Pn.apply(X)[0]
    expect = Pn.project_vector(Pn.precond_diag() * X[0])
    assert np.linalg.norm(y - expect) < 1e-13 * np.linalg.norm(expect)


def test_k1e_is_the_hxc_quadratic_form():
    # <y| K1e x> = int int drho[y] f_Hxc drho[x]  (Eq. 4), evaluated on the grid
    kw = dict(lattice=np.eye(3) * 6.0, grid=(10, 9, 8), ecut=7.0, nocc=(3, 3), seed=5, alpha=0.0)
    Pon, rng = small_problem(**kw)
    Poff, _ = small_problem(use_hartree_fxc=False, **kw)
    X = trial(Pon, rng, 2)
    k1e_x = Pon.apply(X[:1])[0] - Poff.apply(X[:1])[0]
    lhs = Pon.vdot(X[1], k1e_x)
    cx, cy = Pon.prepare(X[0]), Pon.prepare(X[1])
    dx = [np.sum(Pon.phi[s] * cx["a"][s], 0) for s in range(2)]
    dy = [np.sum(Pon.phi[s] * cy["a"][s], 0) for s in range(2)]
    w = Pon.omega / Pon.nr
    rhs = w * np.sum((dy[0] + dy[1]) * Pon.coulomb(dx[0] + dx[1]))
    rhs += w * np.sum(dy[0] * (Pon.fuu * dx[0] + Pon.fud * dx[1]) + dy[1] * (Pon.fud * dx[0] + Pon.fdd * dx[1]))
    assert lhs == pytest.approx(rhs, rel=1e-11)


def test_spin_flip_ignores_hartree_and_fxc():
    # north star: "spin-flip omits the Hartree and f_xc terms" (reading A9)
    kw = dict(lattice=TRI, grid=(6, 5, 4), ecut=6.0, nocc=(3, 2), seed=3)
    Pon, rng = small_problem(**kw)
    Poff, _ = small_problem(use_hartree_fxc=False, **kw)
    X = trial(Pon, rng, 1, lv.SPIN_FLIP)
    assert np.array_equal(Pon.apply(X, lv.SPIN_FLIP), Poff.apply(X, lv.SPIN_FLIP))
    # while the spin-conserving operator does change
    Xc = trial(Pon, rng, 1)
    assert np.linalg.norm(Pon.apply(Xc) - Poff.apply(Xc)) > 1e-6


def test_spin_flip_modes_are_mirror_images():
    kw = dict(lattice=TRI, grid=(6, 5, 4), ecut=6.0, nocc=(3, 2), seed=3, vloc=True)
    P, rng = small_problem(**kw)
    Q = lv.Problem(P.A, P.grid, P.ecut, 2, P.psi[::-1], P.eig[::-1], P.alpha, vloc=P.vloc[::-1])
    X = trial(P, rng, 1, lv.SPIN_FLIP_DOWN_UP)
    assert np.allclose(P.apply(X, lv.SPIN_FLIP_DOWN_UP), Q.apply(X, lv.SPIN_FLIP), rtol=0, atol=1e-14)


def test_closed_shell_equals_duplicated_spin_polarised():
    # reading A6: nspin = 1 is the singlet channel of an nspin = 2 problem with identical spin channels
    lattice, grid, ecut = np.eye(3) * 6.0, (10, 9, 8), 7.0
    miller, g2 = lat.enumerate_half_sphere(lattice, ecut)
    rng = np.random.default_rng(9)
    psi = inputs.orbitals(rng, 3, g2, ecut)
    eig = inputs.eigenvalues(rng, 3)
    P1 = lv.Problem(lattice, grid, ecut, 1, [psi], [eig], 0.25)
    P2 = lv.Problem(lattice, grid, ecut, 2, [psi, psi], [eig, eig], 0.25)
    x = inputs.trial_vectors(rng, [(3, psi)], 1)[0]
    y1 = P1.apply(x[None])[0]
    y2 = P2.apply(np.concatenate([x, x])[None])[0]
    assert np.linalg.norm(y2[: x.size] - y1) < 1e-13 * np.linalg.norm(y1)
    assert np.linalg.norm(y2[x.size:] - y1) < 1e-13 * np.linalg.norm(y1)


def test_projector_properties():
    P, rng = small_problem()
    for s in range(2):
        for c in P.psi[s]:
            assert np.linalg.norm(P.project_c(c, s)) < 1e-13
        y = rng.standard_normal(P.npwh) + 1j * rng.standard_normal(P.npwh)
        y[0] = y[0].real
        py = P.project_c(y, s)
        assert np.linalg.norm(P.project_c(py, s) - py) < 1e-13 * np.linalg.norm(py)


def test_column_matches_apply():
    P, rng = small_problem()
    X = trial(P, rng, 1)
    AX = P.split(P.apply(X)[0], 0)
    ctx = P.prepare(X[0])
    assert np.array_equal(P.column(ctx, 1, 1), AX[1][1])
