"""Pins for the SURVEY 8(f) extensions of the oracle: spin-flip xc kernel (Eqs. 24, 26), near-sightedness truncation and
the rotated K1d (Eqs. 31, 32), ACE exchange in D (Eqs. 28-30) and the off-diagonal block K2e - K2d (Eqs. 5, 7, S7, S9).
Every reference value below comes from explicit plane-wave sums (no FFT, no index maps), closed forms or invariants."""
import numpy as np
import pytest

from oracle import ace, lda, nearsight
from oracle import lattice as lat
from oracle import liouville as lv
import synthetic_inputs as inputs
from test_oracle_liouville import TRI, grid_points, small_problem, trial


class Brute:
    """Explicit cartesian sums on the grid of Problem P: O(N_r^2), independent of oracle/dft.py and of the index maps."""

    def __init__(self, P):
        self.P = P
        r = grid_points(P).reshape(-1, 3)
        self.nr = len(r)
        G = P.miller @ P.B
        self.kin = 0.5 * (G * G).sum(1)
        self.E = np.exp(1j * r @ G.T)
        ms = np.array(np.meshgrid(*lat.grid_miller(P.grid), indexing="ij")).reshape(3, -1).T
        Gg = ms @ P.B
        g2 = (Gg * Gg).sum(1)
        self.Eg = np.exp(1j * r @ Gg.T)
        self.k = np.where(g2 > 1e-12, 4 * np.pi / np.where(g2 > 1e-12, g2, 1.0), 0.0)
        self.phi = [np.array([self.real(c) for c in p]) for p in P.psi]

    def real(self, c):
        return ((self.E @ c) + (np.conj(self.E) @ np.conj(c)) - c[0]).real / np.sqrt(self.P.omega)

    def sphere(self, y):
        return (np.conj(self.E).T @ y) * np.sqrt(self.P.omega) / self.nr

    def coulomb(self, rho):
        return (self.Eg @ (self.k * ((np.conj(self.Eg).T @ rho) / self.nr))).real

    def project(self, yg, s):
        for c in self.P.psi[s]:
            yg = yg - c * (2 * np.real(np.vdot(c, yg)) - c[0].real * yg[0].real)
        return yg


def rel(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


# ---- spin-flip xc kernel ----------------------------------------------------------------------------------------
def test_sf_kernel_exchange_only_closed_form(monkeypatch):
    # Eq. 26 with Slater exchange only: f^SF = -(6/pi)^(1/3) (rho_up^(1/3) - rho_dn^(1/3)) / (rho_up - rho_dn)
    zero = dict(gamma=0.0, beta1=0.0, beta2=0.0, A=0.0, B=0.0, C=0.0, D=0.0)
    monkeypatch.setattr(lda, "PZ_U", zero)
    monkeypatch.setattr(lda, "PZ_P", zero)
    P, _ = small_problem(nocc=(3, 1), sf_xc_kernel=True, sf_cut=1e-3)
    ru, rd = P.rho0
    d = ru - rd
    ok = np.abs(d) >= 1e-3
    assert ok.any() and (~ok).any() or ok.all()
    expect = np.where(ok, -(6 / np.pi) ** (1 / 3) * (np.cbrt(ru) - np.cbrt(rd)) / np.where(ok, d, 1.0), 0.0)
    assert np.max(np.abs(P.fsf - expect)) < 1e-12 * np.max(np.abs(expect))
    assert np.all(P.fsf <= 0)


def test_sf_kernel_cut_zeroes_small_polarisation():
    P, _ = small_problem(nocc=(3, 2), sf_xc_kernel=True, sf_cut=1e9)
    assert np.all(P.fsf == 0.0)
    Q, _ = small_problem(nocc=(3, 2), sf_xc_kernel=True, sf_cut=0.0)
    vu, vd = lda.vxc(Q.rho0[0], Q.rho0[1])
    assert np.allclose(Q.fsf * (Q.rho0[0] - Q.rho0[1]), vu - vd, rtol=1e-12, atol=1e-14)


@pytest.mark.parametrize("mode", [lv.SPIN_FLIP, lv.SPIN_FLIP_DOWN_UP])
def test_sf_k1e_term_equals_brute_force(mode):
    # Eq. 24: (K1e^SF A)_v = P_c,s phi_v,s~ f^SF sum_v' phi_v',s~ a_v'  -- the only difference between kernel on and off
    P, rng = small_problem(nocc=(3, 2), sf_xc_kernel=True, sf_cut=1e-3)
    P0, _ = small_problem(nocc=(3, 2))
    X = trial(P, rng, 1, mode)
    diff = P.apply(X, mode)[0] - P0.apply(X, mode)[0]
    bf = Brute(P)
    so = 0 if mode == lv.SPIN_FLIP else 1
    a = np.array([bf.real(c) for c in P.split(X[0], mode)[0]])
    vu, vd = lda.vxc(*[np.sum(p * p, 0) for p in bf.phi])
    d = np.sum(bf.phi[0] ** 2, 0) - np.sum(bf.phi[1] ** 2, 0)
    fsf = np.where(np.abs(d) >= 1e-3, (vu - vd) / d, 0.0)
    drho = np.sum(bf.phi[so] * a, 0)
    ref = np.concatenate([bf.project(bf.sphere(bf.phi[so][v] * fsf * drho), 1 - so) for v in range(P.nocc[so])])
    assert np.linalg.norm(ref) > 1e-6
    assert rel(diff, ref) < 1e-11


# ---- near-sightedness: Eq. 32 and Eq. 31 --------------------------------------------------------------------------
def test_overlap_function_properties_and_closed_form():
    P, _ = small_problem(lattice=np.eye(3) * 8.0, grid=(12, 12, 12), ecut=6.0, nocc=(4, 3))
    S = nearsight.overlap_matrix(P.phi[0])
    assert np.allclose(np.diag(S), 1.0, rtol=0, atol=1e-14)
    assert np.array_equal(S, S.T) and np.all(S <= 1.0 + 1e-14) and np.all(S >= 0.0)        # Cauchy-Schwarz
    # closed form: phi_1 = Omega^-1/2, phi_2 = sqrt(2/Omega) cos(G.r): densities 1 and 1 + cos(2 G.r) (times 1/Omega),
    # S_12 = <1 * (1 + cos)> / sqrt(<1> <(1 + cos)^2>) = 1 / sqrt(3/2)
    r = grid_points(P)
    G = np.array([1, 2, 0]) @ P.B
    f1 = np.full(P.grid, 1 / np.sqrt(P.omega)); f2 = np.sqrt(2 / P.omega) * np.cos(r @ G)
    S2 = nearsight.overlap_matrix(np.stack([f1, f2]))
    assert S2[0, 1] == pytest.approx(1 / np.sqrt(1.5), rel=1e-13)
    # disjoint supports never overlap
    g1 = np.zeros(P.grid); g2 = np.zeros(P.grid); g1[:4] = 1.0; g2[6:9] = 2.0
    assert nearsight.overlap_matrix(np.stack([g1, g2]))[0, 1] == 0.0
    m = nearsight.pair_mask(S, 0.5)
    assert m.dtype == bool and np.all(np.diag(m)) and np.array_equal(m, S >= 0.5)


def test_masked_k1d_equals_brute_force():
    P0, rng = small_problem(nocc=(3, 2), use_hartree_fxc=False)
    mask = [np.array([[1, 0, 1], [0, 1, 1], [1, 1, 0]], bool), np.array([[1, 0], [0, 1]], bool)]
    P, _ = small_problem(nocc=(3, 2), use_hartree_fxc=False, pair_mask=mask)
    X = trial(P0, rng, 1)
    got = P.apply(X)[0]
    bf = Brute(P)
    xs = P.split(X[0], 0)
    out = []
    for s in range(2):
        a = np.array([bf.real(c) for c in xs[s]])
        for v in range(P.nocc[s]):
            y = np.zeros(bf.nr)
            for vp in range(P.nocc[s]):
                if mask[s][v, vp]:
                    y -= P.alpha * a[vp] * bf.coulomb(bf.phi[s][vp] * bf.phi[s][v])
            out.append(bf.project(bf.sphere(y) + (bf.kin - P.eig[s][v]) * xs[s][v], s))
    assert rel(got, np.concatenate(out)) < 1e-11
    assert rel(got, P0.apply(X)[0]) > 1e-3          # the mask really changes the result


def test_rotated_k1d_full_mask_is_invariant_and_truncated_equals_brute_force():
    # Eq. 31: with every pair kept the rotated evaluation equals the canonical one for ANY orthogonal U
    P0, rng = small_problem(nocc=(3, 2))
    U = [inputs.random_orthogonal(rng, n) for n in P0.nocc]
    X = trial(P0, rng, 1)
    ref = P0.apply(X)[0]
    Pr, _ = small_problem(nocc=(3, 2), wannier_u=U)
    assert rel(Pr.apply(X)[0], ref) < 1e-12
    # truncated: literal Eq. 31 with explicit sums
    mask = [np.array([[1, 1, 0], [1, 1, 0], [0, 0, 1]], bool), np.array([[1, 0], [0, 1]], bool)]
    Pm, _ = small_problem(nocc=(3, 2), use_hartree_fxc=False, wannier_u=U, pair_mask=mask)
    got = Pm.apply(X)[0]
    bf = Brute(Pm)
    xs = Pm.split(X[0], 0)
    out = []
    for s in range(2):
        a = np.array([bf.real(c) for c in xs[s]])
        n = Pm.nocc[s]
        pt = [sum(U[s][v, m] * bf.phi[s][v] for v in range(n)) for m in range(n)]          # phi~_m
        at = [sum(U[s][v, m] * a[v] for v in range(n)) for m in range(n)]                  # a~_m
        g = [sum(at[q] * bf.coulomb(pt[q] * pt[m]) for q in range(n) if mask[s][m, q]) if mask[s][m].any() else 0.0
             for m in range(n)]
        for v in range(n):
            y = -Pm.alpha * sum(U[s][v, m] * g[m] for m in range(n))
            out.append(bf.project(bf.sphere(y) + (bf.kin - Pm.eig[s][v]) * xs[s][v], s))
    assert rel(got, np.concatenate(out)) < 1e-11


# ---- ACE ------------------------------------------------------------------------------------------------------------
def _ace_problem():
    miller, g2 = lat.enumerate_half_sphere(TRI, 6.0)
    rng = np.random.default_rng(11)
    allorb = inputs.orbitals(rng, 5, g2, 6.0)                        # 3 occupied + 2 extra, jointly orthonormal
    psi = [allorb[:3], inputs.orbitals(rng, 2, g2, 6.0)]
    eig = [inputs.eigenvalues(rng, 3), inputs.eigenvalues(rng, 2)]
    P = lv.Problem(TRI, (6, 5, 4), 6.0, 2, psi, eig, 0.3)
    return P, allorb[3:], rng


def test_exchange_operator_equals_brute_force_and_ace_reproduces_it():
    P, extra, rng = _ace_problem()
    bf = Brute(P)
    c = extra[0]
    f = bf.real(c)
    ref = bf.sphere(-sum(bf.phi[0][v] * bf.coulomb(bf.phi[0][v] * f) for v in range(3)))       # Eq. 28
    assert rel(ace.exchange_apply(P, 0, c), ref) < 1e-11
    xi = ace.build(P, 0, extra)
    assert xi.shape == (5, P.npwh)
    for orb in list(P.psi[0]) + list(extra):                       # V_X^ACE phi_i = V_X phi_i on the N_ACE orbitals
        assert rel(ace.ace_apply(xi, orb), ace.exchange_apply(P, 0, orb)) < 1e-10
    # symmetric and negative semi-definite on arbitrary functions
    y = inputs.trial_vectors(rng, [(2, P.psi[0])], 1).reshape(2, -1)
    assert ace.gamma_dot(y[0], ace.ace_apply(xi, y[1])) == pytest.approx(ace.gamma_dot(ace.ace_apply(xi, y[0]), y[1]), rel=1e-12)
    assert ace.gamma_dot(y[0], ace.ace_apply(xi, y[0])) <= 0.0


def test_ace_in_d_term():
    # D with H = T + alpha V_X^ACE: on a function that is one of the extra ACE orbitals the
    # ACE operator is exact, so A_ace x - A x = alpha P_c V_X x with V_X from explicit sums
    P, extra, rng = _ace_problem()
    xi = [ace.build(P, 0, extra), ace.build(P, 1, None)]
    Pa = lv.Problem(TRI, (6, 5, 4), 6.0, 2, P.psi, P.eig, 0.3, ace=xi)
    x = np.zeros(P.vector_len(0), dtype=complex)
    x[P.npwh:2 * P.npwh] = extra[1]                                # block up, v = 1
    diff = (Pa.apply(x[None])[0] - P.apply(x[None])[0])
    bf = Brute(P)
    f = bf.real(extra[1])
    vx = bf.sphere(-sum(bf.phi[0][v] * bf.coulomb(bf.phi[0][v] * f) for v in range(3)))
    ref = np.zeros_like(x)
    ref[P.npwh:2 * P.npwh] = 0.3 * bf.project(vx, 0)
    assert rel(diff, ref) < 1e-10


# ---- off-diagonal block of Eq. 1 ----------------------------------------------------------------------------------
def test_coupling_spin_conserving_brute_force_and_symmetry():
    P, rng = small_problem(nocc=(3, 2))
    X = trial(P, rng, 2)
    BX = P.coupling(X)
    bf = Brute(P)
    rho0 = [np.sum(p * p, 0) for p in bf.phi]
    fuu, fud, fdd = lda.fxc(rho0[0], rho0[1])
    xs = P.split(X[0], 0)
    a = [np.array([bf.real(c) for c in blk]) for blk in xs]
    d = [np.sum(bf.phi[s] * a[s], 0) for s in range(2)]
    vh = bf.coulomb(d[0] + d[1])
    V = [vh + fuu * d[0] + fud * d[1], vh + fud * d[0] + fdd * d[1]]
    out = []
    for s in range(2):
        for v in range(P.nocc[s]):
            y = bf.phi[s][v] * V[s]
            for vp in range(P.nocc[s]):
                y = y - P.alpha * bf.phi[s][vp] * bf.coulomb(a[s][vp] * bf.phi[s][v])      # Eq. 7
            out.append(bf.project(bf.sphere(y), s))
    assert rel(BX[0], np.concatenate(out)) < 1e-11
    # the B block of the Casida matrix is symmetric
    M = np.array([[P.vdot(X[i], BX[j]) for j in range(2)] for i in range(2)])
    assert abs(M[0, 1] - M[1, 0]) < 1e-12 * np.max(np.abs(M))


def test_coupling_semilocal_limit_equals_k1e():
    # alpha = 0: K2d = K1d = 0 and, with real functions, K2e = K1e, so  A x - B x = D x = P_c (T - eps) x
    P, rng = small_problem(nocc=(3, 2), alpha=0.0)
    X = trial(P, rng, 1)
    diff = P.apply(X)[0] - P.coupling(X)[0]
    xs = P.split(X[0], 0)
    ref = np.concatenate([P.project_c((0.5 * P.g2 - P.eig[s][v]) * xs[s][v], s) for s in range(2) for v in range(P.nocc[s])])
    assert rel(diff, ref) < 1e-12


@pytest.mark.parametrize("mode", [lv.SPIN_FLIP, lv.SPIN_FLIP_DOWN_UP])
def test_coupling_spin_flip_brute_force(mode):
    # Eqs. S7, S9: output functions v over occ(s~) living in s; input = the opposite flip direction
    P, rng = small_problem(nocc=(3, 2), sf_xc_kernel=True, sf_cut=1e-3)
    other = lv.SPIN_FLIP_DOWN_UP if mode == lv.SPIN_FLIP else lv.SPIN_FLIP
    X = trial(P, rng, 1, other)
    got = P.coupling(X, mode)[0]
    bf = Brute(P)
    so = 0 if mode == lv.SPIN_FLIP else 1
    st = 1 - so
    a = np.array([bf.real(c) for c in P.split(X[0], other)[0]])           # functions v' over occ(s), living in s~
    vu, vd = lda.vxc(*[np.sum(p * p, 0) for p in bf.phi])
    d = np.sum(bf.phi[0] ** 2, 0) - np.sum(bf.phi[1] ** 2, 0)
    fsf = np.where(np.abs(d) >= 1e-3, (vu - vd) / d, 0.0)
    drho = np.sum(bf.phi[st] * a, 0)
    out = []
    for v in range(P.nocc[so]):
        y = bf.phi[so][v] * fsf * drho
        for vp in range(P.nocc[st]):
            y = y - P.alpha * bf.phi[st][vp] * bf.coulomb(a[vp] * bf.phi[so][v])
        out.append(bf.project(bf.sphere(y), st))
    assert rel(got, np.concatenate(out)) < 1e-11
