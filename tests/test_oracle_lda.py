"""Pins for oracle/lda.py (reading A5: Slater exchange + Perdew-Zunger 1981 correlation)."""
import numpy as np
import pytest

from oracle import lda


def test_exchange_only_closed_forms(monkeypatch):
    zero = dict(gamma=0.0, beta1=0.0, beta2=0.0, A=0.0, B=0.0, C=0.0, D=0.0)
    monkeypatch.setattr(lda, "PZ_U", zero)
    monkeypatch.setattr(lda, "PZ_P", zero)
    # Dirac/Slater: e_x(rho) = -(3/4)(3/pi)^(1/3) rho^(4/3) for an unpolarised gas; the constant is 0.7385587663820224
    assert float(lda.exc_density(0.5, 0.5).f) == pytest.approx(-0.7385587663820224, rel=1e-14)
    ru = np.array([0.013, 0.4, 2.5]); rd = np.array([0.02, 0.1, 3.0])
    vu, vd = lda.vxc(ru, rd)
    assert np.allclose(vu, -(6 * ru / np.pi) ** (1 / 3), rtol=1e-13)
    assert np.allclose(vd, -(6 * rd / np.pi) ** (1 / 3), rtol=1e-13)
    fuu, fud, fdd = lda.fxc(ru, rd)
    assert np.allclose(fuu, -(1 / 3) * (6 / np.pi) ** (1 / 3) * ru ** (-2 / 3), rtol=1e-13)
    assert np.allclose(fdd, -(1 / 3) * (6 / np.pi) ** (1 / 3) * rd ** (-2 / 3), rtol=1e-13)
    assert np.all(fud == 0)


def test_pz81_constants():
    # Ceperley-Alder correlation energies (Ry, unpolarised) that PZ81 fits, rs = 2, 5, 10, 20: fit error < 1.5 %
    for rs, ca_ry in [(2, -0.0902), (5, -0.0563), (10, -0.0372), (20, -0.0230)]:
        assert 2 * lda.eps_c(rs, 0.0) == pytest.approx(ca_ry, rel=0.015)
    # high-density limit: A_U = (1 - ln 2)/pi^2 (Gell-Mann-Brueckner), A_P = A_U / 2
    assert lda.PZ_U["A"] == pytest.approx((1 - np.log(2)) / np.pi ** 2, abs=2e-5)
    assert lda.PZ_P["A"] == pytest.approx(lda.PZ_U["A"] / 2, abs=1e-5)
    # PZ81 matched value and slope of the two branches at rs = 1 (to the digits they print)
    for zeta in (0.0, 1.0):
        lo, hi = lda.eps_c(1 - 1e-9, zeta), lda.eps_c(1 + 1e-9, zeta)
        assert abs(lo - hi) < 5e-5
        dlo = (lda.eps_c(1 - 1e-9, zeta) - lda.eps_c(1 - 1e-4, zeta)) / 1e-4
        dhi = (lda.eps_c(1 + 1e-4, zeta) - lda.eps_c(1 + 1e-9, zeta)) / 1e-4
        assert abs(dlo - dhi) < 2e-4
    # polarised gas correlates less than the unpolarised one
    assert lda.eps_c(2.0, 0.0) < lda.eps_c(2.0, 0.5) < lda.eps_c(2.0, 1.0) < 0


def test_derivatives_by_finite_differences():
    rng = np.random.default_rng(0)
    ru = 10 ** rng.uniform(-3, 0.5, 40)     # spans rs < 1 and rs > 1
    rd = 10 ** rng.uniform(-3, 0.5, 40)
    e = lambda a, b: lda.exc_density(a, b).f
    vu, vd = lda.vxc(ru, rd)
    h = 1e-4 * ru
    fd = (-e(ru + 2 * h, rd) + 8 * e(ru + h, rd) - 8 * e(ru - h, rd) + e(ru - 2 * h, rd)) / (12 * h)
    assert np.allclose(vu, fd, rtol=1e-7, atol=1e-10)
    h = 1e-4 * rd
    fd = (-e(ru, rd + 2 * h) + 8 * e(ru, rd + h) - 8 * e(ru, rd - h) + e(ru, rd - 2 * h)) / (12 * h)
    assert np.allclose(vd, fd, rtol=1e-7, atol=1e-10)
    fuu, fud, fdd = lda.fxc(ru, rd)
    h = 1e-4 * ru
    d = lambda f: (-f(ru + 2 * h, rd) + 8 * f(ru + h, rd) - 8 * f(ru - h, rd) + f(ru - 2 * h, rd)) / (12 * h)
    assert np.allclose(fuu, d(lambda a, b: lda.vxc(a, b)[0]), rtol=1e-6)
    assert np.allclose(fud, d(lambda a, b: lda.vxc(a, b)[1]), rtol=1e-6)
    h = 1e-4 * rd
    d = lambda f: (-f(ru, rd + 2 * h) + 8 * f(ru, rd + h) - 8 * f(ru, rd - h) + f(ru, rd - 2 * h)) / (12 * h)
    assert np.allclose(fdd, d(lambda a, b: lda.vxc(a, b)[1]), rtol=1e-6)
    assert np.allclose(fud, d(lambda a, b: lda.vxc(a, b)[0]), rtol=1e-6)     # f_ud = f_du


def test_spin_exchange_symmetry_and_floor():
    ru = np.array([0.03, 0.7]); rd = np.array([0.2, 0.05])
    a = lda.fxc(ru, rd); b = lda.fxc(rd, ru)
    assert np.allclose(a[0], b[2]) and np.allclose(a[1], b[1]) and np.allclose(a[2], b[0])
    f = lda.fxc(np.array([1e-12, 0.1]), np.array([0.1, 0.1]), rho_floor=1e-10)
    assert f[0][0] == 0 and f[1][0] == 0 and f[2][0] == 0 and f[0][1] != 0


def test_spin_interpolation_normalisation():
    """f(zeta) of reading A5 is normalised so that f(0) = 0 and f(1) = 1: the fully polarised gas has exactly the
    PZ81 'P' correlation energy, the unpolarised one exactly 'U' (PAPER.md:770, :915 cite PZ81).  A wrong denominator
    (2^(1/3) - 1, 2^(4/3) - 1, ...) passes the continuity / ordering checks above but fails here."""
    for rs in (0.3, 1.0, 2.0, 7.5):
        hd = lda.HyperDual(np.float64(rs))
        eu, ep = float(lda._eps_c_pz(hd, lda.PZ_U).f), float(lda._eps_c_pz(hd, lda.PZ_P).f)
        assert lda.eps_c(rs, 0.0) == eu
        assert lda.eps_c(rs, 1.0) == pytest.approx(ep, rel=1e-15)
        assert lda.eps_c(rs, -1.0) == pytest.approx(ep, rel=1e-15)
        # the same through exc_density itself (the function fxc differentiates): e_xc - e_x = rho eps_c
        rho = 3.0 / (4.0 * np.pi * rs ** 3)
        ex_pol = -0.75 * (6.0 / np.pi) ** (1.0 / 3.0) * rho ** (4.0 / 3.0)
        assert float(lda.exc_density(rho, 0.0).f) - ex_pol == pytest.approx(rho * ep, rel=1e-12)
        ex_unp = -0.75 * (6.0 / np.pi) ** (1.0 / 3.0) * 2.0 * (rho / 2.0) ** (4.0 / 3.0)
        assert float(lda.exc_density(rho / 2.0, rho / 2.0).f) - ex_unp == pytest.approx(rho * eu, rel=1e-12)
    # value typed from the PZ81 formula: f(1/2) = [(3/2)^(4/3) + (1/2)^(4/3) - 2] / (2^(4/3) - 2) = 0.11394 / 0.51984 = 0.2191
    hd = lda.HyperDual(np.float64(2.0))
    eu, ep = float(lda._eps_c_pz(hd, lda.PZ_U).f), float(lda._eps_c_pz(hd, lda.PZ_P).f)
    f_half = (1.5 ** (4.0 / 3.0) + 0.5 ** (4.0 / 3.0) - 2.0) / (2.0 ** (4.0 / 3.0) - 2.0)
    assert f_half == pytest.approx(0.2191, abs=1e-4)
    assert lda.eps_c(2.0, 0.5) == pytest.approx(eu + f_half * (ep - eu), rel=1e-14)
