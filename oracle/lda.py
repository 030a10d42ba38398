"""Spin-polarised LDA (Slater exchange + Perdew-Zunger 1981 correlation) and its
first and second density derivatives, for the oracle.

Test infrastructure only (see oracle/__init__.py).

The paper defines f_xc = delta V_xc / delta rho at the ground-state density
(Eq. 8) and names only "LDA" with SI ref. 10 = Perdew-Zunger
1981.  Reading A5 of DESIGN.md fixes the functional:
Hartree units,
  e_x(rho_up, rho_dn) = -(3/4) (6/pi)^(1/3) (rho_up^(4/3) + rho_dn^(4/3)),
  e_c = rho * [eps_c^U(rs) + f(zeta) (eps_c^P(rs) - eps_c^U(rs))],
  rs = (3 / (4 pi rho))^(1/3), zeta = (rho_up - rho_dn)/rho,
  f(zeta) = [(1+zeta)^(4/3) + (1-zeta)^(4/3) - 2] / (2^(4/3) - 2),
  eps_c^i = gamma_i / (1 + beta1_i sqrt(rs) + beta2_i rs)              rs >= 1
          = A_i ln rs + B_i + C_i rs ln rs + D_i rs                     rs <  1.
v_xc,s = d e_xc / d rho_s and f_xc,ss' = d^2 e_xc / d rho_s d rho_s' are obtained
by hyper-dual-number differentiation of e_xc itself (exact to rounding; no
hand-derived derivative formula appears here, so the CUDA side's hand-derived
formulas are an independent derivation).
Pins: tests/test_oracle_lda.py (exchange closed forms, eps_c values from the
PZ81 formula at rs = 1, 2, 5 typed in by hand, finite differences of e_xc and
v_xc, symmetry f_ud = f_du, spin-exchange symmetry).
"""
import numpy as np

# Perdew-Zunger 1981 parameters (Hartree), unpolarised (U) and polarised (P)
PZ_U = dict(gamma=-0.1423, beta1=1.0529, beta2=0.3334, A=0.0311, B=-0.048, C=0.0020, D=-0.0116)
PZ_P = dict(gamma=-0.0843, beta1=1.3981, beta2=0.2611, A=0.01555, B=-0.0269, C=0.0007, D=-0.0048)


class HyperDual:
    """f + f1 e1 + f2 e2 + f12 e1 e2 with e1^2 = e2^2 = 0: carries d/dx1, d/dx2, d2/dx1dx2."""

    __slots__ = ("f", "f1", "f2", "f12")

    def __init__(self, f, f1=0.0, f2=0.0, f12=0.0):
        self.f = np.asarray(f, dtype=np.float64)
        z = np.zeros_like(self.f)
        self.f1 = z + f1
        self.f2 = z + f2
        self.f12 = z + f12

    @staticmethod
    def lift(x):
        return x if isinstance(x, HyperDual) else HyperDual(x)

    def __add__(self, o):
        o = HyperDual.lift(o)
        return HyperDual(self.f + o.f, self.f1 + o.f1, self.f2 + o.f2, self.f12 + o.f12)

    __radd__ = __add__

    def __neg__(self):
        return HyperDual(-self.f, -self.f1, -self.f2, -self.f12)

    def __sub__(self, o):
        return self + (-HyperDual.lift(o))

    def __rsub__(self, o):
        return HyperDual.lift(o) + (-self)

    def __mul__(self, o):
        o = HyperDual.lift(o)
        return HyperDual(self.f * o.f,
                         self.f1 * o.f + self.f * o.f1,
                         self.f2 * o.f + self.f * o.f2,
                         self.f12 * o.f + self.f1 * o.f2 + self.f2 * o.f1 + self.f * o.f12)

    __rmul__ = __mul__

    def apply(self, g, dg, d2g):
        """Compose with a scalar function given its value and two derivatives at self.f."""
        return HyperDual(g, dg * self.f1, dg * self.f2, dg * self.f12 + d2g * self.f1 * self.f2)

    def __truediv__(self, o):
        o = HyperDual.lift(o)
        inv = o.apply(1.0 / o.f, -1.0 / o.f ** 2, 2.0 / o.f ** 3)
        return self * inv

    def __rtruediv__(self, o):
        return HyperDual.lift(o) / self

    def pow(self, a):
        x = self.f
        return self.apply(x ** a, a * x ** (a - 1.0), a * (a - 1.0) * x ** (a - 2.0))

    def log(self):
        x = self.f
        return self.apply(np.log(x), 1.0 / x, -1.0 / x ** 2)

    def sqrt(self):
        return self.pow(0.5)


def _where(cond, a, b):
    return HyperDual(np.where(cond, a.f, b.f), np.where(cond, a.f1, b.f1),
                     np.where(cond, a.f2, b.f2), np.where(cond, a.f12, b.f12))


def _eps_c_pz(rs, par):
    """PZ81 correlation energy per electron for one polarisation state; rs may be HyperDual."""
    hi = par["gamma"] / (1.0 + par["beta1"] * rs.sqrt() + par["beta2"] * rs)
    lnrs = rs.log()
    lo = par["A"] * lnrs + par["B"] + par["C"] * rs * lnrs + par["D"] * rs
    return _where(rs.f >= 1.0, hi, lo)


def exc_density(rho_up, rho_dn):
    """e_xc(rho_up, rho_dn) per unit volume (Hartree/bohr^3); arguments may be HyperDual."""
    ru = HyperDual.lift(rho_up)
    rd = HyperDual.lift(rho_dn)
    ex = -0.75 * (6.0 / np.pi) ** (1.0 / 3.0) * (ru.pow(4.0 / 3.0) + rd.pow(4.0 / 3.0))
    rho = ru + rd
    rs = (3.0 / (4.0 * np.pi * rho)).pow(1.0 / 3.0)
    zeta = (ru - rd) / rho
    fz = ((1.0 + zeta).pow(4.0 / 3.0) + (1.0 - zeta).pow(4.0 / 3.0) - 2.0) / (2.0 ** (4.0 / 3.0) - 2.0)
    ecu = _eps_c_pz(rs, PZ_U)
    ecp = _eps_c_pz(rs, PZ_P)
    ec = rho * (ecu + fz * (ecp - ecu))
    return ex + ec


def eps_c(rs, zeta):
    """PZ81 correlation energy per electron at (rs, zeta): plain floats, for the pins."""
    rs = HyperDual(np.float64(rs))
    fz = ((1 + zeta) ** (4 / 3) + (1 - zeta) ** (4 / 3) - 2) / (2 ** (4 / 3) - 2)
    u = _eps_c_pz(rs, PZ_U).f
    p = _eps_c_pz(rs, PZ_P).f
    return float(u + fz * (p - u))


def vxc(rho_up, rho_dn):
    """(v_xc,up, v_xc,dn) = d e_xc / d rho_s."""
    ru = np.asarray(rho_up, dtype=np.float64)
    rd = np.asarray(rho_dn, dtype=np.float64)
    e = exc_density(HyperDual(ru, 1.0, 0.0), HyperDual(rd, 0.0, 1.0))
    return e.f1, e.f2


def fxc(rho_up, rho_dn, rho_floor=1e-10):
    """(f_uu, f_ud, f_dd) = d^2 e_xc / d rho_s d rho_s' at the given densities.

    Points where either spin density is below rho_floor get f_xc = 0 (reading A5)."""
    ru = np.asarray(rho_up, dtype=np.float64)
    rd = np.asarray(rho_dn, dtype=np.float64)
    ok = (ru >= rho_floor) & (rd >= rho_floor)
    su = np.where(ok, ru, 1.0)
    sd = np.where(ok, rd, 1.0)
    fuu = exc_density(HyperDual(su, 1.0, 1.0), HyperDual(sd, 0.0, 0.0)).f12
    fud = exc_density(HyperDual(su, 1.0, 0.0), HyperDual(sd, 0.0, 1.0)).f12
    fdd = exc_density(HyperDual(su, 0.0, 0.0), HyperDual(sd, 1.0, 1.0)).f12
    z = np.zeros_like(ru)
    return np.where(ok, fuu, z), np.where(ok, fud, z), np.where(ok, fdd, z)
