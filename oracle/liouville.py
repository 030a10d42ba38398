"""The TDA Liouville (Casida-A) operator  A = D + K1e - K1d  on a real-space grid,
spin-conserving (Eq. 9) and spin-flip (Eq. 21).

Test infrastructure only (see oracle/__init__.py).

Every step is the plain grid-discrete definition, in the paper's order:
  O0  reciprocal lattice, plane-wave half sphere (oracle/lattice.py, reading A7)
  O1  phi_vs(r_j) = Omega^-1/2 sum_G c_vs(G) exp(i G.r_j)           (Gamma, real orbitals)
  O2  rho0_s = sum_v phi_vs^2 ;  f_xc,ss' = d^2 e_xc / d rho_s d rho_s' (Eq. 8)
  O3  a_vs(r) from the trial vector as in O1                          (Eq. 2)
  O4  drho_s(r) = sum_v phi_vs(r) a_vs(r)                             (inner sum of Eq. 4)
  O5  V_s(r) = C[drho_up + drho_dn](r) + sum_s' f_xc,ss'(r) drho_s'(r) (f_Hxc = v_c + f_xc)
  O6  y(r) = phi_vs(r) V_s(r) - alpha sum_v' a_v's(r) C[phi_vs phi_v's](r)   (Eq. 4 minus Eq. 6, PAPER.md:82-93;
                                                                        tau_vv's = C[phi_v's phi_vs])
  O7  y(G) = (Omega^1/2 / N_r) sum_j y(r_j) exp(-i G.r_j),  G in the half sphere
  O8  y(G) += (|G|^2/2 - eps_vs) x_vs(G)   [+ V_loc,s a_vs on the grid, model H of reading A4]   (Eq. 3)
  O9  y <- y - sum_u c_us <c_us|y>          (P^c_s = 1 - sum_v |phi_v><phi_v|)
C[rho](r_j) = Re sum_{G != 0} (4 pi/|G|^2) rho~(G) exp(i G.r_j), rho~(G) = N_r^-1 sum_j rho(r_j) exp(-i G.r_j),
G over the whole FFT grid, G = 0 term zero (readings A10, A13, A17).

Spin flip, up-occupied -> down-virtual (Eqs. 21, 23, 25; readings A9, A16):
vector {x_v : v = 1..N_up}; y(r) = -alpha sum_v' a_v'(r) C[phi_v,up phi_v',up](r);
y(G) += (|G|^2/2 - eps_v,up) x_v(G) [+ V_loc,dn a_v]; projected with Phi_dn.  No Hartree, no f_xc (north star).

Vector layout (same as the C ABI): one trial vector = [spin][v][g] complex, contiguous;
a block is [k][spin][v][g].

Pins: tests/test_oracle_liouville.py.  Parity against numbers printed by the paper: unpinned
(the paper prints none for this operator); pinned instead by closed forms (plane-wave pair potential,
Hartree of a cosine, D on plane-wave orbitals), brute-force O(N_r^2) evaluation, Eq. 31 invariance,
symmetry of A, linearity in alpha, nspin=1 vs duplicated nspin=2.
"""
import numpy as np

from . import lattice as lat
from . import lda
from .dft import fft3

SPIN_CONSERVING = 0
SPIN_FLIP = 1           # up occupied -> down virtual
SPIN_FLIP_DOWN_UP = 2   # down occupied -> up virtual


class Problem:
    def __init__(self, lattice, grid, ecut_ry, nspin, psi, eig, alpha,
                 use_hartree_fxc=True, rho_floor=1e-10, vloc=None, fft_backend="radix"):
        self.A = np.asarray(lattice, dtype=np.float64).reshape(3, 3)
        self.grid = tuple(int(n) for n in grid)
        self.nr = self.grid[0] * self.grid[1] * self.grid[2]
        self.ecut = float(ecut_ry)
        self.nspin = int(nspin)
        self.alpha = float(alpha)
        self.use_hartree_fxc = bool(use_hartree_fxc)
        self.fft_backend = fft_backend
        # O0
        self.B, self.omega = lat.reciprocal(self.A)
        self.miller, self.g2 = lat.enumerate_half_sphere(self.A, self.ecut)
        self.npwh = len(self.miller)
        if not lat.check_grid_holds_sphere(self.miller, self.grid):
            raise ValueError("FFT grid does not hold the plane-wave sphere")
        n = np.array(self.grid)
        jp = np.mod(self.miller, n)                 # grid index of  G
        jm = np.mod(-self.miller, n)                # grid index of -G
        self.idx_p = (jp[:, 0] * n[1] + jp[:, 1]) * n[2] + jp[:, 2]
        self.idx_m = (jm[:, 0] * n[1] + jm[:, 1]) * n[2] + jm[:, 2]
        g2grid = lat.grid_g2(self.A, self.grid)
        with np.errstate(divide="ignore"):
            self.vc = np.where(g2grid > 0, 4.0 * np.pi / g2grid, 0.0)   # G = 0 zeroed
        self.vc[0, 0, 0] = 0.0
        # orbitals
        self.psi = [np.asarray(p, dtype=np.complex128) for p in psi]
        self.eig = [np.asarray(e, dtype=np.float64) for e in eig]
        assert len(self.psi) == self.nspin and len(self.eig) == self.nspin
        self.nocc = [p.shape[0] for p in self.psi]
        self.vloc = None if vloc is None else [np.asarray(v, dtype=np.float64).reshape(self.grid) for v in vloc]
        # O1
        self.phi = [np.stack([self.to_real(c) for c in p]) for p in self.psi]
        # O2
        rho = [np.sum(ph * ph, axis=0) for ph in self.phi]
        if self.nspin == 1:
            # closed shell: rho_up = rho_dn = sum_v phi_v^2 (each orbital holds one electron per spin)
            self.rho0 = [rho[0], rho[0]]
        else:
            self.rho0 = rho
        self.fuu, self.fud, self.fdd = lda.fxc(self.rho0[0], self.rho0[1], rho_floor)

    # ---- representation changes -------------------------------------------------
    def to_real(self, c):
        """O1/O3: f(r_j) = Omega^-1/2 sum_{G in sphere} c(G) exp(i G.r_j), c(-G) = conj c(G)."""
        full = np.zeros(self.nr, dtype=np.complex128)
        full[self.idx_m] = np.conj(c)
        full[self.idx_p] = c                       # G = 0 written last with c(0) itself
        f = fft3(full.reshape(self.grid), +1, self.fft_backend) / np.sqrt(self.omega)
        return f.real

    def to_sphere(self, y):
        """O7: y(G) = (Omega^1/2 / N_r) sum_j y(r_j) exp(-i G.r_j), G in the half sphere."""
        Y = fft3(y, -1, self.fft_backend).reshape(-1)
        return Y[self.idx_p] * (np.sqrt(self.omega) / self.nr)

    def coulomb(self, rho):
        """C[rho](r) = Re sum_{G != 0} 4 pi/|G|^2 rho~(G) exp(i G.r)."""
        rt = fft3(rho, -1, self.fft_backend) / self.nr
        return fft3(self.vc * rt, +1, self.fft_backend).real

    def project_c(self, y, s):
        """O9: y - sum_u c_us <c_us|y>."""
        out = y.copy()
        for c in self.psi[s]:
            out = out - c * (2.0 * np.real(np.vdot(c, y)) - c[0].real * y[0].real)
        return out

    # ---- layouts ------------------------------------------------------------------
    def vector_len(self, mode):
        if mode == SPIN_CONSERVING:
            return sum(self.nocc) * self.npwh
        if self.nspin != 2:
            raise ValueError("spin flip needs nspin = 2")
        src = 0 if mode == SPIN_FLIP else 1
        return self.nocc[src] * self.npwh

    def split(self, x, mode):
        """One trial vector -> list over spin blocks of [nocc, npwh] arrays."""
        x = np.asarray(x, dtype=np.complex128).reshape(-1)
        assert x.size == self.vector_len(mode)
        if mode == SPIN_CONSERVING:
            out, o = [], 0
            for s in range(self.nspin):
                out.append(x[o:o + self.nocc[s] * self.npwh].reshape(self.nocc[s], self.npwh))
                o += self.nocc[s] * self.npwh
            return out
        return [x.reshape(-1, self.npwh)]

    # ---- the operator ------------------------------------------------------------
    def prepare(self, x, mode=SPIN_CONSERVING):
        """O3-O5 for one trial vector: everything a column of A x needs that is shared by all columns."""
        xs = self.split(x, mode)
        a = [np.stack([self.to_real(c) for c in blk]) for blk in xs]          # O3
        ctx = dict(mode=mode, x=xs, a=a, V=None)
        if mode == SPIN_CONSERVING and self.use_hartree_fxc:
            drho = [np.sum(self.phi[s] * a[s], axis=0) for s in range(self.nspin)]   # O4
            if self.nspin == 2:
                vh = self.coulomb(drho[0] + drho[1])
                ctx["V"] = [vh + self.fuu * drho[0] + self.fud * drho[1],            # O5
                            vh + self.fud * drho[0] + self.fdd * drho[1]]
            else:
                # reading A6: singlet channel a_up = a_dn = a
                ctx["V"] = [self.coulomb(2.0 * drho[0]) + (self.fuu + self.fud) * drho[0]]
        return ctx

    def column(self, ctx, s, v):
        """O6-O9: the (spin block s, orbital v) component of A x for the prepared trial vector.

        Spin conserving: s is the spin.  Spin flip: s must be 0 (the only block)."""
        mode = ctx["mode"]
        if mode == SPIN_CONSERVING:
            s_occ, s_tgt, blk = s, s, s
        else:
            assert s == 0
            s_occ = 0 if mode == SPIN_FLIP else 1     # spin of the occupied orbitals (sigma-tilde)
            s_tgt = 1 - s_occ                          # spin of H, V_loc and P_c (sigma)
            blk = 0
        phi = self.phi[s_occ]
        a = ctx["a"][blk]
        y = np.zeros(self.grid)
        if ctx["V"] is not None:
            y += phi[v] * ctx["V"][s]
        for vp in range(self.nocc[s_occ]):                                            # O6
            tau = self.coulomb(phi[v] * phi[vp])
            y -= self.alpha * a[vp] * tau
        if self.vloc is not None:
            y += self.vloc[s_tgt] * a[v]
        yg = self.to_sphere(y)                                                        # O7
        yg = yg + (0.5 * self.g2 - self.eig[s_occ][v]) * ctx["x"][blk][v]             # O8
        return self.project_c(yg, s_tgt)                                              # O9

    def apply(self, X, mode=SPIN_CONSERVING):
        """A applied to a block X[k] of trial vectors; returns the same layout."""
        X = np.asarray(X, dtype=np.complex128)
        L = self.vector_len(mode)
        X = X.reshape(-1, L)
        out = np.zeros_like(X)
        for k in range(X.shape[0]):
            ctx = self.prepare(X[k], mode)
            o = 0
            for s in range(len(ctx["x"])):
                for v in range(ctx["x"][s].shape[0]):
                    out[k, o:o + self.npwh] = self.column(ctx, s, v)
                    o += self.npwh
        return out

    # ---- helpers for full vectors ----------------------------------------------
    def vdot(self, x, y):
        """Gamma inner product of two full trial vectors (sums over v and spin)."""
        x = np.asarray(x).reshape(-1, self.npwh)
        y = np.asarray(y).reshape(-1, self.npwh)
        return float(2.0 * np.real(np.vdot(x, y)) - np.sum(x[:, 0].real * y[:, 0].real))

    def project_vector(self, x, mode=SPIN_CONSERVING):
        """P_c applied block by block to a full trial vector (used to prepare inputs and in Davidson)."""
        xs = self.split(x, mode)
        out = []
        for b, blk in enumerate(xs):
            if mode == SPIN_CONSERVING:
                s_tgt = b
            else:
                s_tgt = 1 if mode == SPIN_FLIP else 0
            out.append(np.stack([self.project_c(c, s_tgt) for c in blk]).reshape(-1))
        return np.concatenate(out)

    def precond_diag(self, mode=SPIN_CONSERVING):
        """|G|^2/2 - eps_v for every element of a trial vector (the diagonal of the kinetic D)."""
        out = []
        if mode == SPIN_CONSERVING:
            for s in range(self.nspin):
                out.append((0.5 * self.g2[None, :] - self.eig[s][:, None]).reshape(-1))
        else:
            s_occ = 0 if mode == SPIN_FLIP else 1
            out.append((0.5 * self.g2[None, :] - self.eig[s_occ][:, None]).reshape(-1))
        return np.concatenate(out)
