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

Options beyond the TDA north-star path (each default reproduces the path above exactly):
  sf_xc_kernel  spin flip keeps K1e^SF (Eq. 24) with the kernel of Eq. 26,
                f^SF(r) = (V_xc,s(r) - V_xc,s~(r)) / (rho_s(r) - rho_s~(r)), set to zero where |rho_up - rho_dn| < sf_cut
                ("1e-3", no unit given; reading A9 takes e/bohr^3):
                y(r) += phi_v,s~(r) f^SF(r) sum_v' phi_v',s~(r) a_v'(r)
  pair_mask     near-sightedness truncation: the pair potentials tau_mn with mask[m, n] False are
                taken as zero in K1d
  wannier_u     Eq. 31: phi_v = sum_n U_vn phi~_n; K1d is evaluated with the rotated orbitals,
                (K1d A)_v = alpha P_c sum_m U_vm { sum_n a~_n tau~_mn },  a~_n = sum_v' U_v'n a_v' (real U), and the
                mask then refers to pairs (m, n) of ROTATED orbitals, as in the paper
  ace           D uses H = T + V_loc + alpha V_X^ACE (Eqs. 28-30; oracle/ace.py)
`coupling` is the off-diagonal block K2e - K2d of Eq. 1 (Eqs. 5, 7; at Gamma with real functions
K2e = K1e; spin flip: Eqs. S7, S9, which read the trial vector of the OPPOSITE flip direction).

Vector layout (same as the C ABI): one trial vector = [spin][v][g] complex, contiguous;
a block is [k][spin][v][g].

Pins: tests/test_oracle_liouville.py, tests/test_oracle_extensions.py.  Parity against numbers printed by the paper: unpinned
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
                 use_hartree_fxc=True, rho_floor=1e-10, vloc=None, fft_backend="radix",
                 sf_xc_kernel=False, sf_cut=1e-3, pair_mask=None, wannier_u=None, ace=None):
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
        # options of SURVEY 8(f)
        self.sf_xc_kernel = bool(sf_xc_kernel)
        self.fsf = None
        if self.sf_xc_kernel:                                                       # Eq. 26
            vu, vd = lda.vxc(np.maximum(self.rho0[0], rho_floor), np.maximum(self.rho0[1], rho_floor))
            d = self.rho0[0] - self.rho0[1]
            ok = np.abs(d) >= sf_cut
            self.fsf = np.where(ok, (vu - vd) / np.where(ok, d, 1.0), 0.0)
        self.pair_mask = None if pair_mask is None else [np.asarray(m, dtype=bool) for m in pair_mask]
        self.U = None if wannier_u is None else [np.asarray(u, dtype=np.float64) for u in wannier_u]
        self.phi_rot = None
        if self.U is not None:                                                      # phi~_n = sum_v U_vn phi_v
            self.phi_rot = [np.tensordot(self.U[s].T, self.phi[s], axes=1) for s in range(self.nspin)]
        self.ace = ace          # list over spins of xi [n_ace, npwh] (oracle/ace.py) or None

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
        ctx = dict(mode=mode, x=xs, a=a, V=None, k1d_rot=None, Vsf=None)
        if self.U is not None and self.alpha != 0.0:
            # Eq. 31: g_m(r) = sum_n a~_n(r) tau~_mn(r) for every rotated orbital m of each block (N^2 pair potentials)
            ctx["k1d_rot"] = []
            for b in range(len(xs)):
                s_occ = b if mode == SPIN_CONSERVING else (0 if mode == SPIN_FLIP else 1)
                U, pr = self.U[s_occ], self.phi_rot[s_occ]
                at = np.tensordot(U.T, a[b], axes=1)                                  # a~_n = sum_v' U_v'n a_v'
                g = np.zeros_like(at)
                for m in range(self.nocc[s_occ]):
                    for n in range(self.nocc[s_occ]):
                        if self.pair_mask is not None and not self.pair_mask[s_occ][m, n]:
                            continue
                        g[m] += at[n] * self.coulomb(pr[m] * pr[n])
                ctx["k1d_rot"].append(g)
        if mode != SPIN_CONSERVING and self.sf_xc_kernel:                            # Eq. 22 and Eq. 24
            s_occ = 0 if mode == SPIN_FLIP else 1
            ctx["Vsf"] = self.fsf * np.sum(self.phi[s_occ] * a[0], axis=0)
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
        if ctx["Vsf"] is not None:
            y += phi[v] * ctx["Vsf"]
        if ctx["k1d_rot"] is not None:                                                # Eq. 31, outer sum over m
            y -= self.alpha * np.tensordot(self.U[s_occ][v], ctx["k1d_rot"][blk], axes=1)
        elif self.alpha != 0.0:
            for vp in range(self.nocc[s_occ]):                                        # O6
                if self.pair_mask is not None and not self.pair_mask[s_occ][v, vp]:
                    continue
                tau = self.coulomb(phi[v] * phi[vp])
                y -= self.alpha * a[vp] * tau
        if self.vloc is not None:
            y += self.vloc[s_tgt] * a[v]
        yg = self.to_sphere(y)                                                        # O7
        yg = yg + (0.5 * self.g2 - self.eig[s_occ][v]) * ctx["x"][blk][v]             # O8
        if self.ace is not None:                                                      # alpha V_X^ACE a_v, Eq. 29
            xv = ctx["x"][blk][v]
            for xi in self.ace[s_tgt]:
                yg = yg - self.alpha * xi * (2.0 * np.real(np.vdot(xi, xv)) - xi[0].real * xv[0].real)
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

    # ---- off-diagonal block of Eq. 1 ------------------------------------------------
    def coupling(self, X, mode=SPIN_CONSERVING):
        """(K2e - K2d) X, block of trial vectors (Eqs. 5, 7; spin flip Eqs. S7, S9).

        Spin conserving: (K2e X)_v = P_c phi_v V[X] with the same V as K1e (real functions: a* phi = phi* a);
        (K2d X)_v = alpha P_c sum_v' phi_v'(r) C[a_v' phi_v](r).
        Spin flip, output in the layout of `mode` (functions v over the occupied orbitals of s~, living in s): the input X
        is a block of trial vectors of the OPPOSITE flip direction (functions v' over the occupied orbitals of s, living in
        s~):  (K2d X)_v = alpha P_c,s sum_{v' in occ s} phi_v's(r) C[a_v' phi_v,s~](r), and with sf_xc_kernel
        (K2e X)_v = P_c,s phi_v,s~ f^SF sum_{v' in occ s} a_v' phi_v's."""
        X = np.asarray(X, dtype=np.complex128)
        in_mode = mode if mode == SPIN_CONSERVING else (SPIN_FLIP_DOWN_UP if mode == SPIN_FLIP else SPIN_FLIP)
        X = X.reshape(-1, self.vector_len(in_mode))
        out = np.zeros((X.shape[0], self.vector_len(mode)), dtype=np.complex128)
        for k in range(X.shape[0]):
            xs = self.split(X[k], in_mode)
            a = [np.stack([self.to_real(c) for c in blk]) for blk in xs]
            o = 0
            if mode == SPIN_CONSERVING:
                V = self.prepare(X[k], mode)["V"]
                for s in range(self.nspin):
                    for v in range(self.nocc[s]):
                        y = np.zeros(self.grid)
                        if V is not None:
                            y += self.phi[s][v] * V[s]
                        for vp in range(self.nocc[s]):
                            y -= self.alpha * self.phi[s][vp] * self.coulomb(a[s][vp] * self.phi[s][v])
                        out[k, o:o + self.npwh] = self.project_c(self.to_sphere(y), s)
                        o += self.npwh
            else:
                s_occ = 0 if mode == SPIN_FLIP else 1       # s~ of the OUTPUT: its functions run over occ(s~), live in s
                s_tgt = 1 - s_occ
                Vsf = None
                if self.sf_xc_kernel:
                    Vsf = self.fsf * np.sum(self.phi[s_tgt] * a[0], axis=0)
                for v in range(self.nocc[s_occ]):
                    y = np.zeros(self.grid)
                    if Vsf is not None:
                        y += self.phi[s_occ][v] * Vsf
                    for vp in range(self.nocc[s_tgt]):
                        y -= self.alpha * self.phi[s_tgt][vp] * self.coulomb(a[0][vp] * self.phi[s_occ][v])
                    out[k, o:o + self.npwh] = self.project_c(self.to_sphere(y), s_tgt)
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
