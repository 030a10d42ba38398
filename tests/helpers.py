"""Shared set-up for the parity tests: one seeded problem handed to both the oracle and the CUDA library."""
import numpy as np

from oracle import lattice as olat
from oracle import liouville as olv
import synthetic_inputs as inputs


class Case:
    """Holds the same inputs for both sides.  The CUDA side is created lazily (needs a GPU)."""

    def __init__(self, lattice, grid, ecut, nspin, nocc, alpha, seed, envelope=True, ortho="lowdin",
                 vloc=False, use_hartree_fxc=True, fft_backend="radix", oracle=True, oracle_opts=None, psi=None, **gpu_opts):
        self.lattice = np.asarray(lattice, dtype=np.float64).reshape(3, 3)
        self.grid = tuple(grid); self.ecut = ecut; self.nspin = nspin; self.nocc = tuple(nocc); self.alpha = alpha
        self.use_hartree_fxc = use_hartree_fxc
        self.gpu_opts = gpu_opts
        self.miller, self.g2 = olat.enumerate_half_sphere(self.lattice, ecut)
        self.npwh = len(self.miller)
        self.rng = np.random.Generator(np.random.PCG64(seed))
        self.psi = psi if psi is not None else [inputs.orbitals(self.rng, nocc[s], self.g2, ecut, envelope, ortho) for s in range(nspin)]
        self.eig = [inputs.eigenvalues(self.rng, nocc[s]) for s in range(nspin)]
        self.vloc = None
        if vloc:
            nr = int(np.prod(grid))
            self.vloc = [0.3 * self.rng.standard_normal(nr) for _ in range(2)]
        self.oracle = None
        if oracle:
            self.oracle = olv.Problem(self.lattice, self.grid, ecut, nspin, self.psi, self.eig, alpha,
                                      use_hartree_fxc=use_hartree_fxc, vloc=self.vloc, fft_backend=fft_backend, **(oracle_opts or {}))
        self._ctx = None

    @classmethod
    def from_config(cls, config_id, nocc=None, **kw):
        c = inputs.config(config_id)
        return cls(c["lattice"], c["grid"], c["ecut"], c["nspin"], nocc or c["nocc"], c["alpha"], c["seed"],
                   envelope=c["envelope"], ortho=c["ortho"], **kw)

    def blocks(self, mode):
        if mode == 0:
            return [(self.nocc[s], self.psi[s]) for s in range(self.nspin)]
        src = 0 if mode == 1 else 1
        return [(self.nocc[src], self.psi[1 - src])]

    def trial(self, nvec, mode=0):
        return inputs.trial_vectors(self.rng, self.blocks(mode), nvec)

    # ---- CUDA side ------------------------------------------------------------------------------
    def ctx(self):
        if self._ctx is None:
            import torch
            from paper_2309_03513_b200 import binding as b
            m, g2 = b.tddft_enumerate_gvectors(self.lattice, self.ecut)
            assert np.array_equal(m, self.miller), "library and oracle disagree on the canonical G order"
            self.d_psi = [torch.from_numpy(p).cuda() for p in self.psi]
            opts = dict(self.gpu_opts)
            opts["use_hartree_fxc"] = 1 if self.use_hartree_fxc else 0
            if self.vloc is not None:
                self.d_vloc = [torch.from_numpy(v).cuda() for v in self.vloc]
                opts["vloc_up"] = self.d_vloc[0]
                opts["vloc_dn"] = self.d_vloc[1] if self.nspin == 2 else None
            self._ctx = b.tddft_init(self.lattice, self.grid, self.ecut, self.nspin, self.nocc, self.d_psi[0],
                                     self.d_psi[1] if self.nspin == 2 else None, self.eig[0],
                                     self.eig[1] if self.nspin == 2 else None, self.alpha, **opts)
        return self._ctx

    def gpu_apply(self, X, mode=0):
        import torch
        from paper_2309_03513_b200 import binding as b
        ctx = self.ctx()
        dX = torch.from_numpy(np.ascontiguousarray(X)).cuda()
        dAX = torch.empty_like(dX)
        b.tddft_apply_liouville(ctx, dX, dAX, X.shape[0], mode)
        torch.cuda.synchronize()
        return dAX.cpu().numpy()


def rel_fro(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))
