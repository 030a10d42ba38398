"""GPU parity of tddft_davidson: lowest eigenvalues against the oracle's Davidson within 1e-8 Ha (north star)."""
import numpy as np
import pytest

from helpers import Case
from oracle.davidson import davidson as oracle_davidson

pytestmark = pytest.mark.gpu

TRI = [[7.0, 0, 0], [0.9, 7.4, 0], [0.5, -0.4, 6.6]]


@pytest.mark.parametrize("mode", [0, 1])
def test_davidson_small_matches_oracle(mode):
    import torch
    from paper_2309_03513_b200 import binding as b
    nroots = 3
    base = Case(TRI, (12, 10, 9), 6.0, 2, (4, 3), 0.3, seed=201)
    x0 = base.trial(2 * nroots, mode)
    ref, _, it_ref, res_ref = oracle_davidson(base.oracle, nroots, x0, mode=mode, tol=1e-7)
    assert np.all(res_ref <= 1e-7)
    d_x0 = torch.from_numpy(x0).cuda()
    gpu = Case(TRI, (12, 10, 9), 6.0, 2, (4, 3), 0.3, seed=201, oracle=False, x0=d_x0, n_x0=2 * nroots, tol=1e-7)
    L = b.tddft_vector_len(gpu.ctx(), mode)
    evecs = torch.zeros((nroots, L), dtype=torch.complex128, device="cuda")
    ev, iters, res = b.tddft_davidson(gpu.ctx(), nroots, mode, evecs=evecs)
    assert np.all(res <= 1e-7)
    assert np.max(np.abs(ev - ref)) < 1e-8
    # the returned vectors are eigenvectors of the ORACLE operator: ||A x - theta x|| small, x^T A x = theta
    Xh = evecs.cpu().numpy()
    AX = base.oracle.apply(Xh, mode)
    for i in range(nroots):
        assert np.sqrt(base.oracle.vdot(AX[i] - ev[i] * Xh[i], AX[i] - ev[i] * Xh[i])) < 5e-7
        assert base.oracle.vdot(Xh[i], AX[i]) == pytest.approx(ev[i], abs=1e-10)
        assert base.oracle.vdot(Xh[i], Xh[i]) == pytest.approx(1.0, abs=1e-10)


def test_davidson_config1_restart_and_own_start():
    # BASELINE.json configs[0] (toy cell), lowest 3 singlet roots, three ways:
    # oracle with lowest-diagonal start vectors; CUDA with the same start vectors and a subspace small enough to
    # force restarts; CUDA with the library's own start vectors.  All must give the same eigenvalues.
    import torch
    from paper_2309_03513_b200 import binding as b
    import synthetic_inputs as inputs
    nroots = 3
    base = Case.from_config(1)
    x0 = inputs.diagonal_guess(base.rng, base.oracle.precond_diag(0), base.npwh, 2 * nroots)
    ref, _, it_ref, res_ref = oracle_davidson(base.oracle, nroots, x0, tol=1e-6)
    assert np.all(res_ref <= 1e-6)
    d_x0 = torch.from_numpy(x0).cuda()
    gpu = Case.from_config(1, oracle=False, x0=d_x0, n_x0=2 * nroots, max_subspace=9)
    ev, iters, res = b.tddft_davidson(gpu.ctx(), nroots, 0)
    assert np.all(res <= 1e-6)
    assert np.max(np.abs(ev - ref)) < 1e-8
    own = Case.from_config(1, oracle=False)
    ev2, iters2, res2 = b.tddft_davidson(own.ctx(), nroots, 0)
    assert np.all(res2 <= 1e-6)
    assert np.max(np.abs(ev2 - ref)) < 1e-8
