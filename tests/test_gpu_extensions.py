"""GPU parity of the SURVEY 8(f) rows and of the stand-alone ABI pieces, through the C ABI against the oracle.
Tolerance 1e-10 relative Frobenius (north star), FP64."""
import numpy as np
import pytest

from helpers import Case, rel_fro
from oracle import ace as oace
from oracle import nearsight
import synthetic_inputs as inputs

pytestmark = pytest.mark.gpu

TOL = 1e-10
TRI = [[7.0, 0, 0], [0.9, 7.4, 0], [0.5, -0.4, 6.6]]


def _mask_to_list(mask):
    n = len(mask)
    return [(i, j) for i in range(n) for j in range(i, n) if mask[i, j]]


def _random_mask(rng, n, keep=0.5):
    m = rng.uniform(size=(n, n)) < keep
    m = np.triu(m) | np.triu(m).T
    return m


# ---- stand-alone pieces (include/tddft.h: tddft_project, tddft_gram) ------------------------------------------
@pytest.mark.parametrize("nfun", [3, 130])
def test_project_matches_oracle(nfun):
    import torch
    from paper_2309_03513_b200 import binding as b
    case = Case(TRI, (12, 10, 9), 6.0, 2, (5, 4), 0.3, seed=301)
    y = (case.rng.standard_normal((nfun, case.npwh)) + 1j * case.rng.standard_normal((nfun, case.npwh)))
    y[:, 0] = y[:, 0].real
    for s in range(2):
        dY = torch.from_numpy(y.copy()).cuda()
        b.tddft_project(case.ctx(), s, dY, nfun)
        torch.cuda.synchronize()
        ref = np.stack([case.oracle.project_c(f, s) for f in y])
        assert rel_fro(dY.cpu().numpy(), ref) < 1e-12


@pytest.mark.parametrize("m", [1, 5, 70])
def test_gram_matches_oracle(m):
    import torch
    from paper_2309_03513_b200 import binding as b
    case = Case(TRI, (12, 10, 9), 6.0, 2, (5, 4), 0.3, seed=302)
    L = case.oracle.vector_len(0)
    V = case.rng.standard_normal((m, L)) + 1j * case.rng.standard_normal((m, L))
    W = case.rng.standard_normal((m, L)) + 1j * case.rng.standard_normal((m, L))
    for A in (V, W):
        A.reshape(m, -1, case.npwh)[:, :, 0] = A.reshape(m, -1, case.npwh)[:, :, 0].real
    G = b.tddft_gram(case.ctx(), torch.from_numpy(V).cuda(), torch.from_numpy(W).cuda(), m, L)
    ref = np.array([[case.oracle.vdot(V[i], W[j]) for j in range(m)] for i in range(m)])
    assert np.max(np.abs(G - ref)) < 1e-12 * np.max(np.abs(ref))


def test_custom_nonblocking_stream():
    # the library's work is ordered on the caller's stream only (no reliance on the legacy default stream)
    import torch
    from paper_2309_03513_b200 import binding as b
    st = torch.cuda.Stream()
    case = Case(TRI, (12, 18, 20), 6.0, 2, (5, 4), 0.3, seed=303, cuda_stream=st.cuda_stream)
    X = case.trial(2, 0)
    with torch.cuda.stream(st):
        dX = torch.from_numpy(X).cuda(non_blocking=False)
        dAX = torch.empty_like(dX)
        st.synchronize()
        b.tddft_apply_liouville(case.ctx(), dX, dAX, 2, 0)
        st.synchronize()
    assert rel_fro(dAX.cpu().numpy(), case.oracle.apply(X, 0)) < TOL


# ---- spin-flip xc kernel (Eqs. 24, 26) ---------------------------------------------------------------------------
@pytest.mark.parametrize("mode", [1, 2])
@pytest.mark.parametrize("grid", [(12, 10, 9), (12, 18, 20)])
def test_spin_flip_xc_kernel(mode, grid):
    case = Case(TRI, grid, 6.0, 2, (5, 3), 0.3, seed=311, oracle_opts=dict(sf_xc_kernel=True, sf_cut=1e-3), sf_xc_kernel=1, sf_cut=1e-3)
    X = case.trial(3, mode)
    ref = case.oracle.apply(X, mode)
    assert rel_fro(case.gpu_apply(X, mode), ref) < TOL
    off = Case(TRI, grid, 6.0, 2, (5, 3), 0.3, seed=311, oracle=False)
    assert rel_fro(off.gpu_apply(X, mode), ref) > 1e-4          # the kernel matters on this input


# ---- near-sightedness (Eqs. 31, 32) ---------------------------------------------------------------------------------
def test_full_pair_list_is_bit_identical_and_random_mask_matches_oracle():
    base = Case(TRI, (12, 10, 9), 6.0, 2, (7, 5), 0.3, seed=321, pair_tile=3, fft_batch=2)
    X = base.trial(3, 0)
    ref_gpu = base.gpu_apply(X, 0)
    full = [[(i, j) for i in range(n) for j in range(i, n)] for n in (7, 5)]
    listed = Case(TRI, (12, 10, 9), 6.0, 2, (7, 5), 0.3, seed=321, oracle=False, pair_tile=3, fft_batch=2,
                  pair_list_up=full[0], pair_list_dn=full[1])
    assert np.array_equal(listed.gpu_apply(X, 0), ref_gpu)
    rng = np.random.default_rng(5)
    mask = [_random_mask(rng, 7), _random_mask(rng, 5)]
    for tile in (3, 0):
        masked = Case(TRI, (12, 10, 9), 6.0, 2, (7, 5), 0.3, seed=321, oracle_opts=dict(pair_mask=mask), pair_tile=tile,
                      pair_list_up=_mask_to_list(mask[0]), pair_list_dn=_mask_to_list(mask[1]))
        for mode in (0, 1):
            Xm = masked.trial(2, mode)
            assert rel_fro(masked.gpu_apply(Xm, mode), masked.oracle.apply(Xm, mode)) < TOL


@pytest.mark.parametrize("vloc", [False, True])
def test_rotated_orbitals_eq31(vloc):
    rng = np.random.default_rng(6)
    U = [inputs.random_orthogonal(rng, 6), inputs.random_orthogonal(rng, 4)]
    mask = [_random_mask(rng, 6, 0.6), _random_mask(rng, 4, 0.6)]
    # all pairs kept: any rotation gives the canonical result (oracle without rotation)
    plain = Case(TRI, (12, 18, 20), 6.0, 2, (6, 4), 0.3, seed=322, vloc=vloc, wannier_u_up=U[0], wannier_u_dn=U[1])
    X = plain.trial(2, 0)
    assert rel_fro(plain.gpu_apply(X, 0), plain.oracle.apply(X, 0)) < TOL
    # truncated pairs of the rotated orbitals: literal Eq. 31 in the oracle
    trunc = Case(TRI, (12, 18, 20), 6.0, 2, (6, 4), 0.3, seed=322, vloc=vloc, oracle_opts=dict(wannier_u=U, pair_mask=mask),
                 wannier_u_up=U[0], wannier_u_dn=U[1], pair_list_up=_mask_to_list(mask[0]), pair_list_dn=_mask_to_list(mask[1]))
    for mode in (0, 2):
        Xm = trunc.trial(2, mode)
        assert rel_fro(trunc.gpu_apply(Xm, mode), trunc.oracle.apply(Xm, mode)) < TOL


def test_overlap_function_and_threshold():
    from paper_2309_03513_b200 import binding as b
    rng = np.random.default_rng(7)
    from oracle import lattice as olat
    miller, g2 = olat.enumerate_half_sphere(TRI, 9.0)
    psi = [inputs.localized_orbitals(rng, 9, miller, g2, width=1.1), inputs.localized_orbitals(rng, 8, miller, g2, width=1.1)]
    probe = Case(TRI, (16, 18, 20), 9.0, 2, (9, 8), 0.3, seed=323, psi=psi)
    S_ref = [nearsight.overlap_matrix(probe.oracle.phi[s]) for s in range(2)]
    for s in range(2):
        S = b.tddft_orbital_overlap(probe.ctx(), s, probe.nocc[s])
        assert np.max(np.abs(S - S_ref[s])) < 1e-12
    thr = float(np.median(np.concatenate([S_ref[0][np.triu_indices(9, 1)], S_ref[1][np.triu_indices(8, 1)]])))
    mask = [nearsight.pair_mask(S_ref[s], thr) for s in range(2)]
    assert 0.2 < np.mean(mask[0]) < 0.9
    case = Case(TRI, (16, 18, 20), 9.0, 2, (9, 8), 0.3, seed=323, psi=psi, oracle_opts=dict(pair_mask=mask), s_thr=thr)
    X = case.trial(2, 0)
    assert rel_fro(case.gpu_apply(X, 0), case.oracle.apply(X, 0)) < TOL


# ---- exact exchange and ACE (Eqs. 28-30) ------------------------------------------------------------------------------
def _ace_case(**kw):
    from oracle import lattice as olat
    miller, g2 = olat.enumerate_half_sphere(TRI, 6.0)
    rng = np.random.default_rng(8)
    up = inputs.orbitals(rng, 8, g2, 6.0)            # 5 occupied + 3 extra, jointly orthonormal
    dn = inputs.orbitals(rng, 6, g2, 6.0)            # 4 occupied + 2 extra
    case = Case(TRI, (12, 18, 20), 6.0, 2, (5, 4), 0.3, seed=331, psi=[up[:5].copy(), dn[:4].copy()], **kw)
    return case, [up[5:].copy(), dn[4:].copy()]


def test_exchange_operator_and_ace_against_oracle():
    import torch
    from paper_2309_03513_b200 import binding as b
    case0, extra = _ace_case()
    d_extra = [torch.from_numpy(e).cuda() for e in extra]
    case, _ = _ace_case(ace=1, psi_ace_up=d_extra[0], psi_ace_dn=d_extra[1])
    o = case.oracle
    y = case.rng.standard_normal((3, case.npwh)) + 1j * case.rng.standard_normal((3, case.npwh))
    y[:, 0] = y[:, 0].real
    for s in range(2):
        dY = torch.from_numpy(y).cuda(); dV = torch.empty_like(dY)
        b.tddft_exchange_apply(case.ctx(), s, dY, dV, 3)
        torch.cuda.synchronize()
        ref = np.stack([oace.exchange_apply(o, s, f) for f in y])
        assert rel_fro(dV.cpu().numpy(), ref) < TOL
        xi = oace.build(o, s, extra[s])
        b.tddft_exchange_apply(case.ctx(), s, dY, dV, 3, use_ace=True)
        torch.cuda.synchronize()
        ref = np.stack([oace.ace_apply(xi, f) for f in y])
        assert rel_fro(dV.cpu().numpy(), ref) < 1e-9          # through a Cholesky factor of <phi|V_X|phi>
    # D with H = T + alpha V_X^ACE
    xis = [oace.build(o, s, extra[s]) for s in range(2)]
    ca, _ = _ace_case(oracle_opts=dict(ace=xis), ace=1, psi_ace_up=d_extra[0], psi_ace_dn=d_extra[1])
    for mode in (0, 1):
        X = ca.trial(2, mode)
        assert rel_fro(ca.gpu_apply(X, mode), ca.oracle.apply(X, mode)) < 1e-9


# ---- off-diagonal block of Eq. 1 ------------------------------------------------------------------------------------
@pytest.mark.parametrize("mode", [0, 1, 2])
def test_coupling_block(mode):
    import torch
    from paper_2309_03513_b200 import binding as b
    case = Case(TRI, (12, 18, 20), 6.0, 2, (5, 4), 0.3, seed=341, oracle_opts=dict(sf_xc_kernel=True), sf_xc_kernel=1)
    other = {0: 0, 1: 2, 2: 1}[mode]
    X = case.trial(3, other)
    dX = torch.from_numpy(X).cuda()
    Lout = b.tddft_vector_len(case.ctx(), mode)
    dB = torch.empty((3, Lout), dtype=torch.complex128, device="cuda")
    b.tddft_apply_coupling(case.ctx(), dX, dB, 3, mode)
    torch.cuda.synchronize()
    assert rel_fro(dB.cpu().numpy(), case.oracle.coupling(X, mode)) < TOL


def test_coupling_closed_shell_and_k_chunks():
    import torch
    from paper_2309_03513_b200 import binding as b
    case = Case.from_config(1)
    X = case.trial(3, 0)
    ref = case.oracle.coupling(X, 0)
    for opts in ({}, dict(workspace_gb=0.02)):
        cc = Case.from_config(1, oracle=False, **opts)
        dX = torch.from_numpy(X).cuda(); dB = torch.empty_like(dX)
        b.tddft_apply_coupling(cc.ctx(), dX, dB, 3, 0)
        torch.cuda.synchronize()
        assert rel_fro(dB.cpu().numpy(), ref) < TOL


# ---- the 8(f) rows under the streamed plan (api.cu: apply_streamed: tile loop outermost, contributions added in the sphere) ------
def test_streamed_plan_rotation_truncation_sf_kernel_and_ace():
    import torch
    from paper_2309_03513_b200 import binding as b
    cap = dict(plan=2, pair_tile=4)          # all vectors at once: the row-resident mode of the streamed plan
    rng = np.random.default_rng(16)
    U = [inputs.random_orthogonal(rng, 6), inputs.random_orthogonal(rng, 4)]
    mask = [_random_mask(rng, 6, 0.6), _random_mask(rng, 4, 0.6)]
    trunc = Case(TRI, (12, 18, 20), 6.0, 2, (6, 4), 0.3, seed=352, vloc=True, oracle_opts=dict(wannier_u=U, pair_mask=mask),
                 wannier_u_up=U[0], wannier_u_dn=U[1], pair_list_up=_mask_to_list(mask[0]), pair_list_dn=_mask_to_list(mask[1]), **cap)
    for mode in (0, 2):
        X = trunc.trial(4, mode)
        got = trunc.gpu_apply(X, mode)
        assert mode != 0 or b.tddft_get_stats(trunc.ctx())["blocks_resident"] == 0
        assert rel_fro(got, trunc.oracle.apply(X, mode)) < TOL
    sf = Case(TRI, (12, 18, 20), 6.0, 2, (5, 3), 0.3, seed=353, oracle_opts=dict(sf_xc_kernel=True, sf_cut=1e-3), sf_xc_kernel=1, sf_cut=1e-3, workspace_gb=0.0015, pair_tile=4)
    X = sf.trial(4, 1)
    got = sf.gpu_apply(X, 1)
    assert b.tddft_get_stats(sf.ctx())["blocks_resident"] == 0
    assert rel_fro(got, sf.oracle.apply(X, 1)) < TOL
    case0, extra = _ace_case()
    d_extra = [torch.from_numpy(e).cuda() for e in extra]
    xis = [oace.build(case0.oracle, s, extra[s]) for s in range(2)]
    ca, _ = _ace_case(oracle_opts=dict(ace=xis), ace=1, psi_ace_up=d_extra[0], psi_ace_dn=d_extra[1], workspace_gb=0.002, pair_tile=4)
    X = ca.trial(4, 0)
    got = ca.gpu_apply(X, 0)
    assert b.tddft_get_stats(ca.ctx())["blocks_resident"] == 0
    assert rel_fro(got, ca.oracle.apply(X, 0)) < 1e-9
