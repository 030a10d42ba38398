"""GPU parity: the CUDA path (through the C ABI) against the oracle, element by element, on the same seeded inputs.

Tolerance: relative Frobenius error <= 1e-10 on AX (BASELINE.json north_star), FP64 everywhere.
"""
import math

import numpy as np
import pytest

from helpers import Case, rel_fro

pytestmark = pytest.mark.gpu

TOL = 1e-10
TRI = [[7.0, 0, 0], [0.9, 7.4, 0], [0.5, -0.4, 6.6]]
HEX = [[9.0, 0, 0], [-4.5, 9.0 * math.sqrt(3) / 2, 0], [0, 0, 7.0]]


def test_orbitals_and_pair_potentials_small():
    import torch
    from paper_2309_03513_b200 import binding as b
    case = Case(TRI, (12, 10, 9), 6.0, 2, (5, 4), 0.3, seed=101)
    ctx = case.ctx()
    nr = int(np.prod(case.grid))
    out = torch.empty(nr, dtype=torch.float64, device="cuda")
    for s in range(2):
        for v in range(case.nocc[s]):
            b.tddft_orbital_real_space(ctx, s, v, out)
            torch.cuda.synchronize()
            ref = case.oracle.phi[s][v].reshape(-1)
            assert rel_fro(out.cpu().numpy(), ref) < 1e-13
    pairs = [(i, j) for i in range(5) for j in range(i, 5)]          # odd count: ragged packing tail
    tau = torch.empty((len(pairs), nr), dtype=torch.float64, device="cuda")
    b.tddft_pair_potentials(ctx, 0, pairs, tau)
    tau = tau.cpu().numpy()
    for p, (i, j) in enumerate(pairs):
        ref = case.oracle.coulomb(case.oracle.phi[0][i] * case.oracle.phi[0][j]).reshape(-1)
        assert rel_fro(tau[p], ref) < 1e-12


@pytest.mark.parametrize("mode", [0, 1, 2])
@pytest.mark.parametrize("vloc", [False, True])
def test_apply_small_triclinic(mode, vloc):
    case = Case(TRI, (12, 10, 9), 6.0, 2, (5, 4), 0.3, seed=102, vloc=vloc)
    X = case.trial(3, mode)
    ref = case.oracle.apply(X, mode)
    got = case.gpu_apply(X, mode)
    assert rel_fro(got, ref) < TOL


def test_apply_hexagonal_mixed_radix():
    case = Case(HEX, (20, 18, 15), 5.0, 2, (6, 5), 0.2, seed=103)
    X = case.trial(2, 0)
    assert rel_fro(case.gpu_apply(X, 0), case.oracle.apply(X, 0)) < TOL


def test_apply_config1_full():
    # BASELINE.json configs[0]: toy 24^3 cell, closed shell, 8 orbitals, 4 trial vectors, alpha = 0.25
    case = Case.from_config(1)
    X = case.trial(4, 0)
    ref = case.oracle.apply(X, 0)
    got = case.gpu_apply(X, 0)
    assert rel_fro(got, ref) < TOL
    # the invariants on the GPU result itself
    o = case.oracle
    M = np.array([[o.vdot(X[i], got[j]) for j in range(4)] for i in range(4)])
    assert np.max(np.abs(M - M.T)) < 1e-11 * np.max(np.abs(M))


def test_apply_options_no_hxc_and_alpha_zero():
    case = Case(TRI, (12, 10, 9), 6.0, 2, (5, 4), 0.0, seed=104, use_hartree_fxc=False)
    X = case.trial(2, 0)
    assert rel_fro(case.gpu_apply(X, 0), case.oracle.apply(X, 0)) < TOL


def test_tiling_and_k_chunking_do_not_change_the_result():
    # small tiles (ragged last tile) and a workspace cap that forces chunking over trial vectors
    base = Case(TRI, (12, 10, 9), 6.0, 2, (7, 5), 0.3, seed=105)
    X = base.trial(5, 0)
    ref = base.oracle.apply(X, 0)
    tiled = Case(TRI, (12, 10, 9), 6.0, 2, (7, 5), 0.3, seed=105, oracle=False, pair_tile=3, fft_batch=2)
    assert rel_fro(tiled.gpu_apply(X, 0), ref) < TOL
    capped = Case(TRI, (12, 10, 9), 6.0, 2, (7, 5), 0.3, seed=105, oracle=False, workspace_gb=0.0007)
    assert rel_fro(capped.gpu_apply(X, 0), ref) < TOL


@pytest.mark.parametrize("mode", [0, 1])
def test_host_buffer_entry_point_equals_device_path(mode):
    # tddft_apply_liouville_host copies block by block on its own stream behind the kernels: same bits as the device call,
    # from pageable numpy buffers and from pinned ones, and repeatable
    import torch
    from paper_2309_03513_b200 import binding as b
    case = Case(TRI, (12, 18, 20), 6.0, 2, (5, 4), 0.3, seed=106)
    X = case.trial(3, mode)
    ref = case.gpu_apply(X, mode)
    assert rel_fro(ref, case.oracle.apply(X, mode)) < TOL
    out = np.empty_like(X)
    b.tddft_apply_liouville_host(case.ctx(), np.ascontiguousarray(X), out, 3, mode)
    assert np.array_equal(out, ref)
    Xp = torch.from_numpy(X).pin_memory(); AXp = torch.empty_like(Xp).pin_memory()
    for _ in range(2):
        AXp.zero_()
        b.tddft_apply_liouville_host(case.ctx(), Xp, AXp, 3, mode)
        assert np.array_equal(AXp.numpy(), ref)


@pytest.mark.parametrize("cap", [dict(workspace_gb=0.002), dict(plan=2)])      # vectors in inner chunks / all vectors at once (row-resident mode)
@pytest.mark.parametrize("mode", [0, 1, 2])
def test_streamed_plan_forms_tau_once(mode, cap):
    # A workspace cap under which a(r) / out(r) of a spin block do not fit for all trial vectors: the tile loop runs outermost
    # (api.cu: apply_streamed), tau is formed once whatever the number of vectors (Eq. 6), a(r) is recomputed per tile
    # and the tile contributions are added in the sphere.  Same operator: V_loc, Hxc, ragged tiles, vectors in inner chunks.
    from paper_2309_03513_b200 import binding as b
    case = Case(TRI, (12, 18, 20), 6.0, 2, (9, 7), 0.3, seed=131, vloc=True, pair_tile=4, **cap)
    X = case.trial(5, mode)
    got = case.gpu_apply(X, mode)
    st = b.tddft_get_stats(case.ctx())
    n = [9, 7]
    unique = sum(k * (k + 1) // 2 for k in (n if mode == 0 else [n[mode - 1]]))
    assert st["blocks_resident"] == 0 and st["pair_ffts"] == unique and (st["k_chunk"] == 5) == ("plan" in cap), st
    assert rel_fro(got, case.oracle.apply(X, mode)) < TOL


def test_streamed_plan_closed_shell_and_no_exchange():
    case = Case(TRI, (12, 10, 9), 6.0, 1, (6,), 0.0, seed=132, workspace_gb=0.0004)
    X = case.trial(4, 0)
    assert rel_fro(case.gpu_apply(X, 0), case.oracle.apply(X, 0)) < TOL


@pytest.mark.parametrize("plan", [1, 2])
@pytest.mark.parametrize("mode", [0, 1])
def test_sharded_apply_partial_results_sum_to_the_full_operator(mode, plan):
    # one apply sharded over GPUs.  Each shard applies the exchange tiles it owns, shard 0 adds D, K1e and V_loc, every
    # shard projects its part; the sum over shards (one all-reduce of AX in tddft_apply_liouville_sharded) is A X.  Here the three
    # shards run one after the other on the same GPU and the sum is taken on the host: the partition logic, without the collective.
    full = Case(TRI, (12, 18, 20), 6.0, 2, (9, 7), 0.3, seed=141, vloc=True, pair_tile=4, plan=plan)
    X = full.trial(3, mode)
    ref = full.oracle.apply(X, mode)
    total = np.zeros_like(ref)
    for r in range(3):
        shard = Case(TRI, (12, 18, 20), 6.0, 2, (9, 7), 0.3, seed=141, vloc=True, oracle=False, pair_tile=4, plan=plan, shard_rank=r, shard_count=3)
        part = shard.gpu_apply(X, mode)
        assert np.linalg.norm(part) > 0
        total += part
    assert rel_fro(total, ref) < TOL
    assert rel_fro(full.gpu_apply(X, mode), ref) < TOL
