"""GPU parity at the BASELINE.json sizes, in the launch configuration bench.py times (reading A19).

The oracle needs N_occ pair potentials per output column, so at configs 2 and 3 it computes a seeded sample of the
columns (spin, v, k) of AX one by one (`Problem.column`); the full GPU result is checked against the invariants that
hold at any size: symmetry <Y|AX> = <AY|X> and P_c AX = AX.  Tolerance 1e-10 relative (north star), FP64.
"""
import numpy as np
import pytest

from helpers import Case, rel_fro

pytestmark = pytest.mark.gpu

TOL = 1e-10
TRI = [[7.0, 0, 0], [0.9, 7.4, 0], [0.5, -0.4, 6.6]]


def _sampled_columns(case, X, got, mode, samples):
    o = case.oracle
    L = o.vector_len(mode)
    got = got.reshape(X.shape[0], L)
    off = [0]
    if mode == 0:
        for s in range(o.nspin - 1):
            off.append(off[-1] + o.nocc[s] * o.npwh)
    worst = 0.0
    for k in sorted({k for k, _, _ in samples}):
        ctx = o.prepare(X[k], mode)
        for kk, s, v in samples:
            if kk != k:
                continue
            ref = o.column(ctx, s, v)
            a = off[s] + v * o.npwh
            worst = max(worst, rel_fro(got[k, a:a + o.npwh], ref))
    return worst


def _invariants(case, X, got, mode):
    o = case.oracle
    n = X.shape[0]
    M = np.array([[o.vdot(X[i], got[j]) for j in range(n)] for i in range(n)])
    assert np.max(np.abs(M - M.T)) < 1e-11 * np.max(np.abs(M)), "A is not symmetric on the GPU result"
    for k in (0, n - 1):
        p = o.project_vector(got[k], mode)
        assert rel_fro(p, got[k].reshape(-1)) < 1e-12, "P_c AX != AX"


@pytest.mark.parametrize("fft_path", [0, 1])
def test_pair_potentials_fused_and_general_paths(fft_path):
    # (12,18,20): radices 3,4 / 3,6 / 5,4 -- a shape with fused plane and x kernels, NY != NZ, ragged x tiles
    import torch
    from paper_2309_03513_b200 import binding as b
    case = Case(TRI, (12, 18, 20), 6.0, 2, (5, 4), 0.3, seed=201, fft_path=fft_path, fft_batch=2)
    ctx = case.ctx()
    nr = int(np.prod(case.grid))
    pairs = [(i, j) for i in range(5) for j in range(i, 5)]
    tau = torch.empty((len(pairs), nr), dtype=torch.float64, device="cuda")
    b.tddft_pair_potentials(ctx, 0, pairs, tau)
    tau = tau.cpu().numpy()
    for p, (i, j) in enumerate(pairs):
        ref = case.oracle.coulomb(case.oracle.phi[0][i] * case.oracle.phi[0][j]).reshape(-1)
        assert rel_fro(tau[p], ref) < 1e-12


@pytest.mark.parametrize("mode", [0, 1])
def test_apply_fused_shape_triclinic(mode):
    case = Case(TRI, (12, 18, 20), 6.0, 2, (5, 4), 0.3, seed=202, vloc=True)
    X = case.trial(3, mode)
    assert rel_fro(case.gpu_apply(X, mode), case.oracle.apply(X, mode)) < TOL


def test_apply_config1_general_path_equals_fused():
    fused = Case.from_config(1)
    X = fused.trial(4, 0)
    ref = fused.oracle.apply(X, 0)
    assert rel_fro(fused.gpu_apply(X, 0), ref) < TOL
    general = Case.from_config(1, oracle=False, fft_path=1)
    assert rel_fro(general.gpu_apply(X, 0), ref) < TOL


def test_apply_config2_sampled_columns():
    # BASELINE.json configs[1]: 48^3, 129/127 orbitals, 8 trial vectors, alpha = 0.18
    case = Case.from_config(2)
    X = case.trial(8, 0)
    got = case.gpu_apply(X, 0)
    samples = [(0, 0, 0), (0, 0, 128), (0, 1, 63), (5, 0, 77), (5, 1, 126), (7, 1, 0)]
    assert _sampled_columns(case, X, got, 0, samples) < TOL
    _invariants(case, X, got, 0)


# Columns (k, spin block, v) sampled at config 3.  The tau tiles are 108 orbitals wide (432 = 4 x 108; spin down 430 = 3 x 108 + 106,
# a ragged last tile): the v values hit every row-tile class 0-107, 108-215, 216-323, 324-431 of spin up, both ends of the ragged
# last block of spin down (v = 324..429), the first and last orbital, and k covers both halves of the 16-vector DMMA batch
# (k = 0, 7, 8, 15).  One column per mode is computed with the oracle's own radix FFT instead of the library transform.
CFG3_COLUMNS = {
    0: [(0, 0, 0), (0, 0, 431), (7, 0, 107), (7, 0, 108), (8, 0, 215), (8, 0, 216), (15, 0, 323), (15, 0, 324),
        (0, 1, 0), (7, 1, 150), (8, 1, 324), (15, 1, 429)],
    1: [(0, 0, 0), (0, 0, 431), (7, 0, 107), (7, 0, 200), (8, 0, 216), (8, 0, 323), (15, 0, 324), (15, 0, 108)],
}
CFG3_RADIX_COLUMN = {0: (8, 1, 324), 1: (7, 0, 200)}


@pytest.mark.parametrize("mode", [0, 1])
def test_apply_config3_sampled_columns(mode):
    # BASELINE.json configs[2], the bench workload: 72^3, 432/430 orbitals, 16 trial vectors, both modes
    case = Case.from_config(3, fft_backend="numpy")   # library FFT as the oracle's transform step (pinned equal to the radix FFT at 72^3)
    X = case.trial(16, mode)
    got = case.gpu_apply(X, mode)
    assert _sampled_columns(case, X, got, mode, CFG3_COLUMNS[mode]) < TOL
    _invariants(case, X, got, mode)
    # one column through the oracle's own radix transform
    o = case.oracle
    k, s, v = CFG3_RADIX_COLUMN[mode]
    ctx = o.prepare(X[k], mode)
    o.fft_backend = "radix"
    ref = o.column(ctx, s, v)
    o.fft_backend = "numpy"
    a = (o.nocc[0] * o.npwh if (mode == 0 and s == 1) else 0) + v * o.npwh
    assert rel_fro(got.reshape(16, -1)[k, a:a + o.npwh], ref) < TOL


@pytest.mark.parametrize("grid,lattice,ecut,nocc,nvec", [
    # the large plans, never reached by the smaller grids: 96 = 12*8, 100 = 10*10 (fused kernels and general path), 108 = 3*6*6,
    # 128 = 8*4*4 (fft_core.cuh); the shapes of BASELINE.json configs[3] (hexagonal) and [4] and of the 60 Ry workload
    ((96, 96, 100), [[12.0, 0, 0], [-6.0, 12.0 * 0.8660254037844386, 0], [0, 0, 8.0]], 5.0, (4, 3), 2),
    ((108, 108, 108), [[9.0, 0, 0], [0, 9.0, 0], [0, 0, 9.0]], 8.0, (4, 3), 2),
    ((128, 128, 128), [[9.0, 0, 0], [0, 9.0, 0], [0, 0, 9.0]], 8.0, (3, 2), 1),
])
def test_apply_large_fft_plans(grid, lattice, ecut, nocc, nvec):
    case = Case(lattice, grid, ecut, 2, nocc, 0.3, seed=sum(grid))      # oracle with its own radix FFT
    general = Case(lattice, grid, ecut, 2, nocc, 0.3, seed=sum(grid), oracle=False, fft_path=1) if grid != (108, 108, 108) else None
    cluster = Case(lattice, grid, ecut, 2, nocc, 0.3, seed=sum(grid), oracle=False, fft_path=2) if grid != (128, 128, 128) else None
    for mode in (0, 1):
        X = case.trial(nvec, mode)
        ref = case.oracle.apply(X, mode)
        # default path: fused plane / x kernels (96 x 100 and 108 x 108: one CTA per SM; 128 x 128: a cluster of two CTAs per plane)
        assert rel_fro(case.gpu_apply(X, mode), ref) < TOL
        if general is not None:
            assert rel_fro(general.gpu_apply(X, mode), ref) < TOL          # the general pass kernels on the same shape
        if cluster is not None:
            assert rel_fro(cluster.gpu_apply(X, mode), ref) < TOL          # the two-CTA cluster plane kernel where the shape has both


def test_apply_config4_shape_with_block_at_a_time_plan():
    # the lattice, grid and cutoff of BASELINE.json configs[3] (hexagonal 4H-SiC shaped cell, 96 x 96 x 100, 20 Ry) with fewer
    # orbitals, under a workspace cap that forces the plan of the full configuration: one spin block resident at a time, trial
    # vectors in chunks (tau recomputed per chunk), small tiles.  Sampled columns + invariants, as at the full sizes.
    from paper_2309_03513_b200 import binding as b
    import synthetic_inputs as inputs
    cfg = inputs.config(4)
    case = Case(cfg["lattice"], cfg["grid"], cfg["ecut"], 2, (40, 38), cfg["alpha"], cfg["seed"], envelope=True, ortho="qr",
                fft_backend="numpy", workspace_gb=3.2)
    X = case.trial(3, 0)
    got = case.gpu_apply(X, 0)
    st = b.tddft_get_stats(case.ctx())
    assert st["k_chunk"] < 3 or st["blocks_resident"] == 0 or st["pair_tile"] < 40, st
    samples = [(0, 0, 0), (0, 1, 37), (2, 0, 39), (2, 1, 16), (1, 0, 17)]
    assert _sampled_columns(case, X, got, 0, samples) < TOL
    _invariants(case, X, got, 0)
