"""Seeded synthetic inputs shaped like the paper's defect supercells.

This module serves BOTH the CUDA path and the oracle (tests, bench) and holds none of the
method's arithmetic: it only draws random plane-wave coefficients, orthonormalises them with
the Gamma-point inner product of the half-sphere storage, and lists the five configurations of
BASELINE.json.  The G-sphere (its size and |G|^2 values) is an INPUT here: the caller gets it
from `tddft_enumerate_gvectors` (CUDA side) or `oracle.lattice` (oracle side).

The inputs stand in for the paper's workloads (Quantum ESPRESSO ground states of NV-/SiV0 in
diamond, VV0 in 4H-SiC), which are not available; recipe in DESIGN.md.
"""
import math

import numpy as np

SEED_BASE = 230903513 * 10

_S3 = math.sqrt(3.0) / 2.0

CONFIGS = {
    # id: lattice rows (bohr), grid, wavefunction cutoff (Ry), nspin, nocc per spin, nvec, alpha
    1: dict(name="toy-24", lattice=[[10.0, 0, 0], [0, 10.0, 0], [0, 0, 10.0]], grid=(24, 24, 24), ecut=10.0,
            nspin=1, nocc=(8,), nvec=4, alpha=0.25, envelope=False, ortho="lowdin", nroots=3),
    2: dict(name="C64-48", lattice=[[13.48, 0, 0], [0, 13.48, 0], [0, 0, 13.48]], grid=(48, 48, 48), ecut=25.0,
            nspin=2, nocc=(129, 127), nvec=8, alpha=0.18, envelope=True, ortho="cholqr", nroots=4),
    3: dict(name="NV215-72", lattice=[[20.2, 0, 0], [0, 20.2, 0], [0, 0, 20.2]], grid=(72, 72, 72), ecut=25.0,
            nspin=2, nocc=(432, 430), nvec=16, alpha=0.18, envelope=True, ortho="cholqr", nroots=6),
    4: dict(name="SiC576-96x96x100", lattice=[[36.9, 0, 0], [-18.45, 36.9 * _S3, 0], [0, 0, 19.5]],
            grid=(96, 96, 100), ecut=20.0, nspin=2, nocc=(1150, 1150), nvec=16, alpha=0.15,
            envelope=True, ortho="cholqr", nroots=6),
    5: dict(name="C1000-128", lattice=[[40.4, 0, 0], [0, 40.4, 0], [0, 0, 40.4]], grid=(128, 128, 128), ecut=25.0,
            nspin=2, nocc=(2000, 2000), nvec=32, alpha=0.25, envelope=True, ortho="cholqr", nroots=6),
}


def config(config_id, **overrides):
    c = dict(CONFIGS[config_id])
    c["id"] = config_id
    c["seed"] = SEED_BASE + config_id
    c.update(overrides)
    return c


def _as_real(c):
    """[.., npwh] complex128 -> [.., 2 npwh] float64 view (re, im interleaved)."""
    c = np.ascontiguousarray(c, dtype=np.complex128)
    return c.view(np.float64).reshape(c.shape[:-1] + (2 * c.shape[-1],))


def gamma_gram(a, b):
    """G[i, j] = 2 Re sum_g conj(a_i(g)) b_j(g) - a_i(0) b_j(0): inner products of half-sphere rows."""
    ar = _as_real(a)
    br = _as_real(b)
    g = 2.0 * (ar @ br.T)
    g -= np.outer(ar[:, 0], br[:, 0])
    return g


def orbitals(rng, nocc, g2_half, ecut, envelope=True, ortho="lowdin"):
    """nocc orthonormal real orbitals as half-sphere coefficients [nocc, npwh] (G = 0 first, Im c(0) = 0)."""
    npwh = len(g2_half)
    c = rng.standard_normal((nocc, npwh)) + 1j * rng.standard_normal((nocc, npwh))
    if envelope:
        c *= np.exp(-np.asarray(g2_half) / ecut)[None, :]
    c[:, 0] = c[:, 0].real
    s = gamma_gram(c, c)
    if ortho == "lowdin":
        w, u = np.linalg.eigh(s)
        t = (u * (1.0 / np.sqrt(w))[None, :]) @ u.T          # S^-1/2
        c = t @ c
    else:                                                     # Cholesky-QR: S = L L^T, C <- L^-1 C
        l = np.linalg.cholesky(s)
        c = np.linalg.solve(l, c)
    # one clean-up pass so that orthonormality holds to rounding
    s = gamma_gram(c, c)
    l = np.linalg.cholesky(s)
    c = np.linalg.solve(l, c)
    c[:, 0] = c[:, 0].real
    return np.ascontiguousarray(c)


def eigenvalues(rng, nocc):
    return np.sort(rng.uniform(-0.5, 0.0, size=nocc))


def trial_vectors(rng, blocks, nvec):
    """nvec orthonormal random trial vectors, each block projected off the given orbitals.

    blocks: list of (n_functions, psi_target) per spin block; psi_target [nocc_t, npwh] are the
    occupied orbitals of the block's TARGET spin (the ones P_c removes).
    Returns complex128 [nvec, sum_b n_functions * npwh].
    """
    npwh = blocks[0][1].shape[1]
    parts = []
    for (nf, psi_t) in blocks:
        x = rng.standard_normal((nvec * nf, npwh)) + 1j * rng.standard_normal((nvec * nf, npwh))
        x[:, 0] = x[:, 0].real
        for _ in range(2):
            x -= gamma_gram(x, psi_t) @ psi_t
        x[:, 0] = x[:, 0].real
        parts.append(x.reshape(nvec, nf * npwh))
    X = np.concatenate(parts, axis=1)
    rows = X.shape[1] // npwh
    for _ in range(2):                                        # Cholesky-orthonormalise the nvec vectors
        Xr = X.reshape(nvec * rows, npwh)
        ar = _as_real(Xr).reshape(nvec, -1)
        g = 2.0 * (ar @ ar.T)
        z = Xr[:, 0].real.reshape(nvec, rows)
        g -= z @ z.T
        l = np.linalg.cholesky(g)
        X = np.linalg.solve(l, X)
    return np.ascontiguousarray(X)


def make_problem_inputs(cfg, g2_half, scale_nocc=None):
    """Draw orbitals, eigenvalues for a configuration.  Returns dict(psi=[..], eig=[..])."""
    rng = np.random.Generator(np.random.PCG64(cfg["seed"]))
    nocc = cfg["nocc"] if scale_nocc is None else scale_nocc
    psi, eig = [], []
    for s in range(cfg["nspin"]):
        psi.append(orbitals(rng, nocc[s], g2_half, cfg["ecut"], cfg["envelope"], cfg["ortho"]))
        eig.append(eigenvalues(rng, nocc[s]))
    return dict(psi=psi, eig=eig, rng=rng)


def make_trial_block(cfg, inputs, nvec, mode):
    """Trial vectors for mode 0 (spin conserving), 1 (up->down flip) or 2 (down->up flip)."""
    psi = inputs["psi"]
    if mode == 0:
        blocks = [(psi[s].shape[0], psi[s]) for s in range(cfg["nspin"])]
    else:
        src = 0 if mode == 1 else 1
        blocks = [(psi[src].shape[0], psi[1 - src])]
    return trial_vectors(inputs["rng"], blocks, nvec)


def diagonal_guess(rng, diag, npwh, nvec, noise=1e-3):
    """Davidson start vectors: unit vectors on the nvec smallest entries of `diag` (the caller's
    |G|^2/2 - eps_v per element of a trial vector) plus seeded noise of 2-norm ~`noise`; Im c(G=0) = 0."""
    diag = np.asarray(diag)
    order = np.argsort(diag, kind="stable")[:nvec]
    L = diag.size
    x0 = noise / np.sqrt(2.0 * L) * (rng.standard_normal((nvec, L)) + 1j * rng.standard_normal((nvec, L)))
    for i, e in enumerate(order):
        x0[i, e] += 1.0
    x0.reshape(nvec, -1, npwh)[:, :, 0] = x0.reshape(nvec, -1, npwh)[:, :, 0].real
    return np.ascontiguousarray(x0)
