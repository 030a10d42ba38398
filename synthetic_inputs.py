"""Seeded synthetic inputs shaped like the paper's defect supercells.

This module serves BOTH the CUDA path and the oracle (tests, bench.py) and sits outside both packages.  It holds
none of the method's arithmetic: it draws random numbers, runs plain Euclidean linear algebra (QR / Cholesky of
real vectors) on them, and lists the five configurations of BASELINE.json.  The only convention it knows is the
STORAGE convention of the C ABI (include/tddft.h): a real function is stored as the npwh complex coefficients of
the canonical half sphere, G = 0 first with Im c(0) = 0.  `to_coords` / `from_coords` re-express that storage as the
2*npwh - 1 real coordinates of the function in the orthonormal basis {1, sqrt2 cos(G.r), sqrt2 sin(G.r)}, where
"orthonormal set of functions" is simply "orthonormal set of real vectors".  The G sphere (its size and |G|^2
values) is an INPUT: the caller gets it from `tddft_enumerate_gvectors` (CUDA side) or `oracle.lattice` (oracle side).

The inputs stand in for the paper's workloads (Quantum ESPRESSO ground states of NV-/SiV0 in diamond, VV0 in 4H-SiC,
PAPER.md:224, :276, :292), which are not available; recipe in DESIGN.md section 4.
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
            nspin=2, nocc=(129, 127), nvec=8, alpha=0.18, envelope=True, ortho="qr", nroots=4),
    3: dict(name="NV215-72", lattice=[[20.2, 0, 0], [0, 20.2, 0], [0, 0, 20.2]], grid=(72, 72, 72), ecut=25.0,
            nspin=2, nocc=(432, 430), nvec=16, alpha=0.18, envelope=True, ortho="qr", nroots=6),
    4: dict(name="SiC576-96x96x100", lattice=[[36.9, 0, 0], [-18.45, 36.9 * _S3, 0], [0, 0, 19.5]],
            grid=(96, 96, 100), ecut=20.0, nspin=2, nocc=(1150, 1150), nvec=16, alpha=0.15,
            envelope=True, ortho="qr", nroots=6),
    5: dict(name="C1000-128", lattice=[[40.4, 0, 0], [0, 40.4, 0], [0, 0, 40.4]], grid=(128, 128, 128), ecut=25.0,
            nspin=2, nocc=(2000, 2000), nvec=32, alpha=0.25, envelope=True, ortho="qr", nroots=6),
    # the paper-faithful 60 Ry cutoff on the 215-atom cell; the paper never states a grid,
    # 108^3 holds the doubled sphere (4*24+1 = 97 <= 108), radix mix 2^2 3^3
    6: dict(name="NV215-108-60Ry", lattice=[[20.2, 0, 0], [0, 20.2, 0], [0, 0, 20.2]], grid=(108, 108, 108), ecut=60.0,
            nspin=2, nocc=(432, 430), nvec=16, alpha=0.18, envelope=True, ortho="qr", nroots=6),
}


def config(config_id, **overrides):
    c = dict(CONFIGS[config_id])
    c["id"] = config_id
    c["seed"] = SEED_BASE + config_id
    c.update(overrides)
    return c


# ---- storage convention <-> real coordinates -------------------------------------------------------------------
def to_coords(c):
    """[.., npwh] complex half-sphere storage -> [.., 2 npwh - 1] real coordinates (c0, sqrt2 Re c, sqrt2 Im c)."""
    c = np.asarray(c, dtype=np.complex128)
    r2 = math.sqrt(2.0)
    return np.concatenate([c[..., :1].real, r2 * c[..., 1:].real, r2 * c[..., 1:].imag], axis=-1)


def from_coords(u):
    """Inverse of to_coords."""
    u = np.asarray(u, dtype=np.float64)
    npwh = (u.shape[-1] + 1) // 2
    c = np.empty(u.shape[:-1] + (npwh,), dtype=np.complex128)
    c[..., 0] = u[..., 0]
    c[..., 1:] = (u[..., 1:npwh] + 1j * u[..., npwh:]) / math.sqrt(2.0)
    return np.ascontiguousarray(c)


def _orthonormal_rows(u, how):
    """Orthonormalise the rows of a real matrix (Euclidean): symmetric (Loewdin) or QR, then one clean-up QR."""
    if how == "lowdin":
        s = u @ u.T
        w, v = np.linalg.eigh(s)
        u = ((v * (1.0 / np.sqrt(w))[None, :]) @ v.T) @ u
    q, r = np.linalg.qr(u.T)
    q = q * np.sign(np.diag(r))[None, :]          # keep the orientation of the input rows
    return np.ascontiguousarray(q.T)


def orbitals(rng, nocc, g2_half, ecut, envelope=True, ortho="lowdin"):
    """nocc orthonormal real orbitals as half-sphere coefficients [nocc, npwh] (G = 0 first, Im c(0) = 0)."""
    npwh = len(g2_half)
    u = rng.standard_normal((nocc, 2 * npwh - 1))
    if envelope:
        w = np.exp(-np.asarray(g2_half) / ecut)
        u *= np.concatenate([w, w[1:]])[None, :]
    return from_coords(_orthonormal_rows(u, ortho))


def eigenvalues(rng, nocc):
    return np.sort(rng.uniform(-0.5, 0.0, size=nocc))


def trial_vectors(rng, blocks, nvec):
    """nvec orthonormal random trial vectors whose functions are orthogonal to the given orbitals.

    blocks: list of (n_functions, psi_target) per spin block; psi_target [nocc_t, npwh] are the occupied orbitals of
    the block's TARGET spin (trial functions live in their orthogonal complement).
    Returns complex128 [nvec, sum_b n_functions * npwh].
    """
    parts = []
    for (nf, psi_t) in blocks:
        ut = to_coords(psi_t)
        x = rng.standard_normal((nvec * nf, ut.shape[1]))
        for _ in range(2):
            x -= (x @ ut.T) @ ut
        parts.append(x.reshape(nvec, nf * ut.shape[1]))
    x = np.concatenate(parts, axis=1)
    q, r = np.linalg.qr(x.T)                                   # orthonormalise the nvec long vectors
    x = (q * np.sign(np.diag(r))[None, :]).T
    out, o = [], 0
    for (nf, psi_t) in blocks:
        w = 2 * psi_t.shape[1] - 1
        out.append(from_coords(x[:, o:o + nf * w].reshape(nvec, nf, w)).reshape(nvec, -1))
        o += nf * w
    return np.ascontiguousarray(np.concatenate(out, axis=1))


def localized_orbitals(rng, nocc, miller, g2_half, width=1.6):
    """nocc orthonormal orbitals localised around random sites (Gaussians of the given width in bohr, symmetrically
    orthonormalised): a stand-in for the maximally localised Wannier functions of PAPER.md:237.

    c_n(G) ~ exp(-|G|^2 width^2 / 2) exp(-i G.R_n): a plain Fourier series of a Gaussian, no method arithmetic."""
    frac = rng.uniform(0.0, 1.0, size=(nocc, 3))
    phase = -2.0 * np.pi * (frac @ np.asarray(miller, dtype=np.float64).T)      # G.R = 2 pi m.f
    c = np.exp(-0.5 * width * width * np.asarray(g2_half))[None, :] * np.exp(1j * phase)
    c[:, 0] = c[:, 0].real
    return from_coords(_orthonormal_rows(to_coords(c), "lowdin"))


def random_orthogonal(rng, n):
    q, r = np.linalg.qr(rng.standard_normal((n, n)))
    return np.ascontiguousarray(q * np.sign(np.diag(r))[None, :])


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
    """Davidson start vectors: unit vectors on the nvec smallest entries of `diag` (the caller's per-element
    diagonal of a trial vector) plus seeded noise of 2-norm ~`noise`; Im c(G=0) = 0."""
    diag = np.asarray(diag)
    order = np.argsort(diag, kind="stable")[:nvec]
    L = diag.size
    x0 = noise / np.sqrt(2.0 * L) * (rng.standard_normal((nvec, L)) + 1j * rng.standard_normal((nvec, L)))
    for i, e in enumerate(order):
        x0[i, e] += 1.0
    x0.reshape(nvec, -1, npwh)[:, :, 0] = x0.reshape(nvec, -1, npwh)[:, :, 0].real
    return np.ascontiguousarray(x0)
