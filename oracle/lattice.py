"""Reciprocal lattice, plane-wave sphere and FFT-grid index maps (oracle side).

Test infrastructure only (see oracle/__init__.py).

Conventions (after SURVEY 8.0; the paper works at the
Gamma point with a plane-wave basis and a kinetic-energy cutoff, PAPER.md:48,
:197, :276):
  lattice rows a_i (bohr), reciprocal rows b_i with b_i . a_j = 2 pi delta_ij,
  G = m1 b1 + m2 b2 + m3 b3, grid point r_j = sum_i (j_i / n_i) a_i.
Sphere membership and ordering follow reading A7 of DESIGN.md.
Pins: tests/test_oracle_lattice.py (b.a = 2 pi delta, plane-wave counts vs the
continuum estimate, -G closure, hexagonal cell).
"""
import numpy as np


def reciprocal(lattice):
    """Rows b_i with b_i . a_j = 2 pi delta_ij; cell volume Omega = |det A|."""
    A = np.asarray(lattice, dtype=np.float64).reshape(3, 3)
    B = 2.0 * np.pi * np.linalg.inv(A).T
    omega = abs(np.linalg.det(A))
    return B, omega


def enumerate_half_sphere(lattice, ecut_ry):
    """Canonical half sphere of plane waves, |G|^2 <= E_cut [Ry] (reading A7).

    Returns (miller[npwh,3] int64, g2[npwh] float64 in bohr^-2 == Ry).
    Half = G=0, then m1>0, or m1=0 and m2>0, or m1=m2=0 and m3>0.
    Order = ascending |G|^2 (values within 1e-12 relative count as equal), then
    lexicographic (m1, m2, m3).
    """
    B, _ = reciprocal(lattice)
    A = np.asarray(lattice, dtype=np.float64).reshape(3, 3)
    gmax = np.sqrt(ecut_ry)
    # |m_i| <= |G| |a_i| / (2 pi) because m_i = G . a_i / (2 pi)
    bound = [int(np.floor(gmax * np.linalg.norm(A[i]) / (2 * np.pi))) + 1 for i in range(3)]
    out = []
    for m1 in range(0, bound[0] + 1):
        for m2 in range(-bound[1], bound[1] + 1):
            for m3 in range(-bound[2], bound[2] + 1):
                if m1 == 0 and (m2 < 0 or (m2 == 0 and m3 < 0)):
                    continue
                g = m1 * B[0] + m2 * B[1] + m3 * B[2]
                g2 = g[0] * g[0] + g[1] * g[1] + g[2] * g[2]
                if g2 <= ecut_ry:
                    out.append((g2, m1, m2, m3))
    out.sort(key=lambda t: t[0])
    # group into shells of (numerically) equal |G|^2, then lexicographic inside a shell
    keyed = []
    shell = 0
    prev = None
    for (g2, m1, m2, m3) in out:
        if prev is not None and g2 - prev > 1e-12 * g2:
            shell += 1
        prev = g2
        keyed.append((shell, m1, m2, m3, g2))
    keyed.sort(key=lambda t: (t[0], t[1], t[2], t[3]))
    miller = np.array([(t[1], t[2], t[3]) for t in keyed], dtype=np.int64)
    g2 = np.array([t[4] for t in keyed], dtype=np.float64)
    return miller, g2


def grid_miller(grid):
    """Signed Miller index of every FFT-grid index: m = j if j < (n+1)//2 else j - n.

    For even n the Nyquist index n/2 gets m = -n/2 (reading A7)."""
    ms = []
    for n in grid:
        j = np.arange(n)
        ms.append(np.where(j < (n + 1) // 2, j, j - n))
    return ms


def grid_g2(lattice, grid):
    """|G|^2 (bohr^-2) for every point of the FFT grid, shape grid."""
    B, _ = reciprocal(lattice)
    m1, m2, m3 = grid_miller(grid)
    M1, M2, M3 = np.meshgrid(m1, m2, m3, indexing="ij")
    gx = M1 * B[0, 0] + M2 * B[1, 0] + M3 * B[2, 0]
    gy = M1 * B[0, 1] + M2 * B[1, 1] + M3 * B[2, 1]
    gz = M1 * B[0, 2] + M2 * B[1, 2] + M3 * B[2, 2]
    return gx * gx + gy * gy + gz * gz


def check_grid_holds_sphere(miller, grid):
    """2 m_max + 1 <= n_i on every axis: the sphere and its mirror fit the grid."""
    mmax = np.abs(miller).max(axis=0) if len(miller) else np.zeros(3, int)
    return all(2 * int(mmax[i]) + 1 <= grid[i] for i in range(3))
