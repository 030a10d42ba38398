"""Pins the fact the CUDA path's pruned frequency-space layout rests on: on an alias-free grid the
discrete spectrum of a product of two sphere functions (a pair density phi_v phi_v', or a response
density, Eq. 4) vanishes outside the sphere of radius 2 sqrt(E_cut), and a sphere function's outside sqrt(E_cut).
Oracle side only (no CUDA): the library's column maps are then exercised by the GPU parity tests."""
import numpy as np

from helpers import Case
from oracle import lattice as olat

HEX = [[9.0, 0, 0], [-4.5, 7.794228634059948, 0], [0, 0, 8.0]]


def test_pair_density_spectrum_is_confined_to_the_doubled_sphere():
    case = Case(HEX, (24, 24, 20), 5.0, 1, (4,), 0.25, seed=301)
    o = case.oracle
    mmax = np.max(np.abs(case.miller), axis=0)
    assert all(4 * mmax[a] + 1 <= case.grid[a] for a in range(3)), "the test grid must be alias free for products"
    g2 = olat.grid_g2(case.lattice, case.grid).reshape(case.grid)
    phi = [np.asarray(p).reshape(case.grid) for p in o.phi[0]]
    for i in range(4):
        spec = np.abs(np.fft.fftn(phi[i]))
        assert spec[g2 > case.ecut * (1 + 1e-9)].max() < 1e-13 * spec.max()
        for j in range(i, 4):
            spec = np.abs(np.fft.fftn(phi[i] * phi[j]))
            outside = g2 > 4.0 * case.ecut * (1 + 1e-9)
            assert outside.any() and spec[outside].max() < 1e-13 * spec.max()
            # ... and the Coulomb potential tau_ij inherits the support (the kernel is diagonal in G)
            tau = np.abs(np.fft.fftn(np.asarray(o.coulomb(phi[i] * phi[j])).reshape(case.grid)))
            assert tau[outside].max() < 1e-13 * tau.max()
