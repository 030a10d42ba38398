"""Pins for oracle/lattice.py: what the mathematics fixes about the reciprocal lattice and the sphere."""
import math

import numpy as np
import pytest

from oracle import lattice as lat

HEX = [[36.9, 0, 0], [-18.45, 36.9 * math.sqrt(3) / 2, 0], [0, 0, 19.5]]
TRI = [[4.0, 0, 0], [0.5, 4.2, 0], [0.3, -0.2, 4.5]]


@pytest.mark.parametrize("A", [np.eye(3) * 10.0, HEX, TRI])
def test_reciprocal_duality(A):
    B, omega = lat.reciprocal(A)
    A = np.asarray(A, float)
    assert np.allclose(B @ A.T, 2 * np.pi * np.eye(3), atol=1e-13)
    assert omega == pytest.approx(abs(np.dot(A[0], np.cross(A[1], A[2]))), rel=1e-14)


def test_hexagonal_first_shell():
    # |b1|^2 = (2 pi / a)^2 * 4/3 for a hexagonal cell, |b3| = 2 pi / c
    B, _ = lat.reciprocal(HEX)
    assert np.dot(B[0], B[0]) == pytest.approx((2 * np.pi / 36.9) ** 2 * 4 / 3, rel=1e-13)
    assert np.linalg.norm(B[2]) == pytest.approx(2 * np.pi / 19.5, rel=1e-13)


@pytest.mark.parametrize("A,ecut,npw", [
    (np.eye(3) * 10.0, 10.0, 515),      # SURVEY 8.0 exact enumeration, config 1
    (np.eye(3) * 13.48, 25.0, 5185),    # config 2
])
def test_sphere_counts(A, ecut, npw):
    miller, g2 = lat.enumerate_half_sphere(A, ecut)
    assert 2 * len(miller) - 1 == npw
    # continuum estimate Omega Gmax^3 / (6 pi^2) within a few percent
    _, omega = lat.reciprocal(A)
    est = omega * ecut ** 1.5 / (6 * np.pi ** 2)
    assert abs(npw - est) / est < 0.06


def test_cubic_sphere_is_integer_ball():
    # cubic cell: |G|^2 = (2 pi / L)^2 |m|^2, so the sphere is exactly the integer ball |m|^2 <= R2
    L, ecut = 10.0, 10.0
    R2 = ecut / (2 * np.pi / L) ** 2
    count = sum(1 for a in range(-6, 7) for b in range(-6, 7) for c in range(-6, 7) if a * a + b * b + c * c <= R2)
    miller, _ = lat.enumerate_half_sphere(np.eye(3) * L, ecut)
    assert 2 * len(miller) - 1 == count


@pytest.mark.parametrize("A,ecut", [(np.eye(3) * 10.0, 10.0), (HEX, 2.0), (TRI, 30.0)])
def test_half_sphere_structure(A, ecut):
    miller, g2 = lat.enumerate_half_sphere(A, ecut)
    B, _ = lat.reciprocal(A)
    assert tuple(miller[0]) == (0, 0, 0) and g2[0] == 0.0
    # |G|^2 reported equals |B^T m|^2 and is within the cutoff, ascending up to the tie tolerance
    G = miller @ B
    assert np.allclose((G * G).sum(1), g2, rtol=1e-13, atol=0)
    assert np.all(g2 <= ecut)
    assert np.all(np.diff(g2) > -1e-12 * g2[1:])
    # half and mirrored half are disjoint apart from G = 0 and together closed under negation
    s = {tuple(m) for m in miller}
    sm = {tuple(-m) for m in miller}
    assert s & sm == {(0, 0, 0)}
    # every |m| beyond the sphere is really outside: test the shell just outside on each axis
    full = s | sm
    mmax = np.abs(miller).max(0)
    for a in range(-mmax[0] - 1, mmax[0] + 2):
        for b in range(-mmax[1] - 1, mmax[1] + 2):
            for c in range(-mmax[2] - 1, mmax[2] + 2):
                g = a * B[0] + b * B[1] + c * B[2]
                assert ((a, b, c) in full) == (np.dot(g, g) <= ecut)
    # ties are ordered lexicographically
    for i in range(1, len(miller)):
        if abs(g2[i] - g2[i - 1]) <= 1e-12 * g2[i]:
            assert tuple(miller[i - 1]) < tuple(miller[i])


def test_grid_miller_nyquist():
    m = lat.grid_miller((6, 5, 4))
    assert list(m[0]) == [0, 1, 2, -3, -2, -1]
    assert list(m[1]) == [0, 1, 2, -2, -1]
    assert list(m[2]) == [0, 1, -2, -1]


def test_grid_g2_matches_direct():
    g2 = lat.grid_g2(TRI, (6, 5, 4))
    B, _ = lat.reciprocal(TRI)
    g = 2 * B[0] - 2 * B[1] + 1 * B[2]      # index (2, 3, 1) -> m = (2, -2, 1)
    assert g2[2, 3, 1] == pytest.approx(np.dot(g, g), rel=1e-14)
    assert g2[0, 0, 0] == 0.0


def test_grid_must_hold_the_sphere():
    """check_grid_holds_sphere: 2 m_max + 1 <= n on every axis, and a grid one point short is refused by Problem."""
    from oracle import liouville as olv
    cubic = [[10.0, 0, 0], [0, 10.0, 0], [0, 0, 10.0]]
    miller, g2 = lat.enumerate_half_sphere(cubic, 10.0)
    mmax = np.abs(miller).max(0)
    assert list(mmax) == [5, 5, 5]            # floor(sqrt(10) * 10 / (2 pi)) = 5
    assert lat.check_grid_holds_sphere(miller, (11, 11, 11))
    for short in [(10, 11, 11), (11, 10, 11), (11, 11, 10)]:
        assert not lat.check_grid_holds_sphere(miller, short)
    psi = [np.zeros((1, len(miller)), dtype=complex)]; psi[0][0, 0] = 1.0
    with pytest.raises(ValueError):
        olv.Problem(cubic, (12, 12, 10), 10.0, 1, psi, [np.array([-0.1])], 0.0)


def test_sphere_counts_match_the_survey_table():
    """tests/golden/gvector_counts.txt: N_pw / N_pwh of the five BASELINE.json configurations."""
    import os
    import synthetic_inputs as inputs
    path = os.path.join(os.path.dirname(__file__), "golden", "gvector_counts.txt")
    rows = [l.split() for l in open(path) if l.strip() and not l.startswith("#")]
    assert len(rows) == 5
    for cid, npw, npwh in rows:
        cfg = inputs.config(int(cid))
        miller, _ = lat.enumerate_half_sphere(np.array(cfg["lattice"], dtype=float), cfg["ecut"])
        assert len(miller) == int(npwh) and 2 * len(miller) - 1 == int(npw)
