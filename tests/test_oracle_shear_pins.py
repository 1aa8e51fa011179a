"""Pins of the sheared-lattice oracle (Eq. 48) against what the
mathematics fixes -- none of them is the oracle re-typed:
gamma = 0 reproduces the pinned cubic oracle; gamma and gamma + 1 describe the same lattice; a shift of a particle by a
lattice vector changes nothing; independence of the splitting parameter; symmetry and positive definiteness of the
assembled grand mobility; spectral convergence of O2 to O1 at the rate of Eq. 79 at the paper's gamma = 0.5."""
import math
import os

import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _gold(name):
    with open(os.path.join(GOLD, name)) as fh:
        rows = [ln.split() for ln in fh if ln.strip() and not ln.startswith("#")]
    return [float(v) for v in rows[0]]


def _rel(a, b):
    return float(np.linalg.norm(np.asarray(a) - np.asarray(b)) / np.linalg.norm(np.asarray(b)))


def _cut(xi, L, digits=6.5):
    return int(math.ceil(digits / xi / L)) + 1, int(math.ceil(xi * L / (2 * math.pi) * 2 * digits)) + 1


def test_zero_strain_reproduces_the_cubic_oracles(oracle, workloads):
    sysm = workloads.random_small_system(2, 8, 10.0)
    xi, L = 0.6, sysm["L"]
    nimg, kmax = _cut(xi, L)
    a, mom = (sysm["pos"], sysm["radii"], L), (sysm["F"], sysm["T"], sysm["S"], sysm["s"])
    ref = oracle.o1_apply(*a, xi, *mom, nimg=nimg, kmax=kmax)
    got = oracle.o1_apply_sheared(*a, 0.0, xi, *mom, nimg=nimg, kmax=kmax)
    for g, r in zip(got, ref):
        assert np.array_equal(g, r)
    ref2 = oracle.o2_apply(*a, xi, 0.5 * L, 32, 12, *mom, want_grids=True)
    got2 = oracle.o2_apply_sheared(*a, 0.0, xi, 0.5 * L, 32, 12, *mom, want_grids=True)
    for key in ("U", "Omega", "E", "s_out", "gridH", "gridOut"):
        assert _rel(got2[key], ref2[key]) <= 1e-13, key


@pytest.mark.parametrize("gamma", [0.3, -0.4])
def test_strain_gamma_and_gamma_plus_one_are_the_same_lattice(oracle, workloads, gamma):
    """a2' = a2 + a1: the same set of lattice points, so the definition O1 must give the same numbers."""
    sysm = workloads.random_small_system(3, 5, 9.0)
    xi, L = 0.7, sysm["L"]
    nimg, kmax = _cut(xi, L)
    a, mom = (sysm["pos"], sysm["radii"], L), (sysm["F"], sysm["T"], sysm["S"], sysm["s"])
    r0 = oracle.o1_apply_sheared(*a, gamma, xi, *mom, nimg=nimg + 1, kmax=kmax + 2)
    r1 = oracle.o1_apply_sheared(*a, gamma + 1.0, xi, *mom, nimg=nimg + 1, kmax=kmax + 2)
    for x, y in zip(r0, r1):
        assert _rel(x, y) <= 1e-12
    # and the strain matters: gamma = 0 gives something else
    rc = oracle.o1_apply(*a, xi, *mom, nimg=nimg, kmax=kmax)
    assert _rel(r0[0], rc[0]) > 1e-4


def test_sheared_total_is_independent_of_xi_symmetric_and_positive_definite(oracle, workloads):
    import scipy.linalg as sl
    from test_oracle_pins import _gram
    sysm = workloads.random_small_system(1, 3, 8.0)
    gamma, L, N = 0.35, sysm["L"], sysm["N"]
    mats = []
    for xi in (0.55, 0.9):
        nimg, kmax = _cut(xi, L)
        mats.append(oracle.o1_matrix_sheared(sysm["pos"], sysm["radii"], L, gamma, xi, nimg=nimg + 1, kmax=kmax + 2))
    A, B = mats
    assert np.abs(A - B).max() / np.abs(A).max() < 1e-12
    Q = _gram(N) @ A
    assert np.abs(Q - Q.T).max() / np.abs(Q).max() < 1e-13
    assert sl.eigh(0.5 * (Q + Q.T), _gram(N), eigvals_only=True).min() > 0


def test_o2_is_periodic_on_the_sheared_lattice(oracle, workloads):
    """Moving particles by lattice vectors (a1, a2 = (gamma L, L, 0), a3) changes neither the wrap, the spreading nor the
    minimum image -- only round-off."""
    sysm = workloads.random_small_system(4, 12, 10.0)
    gamma, L, xi = 0.5, sysm["L"], 0.8
    mom = (sysm["F"], sysm["T"], sysm["S"], sysm["s"])
    base = oracle.o2_apply_sheared(sysm["pos"], sysm["radii"], L, gamma, xi, 0.45 * L, 32, 10, *mom)
    rng = np.random.default_rng(2)
    n = rng.integers(-2, 3, size=(sysm["N"], 3))
    A = L * np.array([[1.0, gamma, 0.0], [0.0, 1.0, 0.0], [0.0, 0.0, 1.0]])
    moved = sysm["pos"] + n @ A.T
    got = oracle.o2_apply_sheared(moved, sysm["radii"], L, gamma, xi, 0.45 * L, 32, 10, *mom)
    for key in ("U", "Omega", "E", "s_out"):
        assert _rel(got[key], base[key]) <= 1e-10, key


def test_o2_converges_spectrally_to_o1_under_shear(oracle, workloads):
    """the accuracy at gamma = 0.5 is that of the orthogonal box; Eq. 79 rate exp(-P pi/2) at m = sqrt(pi P)."""
    _, rate = _gold("paper_accuracy_claims.txt")
    sysm = workloads.random_small_system(2, 10, 10.0)
    gamma, xi, L = 0.5, 0.6, sysm["L"]
    nimg, kmax = _cut(xi, L)
    mom = (sysm["F"], sysm["T"], sysm["S"], sysm["s"])
    ref = oracle.o1_apply_sheared(sysm["pos"], sysm["radii"], L, gamma, xi, *mom, nimg=nimg, kmax=kmax + 4, parts=oracle.PART_WAVE)
    errs = {}
    for P in (8, 16, 20, 24):
        r = oracle.o2_apply_sheared(sysm["pos"], sysm["radii"], L, gamma, xi, 0.5 * L, 40, P, *mom, parts=oracle.PART_WAVE)
        errs[P] = max(_rel(r["U"], ref[0]), _rel(r["Omega"], ref[1]), _rel(r["E"], ref[2]), _rel(r["s_out"], ref[3]))
    slope = -math.log(errs[20] / errs[8]) / 12.0
    assert 0.75 * rate < slope < 1.25 * rate, (errs, slope)
    assert errs[24] < 2e-10, errs
    # full product, converged: real part (sheared minimum image) + wave part + self terms
    xi2 = 1.0
    nimg2, kmax2 = _cut(xi2, L)
    full1 = oracle.o1_apply_sheared(sysm["pos"], sysm["radii"], L, gamma, xi2, *mom, nimg=nimg2, kmax=kmax2 + 6)
    full2 = oracle.o2_apply_sheared(sysm["pos"], sysm["radii"], L, gamma, xi2, 0.5 * L, 64, 24, *mom)
    assert _rel(full2["U"], full1[0]) < 1e-8 and _rel(full2["E"], full1[2]) < 1e-8, (_rel(full2["U"], full1[0]), _rel(full2["E"], full1[2]))
