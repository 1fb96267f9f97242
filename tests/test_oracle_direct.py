"""Pins for oracle O1 (direct Ewald, oracle/direct_ewald.c).  CPU only.

Each pin is independent of the oracle's own formulae: invariants of the exact periodic
sum, a closed-form lattice constant, and a differential identity of Stokes flow.
"""
import numpy as np
import pytest

import oracle


def rel(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


@pytest.fixture(scope="module")
def cloud():
    rng = np.random.default_rng(20261104)
    x = rng.random((40, 3))
    f = rng.standard_normal((40, 3))
    return x, f


def test_xi_independence(cloud):
    """The exact sum does not depend on the split parameter (PAPER.md:49 'xi controls the
    decay of G^N'): a wrong sign/factor in (2.3), (2.4b), the 1/V, or the self term breaks it."""
    x, f = cloud
    u4 = oracle.direct_ewald(x, f, 1.0, 4.0)
    u7 = oracle.direct_ewald(x, f, 1.0, 7.0)
    assert rel(u4, u7) < 1e-13


def test_xi_independence_nonzero_net_force(cloud):
    """Reading S2: dropping k=0 stays xi-independent even when sum f != 0."""
    x, f = cloud
    f = f + np.array([0.7, -0.2, 1.1])
    assert rel(oracle.direct_ewald(x, f, 1.0, 3.5), oracle.direct_ewald(x, f, 1.0, 6.0)) < 1e-13


def test_hasimoto_constant(golden_dir):
    """N=1: u = -(4/3) * 2.8372974795 / L * f  (tests/golden/hasimoto_sc.txt)."""
    val = None
    for line in (golden_dir / "hasimoto_sc.txt").read_text().splitlines():
        if line.startswith("hasimoto_sc"):
            val = float(line.split()[1])
    f = np.array([[1.0, -2.0, 0.5]])
    for L, xi in ((1.0, 3.0), (1.0, 5.0), (2.5, 2.0)):
        u = oracle.direct_ewald(np.array([[0.3, 0.2, 0.9]]) * L, f, L, xi)
        np.testing.assert_allclose(u, -(4.0 / 3.0) * val / L * f, rtol=2e-10)


def test_translation_invariance(cloud):
    x, f = cloud
    s = np.array([0.123456, 0.654321, 0.333])
    u0 = oracle.direct_ewald(x, f, 1.0, 5.0)
    u1 = oracle.direct_ewald(np.mod(x + s, 1.0), f, 1.0, 5.0)
    assert rel(u1, u0) < 1e-12


def test_linearity_and_symmetry(cloud):
    x, f = cloud
    rng = np.random.default_rng(5)
    g = rng.standard_normal(f.shape)
    Mf = oracle.direct_ewald(x, f, 1.0, 5.0)
    Mg = oracle.direct_ewald(x, g, 1.0, 5.0)
    Mfg = oracle.direct_ewald(x, 2.0 * f - 3.0 * g, 1.0, 5.0)
    assert rel(Mfg, 2.0 * Mf - 3.0 * Mg) < 1e-13
    # the Stokeslet is symmetric and even: <g, M f> = <f, M g>
    a, b = np.sum(g * Mf), np.sum(f * Mg)
    assert abs(a - b) < 1e-12 * (abs(a) + abs(b))


def test_length_scaling(cloud):
    """G is homogeneous of degree -1: u(Lx; L, xi/L) = u(x; 1, xi)/L."""
    x, f = cloud
    u1 = oracle.direct_ewald(x, f, 1.0, 5.0)
    u3 = oracle.direct_ewald(3.0 * x, f, 3.0, 5.0 / 3.0)
    assert rel(3.0 * u3, u1) < 1e-13


def test_divergence_free_off_particle(cloud):
    """Stokes flow is incompressible: div u = 0 away from the forces (central differences).
    Catches a wrong weight on the r(x)r term relative to the identity term."""
    x, f = cloud
    t0 = np.array([[0.512, 0.487, 0.531]])
    d = 2e-4
    div = 0.0
    scale = 0.0
    for c in range(3):
        e = np.zeros(3); e[c] = d
        up = oracle.direct_ewald(x, f, 1.0, 5.0, targets=t0 + e)
        um = oracle.direct_ewald(x, f, 1.0, 5.0, targets=t0 - e)
        div += (up[0, c] - um[0, c]) / (2 * d)
        scale += abs(up[0, c] - um[0, c]) / (2 * d)
    grad = np.linalg.norm(oracle.direct_ewald(x, f, 1.0, 5.0, targets=t0)) / 0.05
    assert abs(div) < 1e-5 * max(scale, grad)


def test_two_body_free_space_limit():
    """Two close particles in a huge box: the pair part tends to the free-space Stokeslet
    G(r) f = f/r + r (r.f)/r^3, the rest to the Hasimoto self constants.
    u_1 - [lattice self of f_1] - [lattice 'self-like' regular part applied to f_2] -> G(r) f_2,
    with the regular part varying by O(r^2/L^3): use r/L = 1e-3."""
    L = 1.0
    r = np.array([6e-4, -5e-4, 6.2e-4])
    x = np.array([[0.4, 0.5, 0.6], [0.4, 0.5, 0.6]]) + np.array([r, 0 * r])
    f = np.array([[0.0, 0.0, 0.0], [1.0, -0.5, 2.0]])     # only particle 2 forces
    u = oracle.direct_ewald(x, f, L, 6.0)
    rn = np.linalg.norm(r)
    free = f[1] / rn + r * np.dot(r, f[1]) / rn ** 3
    reg = -(4.0 / 3.0) * 2.8372974795 / L * f[1]
    np.testing.assert_allclose(u[0], free + reg, rtol=0, atol=5e-5 * np.linalg.norm(reg))
