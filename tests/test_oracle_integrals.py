"""Pins for the oracle's integral code against things that are not the oracle:
closed forms, brute-force quadrature, symmetry, inequalities."""
import math

import numpy as np
import pytest
from scipy import special

import oracle
from refquad import cart_components, eri_quadrature
from synth import make_config, subset_atoms


# ------------------------------------------------------------------------------------ normalisation
@pytest.mark.parametrize("n", [1, 2, 4])
def test_unit_self_overlap_every_contracted_component(n):
    """north_star: 'normalisation of contracted shells (unit self-overlap)'; S by eq. 11."""
    prob = make_config(n)
    if n != 1:
        prob = subset_atoms(prob, [0, 1, prob.natoms - 1])
    S = oracle.Oracle(prob).overlap()
    assert np.max(np.abs(np.diag(S) - 1.0)) < 1e-13
    assert np.max(np.abs(S - S.T)) < 1e-14
    assert np.min(np.linalg.eigvalsh(S)) > -1e-12


def test_overlap_two_s_primitives_closed_form():
    """Textbook: <s_a(A)|s_b(B)> = (pi/p)^{3/2} exp(-ab/p R^2) for unnormalised s Gaussians."""
    class P:  # two one-primitive s shells
        xyz = np.array([[0.0, 0.0, 0.0], [0.3, -1.1, 0.7]])
        shell_atom = np.array([0, 1], dtype=np.int32)
        shell_l = np.array([0, 0], dtype=np.int32)
        shell_nprim = np.array([1, 1], dtype=np.int32)
        exponents = np.array([0.8, 1.7])
        coefficients = np.array([1.0, 1.0])
    o = oracle.Oracle(P)
    S = o.overlap()
    a, b = P.exponents
    R2 = np.sum((P.xyz[0] - P.xyz[1]) ** 2)
    Na, Nb = (2 * a / math.pi) ** 0.75, (2 * b / math.pi) ** 0.75
    assert S[0, 1] == pytest.approx(Na * Nb * (math.pi / (a + b)) ** 1.5 * math.exp(-a * b / (a + b) * R2), rel=1e-14)


# ------------------------------------------------------------------------------------------ (ss|ss)
def ssss_closed_form(a, A, b, B, c, C, d, D):
    """eq. 28 with F_0(T) = (1/2) sqrt(pi/T) erf(sqrt T)."""
    A, B, C, D = map(np.asarray, (A, B, C, D))
    p, q = a + b, c + d
    P, Q = (a * A + b * B) / p, (c * C + d * D) / q
    T = p * q / (p + q) * np.sum((P - Q) ** 2)
    F0 = 1.0 if T == 0 else 0.5 * math.sqrt(math.pi / T) * special.erf(math.sqrt(T))
    return (math.exp(-a * b / p * np.sum((A - B) ** 2)) * math.exp(-c * d / q * np.sum((C - D) ** 2))
            * 2 * math.pi ** 2.5 / (p * q * math.sqrt(p + q)) * F0)


def test_ssss_closed_form_random():
    rng = np.random.default_rng(7)
    for _ in range(50):
        ex = np.exp(rng.uniform(math.log(0.05), math.log(50), 4))
        X = rng.uniform(-2.5, 2.5, (4, 3))
        v = oracle.prim_eri_raw(0, ex[0], X[0], 0, ex[1], X[1], 0, ex[2], X[2], 0, ex[3], X[3]).ravel()[0]
        assert v == pytest.approx(ssss_closed_form(ex[0], X[0], ex[1], X[1], ex[2], X[2], ex[3], X[3]), rel=2e-14)


def test_ssss_one_centre_value():
    """Four identical normalised s primitives of exponent a on one centre: 2 sqrt(a/pi)
    (= 1.1283791670955126 at a = 1)."""
    for a in (1.0, 0.2, 13.0):
        N = (2 * a / math.pi) ** 0.75
        v = oracle.prim_eri_raw(0, a, [0, 0, 0], 0, a, [0, 0, 0], 0, a, [0, 0, 0], 0, a, [0, 0, 0]).ravel()[0] * N ** 4
        assert v == pytest.approx(2 * math.sqrt(a / math.pi), rel=1e-14)
    assert 2 * math.sqrt(1 / math.pi) == pytest.approx(1.1283791670955126, rel=1e-15)


# ----------------------------------------------------------------- higher l: brute-force quadrature
QUAD_CASES = [
    # (la, lb, lc, ld) -- every l appears in every position; through (ff|ff)
    (1, 0, 0, 0), (0, 1, 0, 0), (0, 0, 1, 0), (0, 0, 0, 1), (1, 1, 0, 0), (1, 0, 1, 0), (1, 1, 1, 1),
    (2, 0, 0, 0), (0, 2, 1, 0), (2, 1, 0, 1), (2, 2, 0, 0), (0, 0, 2, 2), (2, 2, 2, 2),
    (3, 0, 0, 0), (0, 3, 0, 0), (0, 0, 3, 0), (0, 0, 0, 3), (3, 1, 2, 0), (0, 3, 3, 3), (3, 2, 1, 3), (3, 3, 3, 3),
]


@pytest.mark.parametrize("ls", QUAD_CASES)
def test_primitive_block_vs_bruteforce_quadrature(ls):
    """Sampled components of every class against 6-D quadrature of eq. 27 (no recurrences, no Boys)."""
    rng = np.random.default_rng(1000 + 64 * ls[0] + 16 * ls[1] + 4 * ls[2] + ls[3])
    ex = np.exp(rng.uniform(math.log(0.3), math.log(3.0), 4))
    X = rng.uniform(-1.2, 1.2, (4, 3))
    blk = oracle.prim_eri_raw(ls[0], ex[0], X[0], ls[1], ex[1], X[1], ls[2], ex[2], X[2], ls[3], ex[3], X[3])
    comps = [cart_components(l) for l in ls]
    scale = np.max(np.abs(blk))
    n_samples = min(blk.size, 6)
    flat = rng.choice(blk.size, size=n_samples, replace=False)
    for f in flat:
        i, j, k, l = np.unravel_index(f, blk.shape)
        ref = eri_quadrature(comps[0][i], ex[0], X[0], comps[1][j], ex[1], X[1],
                             comps[2][k], ex[2], X[2], comps[3][l], ex[3], X[3])
        assert abs(blk[i, j, k, l] - ref) <= 5e-11 * scale + 1e-13, (ls, (i, j, k, l), blk[i, j, k, l], ref)


def test_quadrature_helper_reproduces_closed_form_ssss():
    """The quadrature itself is pinned to eq. 28 so that it is a trustworthy second opinion."""
    a, b, c, d = 0.9, 1.4, 0.6, 2.2
    A, B, C, D = [0.1, 0.2, -0.3], [-0.5, 0.4, 0.6], [0.9, -0.7, 0.2], [0.0, 1.0, -1.0]
    z = (0, 0, 0)
    assert eri_quadrature(z, a, A, z, b, B, z, c, C, z, d, D) == pytest.approx(
        ssss_closed_form(a, A, b, B, c, C, d, D), rel=1e-12)


def test_p_integral_vs_derivative_ladder():
    """Unnormalised p_x = (1/2a) d/dA_x s: central differences of the closed-form (ss|ss)."""
    a, b, c, d = 0.7, 1.1, 0.9, 0.5
    A, B, C, D = np.array([0.1, 0.2, -0.3]), np.array([-0.5, 0.4, 0.6]), np.array([0.9, -0.7, 0.2]), np.array([0.0, 1.0, -1.0])
    blk = oracle.prim_eri_raw(1, a, A, 0, b, B, 0, c, C, 0, d, D)
    for x in range(3):
        h = 1e-4
        e = np.zeros(3); e[x] = h
        f = lambda s: ssss_closed_form(a, A + s * e, b, B, c, C, d, D)
        deriv = (8 * (f(1) - f(-1)) - (f(2) - f(-2))) / (12 * h)
        assert blk[x, 0, 0, 0] == pytest.approx(deriv / (2 * a), rel=1e-8)


# ----------------------------------------------------------------------------- symmetry / inequalities
def test_eightfold_symmetry_and_schwarz_on_config1_shells(cfg1):
    """eq. 46 and eq. 45 on contracted shell quartets covering all l."""
    o = oracle.Oracle(cfg1)
    rng = np.random.default_rng(3)
    for _ in range(12):
        A, B, C, D = (int(x) for x in rng.integers(0, o.nshells, 4))
        g = o.eri_shell_quartet(A, B, C, D)
        assert np.allclose(g, o.eri_shell_quartet(B, A, C, D).transpose(1, 0, 2, 3), rtol=0, atol=1e-13)
        assert np.allclose(g, o.eri_shell_quartet(A, B, D, C).transpose(0, 1, 3, 2), rtol=0, atol=1e-13)
        assert np.allclose(g, o.eri_shell_quartet(C, D, A, B).transpose(2, 3, 0, 1), rtol=0, atol=1e-13)
        gab = o.eri_shell_quartet(A, B, A, B)
        gcd = o.eri_shell_quartet(C, D, C, D)
        dab = np.sqrt(np.abs(np.einsum("ijij->ij", gab)))
        dcd = np.sqrt(np.abs(np.einsum("klkl->kl", gcd)))
        assert np.all(np.abs(g) <= dab[:, :, None, None] * dcd[None, None, :, :] * (1 + 1e-10) + 1e-14)


def test_eri_supermatrix_positive_semidefinite(cfg1):
    """(mu nu|lambda sigma) as an N^2 x N^2 matrix is PSD (s,p cut of config 1)."""
    prob = subset_atoms(cfg1, [0, 1, 2], max_l=1)
    o = oracle.Oracle(prob)
    n, off = o.nbf, o.shell_offsets()
    G = np.zeros((n, n, n, n))
    for A in range(o.nshells):
        for B in range(o.nshells):
            for C in range(o.nshells):
                for D in range(o.nshells):
                    G[off[A]:off[A + 1], off[B]:off[B + 1], off[C]:off[C + 1], off[D]:off[D + 1]] = o.eri_shell_quartet(A, B, C, D)
    M = G.reshape(n * n, n * n)
    assert np.max(np.abs(M - M.T)) < 1e-12
    assert np.min(np.linalg.eigvalsh(M)) > -1e-10
