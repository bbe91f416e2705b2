"""Pins for the two SURVEY.md 8f rows the oracle gained in round 2: long-range erf(omega r)/r integrals (eq. 32-33,
P:220-237) and nuclear-attraction integrals (eq. 14-26).  Expected values come from closed forms, limits
and brute-force quadrature (tests/refquad.py), never from the function under test."""
import math

import numpy as np
import pytest
from scipy import special

import oracle
from refquad import cart_components, eri_quadrature, nuclear_quadrature
from synth import Problem, make_config, subset_atoms
from test_oracle_bounds import comp_factors
from test_oracle_integrals import QUAD_CASES, ssss_closed_form


# ------------------------------------------------------------------------------------ long-range ERIs
def ssss_lr_closed_form(a, A, b, B, c, C, d, D, w):
    """Attenuated (ss|ss): eq. 33 at zero angular momentum: K_ab K_cd 2 pi^{5/2} w / (p q sqrt(pq + (p+q) w^2))
    F_0(pq w^2 / (pq + (p+q) w^2) |PQ|^2), F_0(T) = (1/2) sqrt(pi/T) erf(sqrt T)."""
    A, B, C, D = map(np.asarray, (A, B, C, D))
    p, q = a + b, c + d
    P, Q = (a * A + b * B) / p, (c * C + d * D) / q
    den = p * q + (p + q) * w * w
    T = p * q * w * w / den * np.sum((P - Q) ** 2)
    F0 = 1.0 if T == 0 else 0.5 * math.sqrt(math.pi / T) * special.erf(math.sqrt(T))
    return (math.exp(-a * b / p * np.sum((A - B) ** 2)) * math.exp(-c * d / q * np.sum((C - D) ** 2))
            * 2 * math.pi ** 2.5 * w / (p * q * math.sqrt(den)) * F0)


def test_lr_ssss_closed_form_random():
    rng = np.random.default_rng(33)
    for _ in range(50):
        ex = np.exp(rng.uniform(math.log(0.05), math.log(50), 4))
        X = rng.uniform(-2.5, 2.5, (4, 3))
        w = float(np.exp(rng.uniform(math.log(0.05), math.log(5.0))))
        v = oracle.prim_eri_raw(0, ex[0], X[0], 0, ex[1], X[1], 0, ex[2], X[2], 0, ex[3], X[3], omega=w).ravel()[0]
        assert v == pytest.approx(ssss_lr_closed_form(ex[0], X[0], ex[1], X[1], ex[2], X[2], ex[3], X[3], w), rel=2e-14)


def test_lr_one_centre_value_and_limits():
    """Four identical normalised s primitives of exponent a on one centre: the (ss|ss) value 2 sqrt(a/pi) is scaled by
    w / sqrt(a + w^2) (p = q = 2a, T = 0); w -> 0 gives no repulsion, w -> infinity the full-range eq. 28."""
    a = 0.8
    N = (2 * a / math.pi) ** 0.75
    z = [0.0, 0.0, 0.0]
    for w in (0.1, 0.33, 2.0, 40.0):
        v = oracle.prim_eri_raw(0, a, z, 0, a, z, 0, a, z, 0, a, z, omega=w).ravel()[0] * N ** 4
        assert v == pytest.approx(2 * math.sqrt(a / math.pi) * w / math.sqrt(a + w * w), rel=1e-14)


@pytest.mark.parametrize("ls", [(1, 0, 2, 1), (3, 2, 1, 3), (3, 3, 3, 3), (0, 2, 0, 2)])
def test_lr_large_omega_recovers_full_range(ls):
    rng = np.random.default_rng(320 + sum(ls))
    ex = np.exp(rng.uniform(math.log(0.3), math.log(3.0), 4))
    X = rng.uniform(-1.2, 1.2, (4, 3))
    args = (ls[0], ex[0], X[0], ls[1], ex[1], X[1], ls[2], ex[2], X[2], ls[3], ex[3], X[3])
    full = oracle.prim_eri_raw(*args)
    lr = oracle.prim_eri_raw(*args, omega=1e8)     # alpha_w = alpha (1 - alpha/w^2 ...): relative change ~1e-16
    assert np.max(np.abs(lr - full)) <= 1e-12 * np.max(np.abs(full))
    half = oracle.prim_eri_raw(*args, omega=0.4)
    assert np.max(np.abs(half - full)) > 1e-3 * np.max(np.abs(full))      # the operator really changes


@pytest.mark.parametrize("ls", QUAD_CASES[::2])
def test_lr_primitive_block_vs_bruteforce_quadrature(ls):
    """eq. 32 by quadrature: erf(w r)/r = (2/sqrt pi) int_0^w exp(-u^2 r^2) du, no recurrences, no Boys."""
    rng = np.random.default_rng(3200 + 64 * ls[0] + 16 * ls[1] + 4 * ls[2] + ls[3])
    ex = np.exp(rng.uniform(math.log(0.3), math.log(3.0), 4))
    X = rng.uniform(-1.2, 1.2, (4, 3))
    w = float(rng.uniform(0.2, 1.5))
    blk = oracle.prim_eri_raw(ls[0], ex[0], X[0], ls[1], ex[1], X[1], ls[2], ex[2], X[2], ls[3], ex[3], X[3], omega=w)
    comps = [cart_components(l) for l in ls]
    scale = np.max(np.abs(blk))
    for f in rng.choice(blk.size, size=min(blk.size, 5), replace=False):
        i, j, k, l = np.unravel_index(f, blk.shape)
        ref = eri_quadrature(comps[0][i], ex[0], X[0], comps[1][j], ex[1], X[1], comps[2][k], ex[2], X[2],
                             comps[3][l], ex[3], X[3], omega=w)
        assert abs(blk[i, j, k, l] - ref) <= 5e-11 * scale + 1e-13, (ls, (i, j, k, l), blk[i, j, k, l], ref)


def test_lr_jk_builds_o1_o2_dense():
    """J/K with the long-range operator: O2 == O1 == dense einsum over long-range shell blocks assembled from
    prim_eri_raw(omega) in numpy; pair list / Schwarz bounds unchanged by omega (reading 20)."""
    prob = subset_atoms(make_config(1), [0, 1], max_l=2)
    w = 0.33
    o = oracle.Oracle(prob)
    n0 = o.build_pairs(0.0)
    q0 = o.pairs()["bound"].copy()
    o.set_omega(w)
    assert o.build_pairs(0.0) == n0 and np.array_equal(o.pairs()["bound"], q0)
    J1, K1 = o.jk_o1(prob.D, 0.0)
    J2, K2, _ = o.jk_o2(prob.D, 0.0)
    ct = o.norm_coefs()
    off = o.shell_offsets()
    pstart = np.concatenate([[0], np.cumsum(prob.shell_nprim)])
    n = o.nbf
    G = np.zeros((n, n, n, n))
    sh = [(int(prob.shell_l[s]), prob.xyz[int(prob.shell_atom[s])], range(pstart[s], pstart[s + 1])) for s in range(prob.nshells)]
    for A, (la, XA, pa) in enumerate(sh):
        for B, (lb, XB, pb) in enumerate(sh):
            for Cc, (lc, XC, pc) in enumerate(sh):
                for Dd, (ld, XD, pd) in enumerate(sh):
                    blk = 0.0
                    for m in pa:
                        for nn in pb:
                            for r in pc:
                                for s in pd:
                                    blk = blk + ct[m] * ct[nn] * ct[r] * ct[s] * oracle.prim_eri_raw(
                                        la, prob.exponents[m], XA, lb, prob.exponents[nn], XB,
                                        lc, prob.exponents[r], XC, ld, prob.exponents[s], XD, omega=w)
                    blk = blk * comp_factors(la)[:, None, None, None] * comp_factors(lb)[None, :, None, None] \
                        * comp_factors(lc)[None, None, :, None] * comp_factors(ld)[None, None, None, :]
                    G[off[A]:off[A + 1], off[B]:off[B + 1], off[Cc]:off[Cc + 1], off[Dd]:off[Dd + 1]] = blk
    Jd, Kd = np.einsum("ijkl,kl->ij", G, prob.D), np.einsum("ijkl,jl->ik", G, prob.D)
    for X, Y in ((J1, Jd), (K1, Kd), (J2, Jd), (K2, Kd)):
        assert np.max(np.abs(X - Y)) < 1e-12
    o.set_omega(0.0)
    J0, K0, _ = o.jk_o2(prob.D, 0.0)
    assert np.max(np.abs(J0 - J2)) > 1e-3            # and the full-range build is restored by omega = 0
    # Coulomb self-energy ordering: the long-range operator is a positive kernel below 1/r
    assert 0 < np.sum(prob.D * J2) < np.sum(prob.D * J0)


# --------------------------------------------------------------------------------- nuclear attraction
def _one_pair_problem(la, a, A, lb, b, B):
    return Problem(name="pair", xyz=np.array([A, B], dtype=float), shell_atom=np.array([0, 1], np.int32),
                   shell_l=np.array([la, lb], np.int32), shell_nprim=np.array([1, 1], np.int32),
                   exponents=np.array([a, b]), coefficients=np.array([1.0, 1.0]), D=np.zeros((1, 1)), nocc=1,
                   tau_pair=0.0, tau_jk=0.0)


def test_nuclear_ss_closed_form():
    """eq. 17: V_ssC = q_C C_mu C_nu exp(-ab/p |AB|^2) (2 pi / p) F_0(p |PC|^2)."""
    rng = np.random.default_rng(17)
    for _ in range(20):
        a, b = np.exp(rng.uniform(math.log(0.1), math.log(20), 2))
        A, B, C = rng.uniform(-2, 2, (3, 3))
        qc = float(rng.uniform(-8, 3))
        o = oracle.Oracle(_one_pair_problem(0, a, A, 0, b, B))
        o.build_pairs(0.0)
        V = o.nuclear_attraction([C], [qc])
        ct = o.norm_coefs()
        p = a + b
        P = (a * A + b * B) / p
        T = p * np.sum((P - C) ** 2)
        F0 = 0.5 * math.sqrt(math.pi / T) * special.erf(math.sqrt(T))
        ref = qc * ct[0] * ct[1] * math.exp(-a * b / p * np.sum((A - B) ** 2)) * 2 * math.pi / p * F0
        assert V[0, 1] == pytest.approx(ref, rel=1e-13) and V[1, 0] == V[0, 1]


@pytest.mark.parametrize("la,lb", [(0, 1), (1, 1), (0, 2), (2, 1), (2, 2), (0, 3), (1, 3), (3, 2), (3, 3)])
def test_nuclear_vs_bruteforce_quadrature(la, lb):
    rng = np.random.default_rng(140 + 4 * la + lb)
    a, b = np.exp(rng.uniform(math.log(0.3), math.log(3.0), 2))
    A, B = rng.uniform(-1.0, 1.0, (2, 3))
    Cs = rng.uniform(-1.5, 1.5, (3, 3))
    qs = np.array([-1.0, 2.5, -0.3])
    o = oracle.Oracle(_one_pair_problem(la, a, A, lb, b, B))
    o.build_pairs(0.0)
    V = o.nuclear_attraction(Cs, qs)
    ct = o.norm_coefs()
    ca, cb = cart_components(la), cart_components(lb)
    fa, fb = comp_factors(la), comp_factors(lb)
    nA = len(ca)
    blk = V[:nA, nA:]
    scale = np.max(np.abs(blk))
    for f in rng.choice(blk.size, size=min(blk.size, 6), replace=False):
        i, j = np.unravel_index(f, blk.shape)
        ref = sum(q * nuclear_quadrature(ca[i], a, A, cb[j], b, B, C) for q, C in zip(qs, Cs)) * ct[0] * ct[1] * fa[i] * fb[j]
        assert abs(blk[i, j] - ref) <= 5e-11 * scale + 1e-13, ((la, lb), (i, j), blk[i, j], ref)
    assert np.max(np.abs(V - V.T)) < 1e-15


def test_nuclear_equals_tight_s_charge_limit_of_eri():
    """A point charge is the limit of a normalised s charge distribution: V_mu,nu,C = lim_{g->inf}
    (mu nu | s_g s_g) / (pi/2g)^{3/2} with both ket primitives at C (the ERI code is pinned by quadrature)."""
    rng = np.random.default_rng(26)
    la, lb = 2, 3
    a, b = 0.9, 1.3
    A, B, C = rng.uniform(-1.0, 1.0, (3, 3))
    o = oracle.Oracle(_one_pair_problem(la, a, A, lb, b, B))
    o.build_pairs(0.0)
    V = o.nuclear_attraction([C], [1.0])
    ct = o.norm_coefs()
    g = 1e12
    raw = oracle.prim_eri_raw(la, a, A, lb, b, B, 0, g, C, 0, g, C)[:, :, 0, 0] / (math.pi / (2 * g)) ** 1.5
    ref = raw * ct[0] * ct[1] * np.outer(comp_factors(la), comp_factors(lb))
    assert np.max(np.abs(V[:6, 6:] - ref)) <= 1e-10 * np.max(np.abs(ref))


def test_nuclear_contracted_basis_invariants(cfg2):
    """Contracted shells, same-shell pairs (m != n mirrored, m == n once), linearity in the charges, translation."""
    prob = subset_atoms(cfg2, [0, 1, 12])
    o = oracle.Oracle(prob)
    o.build_pairs(0.0)
    C = prob.xyz.copy()
    q = np.array([-6.0, -6.0, -1.0])
    V = o.nuclear_attraction(C, q)
    assert np.max(np.abs(V - V.T)) < 1e-13
    assert np.all(np.linalg.eigvalsh(V) < 0)                       # attraction by negative charges: negative definite
    V1 = o.nuclear_attraction(C[:1], q[:1]) + o.nuclear_attraction(C[1:], q[1:])
    assert np.max(np.abs(V - V1)) < 1e-12
    shift = np.array([2.0, -1.0, 0.5])
    pm = Problem(**{**prob.__dict__, "xyz": prob.xyz + shift})
    om = oracle.Oracle(pm)
    om.build_pairs(0.0)
    assert np.max(np.abs(om.nuclear_attraction(C + shift, q) - V)) < 1e-11
    # diagonal s function, single centre, by quadrature-free closed form: <s|1/r|s> over contracted normalised s
    #   = sum_mn c~_m c~_n (2 pi / p) (normalised primitives share the centre, T = 0, F_0 = 1)
    ct = o.norm_coefs()
    n0 = int(prob.shell_nprim[0])
    ex = prob.exponents[:n0]
    ref = q[0] * sum(ct[m] * ct[n] * 2 * math.pi / (ex[m] + ex[n]) for m in range(n0) for n in range(n0))
    assert o.nuclear_attraction(C[:1], q[:1])[0, 0] == pytest.approx(ref, rel=1e-13)
