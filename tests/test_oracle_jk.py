"""Pins for the oracle's J/K builds (eq. 34, 36, 45-47): the symmetry-unique production oracle O2 against the
definition O1, both against a dense einsum over the explicit ERI tensor, plus invariants that no indexing
or sign mistake survives."""
import numpy as np
import pytest

import oracle
from synth import Problem, make_config, subset_atoms


_G_CACHE = {}


def dense_jk(o, D):
    """J, K by eq. 34 / 36 from the full contracted ERI tensor (no screening, no symmetry)."""
    n, off = o.nbf, o.shell_offsets()
    key = (n, o.ex.tobytes(), o.xyz.tobytes())
    if key in _G_CACHE:
        G = _G_CACHE[key]
        return np.einsum("ijkl,kl->ij", G, D), np.einsum("ijkl,jl->ik", G, D)
    G = _G_CACHE[key] = np.zeros((n, n, n, n))
    for A in range(o.nshells):
        for B in range(o.nshells):
            for C in range(o.nshells):
                for Dd in range(o.nshells):
                    G[off[A]:off[A + 1], off[B]:off[B + 1], off[C]:off[C + 1], off[Dd]:off[Dd + 1]] = \
                        o.eri_shell_quartet(A, B, C, Dd)
    return np.einsum("ijkl,kl->ij", G, D), np.einsum("ijkl,jl->ik", G, D)


@pytest.fixture(scope="module")
def small():
    """2 atoms of config 1: all of s,p,d,f, 3 primitives each, nbf = 40."""
    return subset_atoms(make_config(1), [0, 1])


def test_o1_and_o2_equal_dense_einsum(small):
    o = oracle.Oracle(small)
    o.build_pairs(0.0)
    Jd, Kd = dense_jk(o, small.D)
    J1, K1 = o.jk_o1(small.D, 0.0)
    J2, K2, st = o.jk_o2(small.D, 0.0)
    npair = o.npairs
    assert st["live_quartets"] == npair * (npair + 1) // 2
    for X, Y in ((J1, Jd), (K1, Kd), (J2, Jd), (K2, Kd)):
        assert np.max(np.abs(X - Y)) < 1e-12
    assert np.max(np.abs(J2 - J2.T)) < 1e-13 and np.max(np.abs(K2 - K2.T)) < 1e-13


def test_nonsymmetric_D_exposes_index_conventions(small):
    """O1 takes eq. 34/36 literally, so it must match the dense einsum even for a NON-symmetric D
    (a transposed operand would not)."""
    o = oracle.Oracle(small)
    o.build_pairs(0.0)
    rng = np.random.default_rng(5)
    D = rng.normal(size=(o.nbf, o.nbf))
    G_J, G_K = dense_jk(o, D)
    J1, K1 = o.jk_o1(D, 0.0)
    assert np.max(np.abs(J1 - G_J)) < 1e-11
    assert np.max(np.abs(K1 - G_K)) < 1e-11


@pytest.mark.parametrize("n", [2, 3, 4])
def test_o2_equals_o1_with_screening_on_cuts(n):
    """Same per-term rule in both forms (reading 8) => identical term sets, thresholds 1e-12."""
    full = make_config(n)
    ids = {2: [0, 1, 12, 13], 3: [0, 1, 2, 3, 4, 5], 4: [0, 1, 2, 49]}[n]
    prob = subset_atoms(full, ids, max_l=(2 if n == 4 else None))
    o = oracle.Oracle(prob)
    o.build_pairs(prob.tau_pair)
    J1, K1 = o.jk_o1(prob.D, prob.tau_jk)
    J2, K2, st = o.jk_o2(prob.D, prob.tau_jk)
    scale = max(1.0, np.max(np.abs(J1)))
    assert np.max(np.abs(J1 - J2)) < 1e-12 * scale
    assert np.max(np.abs(K1 - K2)) < 1e-12 * scale
    assert st["live_quartets"] <= st["visited"]


def test_sampled_blocks_equal_full_build(small):
    o = oracle.Oracle(small)
    o.build_pairs(0.0)
    J2, K2, _ = o.jk_o2(small.D, 0.0)
    off = o.shell_offsets()
    for (A, B) in [(0, 5), (3, 2), (7, 7)]:
        assert np.max(np.abs(o.j_block(small.D, 0.0, A, B) - J2[off[A]:off[A + 1], off[B]:off[B + 1]])) < 1e-12
        assert np.max(np.abs(o.k_block(small.D, 0.0, A, B) - K2[off[A]:off[A + 1], off[B]:off[B + 1]])) < 1e-12


def test_trace_positivity_and_linearity(small):
    o = oracle.Oracle(small)
    o.build_pairs(0.0)
    D = small.D
    J, K, _ = o.jk_o2(D, 0.0)
    assert np.sum(D * J) > 0 and np.sum(D * K) > 0
    rng = np.random.default_rng(11)
    X = rng.normal(size=D.shape); X = X + X.T
    Jx, Kx, _ = o.jk_o2(X, 0.0)
    assert np.sum(X * Jx) >= 0          # Tr(XJ[X]) >= 0 for any symmetric X (Coulomb self-energy)
    Js, Ks, _ = o.jk_o2(D + 0.5 * X, 0.0)
    assert np.max(np.abs(Js - (J + 0.5 * Jx))) < 1e-11
    assert np.max(np.abs(Ks - (K + 0.5 * Kx))) < 1e-11


def _moved(prob, R=None, shift=None):
    xyz = prob.xyz.copy()
    if R is not None:
        xyz = xyz @ R.T
    if shift is not None:
        xyz = xyz + shift
    return Problem(**{**prob.__dict__, "xyz": xyz})


def test_translation_invariance(small):
    o = oracle.Oracle(small); o.build_pairs(0.0)
    J, K, _ = o.jk_o2(small.D, 0.0)
    m = _moved(small, shift=np.array([3.1, -2.7, 0.9]))
    om = oracle.Oracle(m); om.build_pairs(0.0)
    Jm, Km, _ = om.jk_o2(small.D, 0.0)
    assert np.max(np.abs(J - Jm)) < 1e-11 and np.max(np.abs(K - Km)) < 1e-11


def test_rotation_invariance_with_inverse_overlap_density(small):
    """With D = S^-1 the scalars Tr(D J[D]) and Tr(D K[D]) depend only on the SPACE spanned by the basis;
    full Cartesian shells span rotation-invariant spaces, so a rigid rotation leaves them unchanged."""
    prob = subset_atoms(make_config(1), [0, 1, 2], max_l=2)
    rng = np.random.default_rng(2)
    Q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    if np.linalg.det(Q) < 0:
        Q[:, 0] *= -1
    vals = []
    for p in (prob, _moved(prob, R=Q)):
        o = oracle.Oracle(p); o.build_pairs(0.0)
        Sinv = np.linalg.inv(o.overlap())
        Sinv = 0.5 * (Sinv + Sinv.T)
        J, K, _ = o.jk_o2(Sinv, 0.0)
        vals.append((np.sum(Sinv * J), np.sum(Sinv * K)))
    assert vals[0][0] == pytest.approx(vals[1][0], rel=1e-10)
    assert vals[0][1] == pytest.approx(vals[1][1], rel=1e-10)


def test_axis_permutation_rotation_permutes_components():
    """Exact 90-degree rotation (x,y,z)->(y,z,x): Tr(DJ), Tr(DK) with the component-permuted D are unchanged."""
    prob = subset_atoms(make_config(1), [0, 1], max_l=2)
    R = np.array([[0, 1, 0], [0, 0, 1], [1, 0, 0]], dtype=float)   # new = R @ old: x'=y, y'=z, z'=x
    o = oracle.Oracle(prob); o.build_pairs(0.0)
    J, K, _ = o.jk_o2(prob.D, 0.0)
    # x = z', y = x', z = y'  =>  old component (ix,iy,iz) is new component (iy,iz,ix)
    from refquad import cart_components
    perm = np.zeros(o.nbf, dtype=int)
    off = o.shell_offsets()
    for s in range(o.nshells):
        comps = cart_components(int(prob.shell_l[s]))
        for i, (ix, iy, iz) in enumerate(comps):
            perm[off[s] + comps.index((iy, iz, ix))] = off[s] + i
    Dp = prob.D[np.ix_(perm, perm)]
    pm = _moved(prob, R=R)
    om = oracle.Oracle(pm); om.build_pairs(0.0)
    Jm, Km, _ = om.jk_o2(Dp, 0.0)
    assert np.max(np.abs(Jm - J[np.ix_(perm, perm)])) < 1e-11
    assert np.max(np.abs(Km - K[np.ix_(perm, perm)])) < 1e-11


def test_pair_list_is_canonical_and_thresholded(cfg2):
    prob = subset_atoms(cfg2, [0, 1, 2, 12, 13, 14])
    o = oracle.Oracle(prob)
    n = o.build_pairs(1e-12)
    pr = o.pairs()
    assert n == len(pr["cls"]) and np.all(pr["bound"] >= 1e-12)
    q_all = o.all_bounds()
    assert n == int(np.sum(q_all >= 1e-12))
    key = list(zip(pr["cls"], pr["shellA"], pr["primA"], pr["shellB"], pr["primB"]))
    assert key == sorted(key) and len(set(key)) == n
    la, lb = prob.shell_l[pr["shellA"]], prob.shell_l[pr["shellB"]]
    assert np.all(la <= lb)
    base = np.array([0, 4, 7, 9])
    assert np.all(pr["cls"] == base[la] + (lb - la))
