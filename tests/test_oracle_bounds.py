"""Pins for the oracle's screening quantities: the Schwarz bound of a primitive
shell pair (eq. 45), the density bounds and the per-term rule (eq. 47; DESIGN.md
readings 7 and 8).  Nothing here calls the function under test to produce its own expected value: the bounds are
re-derived in numpy from raw primitive integrals (pinned by quadrature in test_oracle_integrals.py), normalised
coefficients (pinned by S = 1) and component factors written out below."""
import math

import numpy as np
import pytest

import oracle
from refquad import cart_components
from synth import Problem, make_config, subset_atoms
from test_oracle_integrals import ssss_closed_form


def dfact(n):
    r = 1.0
    while n > 1:
        r *= n
        n -= 2
    return r


def comp_factors(l):
    """f(i) = sqrt((2l-1)!! / ((2ix-1)!!(2iy-1)!!(2iz-1)!!)) (reading 3), lexicographic components."""
    return np.array([math.sqrt(dfact(2 * l - 1) / (dfact(2 * ix - 1) * dfact(2 * iy - 1) * dfact(2 * iz - 1)))
                     for (ix, iy, iz) in cart_components(l)])


def _prim_tables(prob, o):
    """Per global primitive: (l, exponent, centre, normalised coefficient, shell)."""
    ct = o.norm_coefs()
    out, g = [], 0
    for s in range(prob.nshells):
        for k in range(int(prob.shell_nprim[s])):
            out.append((int(prob.shell_l[s]), float(prob.exponents[g]), prob.xyz[int(prob.shell_atom[s])], float(ct[g]), s))
            g += 1
    return out


def schwarz_by_definition(la, a, A, ca, lb, b, B, cb):
    """eq. 45 with reading 7: max over components of sqrt|(mu_i nu_j | mu_i nu_j)|, all coefficients included."""
    raw = oracle.prim_eri_raw(la, a, A, lb, b, B, la, a, A, lb, b, B)
    fa, fb = comp_factors(la), comp_factors(lb)
    diag = np.einsum("ijij->ij", raw) * (ca * cb) ** 2 * np.outer(fa, fb) ** 2
    return math.sqrt(np.max(np.abs(diag)))


@pytest.mark.parametrize("n", [1, 2, 4])
def test_schwarz_bound_equals_definition_every_class(n):
    prob = make_config(n)
    if n == 2:
        prob = subset_atoms(prob, [0, 1, 12])
    if n == 4:
        prob = subset_atoms(prob, [0, 1, 49])          # metal (exponents to 1e5, 8-deep contractions) + C + H
    o = oracle.Oracle(prob)
    o.build_pairs(0.0)
    pr = o.pairs()
    prims = _prim_tables(prob, o)
    pstart = np.concatenate([[0], np.cumsum(prob.shell_nprim)])
    rng = np.random.default_rng(45 + n)
    seen = set()
    for cls in range(10):
        idx = np.flatnonzero(pr["cls"] == cls)
        if idx.size == 0:
            continue
        seen.add(cls)
        for x in rng.choice(idx, size=min(50, idx.size), replace=False):
            m = pstart[pr["shellA"][x]] + pr["primA"][x]
            nn = pstart[pr["shellB"][x]] + pr["primB"][x]
            la, a, A, ca, _ = prims[m]
            lb, b, B, cb, _ = prims[nn]
            ref = schwarz_by_definition(la, a, A, ca, lb, b, B, cb)
            assert pr["bound"][x] == pytest.approx(ref, rel=1e-12), (cls, m, nn)
    assert len(seen) == 10


def test_schwarz_bound_ss_closed_form(cfg2):
    """s-s pair: q = c~_m c~_n sqrt((ss|ss)) with (ss|ss) from eq. 28 on the pair with itself."""
    prob = subset_atoms(cfg2, [0, 1, 12, 13])
    o = oracle.Oracle(prob)
    o.build_pairs(0.0)
    pr = o.pairs()
    prims = _prim_tables(prob, o)
    pstart = np.concatenate([[0], np.cumsum(prob.shell_nprim)])
    ss = np.flatnonzero(pr["cls"] == 0)
    assert ss.size > 100
    for x in ss[:: max(1, ss.size // 200)]:
        m = pstart[pr["shellA"][x]] + pr["primA"][x]
        nn = pstart[pr["shellB"][x]] + pr["primB"][x]
        _, a, A, ca, _ = prims[m]
        _, b, B, cb, _ = prims[nn]
        ref = ca * cb * math.sqrt(ssss_closed_form(a, A, b, B, a, A, b, B))
        assert pr["bound"][x] == pytest.approx(ref, rel=1e-12)


def test_all_bounds_equals_pair_list_bounds(cfg2):
    """orc_all_bounds (guard-band helper) indexes candidates hi*(hi+1)/2+lo: tie it to the pinned per-pair bounds."""
    prob = subset_atoms(cfg2, [0, 12])
    o = oracle.Oracle(prob)
    o.build_pairs(0.0)
    pr = o.pairs()
    q_all = o.all_bounds()
    pstart = np.concatenate([[0], np.cumsum(prob.shell_nprim)])
    m = pstart[pr["shellA"]] + pr["primA"]
    n = pstart[pr["shellB"]] + pr["primB"]
    hi, lo = np.maximum(m, n), np.minimum(m, n)
    assert np.array_equal(q_all[hi * (hi + 1) // 2 + lo], pr["bound"])


def test_density_bounds_equal_numpy_block_max():
    """Dm[X][Y] = max |D| over the block; a NON-symmetric D catches swapped axes, signs catch a missing abs."""
    prob = subset_atoms(make_config(2), [0, 12])
    o = oracle.Oracle(prob)
    rng = np.random.default_rng(387)
    D = rng.normal(size=(o.nbf, o.nbf)) * np.exp(rng.uniform(-12, 2, size=(o.nbf, o.nbf)))
    Dm = o.density_bounds(D)
    off = o.shell_offsets()
    ref = np.array([[np.max(np.abs(D[off[X]:off[X + 1], off[Y]:off[Y + 1]])) for Y in range(o.nshells)]
                    for X in range(o.nshells)])
    assert np.array_equal(Dm, ref)
    assert np.all(o.density_bounds(np.zeros_like(D)) == 0.0)


def test_per_term_rule_against_numpy_transcription():
    """eq. 34 / 36 with the per-term rule of eq. 47 (reading 8) written out in numpy over ORDERED
    primitive pairs of a tiny basis (s with 2 primitives, p with 2, d with 1; three centres), at a threshold
    that drops a sizeable part of the terms: J[A_i,B_j] += [..] D[C_k,D_l] iff q_mn q_rs Dm[C,D] >= tau;
    K[A_i,C_k] += [..] D[B_j,D_l] iff q_mn q_rs Dm[B,D] >= tau."""
    rng = np.random.default_rng(47)
    prob = Problem(name="tiny_spd", xyz=np.array([[0.0, 0.0, 0.0], [1.9, 0.3, -0.4], [-0.7, 2.2, 1.1]]),
                   shell_atom=np.array([0, 1, 2], np.int32), shell_l=np.array([0, 1, 2], np.int32),
                   shell_nprim=np.array([2, 2, 1], np.int32), exponents=np.array([3.1, 0.4, 1.7, 0.35, 0.8]),
                   coefficients=np.array([0.6, 0.9, 0.5, 0.8, 1.0]), D=np.zeros((10, 10)), nocc=1, tau_pair=2e-2, tau_jk=2e-3)
    o = oracle.Oracle(prob)
    nkept = o.build_pairs(prob.tau_pair)
    pr = o.pairs()
    assert 0 < nkept < 15                                  # the pair threshold bites
    D = rng.normal(size=(10, 10)) * np.exp(rng.uniform(-6, 0, size=(10, 10)))
    D = D + D.T
    off = o.shell_offsets()
    Dm = np.array([[np.max(np.abs(D[off[X]:off[X + 1], off[Y]:off[Y + 1]])) for Y in range(3)] for X in range(3)])
    prims = _prim_tables(prob, o)
    pstart = np.concatenate([[0], np.cumsum(prob.shell_nprim)])
    ordered = []
    for x in range(nkept):
        m = pstart[pr["shellA"][x]] + pr["primA"][x]
        n = pstart[pr["shellB"][x]] + pr["primB"][x]
        ordered.append((m, n, pr["bound"][x]))
        if m != n:
            ordered.append((n, m, pr["bound"][x]))
    J, K = np.zeros((10, 10)), np.zeros((10, 10))
    dropped = kept = 0
    for (m, n, qb) in ordered:
        la, a, A, ca, sa = prims[m]
        lb, b, B, cb, sb = prims[n]
        for (r, s, qk) in ordered:
            lc, c, C, cc, sc = prims[r]
            ld, d, Dd, cd, sd = prims[s]
            blk = oracle.prim_eri_raw(la, a, A, lb, b, B, lc, c, C, ld, d, Dd) * ca * cb * cc * cd
            blk = blk * comp_factors(la)[:, None, None, None] * comp_factors(lb)[None, :, None, None] \
                * comp_factors(lc)[None, None, :, None] * comp_factors(ld)[None, None, None, :]
            sA, sB, sC, sD = (slice(off[x], off[x + 1]) for x in (sa, sb, sc, sd))
            if qb * qk * Dm[sc, sd] >= prob.tau_jk:
                J[sA, sB] += np.einsum("ijkl,kl->ij", blk, D[sC, sD]); kept += 1
            else:
                dropped += 1
            if qb * qk * Dm[sb, sd] >= prob.tau_jk:
                K[sA, sC] += np.einsum("ijkl,jl->ik", blk, D[sB, sD]); kept += 1
            else:
                dropped += 1
    assert dropped > 20 and kept > 20                      # both branches of the rule are exercised
    J1, K1 = o.jk_o1(D, prob.tau_jk)
    J2, K2, st = o.jk_o2(D, prob.tau_jk)
    assert np.max(np.abs(J1 - J)) < 1e-13 and np.max(np.abs(K1 - K)) < 1e-13
    assert np.max(np.abs(J2 - J)) < 1e-13 and np.max(np.abs(K2 - K)) < 1e-13
    assert st["live_quartets"] < st["visited"]
