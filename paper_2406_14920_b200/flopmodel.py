"""Algorithmic FP64 flop model of one primitive shell quartet (FMA = 2 flops):
McMurchie-Davidson with separable sparse E, 8-fold-unique evaluation, 2 J + 4 K digestions.  This is the
numerator of the "alu" roofline: it cannot be inflated by recomputation."""
import itertools

CLASS_L = [(0, 0), (0, 1), (0, 2), (0, 3), (1, 1), (1, 2), (1, 3), (2, 2), (2, 3), (3, 3)]


def ncart(l):
    return (l + 1) * (l + 2) // 2


def nherm(L):
    return (L + 1) * (L + 2) * (L + 3) // 6


def _comps(l):
    return [(ix, iy, l - ix - iy) for ix in range(l, -1, -1) for iy in range(l - ix, -1, -1)]


def nnz_e(la, lb):
    """Non-zero Hermite coefficients of a pair class: sum over components of prod_tau (i_tau + j_tau + 1)."""
    return sum((a[0] + b[0] + 1) * (a[1] + b[1] + 1) * (a[2] + b[2] + 1) for a in _comps(la) for b in _comps(lb))


def quartet_flops(la, lb, lc, ld):
    """dict(boys, rbuild, eri, digest, total) for one primitive quartet of class (la lb|lc ld)."""
    L1, L2 = la + lb, lc + ld
    L = L1 + L2
    boys = 30 + 2 * (L + 1)
    rbuild = 3 * sum(((n + 1) * (n + 2) // 2) * (L - n + 1) for n in range(1, L + 1))
    nab, ncd = ncart(la) * ncart(lb), ncart(lc) * ncart(ld)
    eri = 2 * nherm(L1) * nnz_e(lc, ld) + 2 * nnz_e(la, lb) * ncd
    digest = 12 * nab * ncd
    return {"boys": boys, "rbuild": rbuild, "eri": eri, "digest": digest, "total": boys + rbuild + eri + digest}


def class_pair_flops(cb, ck):
    (la, lb), (lc, ld) = CLASS_L[cb], CLASS_L[ck]
    return quartet_flops(la, lb, lc, ld)["total"]


def build_flops(quartets):
    """Total model flops of a build from the 10x10 live-quartet matrix returned by te_jk_stats."""
    return float(sum(int(quartets[cb][ck]) * class_pair_flops(cb, ck) for cb in range(10) for ck in range(cb, 10)))
