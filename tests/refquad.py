"""Brute-force numerical quadrature of ONE primitive electron-repulsion integral, eq. 27 (PAPER.md line
173), with unit coefficients.  Uses no McMurchie-Davidson recurrence and no Boys function:

    1/r12 = (2/sqrt(pi)) int_0^inf exp(-u^2 r12^2) du ;

for each u the 6-D integral factorises into three 2-D integrals over (x1, x2) of
polynomial x exp(-quadratic form); each is done EXACTLY by a 14x14 Gauss-Hermite rule in the eigenbasis
of the quadratic form [[p+u^2, -u^2], [-u^2, q+u^2]], and the outer u integral by Gauss-Legendre in t with
u = sqrt(rho) t / sqrt(1-t^2), rho = pq/(p+q).  Pure numpy; test helper only.
"""
import numpy as np

_GH_X, _GH_W = np.polynomial.hermite.hermgauss(14)


def _dim_integral(u, i, a, A, j, b, B, k, c, C, l, d, D):
    """int int (x1-A)^i (x1-B)^j (x2-C)^k (x2-D)^l exp(-a(x1-A)^2 - b(x1-B)^2 - c(x2-C)^2 - d(x2-D)^2
    - u^2 (x1-x2)^2) dx1 dx2 for an array of u."""
    p, q = a + b, c + d
    P, Q = (a * A + b * B) / p, (c * C + d * D) / q
    pre = np.exp(-a * b / p * (A - B) ** 2 - c * d / q * (C - D) ** 2)
    out = np.empty_like(u)
    for n, uu in enumerate(u):
        M = np.array([[p + uu * uu, -uu * uu], [-uu * uu, q + uu * uu]])
        bvec = np.array([p * P, q * Q])
        x0 = np.linalg.solve(M, bvec)
        c0 = p * P * P + q * Q * Q - bvec @ x0
        lam, V = np.linalg.eigh(M)
        y1 = _GH_X / np.sqrt(lam[0])
        y2 = _GH_X / np.sqrt(lam[1])
        w = np.outer(_GH_W, _GH_W) / np.sqrt(lam[0] * lam[1])
        Y1, Y2 = np.meshgrid(y1, y2, indexing="ij")
        x1 = x0[0] + V[0, 0] * Y1 + V[0, 1] * Y2
        x2 = x0[1] + V[1, 0] * Y1 + V[1, 1] * Y2
        poly = (x1 - A) ** i * (x1 - B) ** j * (x2 - C) ** k * (x2 - D) ** l
        out[n] = pre * np.exp(-c0) * np.sum(w * poly)
    return out


def eri_quadrature(ia, a, A, ib, b, B, ic, c, C, id_, d, D, nodes=120, omega=None):
    """(mu nu | lambda sigma) for unnormalised primitives with Cartesian powers ia, ib, ic, id_ (3-tuples).
    omega: long-range operator erf(omega r)/r = (2/sqrt(pi)) int_0^omega exp(-u^2 r^2) du (eq. 32, PAPER.md
    line 222): the same integrand, the outer integral simply stops at u = omega."""
    p, q = a + b, c + d
    rho = p * q / (p + q)
    x, w = np.polynomial.legendre.leggauss(nodes)
    tmax = 1.0 if omega is None else omega / np.sqrt(rho + omega * omega)   # u = omega  <=>  t = tmax
    t = 0.5 * tmax * (x + 1.0)
    w = 0.5 * tmax * w
    u = np.sqrt(rho) * t / np.sqrt(1.0 - t * t)
    du = np.sqrt(rho) * (1.0 - t * t) ** (-1.5)
    f = np.ones_like(u)
    for dim in range(3):
        f = f * _dim_integral(u, ia[dim], a, A[dim], ib[dim], b, B[dim], ic[dim], c, C[dim], id_[dim], d, D[dim])
    return 2.0 / np.sqrt(np.pi) * np.sum(w * du * f)


def nuclear_quadrature(ia, a, A, ib, b, B, C, nodes=160):
    """int mu(r) nu(r) / |r - C| dr for unnormalised primitives (eq. 15, q_C = 1), with
    1/|r-C| = (2/sqrt(pi)) int_0^inf exp(-u^2 |r-C|^2) du: per u three 1-D integrals of polynomial x Gaussian,
    each exact by Gauss-Hermite; outer integral by Gauss-Legendre in t, u = sqrt(p) t / sqrt(1 - t^2)."""
    p = a + b
    x, w = np.polynomial.legendre.leggauss(nodes)
    t = 0.5 * (x + 1.0)
    w = 0.5 * w
    u = np.sqrt(p) * t / np.sqrt(1.0 - t * t)
    du = np.sqrt(p) * (1.0 - t * t) ** (-1.5)
    f = np.ones_like(u)
    for dim in range(3):
        Ax, Bx, Cx, i, j = A[dim], B[dim], C[dim], ia[dim], ib[dim]
        g = np.empty_like(u)
        for n, uu in enumerate(u):
            s_ = p + uu * uu                                  # exponent of the product Gaussian
            x0 = (a * Ax + b * Bx + uu * uu * Cx) / s_
            c0 = a * Ax * Ax + b * Bx * Bx + uu * uu * Cx * Cx - s_ * x0 * x0
            xs = x0 + _GH_X / np.sqrt(s_)
            g[n] = np.exp(-c0) * np.sum(_GH_W * (xs - Ax) ** i * (xs - Bx) ** j) / np.sqrt(s_)
        f = f * g
    return 2.0 / np.sqrt(np.pi) * np.sum(w * du * f)


def cart_components(l):
    """Lexicographic component order, x^l first (reading 4)."""
    return [(ix, iy, l - ix - iy) for ix in range(l, -1, -1) for iy in range(l - ix, -1, -1)]
