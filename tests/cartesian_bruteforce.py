"""Brute-force evaluation of a P0 element from the UNREDUCED Cartesian form (A7)
(PAPER.md:416): integrals over q, q' and x with the theta-functions kept as they
are printed.  Used only to pin the oracle; shares nothing with oracle/ or the
CUDA path (different variables, no polar transform, no F of (A14)).

  element = (d_i dbar_j d_i' dbar_j')^{-1/2} sum_terms g
            int_a^b dq int_c^d dq' int_{-1}^{1} dx q^{A+1} q'^{B+1} / (pi1^{l'+1} pi2^{l+1})
            P_k(x) theta(pi1 in [L1,U1]) theta(pi2 in [L2,U2])
with A = l1+l1', B = l2+l2' (reading R1 of DESIGN.md).  For fixed (q,q') the
theta-product restricts x to one interval in closed form, because pi1^2 and pi2^2
are linear in x; the x-integral is then a 24-point Gauss rule on that interval and
(q,q') is a composite midpoint grid.
"""
import numpy as np
from numpy.polynomial.legendre import leggauss, legval


def element(a, b, c, d, L1, U1, L2, U2, l, lp, terms, m=240, modulus=False):
    """terms: [(k, l1, l1', g)].  m x m midpoint cells in (q,q').
    modulus=True: every term's integrand is replaced by its modulus (|g| |P_k(x)|, everything else in (A7) is positive):
    the absolute term sum that the oracle reports as `absval` (the scale A_e of DESIGN.md R9)."""
    hq, hqp = (b - a) / m, (d - c) / m
    q = a + (np.arange(m) + 0.5) * hq
    qp = c + (np.arange(m) + 0.5) * hqp
    Q, QP = np.meshgrid(q, qp, indexing="ij")
    e1 = Q * Q + 0.25 * QP * QP
    e2 = 0.25 * Q * Q + QP * QP
    qq = Q * QP
    x_lo = np.maximum(-1.0, np.maximum((L1 * L1 - e1) / qq, (L2 * L2 - e2) / qq))
    x_hi = np.minimum(1.0, np.minimum((U1 * U1 - e1) / qq, (U2 * U2 - e2) / qq))
    ok = x_hi > x_lo
    xi, w = leggauss(24)
    half = np.where(ok, 0.5 * (x_hi - x_lo), 0.0)
    mid = 0.5 * (x_hi + x_lo)
    total = 0.0
    for r in range(len(xi)):
        x = np.where(ok, mid + half * xi[r], 0.0)
        pi1 = np.sqrt(np.maximum(e1 + qq * x, 1e-300))
        pi2 = np.sqrt(np.maximum(e2 + qq * x, 1e-300))
        G = np.zeros_like(x)
        for (k, l1, l1p, g) in terms:
            A = l1 + l1p
            B = (l - l1) + (lp - l1p)
            Pk = legval(x, [0.0] * k + [1.0])
            G += (abs(g) * np.abs(Pk) if modulus else g * Pk) * Q ** (A + 1) * QP ** (B + 1)
        total += np.sum(w[r] * half * G / (pi1 ** (lp + 1) * pi2 ** (l + 1)))
    return total * hq * hqp / np.sqrt((U2 - L2) * (b - a) * (U1 - L1) * (d - c))


def hits(a, b, c, d, L1, U1, L2, U2, m=64):
    """Does any point of an m x m interior sample of the (q,q') rectangle admit an x in
    (-1,1) with pi1 in (L1,U1) and pi2 in (L2,U2)?  (theta-product of A7.)"""
    q = a + (np.arange(m) + 0.5) * (b - a) / m
    qp = c + (np.arange(m) + 0.5) * (d - c) / m
    Q, QP = np.meshgrid(q, qp, indexing="ij")
    e1 = Q * Q + 0.25 * QP * QP
    e2 = 0.25 * Q * Q + QP * QP
    qq = Q * QP
    x_lo = np.maximum(-1.0, np.maximum((L1 * L1 - e1) / qq, (L2 * L2 - e2) / qq))
    x_hi = np.minimum(1.0, np.minimum((U1 * U1 - e1) / qq, (U2 * U2 - e2) / qq))
    return bool(np.any(x_hi > x_lo))
