"""Channel enumeration and algebraic coefficients g of (A4) for the oracle.

TEST INFRASTRUCTURE (see oracle/__init__.py).

Channels: PAPER.md:98-102 (eq. 5): alpha={l,s,j}, beta={lambda,I}, Gamma={J,pi,T};
"the sum l+s+t must be odd"; j <= j_max.
Coefficients: PAPER.md:395 (A4) in the reading of DESIGN.md R1/R2 (labels of A3
vs A4 and the garbled brackets), i.e.

  g^{l1 l1' k}_{gamma gamma'} =
     - sqrt(l^ s^ j^ t^ lam^ I^  l'^ s'^ j'^ t'^ lam'^ I'^)  {1/2 1/2 t; 1/2 T t'}
       * sum_{L,S} L^ S^ {1/2 1/2 s; 1/2 S s'} 9j{l s j; lam 1/2 I; L S J} 9j{l' s' j'; lam' 1/2 I'; L S J}
       * k^ (1/2)^{l2'+l1} sqrt((2l+1)!/((2l1)!(2l2)!)) sqrt((2l'+1)!/((2l1')!(2l2')!))
       * sum_{f,f'} {l1' l2' l'; lam' L f'} {l2 l1 l; lam L f} <l2' 0 lam' 0|f' 0> <l1 0 lam 0|f 0>
                    {f' l1' L; f l2 k} <k 0 l1' 0|f 0> <k 0 l2 0|f' 0>,
  x^ = 2x+1,  l1+l2 = l,  l1'+l2' = l',

multiplying the monomial q^{l1+l1'} q'^{l2+l2'} P_k(x) in (A3) (R1).

Pins (tests/test_oracle_channels.py): 18 channels for J=1/2, j<=2;
s-wave collapse to the textbook doublet/quartet recoupling values; vanishing
order G = O(p^l p'^l') at pi2 -> 0 / pi1 -> 0; G_{gg'}(q,q',x) = G_{g'g}(q',q,x); the
orbital part against a brute-force overlap of bipolar spherical harmonics of the
vectors p = q/2 + q', p' = q + q'/2 (fixes labels, powers of 1/2, the k-range); and, for every factor at
once, the spectrum of the multichannel lattice matrix, which must lie in [-1, 2] and approach both ends
(tests/test_oracle_perm.py::test_multichannel_spectrum_bound).  Parity unpinned: only the relative PHASE
convention between channels (a diagonal +-1 similarity of P0), which needs ref. [11]'s potential matrix.
"""
from math import factorial, sqrt

from .wigner import cg000, nine_j, six_j

MODEL_SPINLESS_SWAVE = 0
MODEL_ND = 1


def enumerate_channels(two_J, parity, j_max):
    """Channels (l, s, j, t, lam, two_I) for total (J, parity), pair j <= j_max.

    Order (the contract order, restated in include/wpcd.h): ascending j, then s,
    then l, then two_I, then lam.  parity is +1 or -1; (-1)^(l+lam) == parity.
    """
    out = []
    for j in range(0, j_max + 1):
        for s in (0, 1):
            for l in range(abs(j - s), j + s + 1):
                t = 1 - ((l + s) % 2)  # l+s+t odd
                for two_I in range(abs(two_J - 2 * j), two_J + 2 * j + 1, 2):
                    for lam in ((two_I - 1) // 2, (two_I + 1) // 2):
                        if lam < 0:
                            continue
                        if (1 if (l + lam) % 2 == 0 else -1) != parity:
                            continue
                        out.append((l, s, j, t, lam, two_I))
    return out


def orbital_coefficient(l, lam, lp, lamp, L, l1, l1p, k):
    """Orbital (third and following lines) part of (A4) for one total orbital momentum L:
    k^ (1/2)^{l2'+l1} sqrt(..) sqrt(..) sum_{ff'} {..}{..}<..><..>{..}<..><..>."""
    l2 = l - l1
    l2p = lp - l1p
    ff = 0.0
    for f in range(abs(l1 - lam), l1 + lam + 1):
        c_f = cg000(l1, lam, f)
        c_kf = cg000(k, l1p, f)
        sj_f = six_j(2 * l2, 2 * l1, 2 * l, 2 * lam, 2 * L, 2 * f)
        if c_f == 0.0 or c_kf == 0.0 or sj_f == 0.0:
            continue
        for fp in range(abs(l2p - lamp), l2p + lamp + 1):
            c_fp = cg000(l2p, lamp, fp)
            c_kfp = cg000(k, l2, fp)
            if c_fp == 0.0 or c_kfp == 0.0:
                continue
            ff += (
                six_j(2 * l1p, 2 * l2p, 2 * lp, 2 * lamp, 2 * L, 2 * fp) * sj_f * c_fp * c_f
                * six_j(2 * fp, 2 * l1p, 2 * L, 2 * f, 2 * l2, 2 * k) * c_kf * c_kfp
            )
    return (
        (2 * k + 1) * 0.5 ** (l2p + l1)
        * sqrt(factorial(2 * l + 1) / (factorial(2 * l1) * factorial(2 * l2)))
        * sqrt(factorial(2 * lp + 1) / (factorial(2 * l1p) * factorial(2 * l2p)))
        * ff
    )


def g_coefficient(ch, chp, two_J, two_T, l1, l1p, k):
    """One coefficient g^{l1 l1' k}_{gamma gamma'} of (A4); ch = gamma (row, unprimed),
    chp = gamma' (column, primed)."""
    l, s, j, t, lam, two_I = ch
    lp, sp, jp, tp, lamp, two_Ip = chp
    hat = lambda x: 2 * x + 1
    pref = -sqrt(
        hat(l) * hat(s) * hat(j) * hat(t) * hat(lam) * (two_I + 1)
        * hat(lp) * hat(sp) * hat(jp) * hat(tp) * hat(lamp) * (two_Ip + 1)
    )
    iso = six_j(1, 1, 2 * t, 1, two_T, 2 * tp)
    if iso == 0.0:
        return 0.0
    total = 0.0
    for L in range(max(abs(l - lam), abs(lp - lamp)), min(l + lam, lp + lamp) + 1):
        for two_S in (1, 3):
            spin = six_j(1, 1, 2 * s, 1, two_S, 2 * sp)
            if spin == 0.0:
                continue
            nj = nine_j(2 * l, 2 * s, 2 * j, 2 * lam, 1, two_I, 2 * L, two_S, two_J)
            if nj == 0.0:
                continue
            njp = nine_j(2 * lp, 2 * sp, 2 * jp, 2 * lamp, 1, two_Ip, 2 * L, two_S, two_J)
            if njp == 0.0:
                continue
            total += (2 * L + 1) * (two_S + 1) * spin * nj * njp * orbital_coefficient(l, lam, lp, lamp, L, l1, l1p, k)
    return pref * iso * total


def g_table(channels, two_J, two_T, zero_tol=1e-14):
    """All coupled channel pairs and their nonzero terms.

    Returns a list of (gamma, gamma', [(k, l1, l1', g), ...]) sorted by (gamma, gamma');
    terms in ascending (l1, l1', k); a pair whose every |g| <= zero_tol is not coupled
    and is left out (R13).  k runs over 0 .. min(l1+lam+l1', l2'+lam'+l2), the
    largest value the triangles (f,l1',k), (f',l2,k) of the last 6j allow (R3).
    """
    pairs = []
    for gi, ch in enumerate(channels):
        for gj, chp in enumerate(channels):
            l, lp = ch[0], chp[0]
            lam, lamp = ch[4], chp[4]
            terms = []
            for l1 in range(0, l + 1):
                for l1p in range(0, lp + 1):
                    l2 = l - l1
                    l2p = lp - l1p
                    for k in range(0, min(l1 + lam + l1p, l2p + lamp + l2) + 1):
                        g = g_coefficient(ch, chp, two_J, two_T, l1, l1p, k)
                        if abs(g) > zero_tol:
                            terms.append((k, l1, l1p, g))
            if terms:
                pairs.append((gi, gj, terms))
    return pairs


def spinless_swave_table(g0):
    """Configs 1-2: one channel l=lam=0 with the single coefficient g0 (k=l1=l1'=0),
    DESIGN.md R4."""
    return [(0, 0, 0, 0, 0, 0)], [(0, 0, [(0, 0, 0, float(g0))])]


def G_function(ch, chp, terms, q, qp, x):
    """G_{gamma gamma'}(q,q',x) of (A3) (reading R1): sum q^{l1+l1'} q'^{l2+l2'} P_k(x) g."""
    from numpy.polynomial.legendre import legval

    l, lp = ch[0], chp[0]
    total = 0.0
    for (k, l1, l1p, g) in terms:
        A = l1 + l1p
        B = (l - l1) + (lp - l1p)
        total += q ** A * qp ** B * legval(x, [0.0] * k + [1.0]) * g
    return total
