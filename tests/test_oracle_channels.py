"""Pins for oracle/channels.py (channel rule of eq. 5 and the coefficients g of A4)."""
import numpy as np
import pytest

from oracle import channels


def test_channel_count_matches_paper_18():
    # PAPER.md:346 "18-channel Faddeev equations for the J=1/2 partial nd elastic amplitude"
    assert len(channels.enumerate_channels(1, +1, 2)) == 18
    assert len(channels.enumerate_channels(1, -1, 2)) == 18


def test_channel_rules():
    for two_J, par, jmax in [(1, 1, 2), (3, -1, 3), (7, 1, 3)]:
        chs = channels.enumerate_channels(two_J, par, jmax)
        assert len(set(chs)) == len(chs)
        for (l, s, j, t, lam, two_I) in chs:
            assert (l + s + t) % 2 == 1
            assert abs(l - s) <= j <= l + s and j <= jmax
            assert abs(2 * lam - 1) <= two_I <= 2 * lam + 1  # I = lam + 1/2 (vector sum)
            assert abs(two_J - 2 * j) <= two_I <= two_J + 2 * j
            assert (-1) ** (l + lam) == par
    # counts for j <= 3 (R12)
    assert [len(channels.enumerate_channels(tj, 1, 3)) for tj in (1, 3, 5, 7)] == [26, 46, 58, 62]


def test_swave_values_doublet_quartet():
    # l=lam=l'=lam'=0: g = -sqrt(s^ s'^ t^ t'^) {1/2 1/2 t;1/2 T t'} {1/2 1/2 s;1/2 J s'}:
    # the textbook spin-isospin recoupling of P12P23+P13P23: doublet [[1/4,-3/4],[-3/4,1/4]], quartet -1/2
    sw = [c for c in channels.enumerate_channels(1, +1, 1) if c[0] == 0 and c[4] == 0]
    assert sw == [(0, 0, 0, 1, 0, 1), (0, 1, 1, 0, 0, 1)]
    g = [[channels.g_coefficient(a, b, 1, 1, 0, 0, 0) for b in sw] for a in sw]
    assert np.allclose(g, [[0.25, -0.75], [-0.75, 0.25]], atol=1e-14)
    q = [c for c in channels.enumerate_channels(3, +1, 1) if c[0] == 0 and c[4] == 0]
    assert q == [(0, 1, 1, 0, 0, 1)]
    assert channels.g_coefficient(q[0], q[0], 3, 1, 0, 0, 0) == pytest.approx(-0.5, abs=1e-14)


@pytest.fixture(scope="module")
def table_half_plus():
    chs = channels.enumerate_channels(1, +1, 2)
    return chs, channels.g_table(chs, 1, 1)


def test_G_vanishing_order(table_half_plus):
    """G_{gg'} carries the solid-harmonic factors p^l p'^l' (A1 divides by p^{l+2} p'^{l'+2} and the
    kernel must stay integrable): at x=-1, q'=q/2+eps gives pi2=eps, so G=O(eps^l); q=q'/2+eps gives
    pi1=eps, so G=O(eps^l').  Fails if (A3)'s labels are read as printed (R1)."""
    chs, tab = table_half_plus
    checked = 0
    for gi, gj, terms in tab:
        l, lp = chs[gi][0], chs[gj][0]
        scale = sum(abs(t[3]) for t in terms)
        for eps in (1e-2, 1e-3):
            if l >= 1:   # pi2 -> 0
                val = channels.G_function(chs[gi], chs[gj], terms, 1.0, 0.5 + eps, -1.0)
                assert abs(val) <= 50 * scale * eps ** l
                checked += 1
            if lp >= 1:  # pi1 -> 0
                val = channels.G_function(chs[gi], chs[gj], terms, 0.5 + eps, 1.0, -1.0)
                assert abs(val) <= 50 * scale * eps ** lp
                checked += 1
    assert checked > 300


def test_G_vanishing_order_is_sharp(table_half_plus):
    # and not identically zero: for some l=2 pair the ratio G(eps)/eps^2 stays finite and nonzero
    chs, tab = table_half_plus
    ratios = []
    for gi, gj, terms in tab:
        if chs[gi][0] == 2 and chs[gj][0] == 0:
            r = [channels.G_function(chs[gi], chs[gj], terms, 1.0, 0.5 + e, -1.0) / e ** 2 for e in (1e-2, 1e-3)]
            ratios.append(r)
    assert any(abs(r[0]) > 1e-3 and abs(r[0] / r[1] - 1) < 0.1 for r in ratios)


def test_G_hermiticity(table_half_plus):
    # <pq g|P|p'q' g'> is real symmetric: G_{gg'}(q,q',x) = G_{g'g}(q',q,x)
    chs, tab = table_half_plus
    lookup = {(gi, gj): terms for gi, gj, terms in tab}
    rng = np.random.default_rng(1)
    for (gi, gj), terms in lookup.items():
        assert (gj, gi) in lookup
        q, qp, x = rng.uniform(0.2, 2.0), rng.uniform(0.2, 2.0), rng.uniform(-1, 1)
        lhs = channels.G_function(chs[gi], chs[gj], terms, q, qp, x)
        rhs = channels.G_function(chs[gj], chs[gi], lookup[(gj, gi)], qp, q, x)
        assert lhs == pytest.approx(rhs, abs=1e-12 * (1 + abs(lhs)))


def test_k_range_complete(table_half_plus):
    # DESIGN.md R3: nothing survives beyond k = min(l1+lam+l1', l2'+lam'+l2); something does
    # survive beyond l1'+l2 (the range a misreading of the last 6j would give)
    chs, _ = table_half_plus
    beyond_small_range = 0
    for a, b in [(chs[-1], chs[-2]), (chs[-3], chs[5]), (chs[7], chs[-1])]:
        l, lp, lam, lamp = a[0], b[0], a[4], b[4]
        for l1 in range(l + 1):
            for l1p in range(lp + 1):
                l2, l2p = l - l1, lp - l1p
                kmax = min(l1 + lam + l1p, l2p + lamp + l2)
                for k in range(0, l + lp + lam + lamp + 3):
                    g = channels.g_coefficient(a, b, 1, 1, l1, l1p, k)
                    if k > kmax:
                        assert g == 0.0
                    elif k > l1p + l2 and g != 0.0:
                        beyond_small_range += 1
    assert beyond_small_range > 0


def _bipolar(l, lam, L, M, pvec, qvec):
    """p^l sum_m <l m lam M-m|L M> Y_lm(p^) Y_lam,M-m(q^)  (library CG and Y_lm)."""
    from scipy.special import sph_harm_y
    from sympy.physics.wigner import clebsch_gordan

    def Y(ll, mm, v):
        r = np.linalg.norm(v)
        return sph_harm_y(ll, mm, np.arccos(v[2] / r), np.arctan2(v[1], v[0]))

    tot = 0.0
    for m in range(-l, l + 1):
        if abs(M - m) <= lam:
            tot += float(clebsch_gordan(l, lam, L, m, M - m, M)) * Y(l, m, pvec) * Y(lam, M - m, qvec)
    return tot * np.linalg.norm(pvec) ** l


@pytest.mark.parametrize("l,lam,lp,lamp", [(1, 1, 0, 2), (2, 2, 1, 1), (1, 2, 2, 1), (2, 1, 2, 3), (3, 1, 1, 1)])
def test_orbital_part_against_bipolar_harmonics(l, lam, lp, lamp):
    """sum_{l1 l1' k} o^{L} q^{l1+l1'} q'^{l2+l2'} P_k(x) must be proportional (one constant per
    (l,lam,l',lam'), the same for every L) to  sum_M [Y_l(p) Y_lam(q^)]^{LM*} [Y_l'(p') Y_lam'(q'^)]^{LM} / (2L+1)
    with the VECTORS p = q/2 + q', p' = q + q'/2 whose lengths are pi2, pi1 of (A2)."""
    from numpy.polynomial.legendre import legval

    rng = np.random.default_rng(5)
    ratios = []
    for L in range(max(abs(l - lam), abs(lp - lamp)), min(l + lam, lp + lamp) + 1):
        for _ in range(3):
            q, qp, x = rng.uniform(0.3, 2.0), rng.uniform(0.3, 2.0), rng.uniform(-0.9, 0.9)
            qv = np.array([0.0, 0.0, q])
            qpv = qp * np.array([np.sqrt(1 - x * x), 0.0, x])
            brute = sum(np.conj(_bipolar(l, lam, L, M, 0.5 * qv + qpv, qv)) * _bipolar(lp, lamp, L, M, qv + 0.5 * qpv, qpv)
                        for M in range(-L, L + 1)).real / (2 * L + 1)
            formula = 0.0
            for l1 in range(l + 1):
                for l1p in range(lp + 1):
                    for k in range(0, l + lp + lam + lamp + 1):
                        o = channels.orbital_coefficient(l, lam, lp, lamp, L, l1, l1p, k)
                        formula += o * q ** (l1 + l1p) * qp ** ((l - l1) + (lp - l1p)) * legval(x, [0.0] * k + [1.0])
            if abs(formula) < 1e-9 and abs(brute) < 1e-9:
                continue
            ratios.append(brute / formula)
    assert len(ratios) >= 3
    assert np.ptp(ratios) < 1e-9 * abs(ratios[0])
