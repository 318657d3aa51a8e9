"""Pins for oracle/perm_oracle.c -- predicate, rule R(n), normalisation, SpMV.

Each test names what it would catch.  None of them re-types the oracle's formulae:
they use the Cartesian form (A7), operator identities of P = P12P23+P13P23
and the survey's worked single-cell example.
"""
import os

import numpy as np
import pytest

import wpcd_inputs as wi
from oracle import channels, perm
from tests import cartesian_bruteforce as brute

GOLD = os.path.join(os.path.dirname(__file__), "golden", "single_cell.txt")


def _dense(row_ptr, col_idx, values):
    n = len(row_ptr) - 1
    M = np.zeros((n, n))
    for r in range(n):
        M[r, col_idx[row_ptr[r]:row_ptr[r + 1]]] = values[row_ptr[r]:row_ptr[r + 1]]
    return M


def test_single_cell_golden_and_scale_free(swave_table):
    gold = dict(line.split() for line in open(GOLD) if line.strip() and not line.startswith("#"))
    for a in (0.37, 1.0, 25.0):
        p = np.array([0.0, a])
        for n in (8, 10, 48):
            v, _ = perm.element_values(p, p, [0], [0], [0], [0], n, swave_table)
            assert v[0, 0] == pytest.approx(float(gold[str(n)]), abs=2e-12)
    v, _ = perm.element_values(np.array([0.0, 1.0]), np.array([0.0, 1.0]), [0], [0], [0], [0], 128, swave_table)
    assert abs(v[0, 0] - float(gold["C1"])) < 3e-4


def test_single_cell_against_cartesian_A7(swave_table):
    # independent value of the same element from the unreduced (q,q',x) integral
    ref = brute.element(0, 1, 0, 1, 0, 1, 0, 1, 0, 0, [(0, 0, 0, 1.0)], m=600)
    v, _ = perm.element_values(np.array([0.0, 1.0]), np.array([0.0, 1.0]), [0], [0], [0], [0], 128, swave_table)
    assert v[0, 0] == pytest.approx(ref, abs=2e-3)


def test_elements_against_cartesian_A7_swave(swave_table):
    """Catches wrong limits / normalisation / F / zeta assignment: every structural element of a
    small jittered lattice against the Cartesian brute force (both converge slowly: F has kinks)."""
    p = wi.tan2_grid(5, 1.0, 0.1, seed=3)
    q = wi.tan2_grid(4, 0.7, 0.1, seed=4)   # different p and q grids: catches p<->q mix-ups
    ptr, col = perm.geo_pattern(p, q)
    n_q = len(q) - 1
    rows = np.repeat(np.arange(len(ptr) - 1), np.diff(ptr))
    v, _ = perm.element_values(p, q, rows // n_q, rows % n_q, col // n_q, col % n_q, 64, swave_table)
    worst = 0.0
    for e in range(len(col)):
        i, j, ip, jp = rows[e] // n_q, rows[e] % n_q, col[e] // n_q, col[e] % n_q
        ref = brute.element(q[j], q[j + 1], q[jp], q[jp + 1], p[ip], p[ip + 1], p[i], p[i + 1], 0, 0, [(0, 0, 0, 1.0)], m=160)
        worst = max(worst, abs(v[e, 0] - ref))
    assert worst < 4e-3 * np.abs(v).max()


def test_elements_against_cartesian_A7_multichannel(nd_half_plus_j1):
    """Catches a dropped term, swapped exponents (A <-> B), wrong zeta powers (l <-> l'), P_k index."""
    tab = nd_half_plus_j1
    p = wi.tan2_grid(3, 1.0, 0.1, seed=5)
    q = wi.tan2_grid(3, 0.8, 0.1, seed=6)
    ptr, col = perm.geo_pattern(p, q)
    n_q = len(q) - 1
    rows = np.repeat(np.arange(len(ptr) - 1), np.diff(ptr))
    # elements away from the first bins (there single terms are singular and brute force is poor)
    sel = [e for e in range(len(col)) if min(rows[e] // n_q, col[e] // n_q) >= 1][:6]
    assert len(sel) >= 4
    v, av = perm.element_values(p, q, rows[sel] // n_q, rows[sel] % n_q, col[sel] // n_q, col[sel] % n_q, 48, tab)
    # a few pairs with l != l', both > 0
    pick = [c for c in range(tab.n_pairs) if tab.pair_l[c] != tab.pair_lp[c] and min(tab.pair_l[c], tab.pair_lp[c]) >= 1][:5]
    pick += [c for c in range(tab.n_pairs) if tab.pair_l[c] == 2 and tab.pair_lp[c] == 0][:2]
    for c in pick:
        terms = [(tab.term_k[t], tab.term_l1[t], tab.term_l1p[t], tab.term_g[t]) for t in range(tab.term_ptr[c], tab.term_ptr[c + 1])]
        for n_e, e in enumerate(sel):
            i, j, ip, jp = rows[e] // n_q, rows[e] % n_q, col[e] // n_q, col[e] % n_q
            ref = brute.element(q[j], q[j + 1], q[jp], q[jp + 1], p[ip], p[ip + 1], p[i], p[i + 1],
                                int(tab.pair_l[c]), int(tab.pair_lp[c]), terms, m=120)
            assert abs(v[n_e, c] - ref) < 1e-2 * max(av[n_e, c], 1e-3), (c, e)


def test_absval_against_cartesian_modulus(nd_half_plus_j1):
    """Pins A_e (`absval`), the scale of every coupled-channel value tolerance (R9): it must be the same integral
    with each term's integrand replaced by its modulus -- evaluated here from the unreduced Cartesian form (A7) -- and for a
    pair with a single k = 0 term it must equal |value| exactly.  Catches an inflated or deflated scale (a modulus taken
    of the sum instead of the terms, a dropped factor, terms counted twice)."""
    tab = nd_half_plus_j1
    p = wi.tan2_grid(3, 1.0, 0.1, seed=5)
    q = wi.tan2_grid(3, 0.8, 0.1, seed=6)
    ptr, col = perm.geo_pattern(p, q)
    n_q = len(q) - 1
    rows = np.repeat(np.arange(len(ptr) - 1), np.diff(ptr))
    sel = [e for e in range(len(col)) if min(rows[e] // n_q, col[e] // n_q) >= 1][:6]
    v, av = perm.element_values(p, q, rows[sel] // n_q, rows[sel] % n_q, col[sel] // n_q, col[sel] % n_q, 48, tab)
    assert np.all(av >= np.abs(v) * (1 - 1e-12))
    n_terms = np.diff(tab.term_ptr)
    # pairs whose terms cancel (several terms of both signs): there A_e differs from |v| and only the modulus integral fixes it
    many = [c for c in range(tab.n_pairs) if n_terms[c] >= 3 and min(tab.pair_l[c], tab.pair_lp[c]) >= 1][:4]
    many += [c for c in range(tab.n_pairs) if n_terms[c] >= 3 and tab.pair_l[c] == 2 and tab.pair_lp[c] == 0][:2]
    assert len(many) >= 4
    ratios = []
    for c in many:
        terms = [(tab.term_k[t], tab.term_l1[t], tab.term_l1p[t], tab.term_g[t]) for t in range(tab.term_ptr[c], tab.term_ptr[c + 1])]
        for n_e, e in enumerate(sel):
            i, j, ip, jp = rows[e] // n_q, rows[e] % n_q, col[e] // n_q, col[e] % n_q
            ref = brute.element(q[j], q[j + 1], q[jp], q[jp + 1], p[ip], p[ip + 1], p[i], p[i + 1],
                                int(tab.pair_l[c]), int(tab.pair_lp[c]), terms, m=120, modulus=True)
            assert abs(av[n_e, c] - ref) < 1e-2 * max(ref, 1e-3), (c, e, av[n_e, c], ref)
            ratios.append(av[n_e, c] / max(abs(v[n_e, c]), 1e-300))
    assert max(ratios) > 1.5            # the sample does contain cancelling pairs (the pin is not vacuous)
    # single-term pairs with k = 0 (P_0 = 1 > 0, every other factor positive): the modulus changes nothing
    single = [c for c in range(tab.n_pairs) if n_terms[c] == 1 and tab.term_k[tab.term_ptr[c]] == 0]
    assert single
    assert np.array_equal(av[:, single], np.abs(v[:, single]))


@pytest.mark.parametrize("two_J,parity,jmax,nb,n", [(1, 1, 2, 12, 8), (7, -1, 3, 8, 10)])
def test_fp64_oracle_against_its_long_double_twin(two_J, parity, jmax, nb, n):
    """The same source compiled with -DWPO_EXTENDED evaluates rule R(n) in long double.  The FP64 oracle must agree with
    it to FP64 rounding of the ABSOLUTE term sum: |v64 - v80| <= 3e-12 A_e (measured worst 7e-13: sliver elements, whose
    integration limits move with the rounding of the polygon angles) -- also on the first-bin cells where single
    terms are huge and the value is small by cancellation, where the plain relative error is O(1).  Fixes the
    meaning of A_e once more (an A_e too small by a factor would fail here) and bounds the oracle's own rounding, which the
    GPU tolerance 1e-11 A_e has to cover with room to spare."""
    chs = channels.enumerate_channels(two_J, parity, jmax)
    tab = perm.PairTable(chs, channels.g_table(chs, two_J, 1))
    p = wi.tan2_grid(nb)
    ptr, col = perm.geo_pattern(p, p)
    rows = np.repeat(np.arange(nb * nb), np.diff(ptr))
    v, a = perm.element_values(p, p, rows // nb, rows % nb, col // nb, col % nb, n, tab)
    ve, ae = perm.element_values(p, p, rows // nb, rows % nb, col // nb, col % nb, n, tab, extended=True)
    assert np.all(np.abs(a - ae) <= 1e-11 * ae)
    err = np.abs(v - ve)
    assert np.all(err <= 3e-12 * a + 1e-300)
    # the ill-conditioned entries are there: relative errors far above 1e-11 although err / A_e stays at rounding level
    rel = err / np.maximum(np.abs(ve), 1e-300)
    assert rel.max() > 1e-9 and np.median(rel) < 1e-13


@pytest.fixture(scope="module")
def swave_matrices(swave_table):
    out = {}
    for N in (10, 20):
        p = wi.tan2_grid(N)
        out[N] = (p, perm.build_csr(p, p, 8, swave_table))
    return out


def test_symmetry(swave_matrices):
    # P is Hermitian and the lattice basis real: M = M^T, pattern exactly
    for N, (p, (rp, ci, v, _)) in swave_matrices.items():
        M = _dense(rp, ci, v)
        pat = np.zeros_like(M, bool)
        for r in range(len(rp) - 1):
            pat[r, ci[rp[r]:rp[r + 1]]] = True
        assert np.array_equal(pat, pat.T)
        assert np.abs(M - M.T).max() < 1e-12


def test_spectrum_bound(swave_matrices):
    # g0=1: spectrum of P = P12P23+P13P23 is {2,-1}; a Galerkin projection keeps it inside [-1,2]
    for N, (p, (rp, ci, v, _)) in swave_matrices.items():
        M = _dense(rp, ci, v)
        ev = np.linalg.eigvalsh(0.5 * (M + M.T))
        assert ev[0] > -1.0 - 0.02 and ev[-1] < 2.0 + 0.02


def _symmetric_state(p, alpha=0.5):
    """Lattice projection of psi = exp(-alpha (p^2 + 3/4 q^2)) (fully symmetric s-wave state):
    v_ij = (d_i d_j)^{-1/2} int p e^{-alpha p^2} dp int q e^{-3 alpha q^2/4} dq  (A5)."""
    ip = (np.exp(-alpha * p[:-1] ** 2) - np.exp(-alpha * p[1:] ** 2)) / (2 * alpha)
    b = 0.75 * alpha
    iq = (np.exp(-b * p[:-1] ** 2) - np.exp(-b * p[1:] ** 2)) / (2 * b)
    d = np.diff(p)
    return np.outer(ip / np.sqrt(d), iq / np.sqrt(d)).reshape(-1)


def test_symmetric_state_eigenvalue_two(swave_matrices):
    """P psi = 2 psi for a totally symmetric state: pins the overall normalisation of (A5)/(A9)/(A15)
    and g0 (R4).  Residual must shrink under refinement."""
    res, rq = [], []
    for N in (10, 20):
        p, (rp, ci, v, _) = swave_matrices[N]
        vec = _symmetric_state(p)
        y = perm.spmv(rp, ci, v, vec)
        rq.append(vec @ y / (vec @ vec))
        res.append(np.linalg.norm(y - 2 * vec) / np.linalg.norm(vec))
    assert abs(rq[1] - 2.0) < 0.1 and abs(rq[1] - 2.0) < abs(rq[0] - 2.0)
    assert res[1] < res[0] and res[1] < 0.12


def test_weak_form_P2_equals_P_plus_2(swave_matrices):
    # <v|(M^2 - M - 2)|v>/<v|v> -> 0 on a smooth symmetric vector (trend only, DESIGN.md pins table)
    vals = []
    for N in (10, 20):
        p, (rp, ci, v, _) = swave_matrices[N]
        vec = _symmetric_state(p)
        y = perm.spmv(rp, ci, v, vec)
        yy = perm.spmv(rp, ci, v, y)
        vals.append(abs(vec @ (yy - y - 2 * vec)) / (vec @ vec))
    assert vals[1] < vals[0] and vals[1] < 0.3


def test_multichannel_matrix_symmetric(nd_half_plus_j1):
    tab = nd_half_plus_j1
    p = wi.tan2_grid(4)
    rp, ci, v, av = perm.build_csr(p, p, 16, tab)
    M = _dense(rp, ci, v)
    A = _dense(rp, ci, av)
    assert np.all(np.abs(M - M.T) <= 1e-10 * np.maximum(A, A.T) + 1e-14)


def test_pattern_against_point_sampling():
    """Predicate S vs the theta-product of (A7) sampled on a dense interior grid: no hit may fall
    outside S, and every pair of S must be hit once sampling is fine enough."""
    p = wi.tan2_grid(7, 1.0, 0.1, seed=11)
    q = wi.tan2_grid(6, 1.3, 0.1, seed=12)
    ptr, col = perm.geo_pattern(p, q)
    n_p, n_q = len(p) - 1, len(q) - 1
    S = np.zeros((n_p * n_q, n_p * n_q), bool)
    for r in range(n_p * n_q):
        S[r, col[ptr[r]:ptr[r + 1]]] = True
    missed = 0
    for r in range(n_p * n_q):
        i, j = divmod(r, n_q)
        for c in range(n_p * n_q):
            ip, jp = divmod(c, n_q)
            args = (q[j], q[j + 1], q[jp], q[jp + 1], p[ip], p[ip + 1], p[i], p[i + 1])
            hit = brute.hits(*args, m=24)
            if hit:
                assert S[r, c], (r, c)
            elif S[r, c]:
                if not brute.hits(*args, m=400):
                    missed += 1
    assert missed == 0


def test_pattern_ties_on_identical_grids():
    # un-jittered p == q grids: touching cells (exact FP ties) are not structural nonzeros,
    # the pattern stays symmetric, and every row has at least one entry
    p = wi.tan2_grid(12)
    ptr, col = perm.geo_pattern(p, p)
    n = 12
    S = np.zeros((n * n, n * n), bool)
    for r in range(n * n):
        S[r, col[ptr[r]:ptr[r + 1]]] = True
        assert np.all(np.diff(col[ptr[r]:ptr[r + 1]]) > 0)
    assert np.array_equal(S, S.T)
    assert np.all(np.diff(ptr) > 0)
    # corner-touching pair (i'=i-1, j'=j-1 has E_hi' == E_lo exactly): never in S
    for i in range(1, n):
        for j in range(1, n):
            assert not S[i * n + j, (i - 1) * n + (j - 1)]


def test_values_zero_outside_pattern_and_superset(swave_table):
    # numerically nonzero elements (any n) all lie inside S: evaluate the rule on ALL cell pairs
    p = wi.tan2_grid(6, 1.0, 0.1, seed=2)
    n = 6
    ptr, col = perm.geo_pattern(p, p)
    S = set()
    for r in range(n * n):
        S.update((r, c) for c in col[ptr[r]:ptr[r + 1]])
    allr, allc = np.divmod(np.arange(n ** 4), n * n)
    # the rule returns 0 for a non-overlapping pair by construction; the independent check is the
    # brute-force Cartesian value
    for r, c in zip(allr[::7], allc[::7]):
        if (r, c) in S:
            continue
        i, j, ip, jp = r // n, r % n, c // n, c % n
        ref = brute.element(p[j], p[j + 1], p[jp], p[jp + 1], p[ip], p[ip + 1], p[i], p[i + 1], 0, 0, [(0, 0, 0, 1.0)], m=40)
        assert ref == 0.0


def test_spmv_against_dense(swave_matrices):
    p, (rp, ci, v, _) = swave_matrices[20]
    x = wi.normal_vector(len(rp) - 1)
    assert np.allclose(perm.spmv(rp, ci, v, x), _dense(rp, ci, v) @ x, rtol=0, atol=1e-12)


def test_full_row_ptr_and_columns(nd_half_plus_j1):
    tab = nd_half_plus_j1
    p = wi.tan2_grid(3)
    geo = perm.geo_pattern(p, p)
    rp, ci, v, _ = perm.build_csr(p, p, 4, tab, geo=geo)
    n_geo = 9
    for g in range(tab.n_ch):
        coupled = np.nonzero(tab.mask[g])[0]
        for r in range(n_geo):
            cols = ci[rp[g * n_geo + r]:rp[g * n_geo + r + 1]]
            gc = geo[1][geo[0][r]:geo[0][r + 1]]
            expect = np.concatenate([gp * n_geo + gc for gp in coupled]) if len(coupled) else np.zeros(0)
            assert np.array_equal(cols, expect)
            assert np.all(np.diff(cols) > 0)
    assert not np.isnan(v).any()


@pytest.mark.parametrize("two_J,parity,jmax", [(1, 1, 1), (3, -1, 1), (1, -1, 2)])
def test_multichannel_spectrum_bound(two_J, parity, jmax):
    """P = P12P23 + P13P23 is Hermitian with spectrum {-1, 2} on the states antisymmetric in the pair (l+s+t odd,
    PAPER.md:62, 102); the lattice matrix of ANY truncated channel set is a compression of it, so its eigenvalues
    must lie in [-1, 2] (up to the quadrature error) and the largest must approach 2 as the lattice is refined.
    This involves every factor of (A4) at once -- spin and isospin 6j, both 9j, prefactor and the orbital part:
    a wrong scale or a global sign leaves the interval at once (factor 2 -> 3.6; sign flip -> -1.8)."""
    chs = channels.enumerate_channels(two_J, parity, jmax)
    tab = perm.PairTable(chs, channels.g_table(chs, two_J, 1))
    top = []
    for N in (5, 7):
        p = wi.tan2_grid(N)
        rp, ci, v, _ = perm.build_csr(p, p, 12, tab)
        M = _dense(rp, ci, v)
        assert np.abs(M - M.T).max() < 1e-9
        w = np.linalg.eigvalsh(0.5 * (M + M.T))
        assert w[0] > -1.0 and w[-1] < 2.0
        assert w[0] < -0.8 and w[-1] > 1.6            # both ends of the exact spectrum are being approached
        top.append(w[-1])
    assert top[1] > top[0]


def test_rule_converges_with_order(swave_table):
    """Accuracy of the contract rule R(n) (R7): the integrand has kinks, so the error falls only
    algebraically -- it must fall monotonically, roughly like n^-1.5 .. n^-2 (2.1e-2 at n = 8, 1e-3 at n = 32)."""
    p = wi.tan2_grid(12, 1.0, 0.1, seed=3)
    geo = perm.geo_pattern(p, p)
    ref = perm.build_csr(p, p, 64, swave_table, geo=geo)[2]
    errs = {}
    for n in (4, 8, 16, 32):
        v = perm.build_csr(p, p, n, swave_table, geo=geo)[2]
        errs[n] = np.linalg.norm(v - ref) / np.linalg.norm(ref)
    assert errs[4] > errs[8] > errs[16] > errs[32]
    assert 1e-2 < errs[8] < 4e-2 and errs[32] < 2e-3
    rate = np.log(errs[8] / errs[32]) / np.log(4.0)
    assert 1.0 < rate < 3.0


# ---- kink-split rule RS(n) (R14; SURVEY.md section 8(c) item 7 "optional refinements", 8(f) item 4) ----
def test_split_rule_converges_faster(swave_table):
    """RS(n) cuts phi at the rectangle-corner angles and u at the crossings of the members of (A14)'s min/max.
    Pins: (1) it converges to the SAME limit as R(n) (a wrong cut or a dropped piece would converge elsewhere);
    (2) the survey's probe figure for this lattice: RS(8) reaches 1.9e-3 where R(8) has 2.1e-2; (3) monotone."""
    p = wi.tan2_grid(12, 1.0, 0.1, seed=3)
    geo = perm.geo_pattern(p, p)
    ref_split = perm.build_csr(p, p, 64, swave_table, geo=geo, split=True)[2]
    ref_plain = perm.build_csr(p, p, 64, swave_table, geo=geo)[2]
    nrm = np.linalg.norm(ref_split)
    assert np.linalg.norm(ref_plain - ref_split) / nrm < 5e-4          # R(64) itself is only good to ~3e-4
    errs, errs_plain = {}, {}
    for n in (4, 8, 16, 32):
        errs[n] = np.linalg.norm(perm.build_csr(p, p, n, swave_table, geo=geo, split=True)[2] - ref_split) / nrm
        errs_plain[n] = np.linalg.norm(perm.build_csr(p, p, n, swave_table, geo=geo)[2] - ref_split) / nrm
    assert errs[4] > errs[8] > errs[16] > errs[32]
    assert 1.5e-3 < errs[8] < 2.3e-3                                    # SURVEY: "with both, n=8 reaches 1.9e-3"
    for n in (4, 8, 16, 32):
        assert errs[n] < errs_plain[n] / 5.0


def test_split_rule_against_cartesian_A7(swave_table, nd_half_plus_j1):
    """The split rule against the unreduced (q,q',x) brute force: s-wave elements of a lattice with different p and q
    grids, and multichannel pairs with l != l' (catches a cut placed with the wrong cell's bounds: such a rule still
    converges, but a piece dropped or counted twice does not)."""
    p = wi.tan2_grid(5, 1.0, 0.1, seed=3)
    q = wi.tan2_grid(4, 0.7, 0.1, seed=4)
    ptr, col = perm.geo_pattern(p, q)
    n_q = len(q) - 1
    rows = np.repeat(np.arange(len(ptr) - 1), np.diff(ptr))
    v, _ = perm.element_values(p, q, rows // n_q, rows % n_q, col // n_q, col % n_q, 16, swave_table, split=True)
    v_ref, _ = perm.element_values(p, q, rows // n_q, rows % n_q, col // n_q, col % n_q, 64, swave_table)
    assert np.abs(v - v_ref).max() < 2e-3 * np.abs(v_ref).max()
    worst = 0.0
    for e in range(0, len(col), 3):
        i, j, ip, jp = rows[e] // n_q, rows[e] % n_q, col[e] // n_q, col[e] % n_q
        ref = brute.element(q[j], q[j + 1], q[jp], q[jp + 1], p[ip], p[ip + 1], p[i], p[i + 1], 0, 0, [(0, 0, 0, 1.0)], m=160)
        worst = max(worst, abs(v[e, 0] - ref))
    assert worst < 4e-3 * np.abs(v).max()
    tab = nd_half_plus_j1
    p3 = wi.tan2_grid(3, 1.0, 0.1, seed=5)
    q3 = wi.tan2_grid(3, 0.8, 0.1, seed=6)
    ptr, col = perm.geo_pattern(p3, q3)
    rows = np.repeat(np.arange(len(ptr) - 1), np.diff(ptr))
    sel = [e for e in range(len(col)) if min(rows[e] // 3, col[e] // 3) >= 1][:6]
    vs, avs = perm.element_values(p3, q3, rows[sel] // 3, rows[sel] % 3, col[sel] // 3, col[sel] % 3, 32, tab, split=True)
    vp, _ = perm.element_values(p3, q3, rows[sel] // 3, rows[sel] % 3, col[sel] // 3, col[sel] % 3, 64, tab)
    assert np.all(np.abs(vs - vp) <= 1.5e-3 * np.maximum(avs, 1e-3))     # same limit as R(n): R(64) is good to ~1e-3 here
    pick = [c for c in range(tab.n_pairs) if tab.pair_l[c] != tab.pair_lp[c] and min(tab.pair_l[c], tab.pair_lp[c]) >= 1][:3]
    for c in pick:
        terms = [(tab.term_k[t], tab.term_l1[t], tab.term_l1p[t], tab.term_g[t]) for t in range(tab.term_ptr[c], tab.term_ptr[c + 1])]
        for n_e, e in enumerate(sel[:3]):
            i, j, ip, jp = rows[e] // 3, rows[e] % 3, col[e] // 3, col[e] % 3
            ref = brute.element(q3[j], q3[j + 1], q3[jp], q3[jp + 1], p3[ip], p3[ip + 1], p3[i], p3[i + 1],
                                int(tab.pair_l[c]), int(tab.pair_lp[c]), terms, m=120)
            assert abs(vs[n_e, c] - ref) < 1e-2 * max(avs[n_e, c], 1e-3), (c, e)


def test_split_rule_single_cell(swave_table):
    """Single cell [0,1]^4 (golden constant C1 = 1.5056 +- 1e-4 of SURVEY.md section 8(c)): RS(n) is closer than R(n)
    at every order and reaches the constant; the 1/zeta corner keeps even RS algebraic."""
    gold = dict(line.split() for line in open(GOLD) if line.strip() and not line.startswith("#"))
    c1 = float(gold["C1"])
    p = np.array([0.0, 1.0])
    for n in (8, 32, 128):
        vs, _ = perm.element_values(p, p, [0], [0], [0], [0], n, swave_table, split=True)
        vp, _ = perm.element_values(p, p, [0], [0], [0], [0], n, swave_table)
        assert abs(vs[0, 0] - c1) < abs(vp[0, 0] - c1) + 1e-4
    assert abs(vs[0, 0] - c1) < 1.5e-4


def test_split_rule_symmetric_matrix(swave_table):
    """P0 is symmetric (same integral with the two Jacobi sets exchanged).  On a q == p lattice the
    exchange maps phi -> pi/2 - phi and every cut of RS(n) onto a cut of the transposed element, so the rule's matrix
    is symmetric to rounding -- a cut taken from the wrong cell's bounds breaks this at the 1e-3 level."""
    p = wi.tan2_grid(10, 1.0, 0.1, seed=11)
    rp, ci, v, _ = perm.build_csr(p, p, 8, swave_table, split=True)
    m = _dense(rp, ci, v)
    assert np.abs(m - m.T).max() < 1e-12 * np.abs(m).max()


# ---- rule RA(n): kink-split in phi and u, exact u-integral for the s-wave term (R15) ----
def test_analytic_u_rule_against_quadrature(swave_table):
    """The closed-form u-integrals of RA(n) against 64-point Gauss-Legendre on the same pieces (RS(64) in u, same phi-nodes):
    a wrong antiderivative, a wrong active member or a swapped zeta shows at once.  At equal n the two rules differ only by
    the u-quadrature error of RS(n), so RA(n) -> RS(n) as the u-order grows: compare at n = 64 (1e-5) and check that the
    phi-convergence is the same (RA(8) within 2x of RS(8)'s error, both against RS(64))."""
    p = wi.tan2_grid(12, 1.0, 0.1, seed=3)
    geo = perm.geo_pattern(p, p)
    rs64 = perm.build_csr(p, p, 64, swave_table, geo=geo, split=1)[2]
    ra64 = perm.build_csr(p, p, 64, swave_table, geo=geo, split=2)[2]
    nrm = np.linalg.norm(rs64)
    assert np.linalg.norm(ra64 - rs64) / nrm < 3e-5
    errs = {n: np.linalg.norm(perm.build_csr(p, p, n, swave_table, geo=geo, split=2)[2] - ra64) / nrm for n in (4, 8, 16, 32)}
    assert errs[4] > errs[8] > errs[16] > errs[32]
    assert errs[8] < 4e-3 and errs[32] < 1.5e-4
    # p != q lattice, element by element against RS(64)
    p5, q4 = wi.tan2_grid(5, 1.0, 0.1, seed=3), wi.tan2_grid(4, 0.7, 0.1, seed=4)
    ptr, col = perm.geo_pattern(p5, q4)
    rows = np.repeat(np.arange(len(ptr) - 1), np.diff(ptr))
    va, _ = perm.element_values(p5, q4, rows // 4, rows % 4, col // 4, col % 4, 64, swave_table, split=2)
    vs, _ = perm.element_values(p5, q4, rows // 4, rows % 4, col // 4, col % 4, 64, swave_table, split=1)
    assert np.abs(va - vs).max() < 5e-5 * np.abs(vs).max()


def test_analytic_u_rule_single_cell_and_cartesian(swave_table):
    """Single cell (C1 = 1.5056 +- 1e-4) and the Cartesian (A7) brute force on a p != q lattice."""
    gold = dict(line.split() for line in open(GOLD) if line.strip() and not line.startswith("#"))
    p1 = np.array([0.0, 1.0])
    v, av = perm.element_values(p1, p1, [0], [0], [0], [0], 128, swave_table, split=2)
    assert abs(v[0, 0] - float(gold["C1"])) < 1e-4 and av[0, 0] == pytest.approx(v[0, 0])
    p = wi.tan2_grid(5, 1.0, 0.1, seed=3)
    q = wi.tan2_grid(4, 0.7, 0.1, seed=4)
    ptr, col = perm.geo_pattern(p, q)
    n_q = len(q) - 1
    rows = np.repeat(np.arange(len(ptr) - 1), np.diff(ptr))
    v, _ = perm.element_values(p, q, rows // n_q, rows % n_q, col // n_q, col % n_q, 32, swave_table, split=2)
    worst = 0.0
    for e in range(0, len(col), 3):
        i, j, ip, jp = rows[e] // n_q, rows[e] % n_q, col[e] // n_q, col[e] % n_q
        ref = brute.element(q[j], q[j + 1], q[jp], q[jp + 1], p[ip], p[ip + 1], p[i], p[i + 1], 0, 0, [(0, 0, 0, 1.0)], m=160)
        worst = max(worst, abs(v[e, 0] - ref))
    assert worst < 4e-3 * np.abs(v).max()
    # symmetric to rounding on a q == p lattice (exchange symmetry of the cuts and of the closed forms, zeta1 <-> zeta2)
    pp = wi.tan2_grid(10, 1.0, 0.1, seed=11)
    rp, ci, vv, _ = perm.build_csr(pp, pp, 8, swave_table, split=2)
    m = _dense(rp, ci, vv)
    assert np.abs(m - m.T).max() < 1e-12 * np.abs(m).max()
