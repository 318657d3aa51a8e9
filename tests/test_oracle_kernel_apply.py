"""Pins for oracle/kernel_apply.py (the factored kernel K = O P0 O^T V1 G1 of eq. 10 and 12)."""
import numpy as np

import wpcd_inputs as wi
from oracle import channels, kernel_apply as ka, perm


def _setup(n=4):
    chs = channels.enumerate_channels(1, 1, 1)
    tab = perm.PairTable(chs, channels.g_table(chs, 1, 1))
    p = wi.tan2_grid(n, 1.0, 0.1, seed=81)
    q = wi.tan2_grid(n - 1, 0.9, 0.1, seed=82)
    rp, ci, v, _ = perm.build_csr(p, q, 6, tab)
    return tab.n_ch, n, n - 1, rp, ci, v


def test_identity_factors_give_the_csr_product():
    n_ch, n_p, n_q, rp, ci, v = _setup()
    rows = n_ch * n_p * n_q
    eye = np.broadcast_to(np.eye(n_p), (n_ch, n_p, n_p)).copy()
    x = wi.normal_vector(rows, k=1)
    y = ka.kernel_apply(rp, ci, v, eye, eye, np.ones(rows), x, n_ch, n_p, n_q)
    assert np.allclose(y, perm.spmv(rp, ci, v, x), rtol=0, atol=1e-13)


def test_against_entrywise_eq10():
    """<Z_kj^g|P|Z_k'j'^g'> = sum_{ii'} O^g_ki O^g'_k'i' P0[(g,i,j),(g',i',j')], assembled with the four-index sum."""
    n_ch, n_p, n_q, rp, ci, v = _setup(3)
    rows = n_ch * n_p * n_q
    o, vv, g1 = wi.kernel_factors(n_ch, n_p, n_q)
    P0 = np.zeros((rows, rows))
    for r in range(rows):
        P0[r, ci[rp[r]:rp[r + 1]]] = v[rp[r]:rp[r + 1]]
    idx = lambda g, i, j: (g * n_p + i) * n_q + j
    P = np.zeros((rows, rows))
    for g in range(n_ch):
        for gp in range(n_ch):
            for k in range(n_p):
                for kp in range(n_p):
                    for j in range(n_q):
                        for jp in range(n_q):
                            s = 0.0
                            for i in range(n_p):
                                for ip in range(n_p):
                                    s += o[g, k, i] * o[gp, kp, ip] * P0[idx(g, i, j), idx(gp, ip, jp)]
                            P[idx(g, k, j), idx(gp, kp, jp)] = s
    V = np.zeros((rows, rows))
    for g in range(n_ch):
        for k in range(n_p):
            for kp in range(n_p):
                for j in range(n_q):
                    V[idx(g, k, j), idx(g, kp, j)] = vv[g, k, kp]
    x = wi.normal_vector(rows, k=2) + 1j * wi.normal_vector(rows, k=3)
    ref = P @ (V @ (g1 * x))
    y = ka.kernel_apply(rp, ci, v, o, vv, g1, x, n_ch, n_p, n_q)
    assert np.allclose(y, ref, rtol=0, atol=1e-12 * np.abs(ref).max())


def test_orthogonal_rotation_keeps_the_spectrum():
    n_ch, n_p, n_q, rp, ci, v = _setup()
    rows = n_ch * n_p * n_q
    o, _, _ = wi.kernel_factors(n_ch, n_p, n_q)
    eye = np.broadcast_to(np.eye(n_p), (n_ch, n_p, n_p)).copy()
    cols = [ka.kernel_apply(rp, ci, v, o, eye, np.ones(rows), np.eye(rows)[:, c], n_ch, n_p, n_q) for c in range(rows)]
    P = np.array(cols).T
    P0 = np.zeros((rows, rows))
    for r in range(rows):
        P0[r, ci[rp[r]:rp[r + 1]]] = v[rp[r]:rp[r + 1]]
    assert np.allclose(P, P.T, atol=1e-12)
    assert np.allclose(np.linalg.eigvalsh(0.5 * (P + P.T)), np.linalg.eigvalsh(0.5 * (P0 + P0.T)), atol=1e-11)
    for g in range(n_ch):
        assert np.allclose(o[g] @ o[g].T, np.eye(n_p), atol=1e-13)


def test_pade_sums_divergent_geometric_and_rational_series():
    # sum r^n = 1/(1-r): exact for the [n/1] approximant, also where the series diverges
    for r in (0.5, -2.0, 3.0 + 1.0j, -0.9j):
        terms = np.array([r ** n for n in range(8)], np.complex128)
        assert abs(ka.pade_sum(terms) - 1.0 / (1.0 - r)) < 1e-9 * max(1.0, abs(1.0 / (1.0 - r)))
    # two poles: sum (c1 r1^n + c2 r2^n) = c1/(1-r1) + c2/(1-r2), exact from [n/2] on
    r1, r2, c1, c2 = -1.7, 0.6 + 0.3j, 2.0, -0.5j
    terms = np.array([c1 * r1 ** n + c2 * r2 ** n for n in range(10)], np.complex128)
    exact = c1 / (1 - r1) + c2 / (1 - r2)
    assert abs(ka.pade_sum(terms) - exact) < 1e-8


def test_iteration_and_pade_against_direct_solve():
    """u = b + K u: the amplitude element of (1 - K)^{-1} b from the Neumann terms + Pade, on a tiny lattice, for a
    kernel inside the unit disc (the plain series converges) and for one scaled beyond it (only Pade does)."""
    n_ch, n_p, n_q, rp, ci, v = _setup(3)
    rows = n_ch * n_p * n_q
    o, vv, g1 = wi.kernel_factors(n_ch, n_p, n_q)
    K = np.array([ka.kernel_apply(rp, ci, v, o, vv, g1, np.eye(rows)[:, c].astype(np.complex128), n_ch, n_p, n_q)
                  for c in range(rows)]).T
    rho = np.abs(np.linalg.eigvals(K)).max()
    b = wi.normal_vector(rows, k=5) + 1j * wi.normal_vector(rows, k=6)
    element = 7
    for target_rho, n_terms, tol in ((0.5, 40, 1e-9), (1.6, 40, 1e-5)):
        scale = target_rho / rho
        exact = np.linalg.solve(np.eye(rows) - scale * K, b)[element]
        terms = ka.neumann_terms(rp, ci, v, o, vv, scale * g1, b, element, n_terms, n_ch, n_p, n_q)
        assert abs(ka.pade_sum(terms) - exact) < tol * max(1.0, abs(exact))
        if target_rho > 1:
            assert abs(np.sum(terms) - exact) > 1e3 * abs(exact)        # the plain series has diverged
