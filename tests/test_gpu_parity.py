"""GPU parity: the CUDA path (through the C-ABI binding) against the CPU oracle, element by
element.  Pattern (row_ptr, col_idx) bit-exact; values within
    1e-11 * max(|v|, A_e) + 1e-13 * V
where A_e is the element's absolute-sum scale computed by the oracle (pinned by tests/test_oracle_perm.py:
test_absval_against_cartesian_modulus, test_fp64_oracle_against_its_long_double_twin) and V = max|v| of the
matrix: the floor covers the ill-conditioned sliver elements next to the pi1 = 0 / pi2 = 0
corners, where rule R(n) itself is only ~1e-8 accurate in double precision (R9).
On top of it every WELL-CONDITIONED entry (A_e < 10 |v|: no cancellation between the terms) must agree to a plain
relative 1e-11, and each comparison records its worst error / tolerance and the histogram of the plain relative errors
(SURVEY 8(c)9); with WPCD_PARITY_REPORT=<file> the records are appended to that file (tests/parity_report.py turns them
into profiles/r02_parity.md).  SpMV within 1e-12 * sum_j |a_ij x_j|."""
import json
import os
import sys

import numpy as np
import pytest

import wpcd_inputs as wi
from oracle import channels as och
from oracle import perm as operm

pytestmark = pytest.mark.gpu

VALUE_RTOL = 1e-11
VALUE_FLOOR = 1e-13   # times max|v| of the matrix
WELL_CONDITIONED = 10.0   # A_e / |v| below this: the plain relative error must be within VALUE_RTOL
_HIST_EDGES = [0.0, 1e-15, 1e-14, 1e-13, 1e-12, 1e-11, 1e-10, 1e-9, 1e-6, 1e-3, np.inf]


class _ValueCheck:
    """Accumulates the element-by-element comparison of one test (possibly over several row samples)."""

    def __init__(self, tag):
        self.tag = tag
        self.n = self.n_well = 0
        self.worst = self.worst_well_rel = self.worst_rel = 0.0
        self.hist = np.zeros(len(_HIST_EDGES) - 1, np.int64)
        self.hist_well = np.zeros(len(_HIST_EDGES) - 1, np.int64)

    def add(self, gv, v, av, vmax, where=""):
        err = np.abs(gv - v)
        tol = VALUE_RTOL * np.maximum(np.abs(v), av) + VALUE_FLOOR * vmax
        ratio = err / np.maximum(tol, 1e-300)
        assert np.all(np.isfinite(gv)), where
        assert np.all(err <= tol), f"{self.tag} {where}: worst err/tol = {ratio.max()}"
        nz = np.abs(v) > 0
        rel = err[nz] / np.abs(v[nz])
        well = av[nz] < WELL_CONDITIONED * np.abs(v[nz])
        # an entry without cancellation between its terms: plain relative error (the floor only where |v| is far below V)
        bad = well & (rel > VALUE_RTOL) & (err[nz] > VALUE_FLOOR * vmax)
        assert not bad.any(), f"{self.tag} {where}: {bad.sum()} well-conditioned entries beyond {VALUE_RTOL} relative, worst {rel[bad].max()}"
        self.n += int(err.size); self.n_well += int(well.sum())
        self.worst = max(self.worst, float(ratio.max()) if err.size else 0.0)
        if rel.size:
            self.worst_rel = max(self.worst_rel, float(rel.max()))
            self.hist += np.histogram(rel, bins=_HIST_EDGES)[0]
        if well.any():
            self.worst_well_rel = max(self.worst_well_rel, float(rel[well].max()))
            self.hist_well += np.histogram(rel[well], bins=_HIST_EDGES)[0]

    def close(self, **extra):
        rec = {"test": self.tag, "entries": self.n, "well_conditioned": self.n_well, "worst_err_over_tol": self.worst,
               "worst_rel_err_well_conditioned": self.worst_well_rel, "worst_rel_err": self.worst_rel,
               "hist_edges": [e if np.isfinite(e) else "inf" for e in _HIST_EDGES],
               "hist_rel_err": self.hist.tolist(), "hist_rel_err_well_conditioned": self.hist_well.tolist()}
        rec.update(extra)
        print("PARITY " + json.dumps(rec))
        path = os.environ.get("WPCD_PARITY_REPORT")
        if path:
            with open(path, "a") as f:
                f.write(json.dumps(rec) + "\n")
        return self.worst


def _caller():
    return sys._getframe(2).f_code.co_name


def _torch():
    import torch

    assert torch.cuda.is_available()
    return torch


def _oracle_table(wl, two_J=None, parity=None):
    if wl.model == "swave":
        ch, pairs = och.spinless_swave_table(wl.g0)
    else:
        ch = och.enumerate_channels(two_J, parity, wl.j_pair_max)
        pairs = och.g_table(ch, two_J, 1)
    return operm.PairTable(ch, pairs)


def _gpu_channels(wpcd, wl, two_J=None, parity=None):
    if wl.model == "swave":
        return wpcd.wpcd_channels_create(wpcd.WPCD_SPINLESS_SWAVE, g0=wl.g0)
    return wpcd.wpcd_channels_create(wpcd.WPCD_ND, two_J=two_J, parity=parity, two_T=1, j_pair_max=wl.j_pair_max)


def _compare_full(wpcd, p, q, n_quad, gch, tab, geo_rows=None, split=False, tag=None):
    grid = wpcd.wpcd_grid_create(p, q)
    flag = {0: 0, 1: wpcd.WPCD_RULE_KINK_SPLIT, 2: wpcd.WPCD_RULE_ANALYTIC_U}[int(split)]
    m = wpcd.build_perm(grid, gch, n_quad | flag)
    _torch().cuda.synchronize()
    geo = operm.geo_pattern(p, q)
    rp, ci, v, av = operm.build_csr(p, q, n_quad, tab, geo=geo, geo_rows=geo_rows, split=split)
    assert m.nnz == rp[-1] and m.nnz_geo == geo[0][-1]
    assert np.array_equal(m.geo_row_ptr.cpu().numpy().astype(np.int64), geo[0])
    assert np.array_equal(m.row_ptr.cpu().numpy(), rp)
    assert np.array_equal(m.col_idx.cpu().numpy(), ci)
    gv = m.values.cpu().numpy()
    sel = ~np.isnan(v)
    assert sel.any()
    chk = _ValueCheck(tag or _caller())
    chk.add(gv[sel], v[sel], av[sel], np.abs(v[sel]).max())
    chk.close(n_p=len(p) - 1, n_q=len(q) - 1, n_quad=n_quad, rule=int(split), nnz=int(m.nnz))
    assert np.all(np.isfinite(gv))
    return m, (rp, ci, v, av)


def test_cfg1_swave_n20(wpcd):
    wl = wi.WORKLOADS["cfg1"]
    p = wl.grid()
    _compare_full(wpcd, p, p, wl.n_quad, _gpu_channels(wpcd, wl), _oracle_table(wl))


def test_cfg2_swave_n100_and_spmv(wpcd):
    torch = _torch()
    wl = wi.WORKLOADS["cfg2"]
    p = wl.grid()
    m, (rp, ci, v, av) = _compare_full(wpcd, p, p, wl.n_quad, _gpu_channels(wpcd, wl), _oracle_table(wl))
    rows = m.rows
    y = torch.empty(rows, dtype=torch.float64, device="cuda")
    gv = m.values.cpu().numpy()   # the product on the SAME matrix: isolates the SpMV kernel
    for k in range(3):
        xh = wi.normal_vector(rows, k=k)
        x = torch.from_numpy(xh).cuda()
        wpcd.wpcd_perm_apply(rows, m.row_ptr, m.col_idx, m.values, x, y)
        ref = operm.spmv(rp, ci, gv, xh)
        scale = operm.spmv(rp, ci, np.abs(gv), np.abs(xh))
        assert np.all(np.abs(y.cpu().numpy() - ref) <= 1e-12 * scale + 1e-300)


@pytest.mark.parametrize("n_quad", [1, 3, 4, 6, 10, 12, 48, 64])
def test_quadrature_orders(wpcd, n_quad):
    p = wi.tan2_grid(9, 1.0, 0.1, seed=21)
    q = wi.tan2_grid(7, 0.6, 0.1, seed=22)
    ch, pairs = och.spinless_swave_table(1.0)
    _compare_full(wpcd, p, q, n_quad, wpcd.wpcd_channels_create(wpcd.WPCD_SPINLESS_SWAVE, g0=1.0), operm.PairTable(ch, pairs))


def test_edge_grids(wpcd):
    ch, pairs = och.spinless_swave_table(0.5)
    tab = operm.PairTable(ch, pairs)
    gch = wpcd.wpcd_channels_create(wpcd.WPCD_SPINLESS_SWAVE, g0=0.5)
    # single cell; grids that do not start at zero; very uneven bins; ragged n_p != n_q
    cases = [
        (np.array([0.0, 0.37]), np.array([0.0, 0.37])),
        (np.array([0.3, 0.5, 2.0]), np.array([0.1, 0.2, 0.9, 4.0])),
        (np.array([0.0, 1e-3, 1.0, 50.0]), np.array([0.0, 2.0])),
        (wi.tan2_grid(33, 2.0, 0.2, seed=5), wi.tan2_grid(5, 0.5, 0.0)),
    ]
    for p, q in cases:
        _compare_full(wpcd, p, q, 8, gch, tab)


def test_disjoint_cells_give_empty_matrix(wpcd):
    # p-cells far above anything q,q' can reach: no structural nonzeros at all
    torch = _torch()
    p = np.array([100.0, 101.0])
    q = np.array([0.0, 1.0])
    grid = wpcd.wpcd_grid_create(p, q)
    gch = wpcd.wpcd_channels_create(wpcd.WPCD_SPINLESS_SWAVE, g0=0.5)
    m = wpcd.build_perm(grid, gch, 8)
    assert m.nnz == 0 and operm.geo_pattern(p, q)[0][-1] == 0
    x = torch.ones(1, dtype=torch.float64, device="cuda")
    y = torch.full((1,), 7.0, dtype=torch.float64, device="cuda")
    wpcd.wpcd_perm_apply(1, m.row_ptr, m.col_idx, m.values, x, y)
    assert y.item() == 0.0


def test_apply_multi_vector_and_host(wpcd):
    torch = _torch()
    p = wi.tan2_grid(24, 1.0, 0.1, seed=8)
    grid = wpcd.wpcd_grid_create(p, p)
    gch = wpcd.wpcd_channels_create(wpcd.WPCD_SPINLESS_SWAVE, g0=0.5)
    m = wpcd.build_perm(grid, gch, 8)
    rows = m.rows
    rp, ci, v = m.row_ptr.cpu().numpy(), m.col_idx.cpu().numpy(), m.values.cpu().numpy()
    for n_vec in (1, 2, 3, 7):
        xh = np.stack([wi.normal_vector(rows, k=10 + k) for k in range(n_vec)])
        x = torch.from_numpy(xh).cuda().contiguous()
        y = torch.empty_like(x)
        wpcd.wpcd_perm_apply(rows, m.row_ptr, m.col_idx, m.values, x, y, n_vec=n_vec)
        for k in range(n_vec):
            ref = operm.spmv(rp, ci, v, xh[k])
            scale = operm.spmv(rp, ci, np.abs(v), np.abs(xh[k]))
            assert np.all(np.abs(y[k].cpu().numpy() - ref) <= 1e-12 * scale)
    xh = torch.from_numpy(wi.normal_vector(rows, k=99)).pin_memory()
    yh = torch.empty(rows, dtype=torch.float64).pin_memory()
    xd = torch.empty(rows, dtype=torch.float64, device="cuda")
    yd = torch.empty_like(xd)
    wpcd.wpcd_perm_apply_host(rows, m.row_ptr, m.col_idx, m.values, xh, yh, xd, yd)
    ref = operm.spmv(rp, ci, v, xh.numpy())
    assert np.all(np.abs(yh.numpy() - ref) <= 1e-12 * operm.spmv(rp, ci, np.abs(v), np.abs(xh.numpy())))
    # several vectors in one host call (bench.py's end-to-end leg): 7 go in one piece, 21 through the pipeline over the copy
    # streams (chunks of 8, 8, 5), twice in a row with the same scratch
    for n_vec, reps in ((7, 1), (21, 2)):
        xh7 = torch.from_numpy(np.stack([wi.normal_vector(rows, k=120 + k) for k in range(n_vec)])).pin_memory()
        yh7 = torch.empty(n_vec, rows, dtype=torch.float64).pin_memory()
        xd7 = torch.empty(n_vec, rows, dtype=torch.float64, device="cuda")
        yd7 = torch.empty_like(xd7)
        for _ in range(reps):
            yh7.fill_(float("nan"))
            wpcd.wpcd_perm_apply_host(rows, m.row_ptr, m.col_idx, m.values, xh7, yh7, xd7, yd7, n_vec=n_vec)
            for k in range(n_vec):
                ref = operm.spmv(rp, ci, v, xh7[k].numpy())
                assert np.all(np.abs(yh7[k].numpy() - ref) <= 1e-12 * operm.spmv(rp, ci, np.abs(v), np.abs(xh7[k].numpy())))


def test_errors_on_device_path(wpcd):
    torch = _torch()
    p = wi.tan2_grid(4)
    grid = wpcd.wpcd_grid_create(p, p)
    gch = wpcd.wpcd_channels_create(wpcd.WPCD_SPINLESS_SWAVE, g0=0.5)
    row_ptr = torch.empty(17, dtype=torch.int64, device="cuda")
    geo = torch.empty(17, dtype=torch.int32, device="cuda")
    with pytest.raises(wpcd.WpcdError, match="n_quad"):
        wpcd.wpcd_perm_count(grid, gch, 0, row_ptr, geo)
    with pytest.raises(wpcd.WpcdError, match="n_quad"):
        wpcd.wpcd_perm_count(grid, gch, 65, row_ptr, geo)
    nnz, nnz_geo = wpcd.wpcd_perm_count(grid, gch, 8, row_ptr, geo)
    col = torch.empty(nnz, dtype=torch.int32, device="cuda")
    val = torch.empty(nnz, dtype=torch.float64, device="cuda")
    small = torch.empty(256, dtype=torch.uint8, device="cuda")
    with pytest.raises(wpcd.WpcdError, match="workspace too small"):
        wpcd.wpcd_perm_build(grid, gch, 8, row_ptr, geo, small, col, val)


def test_fp64_peak_microbenchmark(wpcd):
    flops = wpcd.wpcd_fp64_peak()
    assert 5e12 < flops < 1e14
    assert wpcd.wpcd_launch_count() > 0


# ----------------------------------------------------------------------------- coupled channels
def _compare_sampled(wpcd, p, n_quad, gch, tab, geo_rows, tag=None):
    """Full row_ptr + geometric pattern, and col_idx / values on the sampled geometric rows
    (all channels), without materialising the oracle's full CSR (configs 3-5 sizes)."""
    torch = _torch()
    n = len(p) - 1
    n_geo = n * n
    grid = wpcd.wpcd_grid_create(p, p)
    m = wpcd.build_perm(grid, gch, n_quad)
    torch.cuda.synchronize()
    geo_ptr, geo_col = operm.geo_pattern(p, p)
    assert np.array_equal(m.geo_row_ptr.cpu().numpy().astype(np.int64), geo_ptr)
    rp = operm.full_row_ptr(geo_ptr, tab, n, n)
    assert np.array_equal(m.row_ptr.cpu().numpy(), rp)
    assert m.nnz == rp[-1]
    geo_rows = np.asarray(geo_rows)
    cnt = geo_ptr[geo_rows + 1] - geo_ptr[geo_rows]
    erow = np.repeat(geo_rows, cnt)
    eidx = np.concatenate([np.arange(geo_ptr[r], geo_ptr[r + 1]) for r in geo_rows])
    ecol = geo_col[eidx]
    val, aval = operm.element_values(p, p, erow // n, erow % n, ecol // n, ecol % n, n_quad, tab)
    pair_of = -np.ones((tab.n_ch, tab.n_ch), np.int64)
    pair_of[tab.gamma, tab.gammap] = np.arange(tab.n_pairs)
    vmax = np.abs(val).max()
    off = np.concatenate([[0], np.cumsum(cnt)])
    chk = _ValueCheck(tag or _caller())
    # the products of the full-size matrix (general CSR kernel and the blocked one) on the sampled rows: the oracle's row
    # values times x, summed by the oracle side; the tolerance carries the value tolerance through the sum
    rows_all = m.rows
    xh = wi.normal_vector(rows_all, k=333)
    xd = torch.from_numpy(xh).cuda()
    y_csr, y_blk = torch.empty_like(xd), torch.empty_like(xd)
    wpcd.wpcd_perm_apply(rows_all, m.row_ptr, m.col_idx, m.values, xd, y_csr)
    wpcd.wpcd_perm_apply_blocked(grid, gch, m.row_ptr, m.geo_row_ptr, m.col_idx, m.values, xd, y_blk)
    y_csr, y_blk = y_csr.cpu().numpy(), y_blk.cpu().numpy()
    for g in range(tab.n_ch):
        coupled = np.nonzero(tab.mask[g])[0]
        if len(coupled) == 0:
            continue
        for ri, r in enumerate(geo_rows):
            lo, hi = rp[g * n_geo + r], rp[g * n_geo + r + 1]
            gc = geo_col[geo_ptr[r]:geo_ptr[r + 1]]
            exp_cols = (coupled[:, None].astype(np.int64) * n_geo + gc[None, :]).reshape(-1)
            assert hi - lo == len(exp_cols)
            assert np.array_equal(m.col_idx[lo:hi].cpu().numpy(), exp_cols)
            ev = val[off[ri]:off[ri + 1]][:, pair_of[g, coupled]].T.reshape(-1)
            ea = aval[off[ri]:off[ri + 1]][:, pair_of[g, coupled]].T.reshape(-1)
            gv = m.values[lo:hi].cpu().numpy()
            tol = VALUE_RTOL * np.maximum(np.abs(ev), ea) + VALUE_FLOOR * vmax
            chk.add(gv, ev, ea, vmax, where=f"channel {g} geo row {r}")
            xs = xh[exp_cols]
            y_ref = float(np.dot(ev, xs))
            y_tol = float(np.dot(tol, np.abs(xs))) + 1e-12 * float(np.dot(np.abs(ev), np.abs(xs)))
            assert abs(y_csr[g * n_geo + r] - y_ref) <= y_tol and abs(y_blk[g * n_geo + r] - y_ref) <= y_tol, (g, r)
    worst = chk.close(n_p=n, n_q=n, n_quad=n_quad, rule=0, nnz=int(m.nnz), sampled_geo_rows=int(len(geo_rows)), channels=int(tab.n_ch))
    return m, worst


@pytest.mark.parametrize("two_J,parity,jmax,nb,nq", [(1, 1, 1, 6, 6), (1, -1, 2, 5, 4), (3, 1, 2, 4, 8), (5, -1, 3, 3, 10)])
def test_coupled_small_full(wpcd, two_J, parity, jmax, nb, nq):
    chs = och.enumerate_channels(two_J, parity, jmax)
    tab = operm.PairTable(chs, och.g_table(chs, two_J, 1))
    gch = wpcd.wpcd_channels_create(wpcd.WPCD_ND, two_J=two_J, parity=parity, two_T=1, j_pair_max=jmax)
    p = wi.tan2_grid(nb, 1.0, 0.1, seed=31)
    q = wi.tan2_grid(nb + 1, 0.8, 0.1, seed=32)
    _compare_full(wpcd, p, q, nq, gch, tab)


def test_coupled_from_table_matches_builtin(wpcd):
    torch = _torch()
    chs = och.enumerate_channels(1, 1, 1)
    tab = operm.PairTable(chs, och.g_table(chs, 1, 1))
    gch = wpcd.wpcd_channels_create_from_table(np.array([c[0] for c in chs]), tab.gamma, tab.gammap, tab.term_ptr,
                                               tab.term_k, tab.term_l1, tab.term_l1p, tab.term_g)
    p = wi.tan2_grid(5)
    _compare_full(wpcd, p, p, 8, gch, tab)


def test_cfg3_nd_half_plus_full(wpcd):
    """Config 3 (N = 100, J^pi = 1/2+, j <= 2: 18 channels, 7.9e7 nonzeros): pattern AND values of the whole matrix against
    the oracle (values compared in full on configs 1-3), and the products of the CSR and the blocked kernel on
    the whole matrix against the oracle's sequential product of the GPU values."""
    torch = _torch()
    wl = wi.WORKLOADS["cfg3"]
    (two_J, parity), = wl.jpis
    p = wl.grid()
    n = wl.n_bins
    n_geo = n * n
    tab = _oracle_table(wl, two_J, parity)
    assert tab.n_ch == 18
    gch = _gpu_channels(wpcd, wl, two_J, parity)
    grid = wpcd.wpcd_grid_create(p, p)
    m = wpcd.build_perm(grid, gch, wl.n_quad)
    torch.cuda.synchronize()
    assert m.rows == 18 * 100 * 100
    geo_ptr, geo_col = operm.geo_pattern(p, p)
    assert np.array_equal(m.geo_row_ptr.cpu().numpy().astype(np.int64), geo_ptr)
    rp = operm.full_row_ptr(geo_ptr, tab, n, n)
    assert np.array_equal(m.row_ptr.cpu().numpy(), rp) and m.nnz == rp[-1]
    erow = np.repeat(np.arange(n_geo), np.diff(geo_ptr))
    val, aval = operm.element_values(p, p, erow // n, erow % n, geo_col // n, geo_col % n, wl.n_quad, tab)     # [nnz_geo, pairs]
    gv, gci = m.values.cpu().numpy(), m.col_idx.cpu().numpy()
    pair_of = -np.ones((tab.n_ch, tab.n_ch), np.int64)
    pair_of[tab.gamma, tab.gammap] = np.arange(tab.n_pairs)
    cnt_e, pos_e = (geo_ptr[erow + 1] - geo_ptr[erow]), np.arange(len(erow)) - geo_ptr[erow]
    vmax = np.abs(val).max()
    chk = _ValueCheck("test_cfg3_nd_half_plus_full")
    for g in range(tab.n_ch):
        coupled = np.nonzero(tab.mask[g])[0]
        for t, gp in enumerate(coupled):
            dst = rp[g * n_geo + erow] + t * cnt_e + pos_e                 # where entry (g, r; gp, c) sits in the CSR
            assert np.array_equal(gci[dst], gp * n_geo + geo_col)
            chk.add(gv[dst], val[:, pair_of[g, gp]], aval[:, pair_of[g, gp]], vmax, where=f"pair ({g},{gp})")
    chk.close(n_p=n, n_q=n, n_quad=wl.n_quad, rule=0, nnz=int(m.nnz), channels=18)
    del val, aval
    xh = wi.normal_vector(m.rows, k=333)
    xd = torch.from_numpy(xh).cuda()
    y_csr, y_blk = torch.empty_like(xd), torch.empty_like(xd)
    wpcd.wpcd_perm_apply(m.rows, m.row_ptr, m.col_idx, m.values, xd, y_csr)
    wpcd.wpcd_perm_apply_blocked(grid, gch, m.row_ptr, m.geo_row_ptr, m.col_idx, m.values, xd, y_blk)
    ref = operm.spmv(rp, gci, gv, xh)
    scale = operm.spmv(rp, gci, np.abs(gv), np.abs(xh))
    assert np.all(np.abs(y_csr.cpu().numpy() - ref) <= 1e-12 * scale + 1e-300)
    assert np.all(np.abs(y_blk.cpu().numpy() - ref) <= 1e-12 * scale + 1e-300)


@pytest.mark.parametrize("two_J,parity,stride", [(1, 1, 397), (1, -1, 523), (3, 1, 1499), (3, -1, 1301)])
def test_cfg4_sampled(wpcd, two_J, parity, stride):
    """Config 4 (N = 150, j <= 3): all four J^pi matrices, full pattern, sampled geometric rows of every channel."""
    wl = wi.WORKLOADS["cfg4"]
    p = wl.grid()
    tab = _oracle_table(wl, two_J, parity)
    _compare_sampled(wpcd, p, wl.n_quad, _gpu_channels(wpcd, wl, two_J, parity), tab, np.arange(11, wl.n_bins ** 2, stride),
                     tag=f"test_cfg4_sampled[{two_J}/2,{'+' if parity > 0 else '-'}]")


@pytest.mark.parametrize("two_J,parity,stride", [(1, 1, 1201), (1, -1, 1103), (3, 1, 1801), (3, -1, 1709), (5, 1, 2399), (5, -1, 2203),
                                                 (7, 1, 2609), (7, -1, 2503)])
def test_cfg5_sampled(wpcd, two_J, parity, stride):
    """Config 5 (N = 150, j <= 3): all eight J^pi matrices; 7/2- is the largest (62 channels, 3.2e9 nonzeros, 39 GB: offsets
    beyond 2^31)."""
    wl = wi.WORKLOADS["cfg5"]
    p = wl.grid()
    tab = _oracle_table(wl, two_J, parity)
    m, worst = _compare_sampled(wpcd, p, wl.n_quad, _gpu_channels(wpcd, wl, two_J, parity), tab, np.arange(5, wl.n_bins ** 2, stride),
                                tag=f"test_cfg5_sampled[{two_J}/2,{'+' if parity > 0 else '-'}]")
    if (two_J, parity) == (7, -1):
        assert m.nnz > 2_000_000_000


@pytest.mark.parametrize("two_J,parity,jmax,nb,n", [(7, -1, 3, 8, 10), (1, 1, 2, 12, 8), (5, 1, 3, 6, 10)])
def test_first_bin_cells_against_extended_precision(wpcd, two_J, parity, jmax, nb, n):
    """on cells that touch p = 0 or p' = 0 the single (k,l1,l1') terms of pairs with l, l' >= 2 are huge and
    only their sum is small.  The oracle sums the terms per node, the CUDA path integrates monomial moments first and
    contracts with g afterwards (R8).  Against the SAME rule evaluated in long double (oracle built with
    -DWPO_EXTENDED) the CUDA values must be no further off than FP64 rounding of the absolute term sum allows, and not
    systematically worse than the FP64 oracle's own per-node sum: the moments-then-contract schedule loses no digits."""
    torch = _torch()
    chs = och.enumerate_channels(two_J, parity, jmax)
    tab = operm.PairTable(chs, och.g_table(chs, two_J, 1))
    gch = wpcd.wpcd_channels_create(wpcd.WPCD_ND, two_J=two_J, parity=parity, two_T=1, j_pair_max=jmax)
    p = wi.tan2_grid(nb)
    grid = wpcd.wpcd_grid_create(p, p)
    m = wpcd.build_perm(grid, gch, n)
    torch.cuda.synchronize()
    geo_ptr, geo_col = operm.geo_pattern(p, p)
    n_geo = nb * nb
    erow = np.repeat(np.arange(n_geo), np.diff(geo_ptr))
    v64, a64 = operm.element_values(p, p, erow // nb, erow % nb, geo_col // nb, geo_col % nb, n, tab)
    vex, _ = operm.element_values(p, p, erow // nb, erow % nb, geo_col // nb, geo_col % nb, n, tab, extended=True)
    rp = operm.full_row_ptr(geo_ptr, tab, nb, nb)
    gv = m.values.cpu().numpy()
    cnt_e, pos_e = (geo_ptr[erow + 1] - geo_ptr[erow]), np.arange(len(erow)) - geo_ptr[erow]
    vg = np.empty_like(v64)
    for c in range(tab.n_pairs):
        g, gp = tab.gamma[c], tab.gammap[c]
        t = int(np.nonzero(np.nonzero(tab.mask[g])[0] == gp)[0][0])
        vg[:, c] = gv[rp[g * n_geo + erow] + t * cnt_e + pos_e]
    first_bin = ((erow // nb == 0) | (geo_col // nb == 0))[:, None] & ((tab.pair_l >= 2) & (tab.pair_lp >= 2))[None, :]
    assert first_bin.sum() > 100
    eps = 2.0 ** -53
    e_gpu, e_64 = np.abs(vg - vex)[first_bin], np.abs(v64 - vex)[first_bin]
    ae, vx = a64[first_bin], np.abs(vex)[first_bin]
    cond = ae / np.maximum(vx, 1e-300)
    assert np.median(cond) > 10 and cond.max() > 1e6                   # these ARE the ill-conditioned entries
    # entry by entry: a few dozen roundings of the absolute sum, with the same constant for both FP64 evaluations
    # (measured worst: 13 eps A_e on the device, 9.6 eps A_e for the oracle; the parity tolerance 1e-11 A_e is 9e4 eps A_e)
    assert np.all(e_64 <= 64 * eps * ae) and np.all(e_gpu <= 64 * eps * ae), (np.max(e_64 / (eps * ae)), np.max(e_gpu / (eps * ae)))
    # entry by entry against the oracle's own deviation: |v_gpu - v_ext| <= 1e-11 |v_ext| + c max(|v_64 - v_ext|, eps A_e)
    bound = 1e-11 * vx + 64.0 * np.maximum(e_64, eps * ae)
    assert np.all(e_gpu <= bound), np.max(e_gpu / bound)
    # on the whole: the CUDA schedule is not worse than the per-node sum (rms of the errors in units of eps A_e)
    rms_gpu, rms_64 = np.sqrt(np.mean((e_gpu / (eps * ae)) ** 2)), np.sqrt(np.mean((e_64 / (eps * ae)) ** 2))
    print("PARITY " + json.dumps({"test": "test_first_bin_cells_against_extended_precision", "J2": two_J, "parity": parity, "n_bins": nb,
                                  "entries": int(first_bin.sum()), "median_cond": float(np.median(cond)), "max_cond": float(cond.max()),
                                  "rms_err_gpu_eps_Ae": float(rms_gpu), "rms_err_oracle64_eps_Ae": float(rms_64),
                                  "max_err_gpu_eps_Ae": float(np.max(e_gpu / (eps * ae))), "max_err_oracle64_eps_Ae": float(np.max(e_64 / (eps * ae)))}))
    path = os.environ.get("WPCD_PARITY_REPORT")
    if path:
        with open(path, "a") as f:
            f.write(json.dumps({"test": "first_bin_extended", "J2": two_J, "parity": parity, "n_bins": nb, "entries": int(first_bin.sum()),
                                "median_cond": float(np.median(cond)), "max_cond": float(cond.max()), "rms_err_gpu_eps_Ae": float(rms_gpu),
                                "rms_err_oracle64_eps_Ae": float(rms_64), "max_err_gpu_eps_Ae": float(np.max(e_gpu / (eps * ae))),
                                "max_err_oracle64_eps_Ae": float(np.max(e_64 / (eps * ae)))}) + "\n")
    # measured: 1.0 - 1.2 eps A_e on the device (moments in FP64 MMA order, then the contraction), 0.3 - 0.5 for the per-node sum
    assert rms_gpu <= 2.5 and rms_gpu <= 6.0 * rms_64


def test_coupled_wide_classes_from_table(wpcd):
    """A user table whose (l,l') = (5,5) pair uses far more than 32 distinct (k, A) monomials: the
    contraction cuts such a class into pieces handled in successive passes (store, then add)."""
    rng = np.random.default_rng(20140521)
    chan_l = [5, 2, 0]
    pairs = []
    for ga in range(3):
        for gb in range(3):
            if (ga, gb) == (2, 1):
                continue                      # one uncoupled pair
            l, lp = chan_l[ga], chan_l[gb]
            terms = [(k, l1, l1p, float(rng.uniform(-1, 1)))
                     for l1 in range(l + 1) for l1p in range(lp + 1) for k in range(0, 8)]
            pairs.append((ga, gb, terms))
    chs = [(l, 0, 0, 0, 0, 0) for l in chan_l]
    tab = operm.PairTable(chs, pairs)
    n_mono = len({(t[1] + t[2], t[0]) for t in pairs[0][2]})
    assert n_mono > 64                        # (5,5): A = 0..10, k = 0..7 -> 88 monomials, 3 passes
    gch = wpcd.wpcd_channels_create_from_table(np.array(chan_l), tab.gamma, tab.gammap, tab.term_ptr,
                                               tab.term_k, tab.term_l1, tab.term_l1p, tab.term_g)
    p = wi.tan2_grid(4, 1.0, 0.1, seed=41)
    q = wi.tan2_grid(5, 0.7, 0.1, seed=42)
    _compare_full(wpcd, p, q, 6, gch, tab)


@pytest.mark.parametrize("n_quad", [1, 5, 8, 16, 33, 64])
def test_coupled_quadrature_orders(wpcd, n_quad):
    # phi-node groups, masked MMA rows (n not a multiple of 4), n > 32 lanes
    chs = och.enumerate_channels(3, -1, 2)
    tab = operm.PairTable(chs, och.g_table(chs, 3, 1))
    gch = wpcd.wpcd_channels_create(wpcd.WPCD_ND, two_J=3, parity=-1, two_T=1, j_pair_max=2)
    p = wi.tan2_grid(4, 1.0, 0.1, seed=51)
    _compare_full(wpcd, p, p, n_quad, gch, tab)


def test_apply_long_rows_pipelined(wpcd):
    """Coupled matrix with mean row length >= 128: the software-pipelined SpMV variant (HBM-streaming
    path of configs 3-5), 1, 2 and 4 right-hand sides, against the sequential oracle product."""
    torch = _torch()
    gch = wpcd.wpcd_channels_create(wpcd.WPCD_ND, two_J=3, parity=1, two_T=1, j_pair_max=2)
    p = wi.tan2_grid(10, 1.0, 0.1, seed=61)
    grid = wpcd.wpcd_grid_create(p, p)
    m = wpcd.build_perm(grid, gch, 6)
    rows = m.rows
    assert m.nnz / rows >= 128
    rp, ci, v = m.row_ptr.cpu().numpy(), m.col_idx.cpu().numpy(), m.values.cpu().numpy()
    for n_vec in (1, 2, 4, 5):
        xh = np.stack([wi.normal_vector(rows, k=70 + k) for k in range(n_vec)])
        x = torch.from_numpy(xh).cuda().contiguous()
        y = torch.empty_like(x)
        wpcd.wpcd_perm_apply(rows, m.row_ptr, m.col_idx, m.values, x, y, n_vec=n_vec)
        for k in range(n_vec):
            ref = operm.spmv(rp, ci, v, xh[k])
            scale = operm.spmv(rp, ci, np.abs(v), np.abs(xh[k]))
            assert np.all(np.abs(y[k].cpu().numpy() - ref) <= 1e-12 * scale + 1e-300)


def test_full_size_properties_cfg2_and_cfg3(wpcd):
    """Properties that hold at any size, checked on the GPU result at full size: the matrix of the
    Hermitian operator P in a real basis is symmetric (pattern exactly, values to rounding), the
    columns ascend strictly inside every row, and the spectrum of the s-wave matrix g0*P lies in
    [-g0, 2 g0] (checked through its largest eigenvalue by power iteration with the CUDA SpMV)."""
    torch = _torch()
    import scipy.sparse as sp

    wl = wi.WORKLOADS["cfg2"]
    p = wl.grid()
    grid = wpcd.wpcd_grid_create(p, p)
    m = wpcd.build_perm(grid, _gpu_channels(wpcd, wl), wl.n_quad)
    rp, ci, v = m.row_ptr.cpu().numpy(), m.col_idx.cpu().numpy(), m.values.cpu().numpy()
    assert np.all(np.diff(rp) >= 0)
    inner = np.ones(len(ci), bool)
    inner[rp[:-1][np.diff(rp) > 0]] = False                 # first entry of every non-empty row
    assert np.all(np.diff(ci)[inner[1:]] > 0)               # strictly ascending inside rows
    A = sp.csr_matrix((v, ci, rp), shape=(m.rows, m.rows))
    D = (A - A.T).tocsr()
    assert D.nnz == 0 or np.abs(D.data).max() <= 1e-12 * np.abs(v).max()
    assert (A != 0).astype(np.int8).nnz == ((A + A.T) != 0).astype(np.int8).nnz      # symmetric pattern
    x = torch.from_numpy(wi.normal_vector(m.rows, k=5)).cuda()
    y = torch.empty_like(x)
    lam = 0.0
    for _ in range(60):
        wpcd.wpcd_perm_apply(m.rows, m.row_ptr, m.col_idx, m.values, x, y)
        lam = float(torch.dot(x, y) / torch.dot(x, x))
        x = y / torch.linalg.norm(y)
    assert -wl.g0 - 1e-9 <= lam <= 2.0 * wl.g0 + 1e-9 and lam > 0.9 * wl.g0      # top of the spectrum ~ g0 * 2... of the s-wave block ~ g0
    # cfg3 (18 channels): full pattern symmetry from the row pointer and a symmetric-value sample
    wl3 = wi.WORKLOADS["cfg3"]
    p3 = wl3.grid()
    grid3 = wpcd.wpcd_grid_create(p3, p3)
    m3 = wpcd.build_perm(grid3, _gpu_channels(wpcd, wl3, 1, 1), wl3.n_quad)
    rp3 = m3.row_ptr.cpu().numpy()
    rng = np.random.default_rng(7)
    rows = rng.integers(0, m3.rows, 200)
    # values are symmetric up to the rounding of rule R(n), which on cells touching p = 0 or p' = 0 is
    # amplified by the cancellation between the (k,l1,l1') terms (R8, R9): absolute scale
    vmax = float(m3.values.abs().max().item())
    for r in rows:
        lo, hi = rp3[r], rp3[r + 1]
        if hi == lo:
            continue
        k = int(rng.integers(lo, hi))
        c = int(m3.col_idx[k].item())
        val = float(m3.values[k].item())
        cl, ch = rp3[c], rp3[c + 1]
        cols_c = m3.col_idx[cl:ch].cpu().numpy()
        pos = np.searchsorted(cols_c, r)
        assert pos < len(cols_c) and cols_c[pos] == r                      # (c, r) is stored too
        vt = float(m3.values[cl + pos].item())
        assert abs(vt - val) <= 1e-10 * abs(val) + 1e-6 * vmax


def test_apply_complex(wpcd):
    """y = P0 x for complex vectors (interleaved re/im): against two real oracle products, on a short-row
    s-wave matrix and on a long-row coupled matrix (pipelined variant), with 1 and 3 vectors."""
    torch = _torch()
    cases = []
    p = wi.tan2_grid(24, 1.0, 0.1, seed=8)
    cases.append(wpcd.build_perm(wpcd.wpcd_grid_create(p, p), wpcd.wpcd_channels_create(wpcd.WPCD_SPINLESS_SWAVE, g0=0.5), 8))
    p2 = wi.tan2_grid(10, 1.0, 0.1, seed=61)
    cases.append(wpcd.build_perm(wpcd.wpcd_grid_create(p2, p2),
                                 wpcd.wpcd_channels_create(wpcd.WPCD_ND, two_J=3, parity=1, two_T=1, j_pair_max=2), 6))
    for m in cases:
        rows = m.rows
        rp, ci, v = m.row_ptr.cpu().numpy(), m.col_idx.cpu().numpy(), m.values.cpu().numpy()
        for n_vec in (1, 3):
            xr = np.stack([wi.normal_vector(rows, k=200 + k) for k in range(n_vec)])
            xi_ = np.stack([wi.normal_vector(rows, k=300 + k) for k in range(n_vec)])
            x = torch.from_numpy(xr + 1j * xi_).cuda().contiguous()
            y = torch.empty_like(x)
            wpcd.wpcd_perm_apply_complex(rows, m.row_ptr, m.col_idx, m.values, x, y, n_vec=n_vec)
            yh = y.cpu().numpy()
            for k in range(n_vec):
                for part, src in ((yh[k].real, xr[k]), (yh[k].imag, xi_[k])):
                    ref = operm.spmv(rp, ci, v, src)
                    scale = operm.spmv(rp, ci, np.abs(v), np.abs(src))
                    assert np.all(np.abs(part - ref) <= 1e-12 * scale + 1e-300)


def test_coupled_edge_grids(wpcd):
    """Coupled channels on lattices that do not start at zero, with very uneven bins and n_p != n_q."""
    chs = och.enumerate_channels(1, -1, 1)
    tab = operm.PairTable(chs, och.g_table(chs, 1, 1))
    gch = wpcd.wpcd_channels_create(wpcd.WPCD_ND, two_J=1, parity=-1, two_T=1, j_pair_max=1)
    cases = [
        (np.array([0.3, 0.5, 2.0]), np.array([0.1, 0.2, 0.9, 4.0])),
        (np.array([0.0, 1e-3, 1.0, 50.0]), np.array([0.0, 2.0])),
        (np.array([0.0, 0.37]), np.array([0.0, 0.37])),
    ]
    for p, q in cases:
        _compare_full(wpcd, p, q, 7, gch, tab)


def test_handle_state_between_count_and_build(wpcd):
    """The selection staged in the grid handle by wpcd_perm_count serves any later wpcd_perm_build on that
    grid (the geometric pattern does not depend on the channel set); a handle that was never counted runs
    the selection inside wpcd_perm_build."""
    torch = _torch()
    p = wi.tan2_grid(7, 1.0, 0.1, seed=71)
    q = wi.tan2_grid(6, 0.9, 0.1, seed=72)
    chs_a = och.enumerate_channels(1, 1, 1)
    tab_a = operm.PairTable(chs_a, och.g_table(chs_a, 1, 1))
    ch_s, pairs_s = och.spinless_swave_table(0.5)
    tab_s = operm.PairTable(ch_s, pairs_s)
    g_a = wpcd.wpcd_channels_create(wpcd.WPCD_ND, two_J=1, parity=1, two_T=1, j_pair_max=1)
    g_s = wpcd.wpcd_channels_create(wpcd.WPCD_SPINLESS_SWAVE, g0=0.5)
    grid = wpcd.wpcd_grid_create(p, q)
    n_geo = grid.n_p * grid.n_q

    def buffers(ch):
        rows = wpcd.wpcd_rows(grid, ch)
        return (torch.empty(rows + 1, dtype=torch.int64, device="cuda"), torch.empty(n_geo + 1, dtype=torch.int32, device="cuda"))

    rp_a, geo_a = buffers(g_a)
    rp_s, geo_s = buffers(g_s)
    nnz_a, nnz_geo = wpcd.wpcd_perm_count(grid, g_a, 6, rp_a, geo_a)
    nnz_s, nnz_geo2 = wpcd.wpcd_perm_count(grid, g_s, 6, rp_s, geo_s)     # second count before the first build
    assert nnz_geo == nnz_geo2
    out = {}
    for name, ch, rp, geo, nnz in (("a", g_a, rp_a, geo_a, nnz_a), ("s", g_s, rp_s, geo_s, nnz_s)):
        ws = torch.empty(max(256, wpcd.wpcd_perm_workspace_bytes(ch, nnz_geo)), dtype=torch.uint8, device="cuda")
        col = torch.empty(nnz, dtype=torch.int32, device="cuda")
        val = torch.empty(nnz, dtype=torch.float64, device="cuda")
        wpcd.wpcd_perm_build(grid, ch, 6, rp, geo, ws, col, val)
        out[name] = (rp.cpu().numpy(), col.cpu().numpy(), val.cpu().numpy())
    # a fresh handle on the same nodes, never counted: build must run the selection itself
    grid2 = wpcd.wpcd_grid_create(p, q)
    ws = torch.empty(max(256, wpcd.wpcd_perm_workspace_bytes(g_a, nnz_geo)), dtype=torch.uint8, device="cuda")
    col2 = torch.empty(nnz_a, dtype=torch.int32, device="cuda")
    val2 = torch.empty(nnz_a, dtype=torch.float64, device="cuda")
    wpcd.wpcd_perm_build(grid2, g_a, 6, rp_a, geo_a, ws, col2, val2)
    torch.cuda.synchronize()
    assert np.array_equal(col2.cpu().numpy(), out["a"][1]) and np.array_equal(val2.cpu().numpy(), out["a"][2])
    for name, tab in (("a", tab_a), ("s", tab_s)):
        rp, ci, v, av = operm.build_csr(p, q, 6, tab)
        assert np.array_equal(out[name][0], rp) and np.array_equal(out[name][1], ci)
        tol = VALUE_RTOL * np.maximum(np.abs(v), av) + VALUE_FLOOR * np.abs(v).max()
        assert np.all(np.abs(out[name][2] - v) <= tol)


@pytest.mark.parametrize("n_quad", [2, 5, 8, 16, 33])
def test_split_rule_swave(wpcd, n_quad):
    """the kink-split rule RS(n) (R14), s-wave kernel, same pattern, values 1e-11 against the
    oracle at the same rule: jittered lattices with p != q, first-bin cells, a single cell, grids away from zero."""
    ch, pairs = och.spinless_swave_table(0.5)
    tab = operm.PairTable(ch, pairs)
    gch = wpcd.wpcd_channels_create(wpcd.WPCD_SPINLESS_SWAVE, g0=0.5)
    cases = [(wi.tan2_grid(9, 1.0, 0.1, seed=21), wi.tan2_grid(7, 0.6, 0.1, seed=22)),
             (np.array([0.0, 0.37]), np.array([0.0, 0.37])),
             (np.array([0.3, 0.5, 2.0]), np.array([0.1, 0.2, 0.9, 4.0]))]
    if n_quad == 8:
        wl = wi.WORKLOADS["cfg1"]
        cases.append((wl.grid(), wl.grid()))
    for p, q in cases:
        _compare_full(wpcd, p, q, n_quad, gch, tab, split=True)


@pytest.mark.parametrize("two_J,parity,jmax,nb,nq", [(1, 1, 1, 6, 6), (1, -1, 2, 5, 4), (3, 1, 2, 4, 8), (5, -1, 3, 3, 10), (1, 1, 2, 4, 33)])
def test_split_rule_coupled(wpcd, two_J, parity, jmax, nb, nq):
    """The kink-split rule through the coupled path (moments on the FP64 tensor cores + contraction): the u-pieces of a
    phi-node are staged as extra node slots, several rounds per element."""
    chs = och.enumerate_channels(two_J, parity, jmax)
    tab = operm.PairTable(chs, och.g_table(chs, two_J, 1))
    gch = wpcd.wpcd_channels_create(wpcd.WPCD_ND, two_J=two_J, parity=parity, two_T=1, j_pair_max=jmax)
    p = wi.tan2_grid(nb, 1.0, 0.1, seed=31)
    q = wi.tan2_grid(nb + 1, 0.8, 0.1, seed=32)
    _compare_full(wpcd, p, q, nq, gch, tab, split=True)


@pytest.mark.parametrize("n_quad", [1, 4, 8, 9, 32])
def test_analytic_u_rule_swave(wpcd, n_quad):
    """rule RA(n) (R15), the u-integral of every kink-split piece in closed form; values 1e-11
    against the oracle at the same rule; odd orders put a phi-node on pi/4 (b1 = b2) on the symmetric cells."""
    ch, pairs = och.spinless_swave_table(0.5)
    tab = operm.PairTable(ch, pairs)
    gch = wpcd.wpcd_channels_create(wpcd.WPCD_SPINLESS_SWAVE, g0=0.5)
    cases = [(wi.tan2_grid(9, 1.0, 0.1, seed=21), wi.tan2_grid(7, 0.6, 0.1, seed=22)),
             (np.array([0.0, 0.37]), np.array([0.0, 0.37])),
             (np.array([0.3, 0.5, 2.0]), np.array([0.1, 0.2, 0.9, 4.0])),
             (wi.tan2_grid(12, 1.0, 0.0), wi.tan2_grid(12, 1.0, 0.0))]
    if n_quad == 8:
        wl = wi.WORKLOADS["cfg1"]
        cases.append((wl.grid(), wl.grid()))
    for p, q in cases:
        _compare_full(wpcd, p, q, n_quad, gch, tab, split=2)


def test_analytic_u_rule_needs_swave(wpcd):
    gch = wpcd.wpcd_channels_create(wpcd.WPCD_ND, two_J=1, parity=1, two_T=1, j_pair_max=1)
    p = wi.tan2_grid(4, 1.0, 0.1, seed=1)
    grid = wpcd.wpcd_grid_create(p, p)
    with pytest.raises(wpcd.WpcdError, match="s-wave"):
        wpcd.build_perm(grid, gch, 8 | wpcd.WPCD_RULE_ANALYTIC_U)


def test_split_rule_is_more_accurate(wpcd):
    """RS(8) on the device against the oracle's RS(64): ten times closer than R(8) (the accuracy claim of DESIGN.md R14)."""
    ch, pairs = och.spinless_swave_table(1.0)
    tab = operm.PairTable(ch, pairs)
    gch = wpcd.wpcd_channels_create(wpcd.WPCD_SPINLESS_SWAVE, g0=1.0)
    p = wi.tan2_grid(12, 1.0, 0.1, seed=3)
    ref = operm.build_csr(p, p, 64, tab, split=True)[2]
    grid = wpcd.wpcd_grid_create(p, p)
    plain = wpcd.build_perm(grid, gch, 8).values.cpu().numpy()
    split = wpcd.build_perm(grid, gch, 8 | wpcd.WPCD_RULE_KINK_SPLIT).values.cpu().numpy()
    e_plain = np.linalg.norm(plain - ref) / np.linalg.norm(ref)
    e_split = np.linalg.norm(split - ref) / np.linalg.norm(ref)
    assert 1.5e-3 < e_split < 2.3e-3 and e_plain > 8 * e_split


def test_bound_count_build_callables(wpcd):
    """bind_count_build: the same two C calls with their arguments marshalled once (what bench.py's step loop uses)."""
    torch = _torch()
    gch = wpcd.wpcd_channels_create(wpcd.WPCD_SPINLESS_SWAVE, g0=0.5)
    p = wi.tan2_grid(17, 1.0, 0.1, seed=5)
    grid = wpcd.wpcd_grid_create(p, p)
    ref = wpcd.build_perm(grid, gch, 8)
    row_ptr, geo_row_ptr = torch.zeros_like(ref.row_ptr), torch.zeros_like(ref.geo_row_ptr)
    col_idx, values = torch.zeros_like(ref.col_idx), torch.zeros_like(ref.values)
    workspace = torch.empty(max(wpcd.wpcd_perm_workspace_bytes(gch, ref.nnz_geo), 256), dtype=torch.uint8, device="cuda")
    count, build = wpcd.bind_count_build(grid, gch, 8, row_ptr, geo_row_ptr, workspace, col_idx, values, torch.cuda.current_stream())
    for _ in range(3):
        col_idx.zero_(); values.zero_()
        assert count() == (ref.nnz, ref.nnz_geo)
        build()
        torch.cuda.synchronize()
        assert torch.equal(row_ptr, ref.row_ptr) and torch.equal(col_idx, ref.col_idx) and torch.equal(values, ref.values)


def test_count_and_build_on_different_streams(wpcd):
    """wpcd_perm_count returns once the selection is read back, its row-pointer expansion still queued on the count's stream;
    a build issued on ANOTHER stream is ordered behind it by the library (coupled channels: the contraction reads row_ptr)."""
    torch = _torch()
    gch = wpcd.wpcd_channels_create(wpcd.WPCD_ND, two_J=1, parity=1, two_T=1, j_pair_max=2)
    p = wi.tan2_grid(24, 1.0, 0.1, seed=77)
    grid = wpcd.wpcd_grid_create(p, p)
    ref = wpcd.build_perm(grid, gch, 6)
    torch.cuda.synchronize()
    s_count, s_build = torch.cuda.Stream(), torch.cuda.Stream()
    rows = ref.rows
    for _ in range(5):
        row_ptr = torch.zeros(rows + 1, dtype=torch.int64, device="cuda")
        geo_row_ptr = torch.zeros(24 * 24 + 1, dtype=torch.int32, device="cuda")
        col_idx = torch.zeros(ref.nnz, dtype=torch.int32, device="cuda")
        values = torch.zeros(ref.nnz, dtype=torch.float64, device="cuda")
        workspace = torch.empty(max(wpcd.wpcd_perm_workspace_bytes(gch, ref.nnz_geo), 256), dtype=torch.uint8, device="cuda")
        torch.cuda.synchronize()
        nnz, nnz_geo = wpcd.wpcd_perm_count(grid, gch, 6, row_ptr, geo_row_ptr, s_count)
        assert (nnz, nnz_geo) == (ref.nnz, ref.nnz_geo)
        wpcd.wpcd_perm_build(grid, gch, 6, row_ptr, geo_row_ptr, workspace, col_idx, values, s_build)
        s_build.synchronize()
        s_count.synchronize()
        assert torch.equal(row_ptr, ref.row_ptr) and torch.equal(col_idx, ref.col_idx) and torch.equal(values, ref.values)


def test_concurrent_builds_of_different_orders(wpcd):
    """Two builds with different quadrature orders (8 and 10: configs 1-3 and 4-5) in flight at the same time on two
    streams and two grid handles: each launch carries its own rule, so neither disturbs the other (the rule
    used to sit in one __constant__ bank per translation unit)."""
    torch = _torch()
    gch = wpcd.wpcd_channels_create(wpcd.WPCD_ND, two_J=1, parity=1, two_T=1, j_pair_max=2)
    sw = wpcd.wpcd_channels_create(wpcd.WPCD_SPINLESS_SWAVE, g0=0.5)
    p = wi.tan2_grid(30, 1.0, 0.1, seed=77)
    for ch in (gch, sw):
        grids = [wpcd.wpcd_grid_create(p, p), wpcd.wpcd_grid_create(p, p)]
        refs = [wpcd.build_perm(grids[0], ch, 8), wpcd.build_perm(grids[1], ch, 10)]
        torch.cuda.synchronize()
        assert not torch.equal(refs[0].values, refs[1].values)
        streams = [torch.cuda.Stream(), torch.cuda.Stream()]
        for _ in range(4):
            outs = []
            for k, nq in enumerate((8, 10)):
                rp, geo = torch.empty_like(refs[k].row_ptr), torch.empty_like(refs[k].geo_row_ptr)
                nnz, nnz_geo = wpcd.wpcd_perm_count(grids[k], ch, nq, rp, geo, streams[k])
                ws = torch.empty(max(wpcd.wpcd_perm_workspace_bytes(ch, nnz_geo), 256), dtype=torch.uint8, device="cuda")
                outs.append((rp, geo, ws, torch.zeros(nnz, dtype=torch.int32, device="cuda"), torch.zeros(nnz, dtype=torch.float64, device="cuda")))
            torch.cuda.synchronize()
            for rep in range(3):                  # several builds back to back on both streams, interleaved from the host
                for k, nq in enumerate((8, 10)):
                    rp, geo, ws, ci, va = outs[k]
                    wpcd.wpcd_perm_build(grids[k], ch, nq, rp, geo, ws, ci, va, streams[k])
            torch.cuda.synchronize()
            for k in range(2):
                assert torch.equal(outs[k][3], refs[k].col_idx) and torch.equal(outs[k][4], refs[k].values), k


def test_builds_and_products_from_two_host_threads(wpcd):
    """Two host threads, each with its own stream, grid handle and channel set (different table sizes, so different
    shared-memory sizes of the same kernels), build and multiply at the same time: the results are those of the serial calls
    (the dynamic shared-memory limit of a kernel is only ever raised, under a lock)."""
    import threading

    torch = _torch()
    sets = [dict(two_J=1, parity=1, j_pair_max=1), dict(two_J=5, parity=-1, j_pair_max=3)]
    p = wi.tan2_grid(12, 1.0, 0.1, seed=91)
    work = []
    for kw in sets:
        grid = wpcd.wpcd_grid_create(p, p)
        gch = wpcd.wpcd_channels_create(wpcd.WPCD_ND, two_T=1, **kw)
        ref = wpcd.build_perm(grid, gch, 8)
        x = torch.from_numpy(np.stack([wi.normal_vector(ref.rows, k=1500 + k) for k in range(8)])).cuda()
        y_ref = torch.empty_like(x)
        wpcd.wpcd_perm_apply_blocked(grid, gch, ref.row_ptr, ref.geo_row_ptr, ref.col_idx, ref.values, x, y_ref, n_vec=8)
        work.append((grid, gch, ref, x, y_ref))
    torch.cuda.synchronize()
    errors = []

    def run(k):
        try:
            grid, gch, ref, x, y_ref = work[k]
            st = torch.cuda.Stream()
            with torch.cuda.stream(st):
                for _ in range(6):
                    m = wpcd.build_perm(grid, gch, 8, stream=st)
                    y = torch.empty_like(x)
                    wpcd.wpcd_perm_apply_blocked(grid, gch, m.row_ptr, m.geo_row_ptr, m.col_idx, m.values, x, y, n_vec=8, stream=st)
                    st.synchronize()
                    assert torch.equal(m.col_idx, ref.col_idx) and torch.equal(m.values, ref.values), k
                    assert torch.equal(y, y_ref), k
        except BaseException as e:   # noqa: BLE001 -- reported in the main thread
            errors.append((k, repr(e)))

    threads = [threading.Thread(target=run, args=(k,)) for k in range(2)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert not errors, errors


def test_apply_ignores_columns_a_row_does_not_reference(wpcd):
    """x[0] = inf / nan must not leak into rows that do not reference column 0 (padding slots of the batched loads used to
    multiply 0 * x[0]); every product variant, short and long rows."""
    torch = _torch()
    rng = np.random.default_rng(5)
    for rows, short, long_ in ((300, 3, 70), (400, 9, 300)):
        lens = np.full(rows, short, dtype=np.int64)
        lens[::5] = long_
        rp = np.zeros(rows + 1, dtype=np.int64)
        rp[1:] = np.cumsum(lens)
        nnz = int(rp[-1])
        ci = rng.integers(1, rows, nnz).astype(np.int32)          # no entry in column 0
        v = rng.standard_normal(nnz)
        rpd, cid, vd = torch.from_numpy(rp).cuda(), torch.from_numpy(ci).cuda(), torch.from_numpy(v).cuda()
        for bad in (np.inf, np.nan):
            xs = np.stack([wi.normal_vector(rows, k=40 + k) for k in range(4)])
            xs[:, 0] = bad
            x = torch.from_numpy(xs).cuda()
            for n_vec in (1, 2, 4):
                y = torch.empty(n_vec, rows, dtype=torch.float64, device="cuda")
                wpcd.wpcd_perm_apply(rows, rpd, cid, vd, x[:n_vec].contiguous(), y, n_vec)
                assert torch.isfinite(y).all()
            xc = torch.from_numpy((xs[0] + 1j * xs[1])[None, :].copy()).cuda()
            yc = torch.empty_like(xc)
            wpcd.wpcd_perm_apply_complex(rows, rpd, cid, vd, xc, yc, 1)
            assert torch.isfinite(torch.view_as_real(yc)).all()
            xi = torch.from_numpy(np.ascontiguousarray(xs.T)).cuda()
            yi = torch.empty_like(xi)
            wpcd.wpcd_perm_apply_interleaved(rows, rpd, cid, vd, xi, yi)
            assert torch.isfinite(yi).all()
            ych = torch.empty(3, rows, dtype=torch.float64, device="cuda")
            wpcd.wpcd_perm_apply_chain(rows, rpd, cid, vd, x[0].contiguous(), ych, 1)
            assert torch.isfinite(ych[0]).all()


def test_apply_interleaved(wpcd):
    """Four (and two) real vectors stored interleaved [rows][n_inter]: one gather per entry; short-row and long-row matrices."""
    torch = _torch()
    cases = []
    p = wi.tan2_grid(24, 1.0, 0.1, seed=8)
    cases.append(wpcd.build_perm(wpcd.wpcd_grid_create(p, p), wpcd.wpcd_channels_create(wpcd.WPCD_SPINLESS_SWAVE, g0=0.5), 8))
    p2 = wi.tan2_grid(10, 1.0, 0.1, seed=61)
    cases.append(wpcd.build_perm(wpcd.wpcd_grid_create(p2, p2),
                                 wpcd.wpcd_channels_create(wpcd.WPCD_ND, two_J=3, parity=1, two_T=1, j_pair_max=2), 6))
    for m in cases:
        rows = m.rows
        rp, ci, v = m.row_ptr.cpu().numpy(), m.col_idx.cpu().numpy(), m.values.cpu().numpy()
        for n_inter in (2, 4):
            xh = np.stack([wi.normal_vector(rows, k=500 + k) for k in range(n_inter)], axis=1).copy()    # [rows, n_inter]
            x = torch.from_numpy(xh).cuda().contiguous()
            y = torch.empty_like(x)
            wpcd.wpcd_perm_apply_interleaved(rows, m.row_ptr, m.col_idx, m.values, x, y)
            yh = y.cpu().numpy()
            for k in range(n_inter):
                ref = operm.spmv(rp, ci, v, np.ascontiguousarray(xh[:, k]))
                scale = operm.spmv(rp, ci, np.abs(v), np.abs(np.ascontiguousarray(xh[:, k])))
                assert np.all(np.abs(yh[:, k] - ref) <= 1e-12 * scale + 1e-300)


def test_apply_row_length_sweep(wpcd):
    """Foreign CSR arrays with controlled row lengths (empty rows, one batch, batch boundaries +-1, several batches,
    pipelined long rows): every lane-count variant of the plain, multi-vector, complex and interleaved products
    against the oracle's row-by-row product."""
    torch = _torch()
    rng = np.random.default_rng(77)
    for rows, short, long_ in ((500, 4, 4), (500, 4, 33), (500, 9, 64), (500, 9, 65), (500, 0, 129), (500, 20, 257),
                              (700, 40, 300), (1200, 150, 600)):
        lens = np.full(rows, short, dtype=np.int64)
        lens[::7] = long_
        rp = np.zeros(rows + 1, dtype=np.int64)
        rp[1:] = np.cumsum(lens)
        nnz = int(rp[-1])
        ci = rng.integers(0, rows, nnz).astype(np.int32)
        v = rng.standard_normal(nnz)
        rpd, cid, vd = torch.from_numpy(rp).cuda(), torch.from_numpy(ci).cuda(), torch.from_numpy(v).cuda()
        xs = np.stack([wi.normal_vector(rows, k=700 + k) for k in range(4)])                 # [4, rows]
        refs = [operm.spmv(rp, ci, v, xs[k]) for k in range(4)]
        scales = [operm.spmv(rp, ci, np.abs(v), np.abs(xs[k])) for k in range(4)]

        def check(got, k):
            assert np.all(np.abs(got - refs[k]) <= 1e-12 * scales[k] + 1e-300), (rows, short, long_, k)

        xs11 = np.stack([xs[k % 4] * (1.0 + 0.25 * (k // 4)) for k in range(11)])          # 11 right-hand sides: passes of 4, 4, 2, 1
        x11 = torch.from_numpy(xs11).cuda()
        y11 = torch.full_like(x11, np.nan)
        wpcd.wpcd_perm_apply(rows, rpd, cid, vd, x11, y11, 11)
        for k in range(11):
            got = y11[k].cpu().numpy() / (1.0 + 0.25 * (k // 4))
            assert np.all(np.abs(got - refs[k % 4]) <= 2e-12 * scales[k % 4] + 1e-300), (rows, short, long_, k)
        for n_vec in (1, 2, 3, 4):
            x = torch.from_numpy(xs[:n_vec].copy()).cuda()
            y = torch.full_like(x, np.nan)
            wpcd.wpcd_perm_apply(rows, rpd, cid, vd, x, y, n_vec)
            for k in range(n_vec):
                check(y[k].cpu().numpy(), k)
        xc = torch.from_numpy((xs[0] + 1j * xs[1])[None, :].copy()).cuda()
        yc = torch.full_like(xc, np.nan)
        wpcd.wpcd_perm_apply_complex(rows, rpd, cid, vd, xc, yc, 1)
        check(yc[0].real.cpu().numpy(), 0)
        check(yc[0].imag.cpu().numpy(), 1)
        for n_inter in (2, 4):
            xi = torch.from_numpy(np.ascontiguousarray(xs[:n_inter].T)).cuda()              # [rows, n_inter]
            yi = torch.full_like(xi, np.nan)
            wpcd.wpcd_perm_apply_interleaved(rows, rpd, cid, vd, xi, yi)
            yh = yi.cpu().numpy()
            for k in range(n_inter):
                check(yh[:, k], k)


def test_apply_blocked(wpcd):
    """The product through the block structure of P0 (only the first block's column indices of a row are read): against
    the oracle's row-by-row product on coupled matrices (several J^pi, p != q, few and many geometric entries per row, more
    than 32 coupled channels), the s-wave matrix (one block per row) and a lattice with empty rows."""
    torch = _torch()
    cases = []
    for two_J, parity, jmax, nb in ((1, 1, 1, 6), (3, 1, 2, 9), (5, -1, 3, 4), (1, -1, 2, 14)):
        gch = wpcd.wpcd_channels_create(wpcd.WPCD_ND, two_J=two_J, parity=parity, two_T=1, j_pair_max=jmax)
        cases.append((gch, wi.tan2_grid(nb, 1.0, 0.1, seed=41), wi.tan2_grid(nb + 2, 0.8, 0.1, seed=42), 4))
    sw = wpcd.wpcd_channels_create(wpcd.WPCD_SPINLESS_SWAVE, g0=0.5)
    cases.append((sw, wi.tan2_grid(40, 1.0, 0.1, seed=8), wi.tan2_grid(40, 1.0, 0.1, seed=8), 8))
    cases.append((sw, np.array([0.0, 0.1, 0.2, 5.0, 5.1]), np.array([0.0, 0.05, 3.0]), 8))
    gch = wpcd.wpcd_channels_create(wpcd.WPCD_ND, two_J=1, parity=1, two_T=1, j_pair_max=1)
    cases.append((gch, np.array([0.0, 0.1, 0.2, 5.0, 5.1]), np.array([0.0, 0.05, 3.0]), 4))
    for gch, p, q, n_quad in cases:
        grid = wpcd.wpcd_grid_create(p, q)
        m = wpcd.build_perm(grid, gch, n_quad)
        rp, ci, v = m.row_ptr.cpu().numpy(), m.col_idx.cpu().numpy(), m.values.cpu().numpy()
        xs = np.stack([wi.normal_vector(m.rows, k=800 + k) for k in range(3)])
        x = torch.from_numpy(xs).cuda()
        y = torch.full_like(x, np.nan)
        wpcd.wpcd_perm_apply_blocked(grid, gch, m.row_ptr, m.geo_row_ptr, m.col_idx, m.values, x, y, n_vec=3)
        yh = y.cpu().numpy()
        xh_pin = torch.from_numpy(xs).pin_memory()
        yh_pin = torch.full((3, m.rows), np.nan, dtype=torch.float64).pin_memory()
        wpcd.wpcd_perm_apply_blocked_host(grid, gch, m.row_ptr, m.geo_row_ptr, m.col_idx, m.values, xh_pin, yh_pin, torch.empty_like(x),
                                          torch.empty_like(x), n_vec=3)
        for k in range(3):
            ref = operm.spmv(rp, ci, v, xs[k])
            scale = operm.spmv(rp, ci, np.abs(v), np.abs(xs[k]))
            assert np.all(np.abs(yh[k] - ref) <= 1e-12 * scale + 1e-300), (gch.count, len(p), k)
            assert np.array_equal(yh_pin[k].numpy(), yh[k])            # same kernel, same summation order


def test_apply_blocked_chunked_paths(wpcd):
    """The same product with a tiny x tile (wpcd_debug_set): geometric rows cut into column chunks, channels into channel
    chunks, runs of coupled channels split at chunk boundaries; 1 .. 15 vectors per call (scalar passes of 1 and 2 vectors,
    tensor-core passes of 3 .. 8; with "blocked_no_mma" the scalar passes of 4 and 8 vectors)."""
    torch = _torch()
    gch = wpcd.wpcd_channels_create(wpcd.WPCD_ND, two_J=3, parity=1, two_T=1, j_pair_max=2)
    p, q = wi.tan2_grid(9, 1.0, 0.1, seed=41), wi.tan2_grid(11, 0.8, 0.1, seed=42)
    grid = wpcd.wpcd_grid_create(p, q)
    m = wpcd.build_perm(grid, gch, 4)
    rp, ci, v = m.row_ptr.cpu().numpy(), m.col_idx.cpu().numpy(), m.values.cpu().numpy()
    try:
        for tile, no_mma in ((0, 0), (7, 0), (40, 0), (256, 0), (0, 1), (40, 1)):
            wpcd.wpcd_debug_set("blocked_tile_doubles", tile)
            wpcd.wpcd_debug_set("blocked_no_mma", no_mma)          # 1: the scalar passes of 4 and 8 vectors as well
            for n_vec in (1, 2, 3, 5, 6, 9, 12, 15):
                xs = np.stack([wi.normal_vector(m.rows, k=820 + k) for k in range(n_vec)])
                x = torch.from_numpy(xs).cuda()
                y = torch.full((n_vec + 1, m.rows), np.nan, dtype=torch.float64, device="cuda")    # one guard vector behind
                wpcd.wpcd_perm_apply_blocked(grid, gch, m.row_ptr, m.geo_row_ptr, m.col_idx, m.values, x, y, n_vec=n_vec)
                yh = y.cpu().numpy()
                assert np.all(np.isnan(yh[n_vec])), (tile, n_vec)      # a pass padded to 8 vectors writes only those asked for
                for k in range(n_vec):
                    ref = operm.spmv(rp, ci, v, xs[k])
                    scale = operm.spmv(rp, ci, np.abs(v), np.abs(xs[k]))
                    assert np.all(np.abs(yh[k] - ref) <= 1e-12 * scale + 1e-300), (tile, n_vec, k)
    finally:
        wpcd.wpcd_debug_set("blocked_tile_doubles", 0)
        wpcd.wpcd_debug_set("blocked_no_mma", 0)


def test_dynamic_shared_memory_just_under_the_default_limit(wpcd):
    """A launch whose DYNAMIC shared memory is within a few bytes below 48 KB while static + dynamic is above it: the
    opt-in limit has to be raised although the dynamic part alone would fit the default (10 channels, one vector, x tile of
    4089 doubles: 12 * 4089 + 8 * 10 = 49 148 bytes + 16 static)."""
    torch = _torch()
    gch = wpcd.wpcd_channels_create(wpcd.WPCD_ND, two_J=1, parity=1, two_T=1, j_pair_max=1)
    assert gch.count == 10
    p = wi.tan2_grid(8, 1.0, 0.1, seed=95)
    grid = wpcd.wpcd_grid_create(p, p)
    m = wpcd.build_perm(grid, gch, 4)
    xs = wi.normal_vector(m.rows, k=1700)
    x = torch.from_numpy(xs[None, :].copy()).cuda()
    y0, y1 = torch.empty_like(x), torch.full_like(x, np.nan)
    wpcd.wpcd_perm_apply_blocked(grid, gch, m.row_ptr, m.geo_row_ptr, m.col_idx, m.values, x, y0)
    try:
        wpcd.wpcd_debug_set("blocked_tile_doubles", 4089)
        wpcd.wpcd_perm_apply_blocked(grid, gch, m.row_ptr, m.geo_row_ptr, m.col_idx, m.values, x, y1)
    finally:
        wpcd.wpcd_debug_set("blocked_tile_doubles", 0)
    torch.cuda.synchronize()
    assert torch.equal(y0, y1)


def _chain_check(wpcd, torch, rows, rp, ci, v, rpd, cid, vd, n_iter, tag):
    xh = wi.normal_vector(rows, k=900)
    x = torch.from_numpy(xh).cuda()
    y = torch.full((n_iter, rows), np.nan, dtype=torch.float64, device="cuda")
    wpcd.wpcd_perm_apply_chain(rows, rpd, cid, vd, x, y, n_iter)
    yh = y.cpu().numpy()
    ref, scale = xh, np.abs(xh)
    av = np.abs(v)
    for k in range(n_iter):
        ref = operm.spmv(rp, ci, v, ref)
        scale = operm.spmv(rp, ci, av, scale)                   # |P0|^k |x|: what rounding errors are relative to
        assert np.all(np.abs(yh[k] - ref) <= (k + 1) * 2e-12 * scale + 1e-300), (tag, k)


def test_apply_chain(wpcd):
    """The dependent products y_k = P0 y_{k-1} in one cooperative launch (matrix slices resident in shared memory, grid
    barrier between products) against the oracle's product applied n_iter times; also the slices that do not fit
    (one very long row), empty rows, and a matrix too large for the scheme (ordinary products)."""
    torch = _torch()
    for n_bins, n_iter in ((24, 7), (50, 20), (100, 50)):      # N = 50 lies in the window where the fused launch is the default
        p = wi.tan2_grid(n_bins, 1.0, 0.1, seed=8)
        m = wpcd.build_perm(wpcd.wpcd_grid_create(p, p), wpcd.wpcd_channels_create(wpcd.WPCD_SPINLESS_SWAVE, g0=0.5), 8)
        rp, ci, v = m.row_ptr.cpu().numpy(), m.col_idx.cpu().numpy(), m.values.cpu().numpy()
        _chain_check(wpcd, torch, m.rows, rp, ci, v, m.row_ptr, m.col_idx, m.values, n_iter, ("swave", n_bins))
    p2 = wi.tan2_grid(10, 1.0, 0.1, seed=61)
    m = wpcd.build_perm(wpcd.wpcd_grid_create(p2, p2), wpcd.wpcd_channels_create(wpcd.WPCD_ND, two_J=3, parity=1, two_T=1, j_pair_max=2), 6)
    rp, ci, v = m.row_ptr.cpu().numpy(), m.col_idx.cpu().numpy(), m.values.cpu().numpy()
    _chain_check(wpcd, torch, m.rows, rp, ci, v, m.row_ptr, m.col_idx, m.values, 5, "coupled")
    rng = np.random.default_rng(78)
    for rows, short, long_, every, n_iter, tag in ((3000, 6, 40000, 2999, 4, "one long row"), (5000, 0, 60, 3, 6, "empty rows"),
                                                  (40000, 90, 90, 1, 3, "too large: ordinary products"), (37, 3, 3, 1, 1, "n_iter 1")):
        lens = np.full(rows, short, dtype=np.int64)
        lens[::every] = long_
        rp = np.zeros(rows + 1, dtype=np.int64)
        rp[1:] = np.cumsum(lens)
        nnz = int(rp[-1])
        ci = rng.integers(0, rows, nnz).astype(np.int32)
        v = rng.standard_normal(nnz) / np.sqrt(max(short, 1) + long_ / every)
        _chain_check(wpcd, torch, rows, rp, ci, v, torch.from_numpy(rp).cuda(), torch.from_numpy(ci).cuda(), torch.from_numpy(v).cuda(),
                     n_iter, tag)


def test_apply_chain_fused_everywhere(wpcd):
    """The same chain cases with the fused cooperative launch forced on for every matrix that fits on chip, and forced off."""
    try:
        for mode in (1, 2):
            wpcd.wpcd_debug_set("chain_mode", mode)
            test_apply_chain(wpcd)
    finally:
        wpcd.wpcd_debug_set("chain_mode", 0)


def test_apply_forced_variants(wpcd):
    """Every lanes-per-row variant of the CSR product on the same matrices (wpcd_debug_set), with and without the pipelined
    long-row path and programmatic dependent launch."""
    try:
        for lanes in (4, 8, 16, 32):
            wpcd.wpcd_debug_set("spmv_lanes_per_row", lanes)
            test_apply_multi_vector_and_host(wpcd)
        wpcd.wpcd_debug_set("spmv_lanes_per_row", 0)
        wpcd.wpcd_debug_set("spmv_no_pipeline", 1)
        wpcd.wpcd_debug_set("no_pdl", 1)
        test_apply_long_rows_pipelined(wpcd)
        with pytest.raises(wpcd.WpcdError, match="unknown key"):
            wpcd.wpcd_debug_set("no_such_switch", 1)
    finally:
        for key in ("spmv_lanes_per_row", "spmv_no_pipeline", "no_pdl"):
            wpcd.wpcd_debug_set(key, 0)


def test_block_apply_and_kernel_apply(wpcd):
    """batched dense blocks (FP64 MMA) and the factored kernel K = O P0 O^T V1 G1 against
    the numpy oracle, on a lattice whose block sizes are not multiples of the 32 x 32 tile."""
    torch = _torch()
    from oracle import kernel_apply as oka

    gch = wpcd.wpcd_channels_create(wpcd.WPCD_ND, two_J=1, parity=1, two_T=1, j_pair_max=1)
    p = wi.tan2_grid(37, 1.0, 0.1, seed=91)
    q = wi.tan2_grid(9, 0.8, 0.1, seed=92)
    grid = wpcd.wpcd_grid_create(p, q)
    m = wpcd.build_perm(grid, gch, 4)
    n_ch, n_p, n_q, rows = gch.count, 37, 9, m.rows
    assert rows == n_ch * n_p * n_q
    o, v, g1 = wi.kernel_factors(n_ch, n_p, n_q)
    od, vd = torch.from_numpy(o).cuda(), torch.from_numpy(v).cuda()
    # block apply alone: real and complex, plain and transposed
    xr = wi.normal_vector(rows, k=400)
    xc = xr + 1j * wi.normal_vector(rows, k=401)
    for xh in (xr, xc):
        for tr in (False, True):
            x = torch.from_numpy(xh).cuda()
            y = torch.empty_like(x)
            wpcd.wpcd_block_apply(n_ch, n_p, n_q, od, x, y, transpose=tr)
            ref = oka.block_apply(o, xh, n_ch, n_p, n_q, transpose=tr)
            scale = oka.block_apply(np.abs(o), np.abs(xh), n_ch, n_p, n_q, transpose=tr)
            assert np.all(np.abs(y.cpu().numpy() - ref) <= 1e-13 * scale + 1e-300)
    # the whole kernel, on the GPU-built CSR
    rp, ci, vals = m.row_ptr.cpu().numpy(), m.col_idx.cpu().numpy(), m.values.cpu().numpy()
    x = torch.from_numpy(xc).cuda()
    y = torch.empty_like(x)
    scratch = torch.empty(2 * rows, dtype=torch.complex128, device="cuda")
    wpcd.wpcd_kernel_apply(n_ch, n_p, n_q, m.row_ptr, m.col_idx, m.values, od, vd, torch.from_numpy(g1).cuda(), x, y, scratch)
    ref = oka.kernel_apply(rp, ci, vals, o, v, g1, xc, n_ch, n_p, n_q)
    scale = oka.kernel_apply(rp, ci, np.abs(vals), np.abs(o), np.abs(v), np.abs(g1), np.abs(xc).astype(np.float64), n_ch, n_p, n_q)
    assert np.all(np.abs(y.cpu().numpy() - ref) <= 1e-12 * np.abs(scale) + 1e-300)


def test_neumann_terms_and_pade(wpcd):
    """the iteration of eq. (12) on the device and its Pade sum, against the oracle's terms and
    the direct dense solve, for a kernel scaled beyond the unit disc (the plain series diverges)."""
    torch = _torch()
    from oracle import kernel_apply as oka

    gch = wpcd.wpcd_channels_create(wpcd.WPCD_ND, two_J=1, parity=1, two_T=1, j_pair_max=1)
    p = wi.tan2_grid(4, 1.0, 0.1, seed=81)
    q = wi.tan2_grid(3, 0.9, 0.1, seed=82)
    m = wpcd.build_perm(wpcd.wpcd_grid_create(p, q), gch, 6)
    n_ch, n_p, n_q, rows = gch.count, 4, 3, m.rows
    rp, ci, vals = m.row_ptr.cpu().numpy(), m.col_idx.cpu().numpy(), m.values.cpu().numpy()
    o, v, g1 = wi.kernel_factors(n_ch, n_p, n_q)
    K = np.array([oka.kernel_apply(rp, ci, vals, o, v, g1, np.eye(rows)[:, c].astype(np.complex128), n_ch, n_p, n_q)
                  for c in range(rows)]).T
    rho_scale = 1.3 / np.abs(np.linalg.eigvals(K)).max()
    g1 = g1 * rho_scale
    b = wi.normal_vector(rows, k=5) + 1j * wi.normal_vector(rows, k=6)
    element, n_terms = 7, 36
    terms = wpcd.wpcd_neumann_terms(n_ch, n_p, n_q, m.row_ptr, m.col_idx, m.values, torch.from_numpy(o).cuda(),
                                    torch.from_numpy(v).cuda(), torch.from_numpy(g1).cuda(), torch.from_numpy(b).cuda(),
                                    element, n_terms)
    ref = oka.neumann_terms(rp, ci, vals, o, v, g1, b, element, n_terms, n_ch, n_p, n_q)
    growth = np.maximum.accumulate(np.abs(ref))
    assert np.all(np.abs(terms - ref) <= 1e-10 * growth * np.arange(1, n_terms + 1))
    exact = np.linalg.solve(np.eye(rows) - K * rho_scale, b)[element]
    # same table on both sides for the same input terms; the sum itself is as accurate as an epsilon table of
    # 36 terms can be for 120 poles with |lambda| up to 1.3 (the plain series is off by orders of magnitude)
    assert abs(wpcd.wpcd_pade_sum(terms) - oka.pade_sum(terms)) < 1e-8 * max(1.0, abs(exact))
    assert abs(wpcd.wpcd_pade_sum(terms) - exact) < 2e-3 * max(1.0, abs(exact))
    assert abs(np.sum(terms) - exact) > 1e2 * abs(exact)


def test_coupled_limits_of_the_table(wpcd):
    """The largest orbital momentum and Legendre order the header allows (WPCD_MAX_L = 7, WPCD_MAX_K = 23)."""
    rng = np.random.default_rng(20140522)
    chan_l = [7, 3]
    pairs = []
    for ga in range(2):
        for gb in range(2):
            l, lp = chan_l[ga], chan_l[gb]
            terms = [(k, l1, l1p, float(rng.uniform(-1, 1)))
                     for l1 in range(0, l + 1, 2) for l1p in range(0, lp + 1) for k in (0, 5, 11, 23)]
            pairs.append((ga, gb, terms))
    chs = [(l, 0, 0, 0, 0, 0) for l in chan_l]
    tab = operm.PairTable(chs, pairs)
    gch = wpcd.wpcd_channels_create_from_table(np.array(chan_l), tab.gamma, tab.gammap, tab.term_ptr,
                                               tab.term_k, tab.term_l1, tab.term_l1p, tab.term_g)
    p = np.array([0.2, 0.5, 1.1, 2.0])          # away from p = 0: the single terms of l = 7 are not integrable there
    q = np.array([0.1, 0.6, 1.4])
    _compare_full(wpcd, p, q, 5, gch, tab)


class _Guarded:
    """A device buffer with sentinel bands in front of it and behind it (compute-sanitizer is closed on the GPU pool: this is
    the bounds check the tests can make themselves)."""
    BAND = 4096         # bytes

    def __init__(self, torch, n, dtype):
        self.item = torch.empty(0, dtype=dtype).element_size()
        self.g = self.BAND // self.item
        self.full = torch.empty(n + 2 * self.g, dtype=dtype, device="cuda")
        self.full.view(torch.uint8).fill_(0xA5)
        self.view = self.full[self.g:self.g + n]
        self.torch = torch

    def intact(self):
        b = self.full.view(self.torch.uint8)
        n = self.BAND
        return bool((b[:n] == 0xA5).all().item()) and bool((b[b.numel() - n:] == 0xA5).all().item())


@pytest.mark.parametrize("model", ["swave", "nd"])
def test_no_write_outside_the_buffers(wpcd, model):
    """Every output buffer of count / build / the products sits between sentinel bands that must come back untouched, and
    the matrix built into them is the one of the ordinary path.  Sizes are ragged on purpose (7 x 9 cells, n = 10; the
    coupled set has 18 channels: partial element tiles, a partial moment chunk, partial row groups of the tensor-core product)."""
    torch = _torch()
    p, q = wi.tan2_grid(7, 1.0, 0.1, seed=51), wi.tan2_grid(9, 0.9, 0.1, seed=52)
    grid = wpcd.wpcd_grid_create(p, q)
    if model == "swave":
        gch = wpcd.wpcd_channels_create(wpcd.WPCD_SPINLESS_SWAVE, g0=0.5)
    else:
        gch = wpcd.wpcd_channels_create(wpcd.WPCD_ND, two_J=1, parity=1, two_T=1, j_pair_max=2)
    ref = wpcd.build_perm(grid, gch, 10)
    rows, n_geo = ref.rows, (len(p) - 1) * (len(q) - 1)
    row_ptr, geo_row_ptr = _Guarded(torch, rows + 1, torch.int64), _Guarded(torch, n_geo + 1, torch.int32)
    nnz, nnz_geo = wpcd.wpcd_perm_count(grid, gch, 10, row_ptr.view, geo_row_ptr.view)
    assert (nnz, nnz_geo) == (ref.nnz, ref.nnz_geo)
    col_idx, values = _Guarded(torch, nnz, torch.int32), _Guarded(torch, nnz, torch.float64)
    ws = _Guarded(torch, max(wpcd.wpcd_perm_workspace_bytes(gch, nnz_geo), 256), torch.uint8)
    wpcd.wpcd_perm_build(grid, gch, 10, row_ptr.view, geo_row_ptr.view, ws.view, col_idx.view, values.view)
    torch.cuda.synchronize()
    for name, b in (("row_ptr", row_ptr), ("geo_row_ptr", geo_row_ptr), ("col_idx", col_idx), ("values", values), ("workspace", ws)):
        assert b.intact(), name
    assert torch.equal(row_ptr.view, ref.row_ptr) and torch.equal(geo_row_ptr.view, ref.geo_row_ptr)
    assert torch.equal(col_idx.view, ref.col_idx) and torch.equal(values.view, ref.values)
    # the products: y between bands, every pass width of both products
    for n_vec in (1, 2, 3, 4, 5, 8, 11):
        x = torch.from_numpy(np.stack([wi.normal_vector(rows, k=1300 + k) for k in range(n_vec)])).cuda()
        y = _Guarded(torch, n_vec * rows, torch.float64)
        wpcd.wpcd_perm_apply(rows, row_ptr.view, col_idx.view, values.view, x, y.view, n_vec=n_vec)
        torch.cuda.synchronize()
        assert y.intact(), ("apply", n_vec)
        y_csr = y.view.clone()
        assert bool(torch.isfinite(y_csr).all().item())
        if model == "nd":
            y = _Guarded(torch, n_vec * rows, torch.float64)
            wpcd.wpcd_perm_apply_blocked(grid, gch, row_ptr.view, geo_row_ptr.view, col_idx.view, values.view, x, y.view, n_vec=n_vec)
            torch.cuda.synchronize()
            assert y.intact(), ("apply_blocked", n_vec)
            scale = float(torch.abs(y_csr).max().item())
            assert float(torch.abs(y.view - y_csr).max().item()) <= 1e-12 * max(scale, 1.0) * 50
    y = _Guarded(torch, 6 * rows, torch.float64)
    wpcd.wpcd_perm_apply_chain(rows, row_ptr.view, col_idx.view, values.view, x[0].contiguous(), y.view, 6)
    torch.cuda.synchronize()
    assert y.intact(), "apply_chain"
