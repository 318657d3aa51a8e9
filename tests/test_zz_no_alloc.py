"""wpcd_perm_apply_blocked_noalloc: the blocked product whose scratch is a fixed device array of the library (no cudaMalloc of
any kind inside the call) against the existing path wpcd_perm_apply_blocked, and against the oracle's product.

Collected last on purpose (file name): the suite runs with pytest -x."""
import numpy as np
import pytest

import wpcd_inputs as wi
from oracle import perm as operm

pytestmark = pytest.mark.gpu

SPMV_RTOL = 1e-12       # times sum_j |a_ij x_j|: the tolerance of every product test in tests/test_gpu_parity.py


def _matrix(wpcd, n_p, n_q, two_J, parity, jmax, n_quad, seed):
    p, q = wi.tan2_grid(n_p, 1.0, 0.1, seed=seed), wi.tan2_grid(n_q, 0.9, 0.1, seed=seed + 1)
    grid = wpcd.wpcd_grid_create(p, q)
    gch = wpcd.wpcd_channels_create(wpcd.WPCD_ND, two_J=two_J, parity=parity, two_T=1, j_pair_max=jmax)
    return grid, gch, wpcd.build_perm(grid, gch, n_quad)


def test_noalloc_product_matches_the_existing_path_twice_in_a_row(wpcd):
    import torch

    assert torch.cuda.is_available(), "needs a CUDA device"
    # two matrices of different size, one after the other through the SAME scratch array: the second call must see nothing of
    # the first (18 channels on 11 x 13 cells, then 10 channels on 7 x 9 cells: fewer rows, so stale words lie behind its data)
    cases = [_matrix(wpcd, 11, 13, 1, +1, 2, 8, 61), _matrix(wpcd, 7, 9, 1, +1, 1, 6, 63)]
    for rep in range(2):
        for ci, (grid, gch, m) in enumerate(cases):
            rp, ci_, v = m.row_ptr.cpu().numpy(), m.col_idx.cpu().numpy(), m.values.cpu().numpy()
            for n_vec in (8, 5, 1):
                xs = np.stack([wi.normal_vector(m.rows, k=2000 + 16 * ci + k + rep) for k in range(n_vec)])
                x = torch.from_numpy(xs).cuda()
                y_ref = torch.full((n_vec, m.rows), np.nan, dtype=torch.float64, device="cuda")
                wpcd.wpcd_perm_apply_blocked(grid, gch, m.row_ptr, m.geo_row_ptr, m.col_idx, m.values, x, y_ref, n_vec=n_vec)
                ys = []
                for _ in range(2):                                         # two calls in a row
                    y = torch.full((n_vec + 1, m.rows), np.nan, dtype=torch.float64, device="cuda")   # one guard vector behind
                    wpcd.wpcd_perm_apply_blocked_noalloc(grid, gch, m.row_ptr, m.geo_row_ptr, m.col_idx, m.values, x, y, n_vec=n_vec)
                    ys.append(y.cpu().numpy())
                assert np.array_equal(ys[0], ys[1], equal_nan=True)        # deterministic, nothing left over from the call before
                assert np.all(np.isnan(ys[0][n_vec])), "wrote behind the vectors asked for"
                yr = y_ref.cpu().numpy()
                for k in range(n_vec):
                    ref = operm.spmv(rp, ci_, v, xs[k])
                    scale = operm.spmv(rp, ci_, np.abs(v), np.abs(xs[k]))
                    assert np.all(np.abs(ys[0][k] - yr[k]) <= SPMV_RTOL * scale + 1e-300), (rep, ci, n_vec, k)
                    assert np.all(np.abs(ys[0][k] - ref) <= SPMV_RTOL * scale + 1e-300), (rep, ci, n_vec, k)
                if n_vec >= 3:                                             # the existing path takes the same kernel: same bits
                    assert np.array_equal(ys[0][:n_vec], yr)


def test_noalloc_rejects_what_does_not_fit(wpcd):
    import torch

    grid, gch, m = _matrix(wpcd, 7, 9, 1, +1, 1, 6, 63)
    x = torch.zeros(9, m.rows, dtype=torch.float64, device="cuda")
    y = torch.zeros_like(x)
    with pytest.raises(wpcd.WpcdError, match="at most 8 vectors"):
        wpcd.wpcd_perm_apply_blocked_noalloc(grid, gch, m.row_ptr, m.geo_row_ptr, m.col_idx, m.values, x, y, n_vec=9)
    # 10 channels x 170 x 170 cells = 289 000 rows > WPCD_NOALLOC_MAX_ROWS: refused before any pointer is looked at
    big = wpcd.wpcd_grid_create(wi.tan2_grid(170, 1.0), wi.tan2_grid(170, 1.0))
    assert wpcd.wpcd_rows(big, gch) > wpcd.WPCD_NOALLOC_MAX_ROWS
    with pytest.raises(wpcd.WpcdError, match="WPCD_NOALLOC_MAX_ROWS"):
        wpcd.wpcd_perm_apply_blocked_noalloc(big, gch, m.row_ptr, m.geo_row_ptr, m.col_idx, m.values, x, y, n_vec=1)
    wpcd.wpcd_perm_apply_blocked_noalloc(grid, gch, m.row_ptr, m.geo_row_ptr, m.col_idx, m.values, x, y, n_vec=0)     # nothing to do
