"""paper_1404_5253_b200 -- thin Python binding of libwpcd (include/wpcd.h).

Argument marshalling only: every step of the hot path (pattern selection, scan,
CSR fill by FP64 quadrature of (A15), SpMV) runs in the CUDA kernels of
``csrc/``.  PyTorch is used for device memory and streams, nothing else.
There is no CPU fallback: if ``libwpcd.so`` is missing or no CUDA device is
present, compute calls raise ``WpcdError``.

Function names mirror the C-ABI (PAPER.md citations live in include/wpcd.h):
    wpcd_grid_create, wpcd_channels_create, wpcd_channels_create_from_table,
    wpcd_perm_count, wpcd_perm_workspace_bytes, wpcd_perm_build, wpcd_perm_apply,
    wpcd_perm_apply_host, wpcd_perm_apply_complex, wpcd_fp64_peak, wpcd_launch_count.
``build_perm`` strings count -> allocate -> build together and returns a ``PermCSR``.
"""
import ctypes
import os
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libwpcd.so")

WPCD_SPINLESS_SWAVE = 0
WPCD_ND = 1
WPCD_RULE_KINK_SPLIT = 0x100   # OR into n_quad: kink-split rule RS(n) (R14)
WPCD_RULE_ANALYTIC_U = 0x200   # OR into n_quad: rule RA(n), exact x-integral, s-wave only (R15)
WPCD_MAX_QUAD = 64
WPCD_NOALLOC_MAX_ROWS = 262144   # rows wpcd_perm_apply_blocked_noalloc accepts (its fixed 16 MiB scratch array)

EXPORTS = [
    "wpcd_last_error", "wpcd_grid_create", "wpcd_grid_destroy", "wpcd_channels_create",
    "wpcd_channels_create_from_table", "wpcd_channels_destroy", "wpcd_channels_count", "wpcd_channels_pairs",
    "wpcd_channels_terms", "wpcd_channels_monomials", "wpcd_channels_coefficients", "wpcd_channels_get_quantum_numbers", "wpcd_channels_get_table", "wpcd_rows",
    "wpcd_geo_rows", "wpcd_perm_count", "wpcd_perm_workspace_bytes", "wpcd_perm_build", "wpcd_perm_apply",
    "wpcd_perm_apply_host", "wpcd_perm_apply_complex", "wpcd_perm_apply_interleaved", "wpcd_perm_apply_chain", "wpcd_perm_apply_blocked", "wpcd_perm_apply_blocked_noalloc", "wpcd_perm_apply_blocked_host", "wpcd_block_apply", "wpcd_kernel_apply", "wpcd_neumann_terms",
    "wpcd_pade_sum", "wpcd_fp64_peak", "wpcd_launch_count", "wpcd_trace_enable", "wpcd_trace_read", "wpcd_debug_set",
]
TRACE_STAGES = ["geo_count", "scan", "geo_index", "fill_swave", "moments", "contract"]


class WpcdError(RuntimeError):
    pass


_lib = None


def load():
    """dlopen libwpcd.so (built in-tree by ``paper_1404_5253_b200.build``); fail loudly if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise WpcdError(f"{LIB_PATH} not found: run `python -m paper_1404_5253_b200.build` (nvcc, sm_100a); "
                        "there is no CPU fallback")
    L = ctypes.CDLL(LIB_PATH)
    vp, i32, i64, dbl, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_int64, ctypes.c_double, ctypes.c_size_t
    L.wpcd_last_error.restype = ctypes.c_char_p
    L.wpcd_grid_create.argtypes = [vp, i32, vp, i32, ctypes.POINTER(vp)]
    L.wpcd_grid_destroy.argtypes = [vp]
    L.wpcd_grid_destroy.restype = None
    L.wpcd_channels_create.argtypes = [i32, i32, i32, i32, i32, dbl, ctypes.POINTER(vp)]
    L.wpcd_channels_create_from_table.argtypes = [i32, vp, i32, vp, vp, vp, vp, vp, vp, vp, ctypes.POINTER(vp)]
    L.wpcd_channels_destroy.argtypes = [vp]
    L.wpcd_channels_destroy.restype = None
    L.wpcd_channels_count.argtypes = [vp]
    L.wpcd_channels_pairs.argtypes = [vp]
    L.wpcd_channels_terms.argtypes = [vp]
    L.wpcd_channels_terms.restype = i64
    L.wpcd_channels_monomials.argtypes = [vp]
    L.wpcd_channels_coefficients.argtypes = [vp]
    L.wpcd_channels_coefficients.restype = i64
    L.wpcd_channels_get_quantum_numbers.argtypes = [vp, vp]
    L.wpcd_channels_get_table.argtypes = [vp] * 8
    L.wpcd_rows.argtypes = [vp, vp]
    L.wpcd_rows.restype = i64
    L.wpcd_geo_rows.argtypes = [vp]
    L.wpcd_geo_rows.restype = i64
    L.wpcd_perm_count.argtypes = [vp, vp, i32, vp, vp, vp, ctypes.POINTER(i64), ctypes.POINTER(i64)]
    L.wpcd_perm_workspace_bytes.argtypes = [vp, i64]
    L.wpcd_perm_workspace_bytes.restype = sz
    L.wpcd_perm_build.argtypes = [vp, vp, i32, vp, vp, vp, vp, sz, vp, vp]
    L.wpcd_perm_apply.argtypes = [i64, vp, vp, vp, vp, vp, i32, vp]
    L.wpcd_perm_apply_host.argtypes = [i64, vp, vp, vp, vp, vp, i32, vp, vp, vp]
    L.wpcd_perm_apply_complex.argtypes = [i64, vp, vp, vp, vp, vp, i32, vp]
    L.wpcd_perm_apply_interleaved.argtypes = [i64, vp, vp, vp, vp, vp, i32, vp]
    L.wpcd_perm_apply_blocked.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, i32, vp]
    L.wpcd_perm_apply_blocked_noalloc.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, i32, vp]
    L.wpcd_perm_apply_blocked_host.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, i32, vp, vp, vp]
    L.wpcd_perm_apply_chain.argtypes = [i64, vp, vp, vp, vp, vp, i32, vp]
    L.wpcd_block_apply.argtypes = [i32, i32, i32, vp, i32, vp, vp, i32, vp]
    L.wpcd_kernel_apply.argtypes = [i32, i32, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    L.wpcd_neumann_terms.argtypes = [i32, i32, i32, vp, vp, vp, vp, vp, vp, vp, i64, i32, vp, vp, vp]
    L.wpcd_pade_sum.argtypes = [vp, i32, vp]
    L.wpcd_fp64_peak.argtypes = [vp, ctypes.POINTER(dbl)]
    L.wpcd_launch_count.restype = i64
    L.wpcd_trace_enable.argtypes = [i32]
    L.wpcd_trace_read.argtypes = [vp, vp]
    L.wpcd_debug_set.argtypes = [ctypes.c_char_p, i64]
    _lib = L
    return L


def _check(status):
    if status != 0:
        raise WpcdError(f"wpcd status {status}: {load().wpcd_last_error().decode()}")


def _stream_ptr(stream):
    if stream is None:
        import torch

        return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    if isinstance(stream, int):
        return ctypes.c_void_p(stream)
    return ctypes.c_void_p(stream.cuda_stream)


def _dev_ptr(t, dtype=None):
    if t is None:
        return ctypes.c_void_p(0)
    assert t.is_cuda and t.is_contiguous(), "device tensors must be contiguous CUDA tensors"
    if dtype is not None:
        assert t.dtype == dtype, f"expected {dtype}, got {t.dtype}"
    return ctypes.c_void_p(t.data_ptr())


class Grid:
    def __init__(self, handle, n_p, n_q):
        self.handle, self.n_p, self.n_q = handle, n_p, n_q

    def __del__(self):
        if getattr(self, "handle", None) and _lib is not None:
            _lib.wpcd_grid_destroy(self.handle)
            self.handle = None


class Channels:
    def __init__(self, handle):
        self.handle = handle

    def __del__(self):
        if getattr(self, "handle", None) and _lib is not None:
            _lib.wpcd_channels_destroy(self.handle)
            self.handle = None

    @property
    def count(self):
        return load().wpcd_channels_count(self.handle)

    @property
    def pairs(self):
        return load().wpcd_channels_pairs(self.handle)

    @property
    def terms(self):
        return load().wpcd_channels_terms(self.handle)

    @property
    def monomials(self):
        return load().wpcd_channels_monomials(self.handle)

    @property
    def coefficients(self):
        return load().wpcd_channels_coefficients(self.handle)

    def quantum_numbers(self):
        out = np.zeros((self.count, 6), np.int32)
        _check(load().wpcd_channels_get_quantum_numbers(self.handle, out.ctypes.data))
        return out

    def table(self):
        """(pair_gamma, pair_gammap, term_ptr, term_k, term_l1, term_l1p, term_g) host arrays."""
        npairs, nterms = self.pairs, self.terms
        pg, pgp = np.zeros(npairs, np.int32), np.zeros(npairs, np.int32)
        tp = np.zeros(npairs + 1, np.int64)
        tk, tl1, tl1p = (np.zeros(nterms, np.int32) for _ in range(3))
        tg = np.zeros(nterms, np.float64)
        _check(load().wpcd_channels_get_table(self.handle, pg.ctypes.data, pgp.ctypes.data, tp.ctypes.data,
                                              tk.ctypes.data, tl1.ctypes.data, tl1p.ctypes.data, tg.ctypes.data))
        return pg, pgp, tp, tk, tl1, tl1p, tg


def wpcd_grid_create(p_nodes, q_nodes):
    p = np.ascontiguousarray(p_nodes, np.float64)
    q = np.ascontiguousarray(q_nodes, np.float64)
    h = ctypes.c_void_p()
    _check(load().wpcd_grid_create(p.ctypes.data, len(p) - 1, q.ctypes.data, len(q) - 1, ctypes.byref(h)))
    return Grid(h, len(p) - 1, len(q) - 1)


def wpcd_channels_create(model, two_J=1, parity=1, two_T=1, j_pair_max=0, g0=0.5):
    h = ctypes.c_void_p()
    _check(load().wpcd_channels_create(model, two_J, parity, two_T, j_pair_max, float(g0), ctypes.byref(h)))
    return Channels(h)


def wpcd_channels_create_from_table(channel_l, pair_gamma, pair_gammap, term_ptr, term_k, term_l1, term_l1p, term_g):
    a = [np.ascontiguousarray(channel_l, np.int32), np.ascontiguousarray(pair_gamma, np.int32),
         np.ascontiguousarray(pair_gammap, np.int32), np.ascontiguousarray(term_ptr, np.int64),
         np.ascontiguousarray(term_k, np.int32), np.ascontiguousarray(term_l1, np.int32),
         np.ascontiguousarray(term_l1p, np.int32), np.ascontiguousarray(term_g, np.float64)]
    h = ctypes.c_void_p()
    _check(load().wpcd_channels_create_from_table(len(a[0]), a[0].ctypes.data, len(a[1]), a[1].ctypes.data, a[2].ctypes.data,
                                                  a[3].ctypes.data, a[4].ctypes.data, a[5].ctypes.data, a[6].ctypes.data,
                                                  a[7].ctypes.data, ctypes.byref(h)))
    return Channels(h)


def wpcd_rows(grid, channels):
    return load().wpcd_rows(grid.handle, channels.handle)


def wpcd_perm_count(grid, channels, n_quad, row_ptr, geo_row_ptr, stream=None):
    """row_ptr: int64 CUDA tensor [rows+1]; geo_row_ptr: int32 CUDA tensor [n_p*n_q+1]. Returns (nnz, nnz_geo)."""
    import torch

    nnz, nnz_geo = ctypes.c_int64(0), ctypes.c_int64(0)
    _check(load().wpcd_perm_count(grid.handle, channels.handle, n_quad, _stream_ptr(stream), _dev_ptr(row_ptr, torch.int64),
                                  _dev_ptr(geo_row_ptr, torch.int32), ctypes.byref(nnz), ctypes.byref(nnz_geo)))
    return nnz.value, nnz_geo.value


def bind_count_build(grid, channels, n_quad, row_ptr, geo_row_ptr, workspace, col_idx, values, stream):
    """The same two calls with their arguments marshalled ONCE: returns (count, build), two zero-argument callables for a loop
    that rebuilds into fixed buffers on a fixed stream (`stream`: a torch stream or a raw handle, not None).  count() returns
    (nnz, nnz_geo).  The tensors must stay alive and in place while the callables are used."""
    import torch

    L = load()
    st = _stream_ptr(stream)
    rp, gp = _dev_ptr(row_ptr, torch.int64), _dev_ptr(geo_row_ptr, torch.int32)
    ws, wsb = _dev_ptr(workspace), workspace.numel() * workspace.element_size()
    ci, va = _dev_ptr(col_idx, torch.int32), _dev_ptr(values, torch.float64)
    nnz, nnz_geo = ctypes.c_int64(0), ctypes.c_int64(0)
    p_nnz, p_geo = ctypes.byref(nnz), ctypes.byref(nnz_geo)
    gh, chh = grid.handle, channels.handle
    f_count, f_build = L.wpcd_perm_count, L.wpcd_perm_build

    def count():
        _check(f_count(gh, chh, n_quad, st, rp, gp, p_nnz, p_geo))
        return nnz.value, nnz_geo.value

    def build():
        _check(f_build(gh, chh, n_quad, st, rp, gp, ws, wsb, ci, va))

    return count, build


def wpcd_perm_workspace_bytes(channels, nnz_geo):
    return load().wpcd_perm_workspace_bytes(channels.handle, nnz_geo)


def wpcd_perm_build(grid, channels, n_quad, row_ptr, geo_row_ptr, workspace, col_idx, values, stream=None):
    import torch

    _check(load().wpcd_perm_build(grid.handle, channels.handle, n_quad, _stream_ptr(stream), _dev_ptr(row_ptr, torch.int64),
                                  _dev_ptr(geo_row_ptr, torch.int32), _dev_ptr(workspace),
                                  workspace.numel() * workspace.element_size() if workspace is not None else 0,
                                  _dev_ptr(col_idx, torch.int32), _dev_ptr(values, torch.float64)))


def wpcd_perm_apply(rows, row_ptr, col_idx, values, x, y, n_vec=1, stream=None):
    import torch

    _check(load().wpcd_perm_apply(rows, _dev_ptr(row_ptr, torch.int64), _dev_ptr(col_idx, torch.int32),
                                  _dev_ptr(values, torch.float64), _dev_ptr(x, torch.float64), _dev_ptr(y, torch.float64),
                                  n_vec, _stream_ptr(stream)))


def wpcd_perm_apply_complex(rows, row_ptr, col_idx, values, x, y, n_vec=1, stream=None):
    """x, y: complex128 CUDA tensors [n_vec, rows] (interleaved re/im in memory)."""
    import torch

    assert x.dtype == torch.complex128 and y.dtype == torch.complex128
    _check(load().wpcd_perm_apply_complex(rows, _dev_ptr(row_ptr, torch.int64), _dev_ptr(col_idx, torch.int32),
                                          _dev_ptr(values, torch.float64), _dev_ptr(x), _dev_ptr(y), n_vec, _stream_ptr(stream)))


def wpcd_perm_apply_interleaved(rows, row_ptr, col_idx, values, x, y, stream=None):
    """x, y: float64 CUDA tensors [rows, n_inter] (n_inter = 2 or 4 vectors interleaved)."""
    import torch

    assert x.dtype == torch.float64 and y.dtype == torch.float64 and x.shape == y.shape and x.shape[0] == rows
    _check(load().wpcd_perm_apply_interleaved(rows, _dev_ptr(row_ptr, torch.int64), _dev_ptr(col_idx, torch.int32),
                                              _dev_ptr(values, torch.float64), _dev_ptr(x), _dev_ptr(y), int(x.shape[1]),
                                              _stream_ptr(stream)))


def wpcd_perm_apply_blocked(grid, channels, row_ptr, geo_row_ptr, col_idx, values, x, y, n_vec=1, stream=None):
    """y = P0 x through the block structure of the matrix built on (grid, channels); x, y: float64 [n_vec, rows] (CUDA)."""
    import torch

    _check(load().wpcd_perm_apply_blocked(grid.handle, channels.handle, _dev_ptr(row_ptr, torch.int64), _dev_ptr(geo_row_ptr, torch.int32),
                                          _dev_ptr(col_idx, torch.int32), _dev_ptr(values, torch.float64), _dev_ptr(x, torch.float64),
                                          _dev_ptr(y, torch.float64), n_vec, _stream_ptr(stream)))


def wpcd_perm_apply_blocked_noalloc(grid, channels, row_ptr, geo_row_ptr, col_idx, values, x, y, n_vec=1, stream=None):
    """wpcd_perm_apply_blocked for callers that must not allocate: n_vec <= 8, rows <= WPCD_NOALLOC_MAX_ROWS, scratch in a
    fixed device array of the library (calls that overlap on the GPU race on it)."""
    import torch

    _check(load().wpcd_perm_apply_blocked_noalloc(grid.handle, channels.handle, _dev_ptr(row_ptr, torch.int64), _dev_ptr(geo_row_ptr, torch.int32),
                                                  _dev_ptr(col_idx, torch.int32), _dev_ptr(values, torch.float64), _dev_ptr(x, torch.float64),
                                                  _dev_ptr(y, torch.float64), n_vec, _stream_ptr(stream)))


def wpcd_perm_apply_blocked_host(grid, channels, row_ptr, geo_row_ptr, col_idx, values, x_host, y_host, x_dev, y_dev, n_vec=1, stream=None):
    """wpcd_perm_apply_blocked with CPU float64 tensors x_host / y_host (pinned for async copies); x_dev / y_dev: device scratch."""
    import torch

    assert not x_host.is_cuda and not y_host.is_cuda and x_host.dtype == torch.float64 and y_host.dtype == torch.float64
    _check(load().wpcd_perm_apply_blocked_host(grid.handle, channels.handle, _dev_ptr(row_ptr, torch.int64), _dev_ptr(geo_row_ptr, torch.int32),
                                               _dev_ptr(col_idx, torch.int32), _dev_ptr(values, torch.float64),
                                               ctypes.c_void_p(x_host.data_ptr()), ctypes.c_void_p(y_host.data_ptr()), n_vec,
                                               _dev_ptr(x_dev, torch.float64), _dev_ptr(y_dev, torch.float64), _stream_ptr(stream)))


def wpcd_perm_apply_chain(rows, row_ptr, col_idx, values, x, y, n_iter, stream=None):
    """y[k-1] = P0^k x for k = 1 .. n_iter; x: float64 [rows], y: float64 [n_iter, rows] (CUDA)."""
    import torch

    assert y.numel() >= n_iter * rows and x.numel() >= rows
    _check(load().wpcd_perm_apply_chain(rows, _dev_ptr(row_ptr, torch.int64), _dev_ptr(col_idx, torch.int32),
                                        _dev_ptr(values, torch.float64), _dev_ptr(x, torch.float64), _dev_ptr(y, torch.float64),
                                        n_iter, _stream_ptr(stream)))


def wpcd_block_apply(n_channels, n_p, n_q, a, x, y, transpose=False, stream=None):
    """a: float64 [n_channels, n_p, n_p]; x, y: float64 or complex128 CUDA tensors with n_channels*n_p*n_q elements."""
    import torch

    assert a.dtype == torch.float64 and x.dtype == y.dtype and x.dtype in (torch.float64, torch.complex128)
    _check(load().wpcd_block_apply(n_channels, n_p, n_q, _dev_ptr(a), 1 if transpose else 0, _dev_ptr(x), _dev_ptr(y),
                                   1 if x.dtype == torch.complex128 else 0, _stream_ptr(stream)))


def wpcd_kernel_apply(n_channels, n_p, n_q, row_ptr, col_idx, values, o, v, g1, x, y, scratch, stream=None):
    """y = O P0 O^T V1 (G1 .* x); g1, x, y: complex128 [rows]; scratch: complex128 [2*rows]; o, v: float64 [n_ch, n_p, n_p]."""
    import torch

    assert g1.dtype == x.dtype == y.dtype == scratch.dtype == torch.complex128
    assert scratch.numel() >= 2 * x.numel()
    _check(load().wpcd_kernel_apply(n_channels, n_p, n_q, _dev_ptr(row_ptr, torch.int64), _dev_ptr(col_idx, torch.int32),
                                    _dev_ptr(values, torch.float64), _dev_ptr(o, torch.float64), _dev_ptr(v, torch.float64),
                                    _dev_ptr(g1), _dev_ptr(x), _dev_ptr(y), _dev_ptr(scratch), _stream_ptr(stream)))


def wpcd_neumann_terms(n_channels, n_p, n_q, row_ptr, col_idx, values, o, v, g1, b, element, n_terms, stream=None):
    """Complex terms a_n = (K^n b)[element], n = 0 .. n_terms-1, as a numpy complex128 array."""
    import torch

    rows = n_channels * n_p * n_q
    scratch = torch.empty(4 * rows + n_terms, dtype=torch.complex128, device=b.device)
    terms = np.zeros(n_terms, np.complex128)
    _check(load().wpcd_neumann_terms(n_channels, n_p, n_q, _dev_ptr(row_ptr, torch.int64), _dev_ptr(col_idx, torch.int32),
                                     _dev_ptr(values, torch.float64), _dev_ptr(o, torch.float64), _dev_ptr(v, torch.float64),
                                     _dev_ptr(g1), _dev_ptr(b), int(element), n_terms, terms.ctypes.data, _dev_ptr(scratch),
                                     _stream_ptr(stream)))
    return terms


def wpcd_pade_sum(terms):
    """Pade (Wynn epsilon) sum of the complex series `terms` (host only)."""
    t = np.ascontiguousarray(terms, np.complex128)
    out = np.zeros(1, np.complex128)
    _check(load().wpcd_pade_sum(t.ctypes.data, len(t), out.ctypes.data))
    return complex(out[0])


def wpcd_perm_apply_host(rows, row_ptr, col_idx, values, x_host, y_host, x_dev, y_dev, n_vec=1, stream=None):
    """x_host / y_host: CPU float64 tensors (pinned for async copies); x_dev / y_dev: device scratch."""
    import torch

    assert not x_host.is_cuda and not y_host.is_cuda and x_host.dtype == torch.float64 and y_host.dtype == torch.float64
    _check(load().wpcd_perm_apply_host(rows, _dev_ptr(row_ptr, torch.int64), _dev_ptr(col_idx, torch.int32),
                                       _dev_ptr(values, torch.float64), ctypes.c_void_p(x_host.data_ptr()),
                                       ctypes.c_void_p(y_host.data_ptr()), n_vec, _dev_ptr(x_dev, torch.float64),
                                       _dev_ptr(y_dev, torch.float64), _stream_ptr(stream)))


def wpcd_fp64_peak(stream=None):
    out = ctypes.c_double(0.0)
    _check(load().wpcd_fp64_peak(_stream_ptr(stream), ctypes.byref(out)))
    return out.value


def wpcd_trace_enable(on):
    _check(load().wpcd_trace_enable(1 if on else 0))


def wpcd_trace_read():
    """{stage: (milliseconds, launches)} accumulated since the last read."""
    ms = np.zeros(len(TRACE_STAGES), np.float64)
    n = np.zeros(len(TRACE_STAGES), np.int64)
    _check(load().wpcd_trace_read(ms.ctypes.data, n.ctypes.data))
    return {name: (float(ms[i]), int(n[i])) for i, name in enumerate(TRACE_STAGES)}


def wpcd_debug_set(key, value):
    """Test / diagnosis switch of the library (keys: include/wpcd.h); value 0 restores the library's own choice."""
    _check(load().wpcd_debug_set(key.encode(), int(value)))


def wpcd_launch_count():
    return load().wpcd_launch_count()


@dataclass
class PermCSR:
    rows: int
    nnz: int
    nnz_geo: int
    row_ptr: object     # int64 CUDA tensor [rows+1]
    col_idx: object     # int32 CUDA tensor [nnz]
    values: object      # float64 CUDA tensor [nnz]
    geo_row_ptr: object  # int32 CUDA tensor [n_p*n_q+1]


def build_perm(grid, channels, n_quad, stream=None, device="cuda"):
    """count -> allocate (torch) -> build.  Pure plumbing around the C-ABI calls."""
    import torch

    rows = wpcd_rows(grid, channels)
    row_ptr = torch.empty(rows + 1, dtype=torch.int64, device=device)
    geo_row_ptr = torch.empty(grid.n_p * grid.n_q + 1, dtype=torch.int32, device=device)
    nnz, nnz_geo = wpcd_perm_count(grid, channels, n_quad, row_ptr, geo_row_ptr, stream)
    col_idx = torch.empty(nnz, dtype=torch.int32, device=device)
    values = torch.empty(nnz, dtype=torch.float64, device=device)
    ws_bytes = wpcd_perm_workspace_bytes(channels, nnz_geo)
    workspace = torch.empty(max(ws_bytes, 256), dtype=torch.uint8, device=device)
    wpcd_perm_build(grid, channels, n_quad, row_ptr, geo_row_ptr, workspace, col_idx, values, stream)
    if stream is not None and not isinstance(stream, int) and stream != torch.cuda.current_stream():
        # the tensors were allocated on torch's current stream but are used on `stream`: tell the caching allocator, so that
        # the workspace (dropped on return, while the asynchronous build may still run) is not handed out too early
        for t in (workspace, row_ptr, geo_row_ptr, col_idx, values):
            t.record_stream(stream)
    return PermCSR(rows, nnz, nnz_geo, row_ptr, col_idx, values, geo_row_ptr)
