"""ctypes front end to perm_oracle.c (TEST INFRASTRUCTURE, see oracle/__init__.py).

Follows PAPER.md Appendix A: predicate from the theta-functions of (A7)
(PAPER.md:416), values by (A15) with F of (A14),
normalisation (A5)/(A9).  Gauss-Legendre nodes come from
numpy.polynomial.legendre.leggauss (a library primitive).
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "perm_oracle.c")
_SO = os.path.join(_HERE, "_perm_oracle.so")
_SO_EXT = os.path.join(_HERE, "_perm_oracle_ext.so")      # the same source with -DWPO_EXTENDED (rule arithmetic in long double)
_lib = None
_lib_ext = None

_D = np.ctypeslib.ndpointer(np.float64, flags="C_CONTIGUOUS")
_I32 = np.ctypeslib.ndpointer(np.int32, flags="C_CONTIGUOUS")
_I64 = np.ctypeslib.ndpointer(np.int64, flags="C_CONTIGUOUS")


def build(force=False):
    """Compile perm_oracle.c (gcc, -ffp-contract=off) next to this file: the FP64 oracle and its long-double twin."""
    for so, extra in ((_SO, []), (_SO_EXT, ["-DWPO_EXTENDED"])):
        if force or not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(_SRC):
            cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC"] + extra + [_SRC, "-lm", "-o", so]
            subprocess.check_call(cmd)
    return _SO


def lib_extended():
    """The -DWPO_EXTENDED build: same statements, rule arithmetic in long double (only wpo_elements_rule is used from it)."""
    global _lib_ext
    if _lib_ext is None:
        build()
        L = ctypes.CDLL(_SO_EXT)
        i32, i64 = ctypes.c_int, ctypes.c_int64
        L.wpo_elements_rule.argtypes = [i32, i32, _D, _D, i64, _I32, _I32, _I32, _I32, i32, _D, _D, i32,
                                        i32, _I32, _I32, _I64, _I32, _I32, _I32, _D, _D, _D]
        _lib_ext = L
    return _lib_ext


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        dbl, i32, i64 = ctypes.c_double, ctypes.c_int, ctypes.c_int64
        L.wpo_overlap.restype = ctypes.c_int
        L.wpo_overlap.argtypes = [dbl] * 8 + [ctypes.c_void_p, ctypes.c_void_p]
        L.wpo_geo_count.argtypes = [i32, i32, _D, _D, _I32]
        L.wpo_geo_fill.argtypes = [i32, i32, _D, _D, _I64, _I32]
        L.wpo_elements.argtypes = [i32, i32, _D, _D, i64, _I32, _I32, _I32, _I32, i32, _D, _D,
                                   i32, _I32, _I32, _I64, _I32, _I32, _I32, _D, _D, _D]
        L.wpo_elements_rule.argtypes = [i32, i32, _D, _D, i64, _I32, _I32, _I32, _I32, i32, _D, _D, i32,
                                        i32, _I32, _I32, _I64, _I32, _I32, _I32, _D, _D, _D]
        L.wpo_spmv.argtypes = [i64, _I64, _I32, _D, _D, _D]
        L.wpo_num_threads.restype = ctypes.c_int
        _lib = L
    return _lib


def num_threads():
    return lib().wpo_num_threads()


def overlap(a, b, c, d, L1, U1, L2, U2):
    """Predicate S (R6); returns (bool, polygon vertices array [nv,2])."""
    poly = np.zeros((16, 2))
    nv = ctypes.c_int(0)
    ok = lib().wpo_overlap(a, b, c, d, L1, U1, L2, U2, poly.ctypes.data, ctypes.addressof(nv))
    return bool(ok), poly[: nv.value].copy()


def geo_pattern(p, q):
    """Geometric CSR pattern: (geo_row_ptr int64 [n_p*n_q+1], geo_col int32)."""
    p = np.ascontiguousarray(p, np.float64)
    q = np.ascontiguousarray(q, np.float64)
    n_p, n_q = len(p) - 1, len(q) - 1
    counts = np.zeros(n_p * n_q, np.int32)
    lib().wpo_geo_count(n_p, n_q, p, q, counts)
    ptr = np.zeros(n_p * n_q + 1, np.int64)
    np.cumsum(counts, out=ptr[1:])
    col = np.zeros(int(ptr[-1]), np.int32)
    lib().wpo_geo_fill(n_p, n_q, p, q, ptr, col)
    return ptr, col


class PairTable:
    """Flat arrays of the coupled channel pairs and their (k,l1,l1',g) terms."""

    def __init__(self, channels, pairs):
        self.channels = list(channels)
        self.n_ch = len(self.channels)
        self.gamma = np.array([pr[0] for pr in pairs], np.int32)
        self.gammap = np.array([pr[1] for pr in pairs], np.int32)
        self.pair_l = np.array([self.channels[pr[0]][0] for pr in pairs], np.int32)
        self.pair_lp = np.array([self.channels[pr[1]][0] for pr in pairs], np.int32)
        nt = [len(pr[2]) for pr in pairs]
        self.term_ptr = np.zeros(len(pairs) + 1, np.int64)
        np.cumsum(nt, out=self.term_ptr[1:])
        flat = [t for pr in pairs for t in pr[2]]
        self.term_k = np.array([t[0] for t in flat], np.int32)
        self.term_l1 = np.array([t[1] for t in flat], np.int32)
        self.term_l1p = np.array([t[2] for t in flat], np.int32)
        self.term_g = np.array([t[3] for t in flat], np.float64)
        self.n_pairs = len(pairs)
        # coupling mask [n_ch, n_ch] and per-row coupled column channels (ascending)
        self.mask = np.zeros((self.n_ch, self.n_ch), bool)
        self.mask[self.gamma, self.gammap] = True


def gauss_legendre(n):
    xi, w = np.polynomial.legendre.leggauss(n)
    return np.ascontiguousarray(xi), np.ascontiguousarray(w)


def element_values(p, q, ei, ej, eip, ejp, n_quad, table, split=False, extended=False):
    """Values (A15) by rule R(n_quad) -- the kink-split rule RS(n_quad) if split is True / 1, the rule RA(n_quad) with the
    exact u-integral (s-wave term only) if split == 2 -- of the listed geometric elements, all pairs.
    extended=True: the same rule with its arithmetic in long double (results rounded to double at the end).
    Returns (val, absval), each [n_elem, n_pairs]."""
    if int(split) == 2:
        one = np.diff(table.term_ptr) == 1
        assert one.all() and not table.pair_l.any() and not table.pair_lp.any() and not table.term_k.any(), "RA(n): s-wave term only"
    p = np.ascontiguousarray(p, np.float64)
    q = np.ascontiguousarray(q, np.float64)
    ei, ej, eip, ejp = (np.ascontiguousarray(v, np.int32) for v in (ei, ej, eip, ejp))
    xi, w = gauss_legendre(n_quad)
    ne = len(ei)
    val = np.zeros((ne, table.n_pairs))
    absval = np.zeros((ne, table.n_pairs))
    (lib_extended() if extended else lib()).wpo_elements_rule(len(p) - 1, len(q) - 1, p, q, ne, ei, ej, eip, ejp, n_quad, xi, w, int(split),
                       table.n_pairs, table.pair_l, table.pair_lp, table.term_ptr, table.term_k,
                       table.term_l1, table.term_l1p, table.term_g, val, absval)
    return val, absval


def full_row_ptr(geo_ptr, table, n_p, n_q):
    """row_ptr of the full matrix: row (gamma,i,j) = (gamma*n_p+i)*n_q+j holds
    count(i,j) entries for every gamma' coupled to gamma."""
    geo_cnt = np.diff(geo_ptr)
    ncoupled = table.mask.sum(axis=1).astype(np.int64)
    cnt = (ncoupled[:, None] * geo_cnt[None, :]).reshape(-1)
    ptr = np.zeros(table.n_ch * n_p * n_q + 1, np.int64)
    np.cumsum(cnt, out=ptr[1:])
    return ptr


def build_csr(p, q, n_quad, table, geo=None, geo_rows=None, split=False):
    """Full CSR (row_ptr, col_idx, values, absvalues) of P0.

    If geo_rows is given, values are computed only for those geometric rows (all
    channels) and every other value is NaN; the pattern is always complete.
    """
    n_p, n_q = len(p) - 1, len(q) - 1
    geo_ptr, geo_col = geo if geo is not None else geo_pattern(p, q)
    row_ptr = full_row_ptr(geo_ptr, table, n_p, n_q)
    nnz = int(row_ptr[-1])
    col_idx = np.empty(nnz, np.int32)
    values = np.full(nnz, np.nan)
    absvalues = np.full(nnz, np.nan)
    n_geo = n_p * n_q
    rows = np.arange(n_geo) if geo_rows is None else np.asarray(geo_rows)
    # pair index lookup
    pair_of = -np.ones((table.n_ch, table.n_ch), np.int64)
    pair_of[table.gamma, table.gammap] = np.arange(table.n_pairs)
    # column indices for every row
    for g in range(table.n_ch):
        coupled = np.nonzero(table.mask[g])[0]
        if len(coupled) == 0:
            continue
        for r in range(n_geo):
            gc = geo_col[geo_ptr[r]:geo_ptr[r + 1]]
            base = row_ptr[g * n_geo + r]
            m = len(gc)
            if m == 0:
                continue
            col_idx[base:base + m * len(coupled)] = (coupled[:, None].astype(np.int64) * n_geo + gc[None, :]).reshape(-1)
    # values
    if len(rows):
        cnts = (geo_ptr[rows + 1] - geo_ptr[rows]).astype(np.int64)
        erow = np.repeat(rows, cnts)
        eidx = np.concatenate([np.arange(geo_ptr[r], geo_ptr[r + 1]) for r in rows]) if len(rows) else np.zeros(0, np.int64)
        ecol = geo_col[eidx]
        val, absval = element_values(p, q, erow // n_q, erow % n_q, ecol // n_q, ecol % n_q, n_quad, table, split=split)
        pos_in_row = eidx - geo_ptr[erow]
        for g in range(table.n_ch):
            coupled = np.nonzero(table.mask[g])[0]
            for ci, gp in enumerate(coupled):
                dst = row_ptr[g * n_geo + erow] + ci * cnts_of(geo_ptr, erow) + pos_in_row
                values[dst] = val[:, pair_of[g, gp]]
                absvalues[dst] = absval[:, pair_of[g, gp]]
    return row_ptr, col_idx, values, absvalues


def cnts_of(geo_ptr, erow):
    return geo_ptr[erow + 1] - geo_ptr[erow]


def spmv(row_ptr, col_idx, values, x):
    y = np.zeros(len(row_ptr) - 1)
    lib().wpo_spmv(len(row_ptr) - 1, np.ascontiguousarray(row_ptr, np.int64), np.ascontiguousarray(col_idx, np.int32),
                   np.ascontiguousarray(values, np.float64), np.ascontiguousarray(x, np.float64), y)
    return y
