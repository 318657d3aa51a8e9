"""CPU-side checks of the C-ABI library: it loads, exports every symbol that include/wpcd.h
declares, validates arguments, and its host-side channel/g tables (product code, C++) agree
with the oracle's (Python, exact rationals)."""
import ctypes
import os
import re

import numpy as np
import pytest

from oracle import channels as och

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "wpcd.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(wpcd_[a-z0-9_]+)\s*\(", text)))


def test_exports_every_declared_symbol(wpcd):
    lib = ctypes.CDLL(wpcd.LIB_PATH)
    declared = _declared_symbols()
    assert {"wpcd_grid_create", "wpcd_channels_create", "wpcd_perm_count", "wpcd_perm_build", "wpcd_perm_apply"} <= set(declared)
    for name in declared:
        assert hasattr(lib, name), name
    assert set(wpcd.EXPORTS) == set(declared)


def test_grid_argument_checks(wpcd):
    with pytest.raises(wpcd.WpcdError, match="strictly increasing"):
        wpcd.wpcd_grid_create([0.0, 1.0, 1.0], [0.0, 1.0])
    with pytest.raises(wpcd.WpcdError, match="strictly increasing"):
        wpcd.wpcd_grid_create([-0.1, 1.0], [0.0, 1.0])
    with pytest.raises(wpcd.WpcdError):
        wpcd.wpcd_grid_create([0.0], [0.0, 1.0])
    with pytest.raises(wpcd.WpcdError, match="finite"):
        wpcd.wpcd_grid_create([0.0, float("nan")], [0.0, 1.0])


def test_channel_argument_checks(wpcd):
    with pytest.raises(wpcd.WpcdError):
        wpcd.wpcd_channels_create(7)
    with pytest.raises(wpcd.WpcdError):
        wpcd.wpcd_channels_create(wpcd.WPCD_ND, two_J=2, parity=1, j_pair_max=1)
    with pytest.raises(wpcd.WpcdError):
        wpcd.wpcd_channels_create(wpcd.WPCD_ND, two_J=1, parity=0, j_pair_max=1)
    with pytest.raises(wpcd.WpcdError, match="sorted"):
        wpcd.wpcd_channels_create_from_table([0, 0], [1, 0], [0, 0], [0, 1, 2], [0, 0], [0, 0], [0, 0], [1.0, 1.0])
    with pytest.raises(wpcd.WpcdError, match="WPCD_MAX_K"):
        wpcd.wpcd_channels_create_from_table([0], [0], [0], [0, 1], [99], [0], [0], [1.0])
    with pytest.raises(wpcd.WpcdError, match="no terms"):
        wpcd.wpcd_channels_create_from_table([0, 0], [0, 1], [0, 1], [0, 1, 1], [0], [0], [0], [1.0])


@pytest.mark.parametrize("two_J,parity,jmax", [(1, 1, 2), (1, -1, 2), (3, 1, 2), (5, -1, 3)])
def test_host_g_table_matches_oracle(wpcd, two_J, parity, jmax):
    ch = wpcd.wpcd_channels_create(wpcd.WPCD_ND, two_J=two_J, parity=parity, two_T=1, j_pair_max=jmax)
    ochs = och.enumerate_channels(two_J, parity, jmax)
    assert [tuple(r) for r in ch.quantum_numbers()] == ochs
    otab = och.g_table(ochs, two_J, 1)
    pg, pgp, tp, tk, tl1, tl1p, tg = ch.table()
    assert list(zip(pg, pgp)) == [(a, b) for a, b, _ in otab]
    for c, (_, _, terms) in enumerate(otab):
        mine = {(int(tk[t]), int(tl1[t]), int(tl1p[t])): tg[t] for t in range(tp[c], tp[c + 1])}
        theirs = {(k, l1, l1p): g for k, l1, l1p, g in terms}
        assert mine.keys() == theirs.keys()
        for key in mine:
            assert mine[key] == pytest.approx(theirs[key], rel=1e-12, abs=1e-15)


def test_swave_table(wpcd):
    ch = wpcd.wpcd_channels_create(wpcd.WPCD_SPINLESS_SWAVE, g0=0.5)
    assert (ch.count, ch.pairs, ch.terms) == (1, 1, 1)
    assert ch.table()[6][0] == 0.5


def test_compute_fails_loudly_without_gpu(wpcd):
    import torch

    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(wpcd.WpcdError):
        wpcd.wpcd_grid_create(np.array([0.0, 1.0]), np.array([0.0, 1.0]))


def test_pade_sum_host(wpcd):
    """wpcd_pade_sum is host-only code of the product: against the closed forms and the oracle's epsilon table."""
    import numpy as np
    from oracle import kernel_apply as oka

    for r in (0.5, -2.0, 3.0 + 1.0j):
        terms = np.array([r ** n for n in range(8)], np.complex128)
        assert abs(wpcd.wpcd_pade_sum(terms) - 1.0 / (1.0 - r)) < 1e-9
    rng = np.random.default_rng(3)
    poles = np.array([-1.4, 0.7 + 0.2j, 0.3j])
    coef = rng.standard_normal(3) + 1j * rng.standard_normal(3)
    terms = np.array([np.sum(coef * poles ** n) for n in range(12)], np.complex128)
    exact = np.sum(coef / (1 - poles))
    assert abs(wpcd.wpcd_pade_sum(terms) - exact) < 1e-7
    assert abs(wpcd.wpcd_pade_sum(terms) - oka.pade_sum(terms)) < 1e-7
