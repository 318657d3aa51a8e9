"""Seeded synthetic inputs shared by the oracle tests, the CUDA tests and bench.py.

Holds NONE of the method's arithmetic: only the momentum grids, the five
workload descriptions of BASELINE.json `configs` and the random vectors.
Recipe: nodes p_i = q_i = scale * tan^2(pi i / (2N+2)),
i = 0..N (PAPER.md:92 partitions; the paper does not print its grids), with the
interior jitter of DESIGN.md R10 for configs 1-2.
"""
from dataclasses import dataclass, field

import numpy as np

SEED = 20140521


def tan2_grid(n_bins, scale=1.0, jitter=0.0, seed=SEED):
    """n_bins+1 strictly increasing nodes, first node 0.

    jitter: p_i <- p_i + jitter * u_i * min(p_i - p_{i-1}, p_{i+1} - p_i), u_i ~ U(-1,1),
    i = 1..N-1 (end nodes fixed); monotone for jitter < 0.5.
    """
    i = np.arange(n_bins + 1, dtype=np.float64)
    nodes = scale * np.tan(np.pi * i / (2 * n_bins + 2)) ** 2
    if jitter:
        rng = np.random.default_rng(seed)
        u = rng.uniform(-1.0, 1.0, size=n_bins - 1)
        gap = np.minimum(nodes[1:-1] - nodes[:-2], nodes[2:] - nodes[1:-1])
        nodes = nodes.copy()
        nodes[1:-1] += jitter * u * gap
    assert np.all(np.diff(nodes) > 0)
    return nodes


@dataclass
class Workload:
    name: str
    n_bins: int
    n_quad: int
    jitter: float
    model: str                      # "swave" | "nd"
    g0: float = 0.5
    j_pair_max: int = 0
    jpis: list = field(default_factory=list)   # [(two_J, parity)]
    n_spmv: int = 0
    seed: int = SEED

    def grid(self, seed_offset=0):
        return tan2_grid(self.n_bins, 1.0, self.jitter, self.seed + seed_offset)


_BOTH = lambda twoJs: [(tj, par) for tj in twoJs for par in (+1, -1)]

WORKLOADS = {
    # BASELINE.json configs[0..4]
    "cfg1": Workload("cfg1", 20, 8, 0.1, "swave", n_spmv=0),
    "cfg2": Workload("cfg2", 100, 8, 0.1, "swave", n_spmv=50),
    "cfg3": Workload("cfg3", 100, 8, 0.0, "nd", j_pair_max=2, jpis=[(1, +1)], n_spmv=0),
    "cfg4": Workload("cfg4", 150, 10, 0.0, "nd", j_pair_max=3, jpis=_BOTH([1, 3]), n_spmv=100),
    "cfg5": Workload("cfg5", 150, 10, 0.0, "nd", j_pair_max=3, jpis=_BOTH([1, 3, 5, 7]), n_spmv=20),
    # extra, not a BASELINE.json config: the lattice size of the paper's own s-wave timing (M = N = 400,
    # PAPER.md:334), same node formula, for context beside the paper's 2.3 s on a GTX-670
    "fig4": Workload("fig4", 400, 8, 0.0, "swave", n_spmv=0),
}


def normal_vector(n, seed=SEED, k=0):
    """Seeded N(0,1) vector number k of length n."""
    return np.random.default_rng([seed, 7, k]).standard_normal(n)


def kernel_factors(n_ch, n_p, n_q, seed=SEED):
    """Seeded synthetic factors of the kernel K = O P0 O^T V1 G1 (the real ones need the NN potential, which is
    not available): O[g] a random orthogonal n_p x n_p matrix (QR of a Gaussian matrix), V1[g] a random symmetric
    matrix scaled to spectral radius ~0.5, G1 a complex diagonal with |G1| ~ 1.  No method arithmetic here."""
    rng = np.random.default_rng([seed, 11])
    o = np.empty((n_ch, n_p, n_p))
    v = np.empty((n_ch, n_p, n_p))
    for g in range(n_ch):
        qm, rm = np.linalg.qr(rng.standard_normal((n_p, n_p)))
        o[g] = qm * np.sign(np.diag(rm))
        a = rng.standard_normal((n_p, n_p))
        v[g] = 0.25 * (a + a.T) / np.sqrt(n_p)
    rows = n_ch * n_p * n_q
    g1 = (rng.standard_normal(rows) + 1j * rng.standard_normal(rows)) / np.sqrt(2.0)
    return o, v, g1
