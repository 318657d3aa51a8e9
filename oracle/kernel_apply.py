"""Oracle for one application of the Faddeev kernel in factored form (TEST INFRASTRUCTURE, see oracle/__init__.py).

Eq. (12): U = P V1 + P V1 G1 U; the kernel K = P V1 G1 is kept "as a product of four
matrices: a very sparse matrix P0, a diagonal matrix G1 and two block matrices".  In the
scattering-wave-packet basis |Z_kj> = sum_i O_ki |X_ij> (eq. 8-9) the permutation matrix is

    <Z_kj^gamma | P | Z_k'j'^gamma'> = sum_{i i'} O^gamma_{ki} O^gamma'_{k'i'} [P0]^{gamma gamma'}_{ij,i'j'}      (eq. 10)

so, for a coefficient vector c over (gamma, k, j):   K c = O ( P0 ( O^T ( V1 ( G1 .* c ) ) ) ),
with O, V1 acting on the pair index inside one channel and one q-bin (V1 block-diagonal in the channel:
the uncoupled-pair case), G1 diagonal and complex.  Every step below is the plain definition in numpy
(fp64 / complex128), no blocking.  Index convention: element (gamma, i, j) sits at (gamma*n_p + i)*n_q + j.

Pins (tests/test_oracle_kernel_apply.py): O = V1 = 1, G1 = 1 gives the plain CSR product; the matrix
of eq. (10) assembled entry by entry with its four-index sum on a tiny lattice; an orthogonal O leaves the
spectrum of P0 unchanged.
"""
import numpy as np


def block_apply(a, x, n_ch, n_p, n_q, transpose=False):
    """Y_gamma = A_gamma X_gamma (or A_gamma^T X_gamma): y[(g,k,j)] = sum_i a[g,k,i] x[(g,i,j)]."""
    X = np.asarray(x).reshape(n_ch, n_p, n_q)
    A = np.asarray(a).reshape(n_ch, n_p, n_p)
    Y = np.einsum("gik,gij->gkj", A, X) if transpose else np.einsum("gki,gij->gkj", A, X)
    return Y.reshape(-1)


def csr_apply(row_ptr, col_idx, values, x):
    """y = P0 x for a real or complex x, each row summed sequentially in column order."""
    y = np.zeros(len(row_ptr) - 1, dtype=np.result_type(values.dtype, np.asarray(x).dtype))
    for r in range(len(row_ptr) - 1):
        lo, hi = row_ptr[r], row_ptr[r + 1]
        y[r] = np.sum(values[lo:hi] * x[col_idx[lo:hi]])
    return y


def kernel_apply(row_ptr, col_idx, values, o, v, g1, x, n_ch, n_p, n_q):
    """K x = O ( P0 ( O^T ( V1 ( G1 .* x ) ) ) )."""
    t = np.asarray(g1) * np.asarray(x)                       # diagonal channel resolvent
    t = block_apply(v, t, n_ch, n_p, n_q)                    # pair interaction in the SWP basis
    t = block_apply(o, t, n_ch, n_p, n_q, transpose=True)    # SWP -> lattice basis:  sum_k' O_k'i' c_k'
    t = csr_apply(row_ptr, col_idx, values, t)               # P0
    return block_apply(o, t, n_ch, n_p, n_q)                 # lattice -> SWP basis:  sum_i O_ki


def neumann_terms(row_ptr, col_idx, values, o, v, g1, b, element, n_terms, n_ch, n_p, n_q):
    """a_n = (K^n b)[element], n = 0 .. n_terms-1: the terms of the iterated eq. (12) for the amplitude element
    of eq. (13), "solution ... by iteration"."""
    vec = np.asarray(b, np.complex128).copy()
    out = np.zeros(n_terms, np.complex128)
    for n in range(n_terms):
        out[n] = vec[element]
        if n + 1 < n_terms:
            vec = kernel_apply(row_ptr, col_idx, values, o, v, g1, vec, n_ch, n_p, n_q)
    return out


def pade_sum(terms):
    """Sum of the series by the Pade-approximant technique, in the form of Wynn's epsilon
    algorithm on the partial sums S_n:  eps_{-1} = 0, eps_0^{(n)} = S_n,
        eps_{k+1}^{(n)} = eps_{k-1}^{(n+1)} + 1 / (eps_k^{(n+1)} - eps_k^{(n)}),
    whose even columns eps_{2k}^{(n)} are the Pade approximants [n+k / k] of sum a_n lambda^n at lambda = 1.
    Returns the last entry of the highest even column that could be formed."""
    S = np.cumsum(np.asarray(terms, np.complex128))
    table = [np.zeros(len(S) + 1, np.complex128), S]          # eps_{-1}, eps_0
    best = S[-1]
    while len(table[-1]) > 1:
        cur, prev = table[-1], table[-2]
        d = cur[1:] - cur[:-1]
        if np.any(d == 0):
            break
        table.append(prev[1:len(cur)] + 1.0 / d)
        if (len(table) - 2) % 2 == 0:                          # column index = len(table) - 2
            best = table[-1][-1]
    return complex(best)
