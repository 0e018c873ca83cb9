"""Brute-force references for tiny systems (n <= 12): what the paper and the mathematics fix,
written independently of oracle/ (dense Kronecker products of PAPER.md:40 Eq. 1, Slater-Condon /
second quantisation on occupation bit strings).  Index convention: basis index = sum_j x_j 2^j, so
qubit n-1 is the most significant Kronecker factor (reading A5)."""
import numpy as np

SIGMA = [
    np.array([[1, 0], [0, 1]], dtype=np.complex128),
    np.array([[0, 1], [1, 0]], dtype=np.complex128),
    np.array([[0, -1j], [1j, 0]], dtype=np.complex128),
    np.array([[1, 0], [0, -1]], dtype=np.complex128),
]


def dense_pauli_string(codes_row):
    m = np.array([[1.0 + 0j]])
    for c in codes_row:                 # qubit 0 first -> ends up least significant
        m = np.kron(SIGMA[int(c)], m)
    return m


def dense_pauli_sum(codes, coeffs):
    n = len(codes[0])
    H = np.zeros((2 ** n, 2 ** n), dtype=np.complex128)
    for row, c in zip(codes, coeffs):
        H += c * dense_pauli_string(row)
    return H


def _apply(states, amp, j, create):
    """Apply a_j (create=False) or a+_j (create=True) to basis states (int arrays); returns new states,
    amplitudes (0 where annihilated), fermionic sign (-1)^{# occupied modes below j}."""
    occ = (states >> j) & 1
    ok = (occ == 0) if create else (occ == 1)
    below = states & ((1 << j) - 1)
    sign = 1 - 2 * (np.bitwise_count(below.astype(np.uint64)).astype(np.int64) & 1)
    return states ^ (1 << j), amp * ok * sign


def slater_condon(h, g):
    """Determinant-basis (occupation number) matrix of
    H = sum h_pq a+_ps a_qs + 1/2 sum g_pqrs a+_ps a+_rt a_st a_qs, g = (pq|rs), mode j = 2p + s."""
    N = h.shape[0]
    n = 2 * N
    dim = 2 ** n
    H = np.zeros((dim, dim), dtype=np.float64)
    kets = np.arange(dim, dtype=np.int64)
    one = np.ones(dim, dtype=np.float64)
    for p in range(N):
        for q in range(N):
            for s in range(2):
                st, a = _apply(kets, one, 2 * q + s, False)
                st, a = _apply(st, a, 2 * p + s, True)
                np.add.at(H, (st, kets), h[p, q] * a)
    for p in range(N):
        for q in range(N):
            for r in range(N):
                for s4 in range(N):
                    for s in range(2):
                        for t in range(2):
                            st, a = _apply(kets, one, 2 * q + s, False)
                            st, a = _apply(st, a, 2 * s4 + t, False)
                            st, a = _apply(st, a, 2 * r + t, True)
                            st, a = _apply(st, a, 2 * p + s, True)
                            np.add.at(H, (st, kets), 0.5 * g[p, q, r, s4] * a)
    return H


def number_operator(n):
    return np.diag(np.bitwise_count(np.arange(2 ** n, dtype=np.uint64)).astype(np.float64))


def all_configs(n):
    """uint64 [2^n, 2] packed configurations in index order."""
    out = np.zeros((2 ** n, 2), dtype=np.uint64)
    out[:, 0] = np.arange(2 ** n, dtype=np.uint64)
    return out
