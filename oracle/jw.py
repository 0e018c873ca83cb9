"""Slow symbolic Jordan-Wigner transform by the definition (oracle; test infrastructure).

H = sum_{pq,s} h_pq a+_{ps} a_{qs} + 1/2 sum_{pqrs,s,t} g_pqrs a+_{ps} a+_{rt} a_{st} a_{qs},  g = (pq|rs),
spin-orbital j = 2p + s (Eq. 12), a_j = (prod_{k<j} Z_k)(X_j + iY_j)/2, a+_j = its adjoint
(PAPER.md:49, :216 — OpenFermion's Jordan-Wigner).  Pauli strings are tuples of codes 0..3 multiplied
qubit by qubit with the single-qubit table sigma_a sigma_b = phase * sigma_c of PAPER.md:40 Eq. 1.
Used to pin the fast input generator and, with tests/bruteforce.py, the whole sign convention.
"""
import itertools

# sigma_a * sigma_b = PH[a][b] * sigma_{IDX[a][b]}
_IDX = [[0, 1, 2, 3], [1, 0, 3, 2], [2, 3, 0, 1], [3, 2, 1, 0]]
_PH = [[1, 1, 1, 1], [1, 1, 1j, -1j], [1, -1j, 1, 1j], [1, 1j, -1j, 1]]


def pmul(a, b):
    """(coef_a, string_a) * (coef_b, string_b)."""
    ca, sa = a
    cb, sb = b
    ph = ca * cb
    out = []
    for x, y in zip(sa, sb):
        ph *= _PH[x][y]
        out.append(_IDX[x][y])
    return ph, tuple(out)


def ladder(j, n, dagger):
    """a_j or a+_j as a list of two (coef, string) terms."""
    base = [3] * j + [0] * (n - j)
    sx = list(base); sx[j] = 1
    sy = list(base); sy[j] = 2
    return [(0.5, tuple(sx)), ((-0.5j if dagger else 0.5j), tuple(sy))]


def jw_hamiltonian(h, g, tol=1e-8):
    """Integrals -> dict {pauli string tuple: real coefficient}, |c| < tol dropped, identity kept."""
    N = len(h)
    n = 2 * N
    acc = {}

    def add_product(ops, scale):
        for combo in itertools.product(*ops):
            term = (scale, tuple([0] * n))
            for t in combo:
                term = pmul(term, t)
            acc[term[1]] = acc.get(term[1], 0.0) + term[0]

    cr = [ladder(j, n, True) for j in range(n)]
    an = [ladder(j, n, False) for j in range(n)]
    for p in range(N):
        for q in range(N):
            if h[p][q] != 0.0:
                for s in range(2):
                    add_product([cr[2 * p + s], an[2 * q + s]], float(h[p][q]))
    for p in range(N):
        for q in range(N):
            for r in range(N):
                for s4 in range(N):
                    gv = float(g[p][q][r][s4])
                    if gv == 0.0:
                        continue
                    for s in range(2):
                        for t in range(2):
                            add_product([cr[2 * p + s], cr[2 * r + t], an[2 * s4 + t], an[2 * q + s]], 0.5 * gv)
    out = {}
    for k, v in acc.items():
        if abs(v.imag) > 1e-10:
            raise ValueError("non-real Pauli coefficient: integrals not Hermitian/symmetric")
        if abs(v.real) >= tol:
            out[k] = v.real
    return out
