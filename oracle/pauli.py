"""Pauli-string bookkeeping and the matrix element of PAPER.md:158 Eq. 16 (oracle; test infrastructure).

Conventions (readings A1, A5): qubit j <-> bit j of the configuration; x_j = 1 <-> |1>.
A configuration / mask is a pair of uint64 words (word j//64, bit j%64).  Codes 0..3 = sigma_0..sigma_3
= I, X, Y, Z (Eq. 1).
"""
import numpy as np

U1 = np.uint64(1)


def pack_mask(bits01: np.ndarray) -> np.ndarray:
    """[..., n] 0/1 -> [..., 2] uint64."""
    n = bits01.shape[-1]
    out = np.zeros(bits01.shape[:-1] + (2,), dtype=np.uint64)
    for j in range(n):
        out[..., j // 64] |= bits01[..., j].astype(np.uint64) << np.uint64(j % 64)
    return out


def unpack_mask(packed: np.ndarray, n: int) -> np.ndarray:
    """[..., 2] uint64 -> [..., n] uint8."""
    out = np.zeros(packed.shape[:-1] + (n,), dtype=np.uint8)
    for j in range(n):
        out[..., j] = ((packed[..., j // 64] >> np.uint64(j % 64)) & U1).astype(np.uint8)
    return out


def incidence(codes: np.ndarray):
    """Operator Matrix [K, n] -> (F12, F23, r).

    F^{1,2}[k, j] = 1 where term k holds sigma_1 or sigma_2 (the flip mask), F^{2,3}[k, j] = 1 where it
    holds sigma_2 or sigma_3 (the sign mask) — PAPER.md:101 (Fig. 1), :154-156; r = number of sigma_2
    (PAPER.md:192).  Returned bit-packed: f, s uint64 [K, 2]; r int64 [K].
    """
    codes = np.asarray(codes)
    f12 = ((codes == 1) | (codes == 2)).astype(np.uint8)
    f23 = ((codes == 2) | (codes == 3)).astype(np.uint8)
    r = (codes == 2).sum(axis=1).astype(np.int64)
    return pack_mask(f12), pack_mask(f23), r


def popcount2(a: np.ndarray) -> np.ndarray:
    """popcount of a 2-word mask [..., 2] -> int64 [...]."""
    return np.bitwise_count(a[..., 0]).astype(np.int64) + np.bitwise_count(a[..., 1]).astype(np.int64)


_MINUS_I_POW = np.array([1, -1j, -1, 1j], dtype=np.complex128)   # (-i)^r, r mod 4


def matrix_element(x: np.ndarray, s: np.ndarray, r: np.ndarray) -> np.ndarray:
    """<x|P_p|x^p> = (-i)^r * prod_{k: p_k in {2,3}} (-1)^{x_k}   (Eq. 16).

    The x_k are those of the ROW configuration x (reading A1, pinned against Kronecker products of the
    Eq. 1 matrices in tests/test_oracle_pauli.py).  x [..., 2], s [K, 2] broadcastable; r [K].
    """
    par = popcount2(x & s) & 1
    return _MINUS_I_POW[r % 4] * (1 - 2 * par)
