"""Seeded fixed-Hamming-weight samples + multiplicities (BASELINE.json configs; Eq. 12).

Per row: n_alpha of the N even bits and n_beta of the N odd bits, uniformly; duplicates
rejected when `unique` (cfg 1 cannot be unique: its sector has C(4,2)^2 = 36 states, A16).
Counts uniform integers in [1, max_count].  Bit j of the packed 2 x uint64 word = qubit j.
"""
import numpy as np


def pack_bits(bits: np.ndarray) -> np.ndarray:
    """uint8 [B, n] (0/1, column j = qubit j) -> uint64 [B, 2]."""
    B, n = bits.shape
    out = np.zeros((B, 2), dtype=np.uint64)
    for j in range(n):
        out[:, j // 64] |= bits[:, j].astype(np.uint64) << np.uint64(j % 64)
    return out


def unpack_bits(packed: np.ndarray, n: int) -> np.ndarray:
    """uint64 [B, 2] -> uint8 [B, n]."""
    B = packed.shape[0]
    out = np.zeros((B, n), dtype=np.uint8)
    for j in range(n):
        out[:, j] = ((packed[:, j // 64] >> np.uint64(j % 64)) & np.uint64(1)).astype(np.uint8)
    return out


def make_samples(n_spatial: int, n_alpha: int, n_beta: int, batch: int, max_count: int,
                 seed: int, unique: bool = True):
    """Return (samples uint64[B,2], counts int64[B])."""
    N = int(n_spatial)
    rng = np.random.default_rng(seed)
    rows = []
    seen = set()
    need = int(batch)
    while need > 0:
        m = max(need + need // 8, 64)
        ka = np.argsort(rng.random((m, N)), axis=1)[:, :n_alpha]      # uniform n_alpha-subsets
        kb = np.argsort(rng.random((m, N)), axis=1)[:, :n_beta]
        bits = np.zeros((m, 2 * N), dtype=np.uint8)
        np.put_along_axis(bits, 2 * ka, 1, axis=1)                     # alpha = even spin-orbitals
        np.put_along_axis(bits, 2 * kb + 1, 1, axis=1)                 # beta  = odd
        packed = pack_bits(bits)
        for r in range(m):
            if need == 0:
                break
            key = (int(packed[r, 0]), int(packed[r, 1]))
            if unique:
                if key in seen:
                    continue
                seen.add(key)
            rows.append(packed[r])
            need -= 1
    samples = np.stack(rows).astype(np.uint64)
    counts = rng.integers(1, max_count + 1, size=batch, dtype=np.int64)
    return samples, counts
