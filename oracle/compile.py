"""Grouped Hamiltonian tensors (oracle; test infrastructure) — PAPER.md:154-156: "collect the indices of
sigma_1, sigma_2 operators prior to the training and only keep a buffer of unique flippings and their
corresponding number of occurrences".

Compile rules: (1) per term (f, s), r; (2) terms with identical
(f, s) merged, coefficients summed in fp64 in INPUT order, left to right; (3) nothing dropped except an
exact 0.0 after merging; (4) groups ordered by f ascending as an unsigned 128-bit integer (word 1 major),
terms within a group by s ascending the same way; (5) coef = float32(c) round-to-nearest-even,
ycount = r, offsets = term indices with offsets[G] = K.

Deliberately written with Python dicts/ints (not the sort-based scheme of the C++ compiler).
"""
import numpy as np

from .pauli import incidence


def compile_hamiltonian(codes, coeffs):
    f, s, r = incidence(codes)
    coeffs = np.asarray(coeffs, dtype=np.float64)
    merged = {}                                   # (f128, s128) -> [sum, r]; dict keeps first-seen order
    for k in range(f.shape[0]):
        key = ((int(f[k, 1]) << 64) | int(f[k, 0]), (int(s[k, 1]) << 64) | int(s[k, 0]))
        if key in merged:
            merged[key][0] = merged[key][0] + float(coeffs[k])
        else:
            merged[key] = [float(coeffs[k]), int(r[k])]
    items = sorted((key, v) for key, v in merged.items() if v[0] != 0.0)
    K = len(items)
    zy = np.zeros((K, 2), dtype=np.uint64)
    ycount = np.zeros(K, dtype=np.uint8)
    coef = np.zeros(K, dtype=np.float32)
    flips, offsets = [], []
    last = None
    m64 = (1 << 64) - 1
    for t, ((fk, sk), (c, rr)) in enumerate(items):
        if fk != last:
            flips.append((fk & m64, fk >> 64))
            offsets.append(t)
            last = fk
        zy[t, 0], zy[t, 1] = sk & m64, sk >> 64
        ycount[t] = rr
        coef[t] = np.float32(c)
    offsets.append(K)
    return {
        "flips": np.array(flips, dtype=np.uint64).reshape(-1, 2),
        "offsets": np.array(offsets, dtype=np.uint32),
        "zy": zy, "ycount": ycount, "coef": coef,
        "sum_abs_coeff": float(np.sum(np.abs([v[0] for _, v in items]))) if K else 0.0,
    }
