"""Local energy, term by term (oracle; test infrastructure).

l_theta(x) = sum_{p in S} alpha_p <x|P_p|x^p> f(x^p)/f(x)          (Eq. 15)
following Algorithm 1 in its order: (1) x^p = X xor F^{1,2}; (2) amplitudes f(x),
{f(x^p)}; (3) matrix elements by Eq. 16; (4) the sum.  E_loc is exact (it is (H psi)(x)/psi(x)), so this
IS the plain definition; fp64 throughout.  Terms are taken in input order, ungrouped; chunking over
terms only bounds memory.
"""
import numpy as np

from .pauli import incidence, matrix_element, unpack_mask, pack_mask
from . import made as _made


def local_energy_generic(codes, coeffs, samples, logpsi_fn, term_chunk: int = 16384,
                         memo: bool = False, return_max_ratio: bool = False):
    """E_loc for any wavefunction given as logpsi_fn(configs uint64[M,2]) -> complex128 [M].

    memo=True evaluates logpsi once per distinct x^p within a sample (allowed at the large configs,
    must equal memo=False — tested at cfg 1-2).
    """
    f, s, r = incidence(codes)
    coeffs = np.asarray(coeffs, dtype=np.float64)
    samples = np.asarray(samples, dtype=np.uint64)
    B, K = samples.shape[0], f.shape[0]
    out = np.zeros(B, dtype=np.complex128)
    max_ratio = 0.0
    lp0 = logpsi_fn(samples) if B else np.zeros(0, np.complex128)
    if memo and K:
        fu, inv = np.unique(f, axis=0, return_inverse=True)
        inv = inv.reshape(-1)
    for i in range(B):
        x = samples[i]
        if memo and K:
            lpu = np.concatenate([logpsi_fn(x[None, :] ^ fu[a:a + term_chunk])
                                  for a in range(0, fu.shape[0], term_chunk)])
            ratio_all = np.exp(lpu - lp0[i])[inv]
        E = 0.0 + 0.0j
        for a in range(0, K, term_chunk):
            b = min(K, a + term_chunk)
            xp = x[None, :] ^ f[a:b]                                   # Alg. 1 line 1
            if memo:
                ratio = ratio_all[a:b]
            else:
                ratio = np.exp(logpsi_fn(xp) - lp0[i])                 # Alg. 1 line 2 (log domain, Eq. 10)
            elem = matrix_element(x[None, :], s[a:b], r[a:b])          # Alg. 1 line 3 (Eq. 16)
            E += np.sum(coeffs[a:b] * elem * ratio)                    # Alg. 1 line 4 (Eq. 15)
            if ratio.size:
                max_ratio = max(max_ratio, float(np.max(np.abs(ratio))))
        out[i] = E
    if return_max_ratio:
        return out, max_ratio
    return out


def local_energy(codes, coeffs, params, samples, **kw):
    """E_loc of the MADE wavefunction `params` (oracle.made.logpsi)."""
    return local_energy_generic(codes, coeffs, samples, lambda c: _made.logpsi(params, c), **kw)


def local_energy_loops(codes, coeffs, x_bits, amp_fn):
    """Literal scalar transcription of Algorithm 1 for ONE sample (tiny cases only).

    codes: list of K lists of n ints in 0..3; x_bits: list of n ints; amp_fn(bits) -> complex f(bits).
    """
    n = len(x_bits)
    fx = amp_fn(list(x_bits))
    total = 0.0 + 0.0j
    for p, alpha in zip(codes, coeffs):
        xp = [x_bits[k] ^ (1 if p[k] in (1, 2) else 0) for k in range(n)]       # X xor F^{1,2}
        r = sum(1 for k in range(n) if p[k] == 2)
        elem = (-1j) ** r
        for k in range(n):
            if p[k] in (2, 3):
                elem *= (-1) ** x_bits[k]                                          # Eq. 16
        total += alpha * elem * amp_fn(xp) / fx                                    # Eq. 15
    return total


def weighted_stats(eloc: np.ndarray, counts: np.ndarray, max_ratio: float = float("nan")):
    """Count-weighted statistics of Eq. 17 with repeated samples collapsed:
    [sum n, sum n Re E, sum n Im E, sum n |E|^2, max |ratio|]."""
    c = np.asarray(counts, dtype=np.float64)
    e = np.asarray(eloc, dtype=np.complex128)
    return np.array([c.sum(), (c * e.real).sum(), (c * e.imag).sum(), (c * np.abs(e) ** 2).sum(), max_ratio])
