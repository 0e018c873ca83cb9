"""Pins for oracle/pauli.py, oracle/jw.py and the fast JW input generator (CPU only)."""
import os

import numpy as np
import pytest

from oracle import pauli as opauli
from oracle import jw as ojw
from paper_2208_05637_b200 import workloads as wl
from tests import bruteforce as bf


def test_matrix_element_vs_kronecker_including_odd_Y():
    """PAPER.md:158 Eq. 16 + :150 "exactly one column index x^p": every row x of kron(sigma...) has its
    single nonzero at column x xor F^{1,2}, with value (-i)^r prod (-1)^{x_k}."""
    rng = np.random.default_rng(1)
    for n in (1, 2, 3, 5, 6):
        codes = rng.integers(0, 4, size=(40, n)).astype(np.uint8)
        codes[0] = 2                                    # all-Y string: r = n (odd for odd n)
        f, s, r = opauli.incidence(codes)
        xs = bf.all_configs(n)
        for k in range(codes.shape[0]):
            P = bf.dense_pauli_string(codes[k])
            assert np.count_nonzero(P) == 2 ** n
            cols = (xs[:, 0] ^ f[k, 0]).astype(np.int64)
            vals = P[np.arange(2 ** n), cols]
            me = opauli.matrix_element(xs, s[k][None, :], r[k:k + 1])
            np.testing.assert_allclose(me, vals, atol=0)


def test_pack_unpack_roundtrip_two_words():
    rng = np.random.default_rng(2)
    for n in (1, 63, 64, 65, 76, 128):
        bits = rng.integers(0, 2, size=(17, n)).astype(np.uint8)
        p = opauli.pack_mask(bits)
        assert np.array_equal(opauli.unpack_mask(p, n), bits)
        assert np.array_equal(opauli.popcount2(p), bits.sum(axis=1))


def _dict_from_masks(x, z, c, n):
    codes = wl.masks_to_codes(x, z, n)
    return {tuple(int(v) for v in row): float(cc) for row, cc in zip(codes, c)}


@pytest.mark.parametrize("N", [2, 3, 4])
def test_jw_hermitian_equals_slater_condon_commutes_with_number(N):
    """The JW Pauli sum (oracle.jw, by definition) is Hermitian, equals the determinant-basis
    Hamiltonian built independently on occupation bit strings, commutes with N and S_z; all Y counts even."""
    h, g = wl.make_integrals(N, 1234 + N)
    terms = ojw.jw_hamiltonian(h, g)
    codes = list(terms.keys())
    coeffs = [terms[k] for k in codes]
    assert all(sum(1 for c in k if c == 2) % 2 == 0 for k in codes)
    H = bf.dense_pauli_sum(codes, coeffs)
    n = 2 * N
    np.testing.assert_allclose(H, H.conj().T, atol=1e-12)
    Hsc = bf.slater_condon(h, g)
    np.testing.assert_allclose(H.real, Hsc, atol=1e-7)          # 1e-8 drop tolerance
    np.testing.assert_allclose(H.imag, 0, atol=1e-12)
    Nop = bf.number_operator(n)
    np.testing.assert_allclose(H @ Nop, Nop @ H, atol=1e-10)
    idx = np.arange(2 ** n, dtype=np.uint64)
    sz = np.diag((np.bitwise_count(idx & np.uint64(0x5555555555555555)).astype(float)
                  - np.bitwise_count(idx & np.uint64(0xAAAAAAAAAAAAAAAA)).astype(float)))
    np.testing.assert_allclose(H @ sz, sz @ H, atol=1e-10)


@pytest.mark.parametrize("N", [2, 3, 4, 5])
def test_fast_generator_equals_oracle_jw(N):
    h, g = wl.make_integrals(N, 99 + N)
    x, z, c = wl.jw_pauli_terms(h, g)
    fast = _dict_from_masks(x, z, c, 2 * N)
    slow = ojw.jw_hamiltonian(h, g)
    assert set(fast.keys()) == set(slow.keys())
    for k in slow:
        assert abs(fast[k] - slow[k]) <= 1e-12 * max(1.0, abs(slow[k]))


def test_generator_counts_closed_form():
    """K(N), G(N) for dense integrals: cfg 1 -> 361 / 51."""
    from math import comb
    for N in (2, 3, 4, 5, 6):
        h, g = wl.make_integrals(N, 7 + N)
        x, z, c = wl.jw_pauli_terms(h, g)
        n = 2 * N
        K = 1 + n + comb(n, 2) + 4 * (n - 1) * comb(N, 2) + 4 * comb(N, 2) ** 2 + 12 * comb(N, 4)
        G = 1 + 2 * comb(N, 2) + comb(N, 2) ** 2 + 2 * comb(N, 4)
        assert len(c) == K
        assert len(np.unique(x, axis=0)) == G


def test_h2_shape_golden():
    """tests/golden/h2_shape.txt: H2-symmetric integrals give K = 15 = 1 + 4 Z + 6 ZZ + 4 flips."""
    gold = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "h2_shape.txt")) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            k, *v = line.split()
            gold[k] = v
    h = np.diag([-1.25, -0.47])
    g = np.zeros((2, 2, 2, 2))
    g[0, 0, 0, 0], g[1, 1, 1, 1] = 0.67, 0.70
    g[0, 0, 1, 1] = g[1, 1, 0, 0] = 0.66
    for idx in [(0, 1, 0, 1), (0, 1, 1, 0), (1, 0, 0, 1), (1, 0, 1, 0)]:
        g[idx] = 0.18
    terms = ojw.jw_hamiltonian(h, g)
    assert len(terms) == int(gold["K"][0])
    strs = ["".join("IXYZ"[c] for c in k) for k in terms]
    assert sum(s == "IIII" for s in strs) == int(gold["identity"][0])
    assert sum(sorted(s) == list("IIIZ") for s in strs) == int(gold["single_Z"][0])
    assert sum(sorted(s) == list("IIZZ") for s in strs) == int(gold["double_Z"][0])
    assert sorted(s for s in strs if "X" in s) == sorted(gold["four_flip_strings"])
    x, z, c = wl.jw_pauli_terms(h, g)
    assert len(c) == 15
