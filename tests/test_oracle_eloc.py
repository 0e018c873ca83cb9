"""Pins for oracle/eloc.py (CPU only): E_loc(x) = (H psi)(x)/psi(x) against dense matrices."""
import numpy as np
import pytest

from oracle import eloc as oeloc
from oracle import made as omade
from oracle import jw as ojw
from paper_2208_05637_b200 import workloads as wl
from tests import bruteforce as bf


def _random_pauli_list(n, K, seed):
    rng = np.random.default_rng(seed)
    codes = rng.integers(0, 4, size=(K, n)).astype(np.uint8)
    codes[0] = 0                                            # identity
    codes[1] = 2                                            # all Y (odd r when n odd)
    codes[2] = codes[3]                                     # a duplicate string
    coeffs = rng.standard_normal(K)
    return codes, coeffs


@pytest.mark.parametrize("n", [3, 5, 8])
def test_eloc_equals_Hpsi_over_psi_for_arbitrary_table(n):
    """Pins Alg. 1 / Eq. 15-16 independently of MADE: random complex psi table, generic (odd-Y) Hamiltonian."""
    codes, coeffs = _random_pauli_list(n, 60, n)
    rng = np.random.default_rng(n + 100)
    psi = rng.standard_normal(2 ** n) + 1j * rng.standard_normal(2 ** n)
    H = bf.dense_pauli_sum(codes, coeffs)
    xs = bf.all_configs(n)
    fn = lambda cfg: np.log(psi[cfg[:, 0].astype(np.int64)])
    e = oeloc.local_energy_generic(codes, coeffs, xs, fn, term_chunk=7)
    np.testing.assert_allclose(e, (H @ psi) / psi, rtol=1e-11, atol=1e-11)
    e2 = oeloc.local_energy_generic(codes, coeffs, xs, fn, memo=True)
    np.testing.assert_allclose(e2, e, rtol=1e-12, atol=1e-12)


def test_eloc_diagonal_element():
    """psi = basis state |x>: E_loc(x) = H_xx = sum over f_t = 0 terms of c_t (-1)^{popcount(x & s_t)}."""
    n = 6
    codes, coeffs = _random_pauli_list(n, 80, 5)
    codes[10:30][codes[10:30] == 1] = 0                     # make plenty of diagonal (I/Z only) strings
    codes[10:30][codes[10:30] == 2] = 3
    H = bf.dense_pauli_sum(codes, coeffs)
    xs = bf.all_configs(n)
    for i in (0, 13, 63):
        x = xs[i:i + 1]
        with np.errstate(divide="ignore"):
            fn = lambda cfg: np.where(cfg[:, 0] == x[0, 0], 0.0, -np.inf).astype(np.complex128)
            e = oeloc.local_energy_generic(codes, coeffs, x, fn)
        assert abs(e[0] - H[i, i]) < 1e-12


def test_energy_identity_with_made_wavefunction():
    """sum_x |psi|^2 E_loc / sum_x |psi|^2 = <psi|H|psi>/<psi|psi> on a JW Hamiltonian."""
    N = 3
    n = 2 * N
    h, g = wl.make_integrals(N, 321)
    terms = ojw.jw_hamiltonian(h, g)
    codes = np.array(list(terms.keys()), dtype=np.uint8)
    coeffs = np.array([terms[tuple(k)] for k in codes])
    p = wl.make_made_params(n, 16, 77)
    xs = bf.all_configs(n)
    lp = omade.logpsi(p, xs)
    psi = np.exp(lp)
    e = oeloc.local_energy(codes, coeffs, p, xs)
    w = np.abs(psi) ** 2
    lhs = (w * e).sum() / w.sum()
    H = bf.dense_pauli_sum(codes, coeffs)
    rhs = (psi.conj() @ H @ psi) / (psi.conj() @ psi)
    assert abs(lhs - rhs) < 1e-11
    assert abs(lhs.imag) < 1e-11
    np.testing.assert_allclose(e, (H @ psi) / psi, rtol=1e-10, atol=1e-10)


def test_loops_transcription_equals_vectorised():
    n = 4
    codes, coeffs = _random_pauli_list(n, 25, 8)
    p = wl.make_made_params(n, 8, 5, order="random")
    xs = bf.all_configs(n)
    e = oeloc.local_energy(codes, coeffs, p, xs)

    def amp(bits):
        cfg = np.zeros((1, 2), dtype=np.uint64)
        cfg[0, 0] = sum(int(b) << j for j, b in enumerate(bits))
        return np.exp(omade.logpsi(p, cfg)[0])

    for i in (0, 5, 15):
        bits = [(i >> j) & 1 for j in range(n)]
        el = oeloc.local_energy_loops([list(map(int, r)) for r in codes], list(coeffs), bits, amp)
        assert abs(el - e[i]) < 1e-12


def test_memo_equals_strict_on_cfg1_subset():
    w, (x, z, c), params, samples, counts = wl.make_workload(1, batch=8)
    codes = wl.masks_to_codes(x, z, w.n_qubits)
    e0 = oeloc.local_energy(codes, c, params, samples)
    e1, mr = oeloc.local_energy(codes, c, params, samples, memo=True, return_max_ratio=True)
    np.testing.assert_allclose(e1, e0, rtol=1e-12, atol=1e-12)
    assert mr >= 1.0                                     # the f = 0 terms have ratio exactly 1
    assert np.abs(e0.imag).min() > 1e-3                  # complex psi (phase net): Im E_loc of every sample is nonzero


def test_memo_equals_strict_on_cfg2_subset():
    """BASELINE.md section 3 / SURVEY 8(c): the memoised mode (used for cfg 4-5 and the timed baseline) equals the strict
    term-by-term mode on cfg 1 AND cfg 2."""
    w, (x, z, c), params, samples, counts = wl.make_workload(2, batch=4)
    codes = wl.masks_to_codes(x, z, w.n_qubits)
    e0 = oeloc.local_energy(codes, c, params, samples)
    e1 = oeloc.local_energy(codes, c, params, samples, memo=True)
    np.testing.assert_allclose(e1, e0, rtol=1e-12, atol=1e-12)


def test_weighted_stats():
    e = np.array([1 + 2j, -3 + 0.5j, 0.25j])
    n = np.array([2, 5, 1])
    s = oeloc.weighted_stats(e, n, 1.5)
    assert s[0] == 8 and abs(s[1] - (2 - 15)) < 1e-15 and abs(s[2] - (4 + 2.5 + 0.25)) < 1e-15
    assert abs(s[3] - (2 * 5 + 5 * 9.25 + 0.0625)) < 1e-12 and s[4] == 1.5
