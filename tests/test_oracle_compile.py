"""Pins for oracle/compile.py (CPU only): invariants, closed-form counts, and equality of the grouped
evaluation with the ungrouped E_loc."""
from math import comb

import numpy as np
import pytest

from oracle import compile as ocomp
from oracle import eloc as oeloc
from oracle.pauli import popcount2, matrix_element
from paper_2208_05637_b200 import workloads as wl
from tests import bruteforce as bf


def _invariants(t, K_expected=None):
    off = t["offsets"].astype(np.int64)
    G = len(off) - 1
    K = t["zy"].shape[0]
    assert off[0] == 0 and off[-1] == K and np.all(np.diff(off) > 0)
    if K_expected is not None:
        assert K == K_expected
    f = t["flips"]
    key = [(int(a[1]) << 64) | int(a[0]) for a in f]
    assert all(key[i] < key[i + 1] for i in range(G - 1))                 # strictly ascending flips
    for gi in range(G):
        zy = t["zy"][off[gi]:off[gi + 1]]
        sk = [(int(a[1]) << 64) | int(a[0]) for a in zy]
        assert all(sk[i] < sk[i + 1] for i in range(len(sk) - 1))
        assert np.array_equal(popcount2(zy & f[gi][None, :]), t["ycount"][off[gi]:off[gi + 1]])


def test_merge_drop_sort():
    codes = np.array([[1, 0, 3], [0, 3, 0], [1, 0, 3], [2, 2, 0], [0, 3, 0], [3, 3, 3], [1, 1, 0]], dtype=np.uint8)
    coeffs = np.array([0.5, 1.0, 0.25, -2.0, -1.0, 3.0, 1e-30])
    t = ocomp.compile_hamiltonian(codes, coeffs)
    _invariants(t)
    # [0,3,0] cancels exactly -> dropped; [1,0,3] merged 0.75
    assert t["zy"].shape[0] == 4
    assert t["flips"][:, 0].tolist() == [0, 1, 3]
    assert t["offsets"].tolist() == [0, 1, 2, 4]
    g1 = t["coef"][1]
    assert g1 == np.float32(0.75)
    assert abs(t["sum_abs_coeff"] - (3.0 + 0.75 + 2.0 + 1e-30)) < 1e-12
    # group f=3: XX.(s=0) then YY.(s=3)
    assert t["zy"][2:, 0].tolist() == [0, 3] and t["ycount"].tolist() == [0, 0, 0, 2]


@pytest.mark.parametrize("cfg", [1, 2])
def test_generator_group_structure(cfg):
    """Closed forms: K(N), G(N); f=0 group has 1+n+C(n,2) terms, two-flip groups 2(n-1),
    aabb four-flip groups 4, aaaa/bbbb four-flip groups 6."""
    w = wl.WORKLOADS[cfg]
    h, g = wl.make_integrals(w.n_spatial, w.seed_integrals)
    x, z, c = wl.jw_pauli_terms(h, g)
    codes = wl.masks_to_codes(x, z, w.n_qubits)
    t = ocomp.compile_hamiltonian(codes, c)
    N, n = w.n_spatial, w.n_qubits
    K = 1 + n + comb(n, 2) + 4 * (n - 1) * comb(N, 2) + 4 * comb(N, 2) ** 2 + 12 * comb(N, 4)
    G = 1 + 2 * comb(N, 2) + comb(N, 2) ** 2 + 2 * comb(N, 4)
    _invariants(t, K)
    sizes = np.diff(t["offsets"].astype(np.int64))
    assert len(sizes) == G
    nflip = popcount2(t["flips"])
    assert sizes[nflip == 0].tolist() == [1 + n + comb(n, 2)]
    assert set(sizes[nflip == 2].tolist()) == {2 * (n - 1)} and (nflip == 2).sum() == 2 * comb(N, 2)
    assert set(sizes[nflip == 4].tolist()) <= {4, 6}
    assert (sizes[nflip == 4] == 6).sum() == 2 * comb(N, 4)
    assert abs(t["sum_abs_coeff"] - np.abs(c).sum()) < 1e-9


def test_grouped_evaluation_equals_ungrouped():
    """E_i = sum_g S[i,g] * psi(x^f_g)/psi(x) with S from the grouped tensors == term-by-term E_loc."""
    n = 6
    rng = np.random.default_rng(3)
    codes = rng.integers(0, 4, size=(120, n)).astype(np.uint8)
    coeffs = rng.standard_normal(120)
    t = ocomp.compile_hamiltonian(codes, coeffs)
    _invariants(t)
    psi = rng.standard_normal(2 ** n) + 1j * rng.standard_normal(2 ** n)
    xs = bf.all_configs(n)
    e_ref = oeloc.local_energy_generic(codes, coeffs, xs, lambda cfg: np.log(psi[cfg[:, 0].astype(np.int64)]))
    off = t["offsets"].astype(np.int64)
    e = np.zeros(2 ** n, dtype=np.complex128)
    for gi in range(len(off) - 1):
        sl = slice(off[gi], off[gi + 1])
        S = (t["coef"][sl].astype(np.float64)[None, :]
             * matrix_element(xs[:, None, :], t["zy"][sl][None, :, :], t["ycount"][sl].astype(np.int64))).sum(axis=1)
        xp = (xs[:, 0] ^ t["flips"][gi, 0]).astype(np.int64)
        e += S * psi[xp] / psi
    np.testing.assert_allclose(e, e_ref, rtol=1e-6, atol=1e-6)          # fp32 coefficient cast
