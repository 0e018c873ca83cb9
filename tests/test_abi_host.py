"""CPU-only tests of the C-ABI library: it loads, exports every symbol include/nqs.h declares, and its host
logic (Hamiltonian compile, mask packing, argument checking) matches the oracle bit-exactly.  No compute calls."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_2208_05637_b200 as nqs
from paper_2208_05637_b200 import workloads as wl
from oracle import compile as ocomp
from oracle import made as omade

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "nqs.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = sorted(set(re.findall(r"\b(nqs_[a-z_0-9]+)\s*\(", hdr)))
    assert {"nqs_ham_compile", "nqs_made_logpsi", "nqs_local_energy"} <= set(names)
    L = ctypes.CDLL(nqs.LIB_PATH)
    for nm in names:
        assert hasattr(L, nm), nm


def _assert_same(lib_t, ora_t):
    for k in ("flips", "offsets", "zy", "ycount", "coef"):
        a, b = lib_t[k], ora_t[k]
        assert a.dtype == b.dtype and a.shape == b.shape, k
        assert a.tobytes() == b.tobytes(), k            # bit-exact, including the fp32 cast


@pytest.mark.parametrize("n", [3, 17, 63, 64, 65, 128])
def test_compile_bit_exact_random_lists(n):
    rng = np.random.default_rng(n)
    K = 400
    codes = rng.integers(0, 4, size=(K, n)).astype(np.uint8)
    codes[:, rng.random(n) < 0.6] = 0                       # many identities -> shared flips
    codes[50:60] = codes[40:50]                              # duplicates
    coeffs = rng.standard_normal(K) * 10.0 ** rng.integers(-9, 3, size=K)
    coeffs[55] = -coeffs[45]                                 # exact cancellation
    H = nqs.ham_compile(codes, coeffs)
    ora = ocomp.compile_hamiltonian(codes, coeffs)
    _assert_same(H.export(), ora)
    assert H.K == ora["zy"].shape[0] and H.G == ora["flips"].shape[0]
    assert abs(H.sum_abs_coeff - ora["sum_abs_coeff"]) <= 1e-12 * max(1.0, ora["sum_abs_coeff"])
    # packed entry point gives the same tensors
    from oracle.pauli import incidence
    f, s, _ = incidence(codes)
    _assert_same(nqs.ham_compile_packed(n, f, s, coeffs).export(), ora)


@pytest.mark.parametrize("cfg", [1, 2])
def test_compile_bit_exact_workloads(cfg):
    w = wl.WORKLOADS[cfg]
    h, g = wl.make_integrals(w.n_spatial, w.seed_integrals)
    x, z, c = wl.jw_pauli_terms(h, g)
    codes = wl.masks_to_codes(x, z, w.n_qubits)
    H = nqs.ham_compile(codes, c)
    _assert_same(H.export(), ocomp.compile_hamiltonian(codes, c))
    Hp = nqs.ham_compile_packed(w.n_qubits, x, z, c)
    _assert_same(Hp.export(), H.export())


def _check_compiled_invariants(t, n, exact):
    """SURVEY 8(c) pins of the compiled tensors that need no second implementation: CSR covers every term, flips strictly
    ascending as 128-bit integers (word 1 major), ycount = popcount(flip & zy), and the group sizes of a JW chemistry
    Hamiltonian: 1 + n + C(n,2) diagonal strings, 2(n-1) per same-spin two-flip, 4 per aabb four-flip, 6 per aaaa / bbbb
    four-flip (exactly when nothing fell under the generator's 1e-8 drop, at most that otherwise)."""
    from math import comb
    flips, off, zy, yc = t["flips"], t["offsets"].astype(np.int64), t["zy"], t["ycount"]
    K, G, N = zy.shape[0], flips.shape[0], n // 2
    assert off[0] == 0 and off[-1] == K and np.all(np.diff(off) > 0)
    hi, lo = flips[:, 1], flips[:, 0]
    assert np.all((hi[1:] > hi[:-1]) | ((hi[1:] == hi[:-1]) & (lo[1:] > lo[:-1])))
    grp = np.repeat(np.arange(G), np.diff(off))
    pc = lambda a: np.bitwise_count(a).astype(np.int64)
    assert np.array_equal(pc(flips[grp, 0] & zy[:, 0]) + pc(flips[grp, 1] & zy[:, 1]), yc.astype(np.int64))
    # within a group the sign masks ascend strictly (rule 4; equal masks were merged by rule 2)
    same = grp[1:] == grp[:-1]
    zhi, zlo = zy[:, 1], zy[:, 0]
    assert np.all(~same | (zhi[1:] > zhi[:-1]) | ((zhi[1:] == zhi[:-1]) & (zlo[1:] > zlo[:-1])))
    nflip = pc(flips[:, 0]) + pc(flips[:, 1])
    sizes = np.diff(off)
    assert set(np.unique(nflip)) <= {0, 2, 4} and np.all(yc % 2 == 0)          # real integrals: even Y counts
    even = np.uint64(0x5555555555555555)
    n_even = pc(flips[:, 0] & even) + pc(flips[:, 1] & even)                   # flipped alpha (even) spin-orbitals
    cap = np.where(nflip == 0, 1 + n + comb(n, 2), np.where(nflip == 2, 2 * (n - 1), np.where(n_even == 2, 4, 6)))
    assert np.all(sizes <= cap)
    assert np.all((nflip != 2) | (n_even != 1)) and np.all((nflip != 4) | (n_even % 2 == 0))   # S_z is conserved
    if exact:
        assert np.array_equal(sizes, cap)
        assert G == 1 + 2 * comb(N, 2) + comb(N, 2) ** 2 + 2 * comb(N, 4)
        assert K == 1 + n + comb(n, 2) + 4 * (n - 1) * comb(N, 2) + 4 * comb(N, 2) ** 2 + 12 * comb(N, 4)
    else:
        assert G <= 1 + 2 * comb(N, 2) + comb(N, 2) ** 2 + 2 * comb(N, 4)


@pytest.mark.parametrize("cfg", [3, pytest.param(4, marks=pytest.mark.slow), pytest.param(5, marks=pytest.mark.slow)])
def test_compile_bit_exact_at_the_benchmarked_sizes(cfg):
    """north_star: "grouped tensors and flip masks must match bit-exactly" -- at the sizes that are benchmarked, not only
    cfg 1-2: 73,126 terms (cfg 3), ~0.67 M (cfg 4), ~2.8 M (cfg 5, the bench workload; about 100 s here, most of it
    the dict-based oracle).  PAPER.md:154-156, Fig. 1 (:101)."""
    w = wl.WORKLOADS[cfg]
    h, g = wl.make_integrals(w.n_spatial, w.seed_integrals)
    x, z, c = wl.jw_pauli_terms(h, g)
    H = nqs.ham_compile_packed(w.n_qubits, x, z, c)
    t = H.export()
    ora = ocomp.compile_hamiltonian(wl.masks_to_codes(x, z, w.n_qubits), c)
    _assert_same(t, ora)
    assert (H.K, H.G) == (ora["zy"].shape[0], ora["flips"].shape[0])
    assert abs(H.sum_abs_coeff - ora["sum_abs_coeff"]) <= 1e-12 * ora["sum_abs_coeff"]
    _check_compiled_invariants(t, w.n_qubits, exact=(cfg == 3))
    if cfg == 3:
        assert (H.K, H.G) == (73126, 13966)                                 # closed forms K(15), G(15), SURVEY 8


def test_compile_edge_cases_and_errors():
    L = nqs.lib()
    out = ctypes.c_void_p()
    codes = np.zeros((1, 4), np.uint8)
    co = np.ones(1)
    assert L.nqs_ham_compile(2, 1, codes.ctypes.data, co.ctypes.data, ctypes.byref(out)) == -2      # n < 3
    assert L.nqs_ham_compile(129, 1, codes.ctypes.data, co.ctypes.data, ctypes.byref(out)) == -2
    assert L.nqs_ham_compile(4, -1, codes.ctypes.data, co.ctypes.data, ctypes.byref(out)) == -1
    assert L.nqs_ham_compile(4, 1, None, co.ctypes.data, ctypes.byref(out)) == -1
    bad = np.full((1, 4), 4, np.uint8)
    assert L.nqs_ham_compile(4, 1, bad.ctypes.data, co.ctypes.data, ctypes.byref(out)) == -1       # code > 3
    assert out.value is None                                                                       # untouched
    H = nqs.ham_compile(np.zeros((0, 5), np.uint8), np.zeros(0), n_qubits=5)                        # K = 0 valid
    assert (H.K, H.G) == (0, 0) and H.export()["offsets"].tolist() == [0]
    # bits above n_qubits in packed masks are rejected
    f = np.array([[1 << 5, 0]], np.uint64)
    assert L.nqs_ham_compile_packed(5, 1, f.ctypes.data, f.ctypes.data, co.ctypes.data, ctypes.byref(out)) == -1
    assert nqs.lib().nqs_strerror(-5).decode().startswith("device is not")


@pytest.mark.parametrize("n,h,L,order,rd", [(8, 32, 2, "reverse", False), (13, 48, 1, "random", True),
                                            (76, 64, 2, "reverse", False)])
def test_made_masks_match_oracle(n, h, L, order, rd):
    p = wl.make_made_params(n, h, 3, n_hidden_layers=L, order=order)
    if rd:
        p.deg_hidden = np.random.default_rng(1).integers(1, n, size=(L, h)).astype(np.int32)
    M = nqs.made_create(p)
    masks = omade.build_masks(n, p.deg_hidden)
    for k in range(L + 1):
        expect = (p.weights[k].astype(np.float64) * masks[k]).astype(np.float32)
        assert np.array_equal(M.export_masked(k), expect)
    # NULL degrees = default sorted rule
    q = wl.make_made_params(n, h, 3, n_hidden_layers=L, order=order)
    q.deg_hidden = None
    M2 = nqs.made_create(q)
    dm = omade.build_masks(n, wl.default_degrees(n, h, L))
    assert np.array_equal(M2.export_masked(0), (q.weights[0].astype(np.float64) * dm[0]).astype(np.float32))


def test_made_create_errors():
    p = wl.make_made_params(8, 16, 1)
    p.order = np.array([0, 1, 2, 3, 4, 5, 6, 6], np.int32)            # not a permutation
    with pytest.raises(nqs.NqsError) as e:
        nqs.made_create(p)
    assert e.value.status == -1
    p = wl.make_made_params(8, 16, 1)
    p.deg_hidden = np.full((2, 16), 8, np.int32)                        # degree n is out of range
    with pytest.raises(nqs.NqsError) as e:
        nqs.made_create(p)
    assert e.value.status == -2
    p = wl.make_made_params(8, 16, 1)
    p.n_qubits = 2
    with pytest.raises(nqs.NqsError):
        nqs.made_create(p)


def test_compute_entry_points_fail_loudly_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    w, (x, z, c), params, samples, counts = wl.make_workload(1, batch=4)
    H = nqs.ham_compile_packed(w.n_qubits, x, z, c)
    M = nqs.made_create(params)
    with pytest.raises(nqs.NqsError) as e:
        nqs.local_energy_host(H, M, samples, counts)
    assert e.value.status in (-4, -5)


def test_host_entry_point_rejects_bits_above_n_qubits():
    """include/nqs.h: a sample with a bit >= n_qubits set is NQS_EINVAL; nqs_local_energy_host checks it on the host,
    before any device work (so the check runs here without a GPU)."""
    w, (x, z, c), params, samples, counts = wl.make_workload(1, batch=4)
    H = nqs.ham_compile_packed(w.n_qubits, x, z, c)
    M = nqs.made_create(params)
    bad = samples.copy()
    bad[2, 0] |= np.uint64(1) << np.uint64(w.n_qubits)
    with pytest.raises(nqs.NqsError) as e:
        nqs.local_energy_host(H, M, bad, counts)
    assert e.value.status == -1
    bad = samples.copy()
    bad[1, 1] = 1
    with pytest.raises(nqs.NqsError) as e:
        nqs.local_energy_host(H, M, bad, counts)
    assert e.value.status == -1


def test_tensor_core_path_shape_limits():
    """include/nqs.h: NQS_PATH_TC takes n_hidden_layers in {1, 2}, hidden in [1, 512] and every
    n_qubits in [3, 126] (two operand columns carry the biases: round16(n + 2) <= 128); everything else is
    NQS_EUNSUPPORTED and NQS_PATH_AUTO falls to the fp32 path (host-only query, no GPU needed)."""
    from paper_2208_05637_b200 import workloads as wl
    for n in (3, 4, 14, 15, 16, 17, 64, 76, 77, 80, 96, 112, 126):
        for h in (128, 256, 384, 512):
            for L in (1, 2):
                M = nqs.made_create(wl.make_made_params(n, h, 1, n_hidden_layers=L))
                assert M.resolved_path(nqs.PATH_TC) == nqs.PATH_TC, (n, h, L)
                assert M.resolved_path(nqs.PATH_AUTO) == nqs.PATH_TC
    for n in (127, 128):
        M = nqs.made_create(wl.make_made_params(n, 512, 1))
        with pytest.raises(nqs.NqsError) as ei:
            M.resolved_path(nqs.PATH_TC)
        assert ei.value.status == -6
        assert M.resolved_path(nqs.PATH_AUTO) == nqs.PATH_SIMT
    for n, h in ((20, 64), (20, 192), (8, 32), (20, 1), (20, 500)):                 # padded to a multiple of 128 inside
        M = nqs.made_create(wl.make_made_params(n, h, 1))
        assert M.resolved_path(nqs.PATH_TC) == nqs.PATH_TC and M.resolved_path(nqs.PATH_AUTO) == nqs.PATH_TC
    for n, h in ((20, 640), (20, 513), (20, 1024)):
        M = nqs.made_create(wl.make_made_params(n, h, 1))
        with pytest.raises(nqs.NqsError) as ei:
            M.resolved_path(nqs.PATH_TC)
        assert ei.value.status == -6
        assert M.resolved_path(nqs.PATH_AUTO) == nqs.PATH_SIMT


def test_text_loader_equals_operator_matrix_compile():
    """nqs_ham_compile_text (dense words, sparse factors, OpenFermion-style complex literals, comments) gives the same
    grouped tensors, bit for bit, as nqs_ham_compile on the parsed Operator Matrix."""
    rng = np.random.default_rng(4)
    n, K = 9, 60
    codes = rng.integers(0, 4, size=(K, n)).astype(np.uint8)
    codes[5] = 0
    codes[7] = codes[3]
    coeffs = rng.standard_normal(K)
    letters = "IXYZ"
    lines = ["# a comment line", ""]
    for t in range(K):
        c = repr(float(coeffs[t]))
        if t % 3 == 0:
            lines.append(f"{c} {''.join(letters[v] for v in codes[t])}")
        elif t % 3 == 1:
            lines.append(f"({c}+0j) [" + " ".join(f"{letters[v]}{j}" for j, v in enumerate(codes[t]) if v) + "]  # sparse")
        else:
            lines.append(f"{c} * " + " ".join(f"{letters[v]}{j}" for j, v in reversed(list(enumerate(codes[t]))) if v))
    Ht = nqs.ham_compile_text(n, "\n".join(lines) + "\n")
    Hc = nqs.ham_compile(codes, coeffs)
    a, b = Ht.export(), Hc.export()
    assert (Ht.K, Ht.G) == (Hc.K, Hc.G)
    for k in a:
        assert a[k].tobytes() == b[k].tobytes(), k
    for bad in ("0.5 XX", "0.5 X0 Y0", "(0.5+1j) X0", "abc X0", "0.5 Q1", "0.5 X99",
                # the coefficient is a finite decimal literal: no hex ("0X1 Z2" must not read as 1.0 * Z2), nan, inf, overflow
                "0X1 Z2", "0x1p3 Z2", "nan X0", "inf X0", "-inf X0", "1e400 X0", "0.5X0", ". X0",
                # a qubit named twice is refused whichever factor comes first, identity included
                "0.5 X0 I0", "0.5 I0 X0", "0.5 I3 I3"):
        with pytest.raises(nqs.NqsError):
            nqs.ham_compile_text(n, bad)
    assert nqs.ham_compile_text(n, "# nothing\n").K == 0
    ok = nqs.ham_compile_text(n, "+1.5e-3 X0 I1 Z2\n-.25 Y4\n(2.E0-0.0j) [Z1]\n")
    assert ok.K == 3 and abs(ok.sum_abs_coeff - (1.5e-3 + 0.25 + 2.0)) < 1e-15
