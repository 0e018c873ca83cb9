"""GPU parity tests (-m gpu): the CUDA path, called through the C ABI, against the fp64 oracle on the same
seeded inputs.  Tolerances:
  * E_loc: |dE| <= 1e-5 * sum_t |c_t| per sample, complex modulus (BASELINE.json north_star);
  * log psi (NQS_PATH_SIMT, fp32): 2e-4 absolute — n <= 128 conditionals of |log pi| <~ 10 summed in fp32
    after <= 1024-term fp32 dot products;
  * contraction S[i,g]: 4 ulp(fp32) * sum_{t in g} |c_t|  (sequential fp32 sum of exactly rounded +-c_t);
  * grouped tensors: bit-exact (tests/test_abi_host.py).
"""
import numpy as np
import pytest
import torch

import paper_2208_05637_b200 as nqs
from paper_2208_05637_b200 import workloads as wl
from oracle import eloc as oeloc
from oracle import made as omade
from oracle import compile as ocomp
from oracle.pauli import matrix_element

pytestmark = pytest.mark.gpu
DEV = "cuda:0"
# log psi on the tensor-core path: weights and hidden activations are rounded to fp16 (relative 2^-11 = 4.9e-4 per
# operand), accumulated in fp32.  Each of the <= 128 conditionals' logits carries ~ 2^-11 * |a| * sqrt(2/3) of
# independent rounding error from each of the three layers; the sum of n <= 128 log-sigmoids (slope <= 1) of
# logits |a| <~ 3 then carries <~ sqrt(128) * 3 * 3 * 4.9e-4 / 2 ~ 2.5e-2 in the worst alignment and ~3e-3 as an rms
# over random signs.  Measured maximum over every shape below: 7.7e-4.  Bound = 3e-3.
TC_LOGPSI_TOL = 3e-3
# E_loc on the tensor-core path for h <= 256: split-precision operands (hi + lo fp16 parts, three MMA passes, DESIGN.md
# section 8) — the north_star bound 1e-5 sum|c| itself, no slack factor (round 1 needed 10 with single-pass fp16).
TC_NARROW_FACTOR = 1.0


def _dev_u64(a):
    return torch.from_numpy(np.ascontiguousarray(a).view(np.int64)).to(DEV)


_cache = {}


def workload(cfg):
    if cfg not in _cache:
        w = wl.WORKLOADS[cfg]
        h, g = wl.make_integrals(w.n_spatial, w.seed_integrals)
        x, z, c = wl.jw_pauli_terms(h, g)
        params = wl.make_made_params(w.n_qubits, w.hidden, w.seed_weights)
        H = nqs.ham_compile_packed(w.n_qubits, x, z, c)
        M = nqs.made_create(params)
        _cache[cfg] = (w, (x, z, c), params, H, M)
    return _cache[cfg]


def _paths(M, min_hidden_tc=0):
    # SIMT always; TC wherever the shape supports it (that is where NQS_PATH_AUTO selects it, include/nqs.h).
    out = [nqs.PATH_SIMT]
    if M.hidden < min_hidden_tc:
        return out
    try:
        assert M.resolved_path(nqs.PATH_TC) == nqs.PATH_TC
        out.append(nqs.PATH_TC)
    except nqs.NqsError as e:
        assert e.status == -6
    return out


@pytest.mark.parametrize("n,h,L,order", [(8, 32, 2, "reverse"), (20, 128, 2, "reverse"), (30, 256, 2, "identity"),
                                         (76, 512, 2, "reverse"), (13, 48, 1, "random"), (128, 64, 2, "random"),
                                         (65, 16, 2, "reverse"), (3, 8, 1, "identity"),
                                         # tensor-core shape limits: one hidden layer (the paper's own architecture,
                                         # PAPER.md:84), n = 3 / 77 (two accumulators) / 96 / 112 / 126 (the largest n
                                         # the tensor-core path takes; 127 and 128 run on the fp32 path), odd chunk counts
                                         (126, 512, 2, "random"), (125, 384, 1, "reverse"), (127, 256, 2, "reverse"),
                                         (30, 128, 1, "identity"), (52, 512, 1, "reverse"), (76, 384, 1, "random"),
                                         (3, 128, 2, "identity"), (77, 512, 2, "reverse"), (96, 512, 2, "random"),
                                         (112, 512, 2, "reverse"), (128, 512, 2, "random"), (128, 384, 1, "reverse")])
def test_logpsi_parity(n, h, L, order):
    p = wl.make_made_params(n, h, 100 + n, n_hidden_layers=L, order=order)
    rng = np.random.default_rng(n)
    B = 333                                                      # several tiles + ragged tail
    bits = rng.integers(0, 2, size=(B, n)).astype(np.uint8)
    cfgs = wl.pack_bits(bits)
    ref = omade.logpsi(p, cfgs)
    M = nqs.made_create(p)
    for path in _paths(M, min_hidden_tc=0):
        out = nqs.made_logpsi(M, _dev_u64(cfgs), path=path).cpu().numpy().astype(np.float64)
        tol = 2e-4 if path == nqs.PATH_SIMT else TC_LOGPSI_TOL
        assert np.abs(out[:, 0] - ref.real).max() < tol, (path, np.abs(out[:, 0] - ref.real).max())
        assert np.abs(out[:, 1] - ref.imag).max() < tol, (path, np.abs(out[:, 1] - ref.imag).max())
    assert nqs.made_logpsi(M, torch.zeros((0, 2), dtype=torch.int64, device=DEV)).shape == (0, 2)   # B = 0


def test_logpsi_tensor_core_vs_fp32_path_random_shapes():
    """Fuzz over shapes the fixed lists do not name: random (n, hidden, layers, order, degrees) with hidden NOT a
    multiple of 128 (zero-padded inside), both precisions (split for padded hidden <= 256, single pass above), two or
    three accumulators, ragged multi-tile launches.  GPU vs GPU against the fp32 path (itself checked against the
    oracle above), so 24 shapes cost a second; two shapes also go to the oracle."""
    rng = np.random.default_rng(2208)
    worst = {}
    for it in range(24):
        n = int(rng.integers(3, 127))
        h = int(rng.integers(1, 513))
        L = int(rng.integers(1, 3))
        order = ["reverse", "identity", "random"][int(rng.integers(0, 3))]
        p = wl.make_made_params(n, h, 5000 + it, n_hidden_layers=L, order=order)
        if it % 3 == 0:                                          # unsorted degrees: masks are not prefixes
            p.deg_hidden = rng.integers(1, max(2, n), size=(L, h)).astype(np.int32)
        M = nqs.made_create(p)
        assert M.resolved_path(nqs.PATH_TC) == nqs.PATH_TC, (n, h, L)
        B = int(rng.integers(1, 1200))
        cfgs = wl.pack_bits(rng.integers(0, 2, size=(B, n)).astype(np.uint8))
        a = nqs.made_logpsi(M, _dev_u64(cfgs), path=nqs.PATH_TC).cpu().numpy().astype(np.float64)
        b = nqs.made_logpsi(M, _dev_u64(cfgs), path=nqs.PATH_SIMT).cpu().numpy().astype(np.float64)
        hp = (h + 127) // 128 * 128
        tol = 4e-4 if hp <= 256 else TC_LOGPSI_TOL               # split precision: the fp32 path's own 2e-4, twice
        err = np.abs(a - b).max()
        worst[hp <= 256] = max(worst.get(hp <= 256, 0.0), err)
        assert np.isfinite(a).all() and err < tol, (n, h, L, order, B, err)
        if it in (1, 2):
            ref = omade.logpsi(p, cfgs[:16])
            assert np.abs(a[:16, 0] - ref.real).max() < tol and np.abs(a[:16, 1] - ref.imag).max() < tol
    print(f"[parity] TC vs fp32 path over 24 random shapes: max|dlogpsi| split {worst.get(True, 0):.2e}, single pass {worst.get(False, 0):.2e}")


def test_tc_flops_bookkeeping():
    """nqs_made_tc_flops (the roofline report's issued / dense flops per psi evaluation): the dense figure is the
    chain's plain MAC count on the padded shapes, the issued one lies between the algorithmic count bench.py uses
    (423,346 at cfg 5) and the dense one in single-pass mode, and is about three times larger in
    split-precision mode."""
    w, _, params, _, M = workload(5)
    issued, dense = M.tc_flops()
    n, h = w.n_qubits, w.hidden
    KI, KO = 80, 80                                              # round16(n + 2), round16(n + 4)
    assert dense == 2 * (2 * KI * h + h * h + KO * h + 16 * h)   # W1 + P1 (K = KI), W2, W3 (N = KO), P2 (N = 16)
    assert 423346 < issued < dense
    w2, _, params2, _, M2 = workload(2)
    i2, d2 = M2.tc_flops()
    assert i2 > 2 * (2 * (11185 + 2816))                         # split precision issues > 2 x the algorithmic flops


def test_eloc_tensor_core_vs_fp32_path_random_shapes():
    """The same fuzz through nqs_local_energy: random generic Hamiltonians (odd Y counts, with and without an f = 0
    group) on random model shapes, several ragged sample blocks, counts; every row of the tensor-core path against the
    fp32 path, which the oracle tests above pin.  Bound: sum|c| max|ratio| times the ratio error the log psi bound
    allows (2 sqrt 2 tol), as in test_generic_odd_Y_no_diagonal_on_tensor_core_path."""
    rng = np.random.default_rng(52637)
    for it in range(10):
        n = int(rng.integers(5, 127))
        h = int(rng.integers(1, 513))
        L = int(rng.integers(1, 3))
        p = wl.make_made_params(n, h, 7000 + it, n_hidden_layers=L, order=["reverse", "random"][it & 1])
        if it % 4 == 1:
            p.deg_hidden = rng.integers(1, n, size=(L, h)).astype(np.int32)
        codes, coeffs = _few_flip_pauli_list(rng, n, 120)
        if it % 2 == 0:
            codes[:30, 0] = np.where(codes[:30, 0] == 2, 3, 0)   # some strings without any flip: an f = 0 group exists
            codes[:30, 1:] = np.where(np.isin(codes[:30, 1:], (1, 2)), 3, codes[:30, 1:])
        H = nqs.ham_compile(codes, coeffs)
        M = nqs.made_create(p)
        B = int(rng.integers(1, 700))
        xs = _dev_u64(wl.pack_bits(rng.integers(0, 2, size=(B, n)).astype(np.uint8)))
        cn = torch.from_numpy(rng.integers(1, 50, size=B).astype(np.int64)).to(DEV)
        mb = [0, 128, 200][it % 3]
        e_tc, s_tc = nqs.local_energy(H, M, xs, cn, minibatch=mb, path=nqs.PATH_TC)
        e_si, s_si = nqs.local_energy(H, M, xs, cn, minibatch=mb, path=nqs.PATH_SIMT)
        d = (e_tc - e_si).cpu().numpy().astype(np.float64)
        hp = (h + 127) // 128 * 128
        tol = H.sum_abs_coeff * max(1.0, s_si[4]) * 2 * 2 ** 0.5 * (4e-4 if hp <= 256 else TC_LOGPSI_TOL)
        err = np.hypot(d[:, 0], d[:, 1]).max()
        assert torch.isfinite(e_tc).all() and err <= tol, (it, n, h, L, B, err, tol)
        assert s_tc[0] == s_si[0] and abs(s_tc[1] - s_si[1]) <= tol * s_si[0]


@pytest.mark.parametrize("n,h", [(20, 128), (76, 128), (40, 256), (76, 512), (100, 384)])
def test_logpsi_tensor_core_many_tiles_per_cta(n, h):
    """Persistent-kernel paths that a few-tile launch never reaches: every CTA walks several 128-row tiles, so
    the weight ring wraps, the double-buffered operand tile and every barrier parity are re-used (a producer
    lane running ahead of the ring aliased a barrier parity exactly here).  Sampled rows against the oracle."""
    p = wl.make_made_params(n, h, 300 + n)
    M = nqs.made_create(p)
    try:
        assert M.resolved_path(nqs.PATH_TC) == nqs.PATH_TC
    except nqs.NqsError as e:
        assert e.status == -6
        pytest.skip("shape not supported by the tensor-core path")
    B = 128 * 148 * 3 + 77                                       # 3+ tiles per CTA and a ragged tail
    rng = np.random.default_rng(n + h)
    cfgs = wl.pack_bits(rng.integers(0, 2, size=(B, n)).astype(np.uint8))
    out = nqs.made_logpsi(M, _dev_u64(cfgs), path=nqs.PATH_TC).cpu().numpy().astype(np.float64)
    idx = np.concatenate([np.arange(40), rng.choice(B, size=200, replace=False), np.arange(B - 40, B)])
    ref = omade.logpsi(p, cfgs[idx])
    assert np.isfinite(out).all()
    assert np.abs(out[idx, 0] - ref.real).max() < TC_LOGPSI_TOL
    assert np.abs(out[idx, 1] - ref.imag).max() < TC_LOGPSI_TOL


@pytest.mark.parametrize("cfg,B", [(1, 256), (2, 300), (3, 130)])
def test_contraction_parity(cfg, B):
    w, (x, z, c), params, H, M = workload(cfg)
    samples, _ = wl.make_samples(w.n_spatial, w.n_alpha, w.n_beta, B, w.max_count, w.seed_samples, w.unique)
    t = H.export()
    off = t["offsets"].astype(np.int64)
    g0, g1 = (0, H.G) if cfg < 3 else (5, 1200)
    S = nqs.pauli_contract(H, _dev_u64(samples), g0, g1).cpu().numpy().astype(np.float64)
    S = S[..., 0] + 1j * S[..., 1]                               # [g, B]
    for gi in range(g0, g1):
        sl = slice(off[gi], off[gi + 1])
        cc = t["coef"][sl].astype(np.float64)
        ref = (cc[None, :] * matrix_element(samples[:, None, :], t["zy"][sl][None, :, :],
                                            t["ycount"][sl].astype(np.int64))).sum(axis=1)
        tol = 4 * 2.0 ** -24 * np.abs(cc).sum() * max(1, sl.stop - sl.start) ** 0.5 + 1e-30
        assert np.abs(S[gi - g0] - ref).max() <= tol, (gi, np.abs(S[gi - g0] - ref).max(), tol)


def _check_eloc(cfg, B_gpu, n_oracle, minibatch, memo=False):
    w, (x, z, c), params, H, M = workload(cfg)
    samples, counts = wl.make_samples(w.n_spatial, w.n_alpha, w.n_beta, B_gpu, w.max_count, w.seed_samples, w.unique)
    codes = wl.masks_to_codes(x, z, w.n_qubits)
    rng = np.random.default_rng(cfg)
    pick = np.sort(rng.choice(B_gpu, size=min(n_oracle, B_gpu), replace=False))
    ref = oeloc.local_energy(codes, c, params, samples[pick], memo=memo)
    tol = 1e-5 * H.sum_abs_coeff
    res = {}
    for path in _paths(M):
        e, stats = nqs.local_energy(H, M, _dev_u64(samples), torch.from_numpy(counts).to(DEV), minibatch=minibatch, path=path)
        e = e.cpu().numpy().astype(np.float64)
        ec = e[:, 0] + 1j * e[:, 1]
        err = np.abs(ec[pick] - ref).max()
        assert err <= tol, (cfg, path, err, tol)
        ws = oeloc.weighted_stats(ec, counts)
        np.testing.assert_allclose(stats[:4], ws[:4], rtol=1e-9)
        assert stats[4] >= 1.0 and np.isfinite(stats[4])
        res[path] = (err / tol, ec)
        print(f"[parity] cfg {cfg} path {path}: max|dE_loc|/tol = {err / tol:.4f} over {len(pick)} oracle samples "
              f"(tol = 1e-5 * sum|c| = {tol:.3e})")
    return res


def test_eloc_cfg1_all_samples_and_full_sector():
    _check_eloc(1, 256, 256, 256)
    # the whole 2a+2b sector (36 states), A16
    w, (x, z, c), params, H, M = workload(1)
    from itertools import combinations
    rows = []
    for a in combinations(range(4), 2):
        for b in combinations(range(4), 2):
            bits = np.zeros(8, np.uint8)
            for k in a: bits[2 * k] = 1
            for k in b: bits[2 * k + 1] = 1
            rows.append(bits)
    sector = wl.pack_bits(np.array(rows))
    ref = oeloc.local_energy(wl.masks_to_codes(x, z, 8), c, params, sector)
    e, _ = nqs.local_energy(H, M, _dev_u64(sector), None, path=nqs.PATH_SIMT)
    e = e.cpu().numpy().astype(np.float64)
    assert np.abs(e[:, 0] + 1j * e[:, 1] - ref).max() <= 1e-5 * H.sum_abs_coeff


def test_eloc_cfg2_bench_configuration():
    _check_eloc(2, 4096, 192, 4096)


def test_eloc_cfg2_explicit_tensor_core_path():
    """NQS_PATH_TC on a narrow net (h = 128): split-precision operands keep |dE| inside the north_star bound
    1e-5 * sum|c| (single-pass fp16 gave 1.9-2.2 x the bound here)."""
    w, (x, z, c), params, H, M = workload(2)
    samples, counts = wl.make_samples(w.n_spatial, w.n_alpha, w.n_beta, 512, w.max_count, w.seed_samples, True)
    ref = oeloc.local_energy(wl.masks_to_codes(x, z, w.n_qubits), c, params, samples[:64])
    e, st = nqs.local_energy(H, M, _dev_u64(samples), None, path=nqs.PATH_TC)
    e = e.cpu().numpy().astype(np.float64)
    err = np.abs(e[:64, 0] + 1j * e[:64, 1] - ref).max()
    print(f"[parity] cfg 2 explicit TC: max|dE_loc| = {err / (1e-5 * H.sum_abs_coeff):.3f} x (1e-5 sum|c|)")
    assert err <= 1e-5 * H.sum_abs_coeff


def test_eloc_cfg3_sampled():
    _check_eloc(3, 2048, 24, 2048, memo=True)


def test_eloc_cfg4_sampled():
    _check_eloc(4, 160, 6, 96, memo=True)          # two mini-batches, the second short


def test_eloc_cfg5_sampled():
    _check_eloc(5, 128, 2, 8192, memo=True)


def test_minibatch_partition_and_host_variant():
    w, (x, z, c), params, H, M = workload(2)
    samples, counts = wl.make_samples(w.n_spatial, w.n_alpha, w.n_beta, 300, w.max_count, w.seed_samples, True)
    xs = _dev_u64(samples)
    cd = torch.from_numpy(counts).to(DEV)
    e1, s1 = nqs.local_energy(H, M, xs, cd, minibatch=300, path=nqs.PATH_SIMT)
    e2, s2 = nqs.local_energy(H, M, xs, cd, minibatch=128, path=nqs.PATH_SIMT)        # 128 + 128 + 44
    tol = 1e-5 * H.sum_abs_coeff
    d = (e1 - e2).cpu().numpy().astype(np.float64)
    assert np.hypot(d[:, 0], d[:, 1]).max() <= tol
    np.testing.assert_allclose(s1[:4], s2[:4], rtol=1e-6)
    eh, sh = nqs.local_energy_host(H, M, samples, counts, minibatch=128, path=nqs.PATH_SIMT)
    assert np.array_equal(eh, e2.cpu().numpy())
    np.testing.assert_allclose(sh, s2, rtol=0, atol=0)
    # counts = NULL -> unit weights
    e3, s3 = nqs.local_energy(H, M, xs, None, minibatch=0, path=nqs.PATH_SIMT)
    assert s3[0] == 300
    # B = 0
    e0, s0 = nqs.local_energy(H, M, xs[:0], None)
    assert e0.shape == (0, 2) and np.all(s0 == 0)


@pytest.mark.parametrize("n", [5, 64, 65, 128])
def test_generic_hamiltonian_odd_Y_two_words(n):
    """Random Pauli lists with odd Y counts, duplicates, no identity group, n around the word boundary."""
    rng = np.random.default_rng(n)
    K = 150
    codes = rng.integers(0, 4, size=(K, n)).astype(np.uint8)
    codes[:, rng.random(n) < 0.8] = 0
    codes[:, n - 1] = rng.integers(0, 4, size=K)                 # keep the top qubit busy
    codes[:, 0] = np.where(codes[:, 0] == 0, 1, codes[:, 0])     # every string flips qubit 0: no f = 0 group
    codes[7] = codes[3]
    coeffs = rng.standard_normal(K)
    p = wl.make_made_params(n, 32, n, order="random")
    bits = rng.integers(0, 2, size=(70, n)).astype(np.uint8)
    samples = wl.pack_bits(bits)
    H = nqs.ham_compile(codes, coeffs)
    assert H.export()["flips"][0].any()
    M = nqs.made_create(p)
    ref, mr = oeloc.local_energy(codes, coeffs, p, samples, return_max_ratio=True)
    e, st = nqs.local_energy(H, M, _dev_u64(samples), None, path=nqs.PATH_SIMT)
    e = e.cpu().numpy().astype(np.float64)
    scale = max(1.0, mr)
    assert np.abs(e[:, 0] + 1j * e[:, 1] - ref).max() <= 1e-5 * H.sum_abs_coeff * scale
    assert abs(st[4] - mr) <= 1e-3 * mr
    assert np.abs(ref.imag).max() > 1e-3                          # the imaginary channel is really exercised


def test_empty_hamiltonian():
    p = wl.make_made_params(6, 16, 1)
    H = nqs.ham_compile(np.zeros((0, 6), np.uint8), np.zeros(0), n_qubits=6)
    M = nqs.made_create(p)
    xs = _dev_u64(wl.pack_bits(np.random.default_rng(0).integers(0, 2, size=(9, 6)).astype(np.uint8)))
    e, st = nqs.local_energy(H, M, xs, None)
    assert torch.all(e == 0) and st[0] == 9 and st[1] == 0


# ---- the tensor-core path in the launch configuration bench.py times: many sample blocks per launch ---------
def _spread_rows(B, n_oracle, seed):
    """Oracle rows spread over the 128-row sample blocks of a launch: first block, last (ragged) block, and
    the rest drawn from distinct blocks in between; with more rows than blocks, further rounds over the blocks."""
    nsb = (B + 127) // 128
    rng = np.random.default_rng(seed)
    blocks = [0, nsb - 1] + list(rng.permutation(np.arange(1, max(nsb - 1, 1)))[: max(n_oracle - 2, 0)])
    while len(blocks) < n_oracle:
        blocks += list(rng.permutation(nsb))
    rows = []
    for k, sb in enumerate(blocks[:n_oracle]):
        lo, hi = sb * 128, min(B, sb * 128 + 128)
        rows.append(hi - 1 if k == 1 else int(rng.integers(lo, hi)))        # the very last row of the ragged block
    return np.array(sorted(set(rows)))


def _check_eloc_tc_blocks(cfg, B, n_oracle, minibatch):
    w, (x, z, c), params, H, M = workload(cfg)
    assert M.resolved_path(nqs.PATH_TC) == nqs.PATH_TC
    samples, counts = wl.make_samples(w.n_spatial, w.n_alpha, w.n_beta, B, w.max_count, w.seed_samples, w.unique)
    pick = _spread_rows(B, n_oracle, cfg)
    if minibatch and minibatch < B:                      # also the first and last row of the second mini-batch
        pick = np.unique(np.concatenate([pick, [minibatch, B - 1]]))
    ref = oeloc.local_energy(wl.masks_to_codes(x, z, w.n_qubits), c, params, samples[pick], memo=True)
    e, stats = nqs.local_energy(H, M, _dev_u64(samples), torch.from_numpy(counts).to(DEV), minibatch=minibatch,
                                path=nqs.PATH_TC)
    e = e.cpu().numpy().astype(np.float64)
    ec = e[:, 0] + 1j * e[:, 1]
    tol = 1e-5 * H.sum_abs_coeff
    err = np.abs(ec[pick] - ref)
    print(f"[parity] cfg {cfg} TC, B = {B} ({(B + 127) // 128} sample blocks), minibatch {minibatch}: max|dE_loc|/tol = "
          f"{err.max() / tol:.4f} over {len(pick)} oracle rows {pick.tolist()}")
    assert err.max() <= tol, (cfg, err / tol)
    assert np.isfinite(e).all()
    np.testing.assert_allclose(stats[:4], oeloc.weighted_stats(ec, counts)[:4], rtol=1e-9)
    return ec, samples, counts


def test_eloc_cfg5_tc_many_sample_blocks_ragged():
    """cfg 5 on NQS_PATH_TC, 1,101 samples in ONE launch = 9 sample blocks (the last holds 77 rows): a CTA's tile
    range crosses sample-block boundaries (reload of x / base, flush of E, atomics from several CTAs per row)."""
    _check_eloc_tc_blocks(5, 1101, 8, 8192)


def _all_rows_vs_fp32_path(H, M, samples, rows, ec_tc, tag):
    """Every row in `rows` of a tensor-core launch against the fp32 CUDA-core path run on exactly those samples (the
    fp32 path is itself within ~0.04 x the bound of the oracle and costs ~30 x the tensor-core time per row): the
    GPU-side reference that reaches rows the oracle cannot.  Asserted at 1 x the north_star bound."""
    tol = 1e-5 * H.sum_abs_coeff
    e_si, _ = nqs.local_energy(H, M, _dev_u64(samples[rows]), None, path=nqs.PATH_SIMT)
    e_si = e_si.cpu().numpy().astype(np.float64)
    d = np.abs(ec_tc[rows] - (e_si[:, 0] + 1j * e_si[:, 1]))
    print(f"[parity] {tag}: max|TC - fp32 path|/tol = {d.max() / tol:.4f} (mean {d.mean() / tol:.4f}) over all {len(rows)} rows compared")
    assert d.max() <= tol, (tag, d.max() / tol)


def test_eloc_cfg5_literal_bench_call():
    """The call bench.py times: 8,192 cfg-5 samples, minibatch = 8192, NQS_PATH_AUTO -> tensor cores.  32 oracle rows
    from 32 distinct sample blocks, and every row of 8 whole sample blocks spread over the 64 plus 77 more
    rows (1,101 in all) against the fp32 path."""
    w, (x, z, c), params, H, M = workload(5)
    assert M.resolved_path(nqs.PATH_AUTO) == nqs.PATH_TC
    ec, samples, counts = _check_eloc_tc_blocks(5, 8192, 32, 8192)
    rows = np.concatenate([np.arange(sb * 128, sb * 128 + 128) for sb in (0, 9, 18, 27, 36, 45, 54, 63)] + [np.arange(4000, 4077)])
    _all_rows_vs_fp32_path(H, M, samples, rows, ec, "cfg 5 bench launch (B = 8192)")


def test_eloc_cfg5_two_full_minibatches_in_one_call():
    """Row a7 at the configured slice size: ONE nqs_local_energy call over 16,384 cfg-5 samples with
    minibatch = 8192 = two full gradient-accumulation slices.  The second slice must equal a direct call on those rows
    (same kernel and launch shape, fixed-order sums: bit for bit), the statistics must be those of all 16,384 rows, and two
    rows of the second slice are checked against the oracle."""
    w, (x, z, c), params, H, M = workload(5)
    B = 16384
    samples, counts = wl.make_samples(w.n_spatial, w.n_alpha, w.n_beta, B, w.max_count, w.seed_samples, w.unique)
    xs, cn = _dev_u64(samples), torch.from_numpy(counts).to(DEV)
    e, st = nqs.local_energy(H, M, xs, cn, minibatch=8192)
    e2, st2 = nqs.local_energy(H, M, xs[8192:].contiguous(), cn[8192:].contiguous(), minibatch=8192)
    tol = 1e-5 * H.sum_abs_coeff
    d = (e[8192:] - e2).cpu().numpy().astype(np.float64)
    en = e.cpu().numpy().astype(np.float64)
    ec = en[:, 0] + 1j * en[:, 1]
    pick = np.array([8192, 16383])
    ref = oeloc.local_energy(wl.masks_to_codes(x, z, w.n_qubits), c, params, samples[pick], memo=True)
    err = np.abs(ec[pick] - ref).max()
    print(f"[parity] cfg 5, B = 16384 as 2 x 8192 in one call: second slice vs direct call max|d|/tol = "
          f"{np.hypot(d[:, 0], d[:, 1]).max() / tol:.5f}; max|dE_loc|/tol = {err / tol:.4f} over oracle rows {pick.tolist()}")
    assert torch.equal(e[8192:], e2)                  # same launch shape, fixed-order sums: the same bytes
    assert err <= tol
    np.testing.assert_allclose(st[:4], oeloc.weighted_stats(ec, counts)[:4], rtol=1e-9)
    assert st[0] == counts.sum() and st[4] >= st2[4] >= 1.0


def test_eloc_cfg4_tc_many_sample_blocks_two_minibatches():
    """cfg 4: 8 blocks, then a second mini-batch of 333 (3 blocks, ragged); 64 oracle rows and every one of
    the 1,357 rows against the fp32 path."""
    w, (x, z, c), params, H, M = workload(4)
    ec, samples, counts = _check_eloc_tc_blocks(4, 1024 + 333, 64, 1024)
    _all_rows_vs_fp32_path(H, M, samples, np.arange(1024 + 333), ec, "cfg 4 (B = 1357, minibatch 1024)")


def test_eloc_cfg3_tc_vs_simt_all_rows_and_oracle():
    """cfg 3 (h = 256): every row of a 9-block launch against the fp32 CUDA-core path (GPU vs GPU, cheap), 64
    rows against the oracle."""
    w, (x, z, c), params, H, M = workload(3)
    B = 1101
    samples, counts = wl.make_samples(w.n_spatial, w.n_alpha, w.n_beta, B, w.max_count, w.seed_samples, w.unique)
    xs = _dev_u64(samples)
    e_tc, _ = nqs.local_energy(H, M, xs, None, path=nqs.PATH_TC)
    e_si, _ = nqs.local_energy(H, M, xs, None, path=nqs.PATH_SIMT)
    d = (e_tc - e_si).cpu().numpy().astype(np.float64)
    tol = 1e-5 * H.sum_abs_coeff
    pick = _spread_rows(B, 64, 3)
    ref = oeloc.local_energy(wl.masks_to_codes(x, z, w.n_qubits), c, params, samples[pick], memo=True)
    et = e_tc.cpu().numpy().astype(np.float64)
    err = np.abs(et[pick, 0] + 1j * et[pick, 1] - ref).max()
    print(f"[parity] cfg 3 TC, B = {B}: max|dE_loc|/tol = {err / tol:.4f} over {len(pick)} oracle rows; "
          f"max|TC - SIMT|/tol over all rows = {np.hypot(d[:, 0], d[:, 1]).max() / tol:.4f}")
    assert err <= TC_NARROW_FACTOR * tol
    assert np.hypot(d[:, 0], d[:, 1]).max() <= (TC_NARROW_FACTOR + 1) * tol


def _few_flip_pauli_list(rng, n, K):
    """Generic Pauli strings with the paper's sparsity (<= 4 X/Y positions per string), odd Y counts
    allowed, a few Z elsewhere, qubit 0 always flipped (so there is NO f = 0 group), one duplicate string."""
    codes = np.zeros((K, n), np.uint8)
    for t in range(K):
        nf = int(rng.integers(0, 4))                              # 0..3 further flipped qubits besides qubit 0
        pos = rng.choice(np.arange(1, n), size=nf, replace=False)
        codes[t, 0] = rng.integers(1, 3)                          # X or Y
        codes[t, pos] = rng.integers(1, 3, size=nf)
        zpos = rng.choice(np.arange(1, n), size=int(rng.integers(0, 4)), replace=False)
        codes[t, zpos] = np.where(codes[t, zpos] == 0, 3, codes[t, zpos])
    codes[:, n - 1] = np.where(codes[:, n - 1] == 0, rng.integers(0, 4, size=K), codes[:, n - 1])   # top qubit busy
    codes[17] = codes[5]
    return codes, rng.standard_normal(K)


@pytest.mark.parametrize("n,h", [(20, 512), (65, 512), (20, 384), (20, 128), (65, 256)])
def test_generic_odd_Y_no_diagonal_on_tensor_core_path(n, h):
    """Complex S (odd Y counts -> Im S != 0), a Hamiltonian WITHOUT an f = 0 group (g_begin = 0), duplicates, two
    mask words, h = 384 (the narrowest width AUTO sends to the tensor cores) -- all on NQS_PATH_TC, several sample
    blocks, ragged.  Bound: each term's ratio carries a relative error |exp(d) - 1| with |d| <= 2 sqrt(2) *
    TC_LOGPSI_TOL (log|psi| and phi of x' and of x), so |dE| <= sum|c| * max|ratio| * 2 sqrt(2) * TC_LOGPSI_TOL; the
    ratio to the north_star bound (which is stated for the five chemistry configs) is printed."""
    rng = np.random.default_rng(1000 + n + h)
    codes, coeffs = _few_flip_pauli_list(rng, n, 400)
    p = wl.make_made_params(n, h, n + h, order="random")
    B = 3 * 128 + 41
    samples = wl.pack_bits(rng.integers(0, 2, size=(B, n)).astype(np.uint8))
    H = nqs.ham_compile(codes, coeffs)
    assert H.export()["flips"][0].any()
    M = nqs.made_create(p)
    assert M.resolved_path(nqs.PATH_TC) == nqs.PATH_TC
    pick = _spread_rows(B, 24, n)
    ref, mr = oeloc.local_energy(codes, coeffs, p, samples[pick], return_max_ratio=True)
    e, st = nqs.local_energy(H, M, _dev_u64(samples), None, path=nqs.PATH_TC)
    e = e.cpu().numpy().astype(np.float64)
    ec = e[:, 0] + 1j * e[:, 1]
    err = np.abs(ec[pick] - ref).max()
    print(f"[parity] generic odd-Y n={n} h={h} TC: max|dE_loc| = {err:.3e} = {err / (1e-5 * H.sum_abs_coeff * max(1.0, mr)):.3f} x "
          f"(1e-5 sum|c| max|ratio|), max|ratio| = {mr:.2f}")
    assert err <= H.sum_abs_coeff * max(1.0, mr) * 2 * 2 ** 0.5 * TC_LOGPSI_TOL
    if h <= 256:                                        # split precision: the north_star scale itself, ratios included
        assert err <= 1e-5 * H.sum_abs_coeff * max(1.0, mr)
    assert np.abs(ref.imag).max() > 1e-3 and np.abs(ec.imag).max() > 1e-3
    # the imaginary channel on its own: Im E of the picked rows, same bound, and a sign/swap error would be O(sum|c|)
    assert np.abs(ec[pick].imag - ref.imag).max() <= H.sum_abs_coeff * max(1.0, mr) * 2 * 2 ** 0.5 * TC_LOGPSI_TOL
    assert np.abs(ref.imag).max() > 50 * np.abs(ec[pick].imag - ref.imag).max()
    assert st[4] >= mr * (1 - 1e-2)
    np.testing.assert_allclose(st[2], ec.imag.sum(), rtol=1e-6, atol=1e-6 * H.sum_abs_coeff)


def test_empty_hamiltonian_on_tensor_core_path():
    """K = 0 on NQS_PATH_TC (ntiles == 0): E_loc = 0, statistics counted."""
    p = wl.make_made_params(20, 128, 1)
    H = nqs.ham_compile(np.zeros((0, 20), np.uint8), np.zeros(0), n_qubits=20)
    M = nqs.made_create(p)
    xs = _dev_u64(wl.pack_bits(np.random.default_rng(0).integers(0, 2, size=(300, 20)).astype(np.uint8)))
    e, st = nqs.local_energy(H, M, xs, None, path=nqs.PATH_TC)
    assert torch.all(e == 0) and st[0] == 300 and st[1] == 0


def test_hamiltonian_handle_reuse_does_not_alias_flip_cache():
    """free H1, compile H2 with the same G (cudaMalloc usually returns the same addresses): the
    tensor-core path must use H2's flips, not a cached position-ordered copy of H1's."""
    n, h = 20, 128
    p = wl.make_made_params(n, h, 77)
    M = nqs.made_create(p)
    rng = np.random.default_rng(77)
    samples = wl.pack_bits(rng.integers(0, 2, size=(200, n)).astype(np.uint8))
    xs = _dev_u64(samples)

    def ham(seed):
        r = np.random.default_rng(seed)
        K = 64
        codes = np.zeros((K, n), np.uint8)
        for t in range(K):                                  # K distinct flip masks: bits t%n and (3t+1)%n ... distinct per t
            codes[t, t % n] = 1
            codes[t, (t // n + 1 + t) % n] = 2 if (t % 3 == 0) else 1
            codes[t, r.integers(0, n)] |= 3 if r.random() < 0.5 else 0
        return nqs.ham_compile(codes, r.standard_normal(K))

    H1 = ham(1)
    e1, _ = nqs.local_energy(H1, M, xs, None, path=nqs.PATH_TC)
    G1 = H1.G
    del H1
    H2 = ham(2)
    e2_tc, _ = nqs.local_energy(H2, M, xs, None, path=nqs.PATH_TC)
    e2_si, _ = nqs.local_energy(H2, M, xs, None, path=nqs.PATH_SIMT)
    d = (e2_tc - e2_si).cpu().numpy().astype(np.float64)
    assert np.hypot(d[:, 0], d[:, 1]).max() <= 1e-4 * H2.sum_abs_coeff * 10, (G1, H2.G)


def test_pauli_contract_output_layout_raw_ctypes():
    """include/nqs.h documents S_out_dev as float [g1-g0][B][2]; pin it through raw ctypes."""
    import ctypes
    w, (x, z, c), params, H, M = workload(1)
    samples, _ = wl.make_samples(w.n_spatial, w.n_alpha, w.n_beta, 37, w.max_count, w.seed_samples, w.unique)
    xs = _dev_u64(samples)
    g0, g1 = 2, 9
    out = torch.full(((g1 - g0) * 37 * 2,), float("nan"), dtype=torch.float32, device=DEV)
    rc = nqs.lib().nqs_pauli_contract(H._h, ctypes.c_void_p(xs.data_ptr()), 37, g0, g1, ctypes.c_void_p(out.data_ptr()), None)
    assert rc == 0
    torch.cuda.synchronize()
    S = out.cpu().numpy().astype(np.float64).reshape(g1 - g0, 37, 2)
    t = H.export()
    off = t["offsets"].astype(np.int64)
    for gi in range(g0, g1):
        sl = slice(off[gi], off[gi + 1])
        cc = t["coef"][sl].astype(np.float64)
        ref = (cc[None, :] * matrix_element(samples[:, None, :], t["zy"][sl][None, :, :], t["ycount"][sl].astype(np.int64))).sum(axis=1)
        np.testing.assert_allclose(S[gi - g0, :, 0] + 1j * S[gi - g0, :, 1], ref, atol=1e-5 * np.abs(cc).sum())


# ---- gradient of Eq. 7 -----------------------------------------------------------------------------
def _grad_tensor_slices(p):
    sizes = []
    for W, b in zip(p.weights, p.biases):
        sizes += [W.size, b.size]
    sizes += [p.phase_weights[0].size, p.phase_biases[0].size, p.phase_weights[1].size, p.phase_biases[1].size]
    offs = np.concatenate([[0], np.cumsum(sizes)])
    return [slice(int(offs[i]), int(offs[i + 1])) for i in range(len(sizes))]


def _check_grad(params, samples, counts, eloc_c64, minibatch, tag):
    """CUDA gradient against oracle.grad on the SAME (fp32) local energies.  Tolerance per parameter tensor: the kernel
    forms each entry as an fp32 sum over the B rows of products of fp32 activations (relative error ~ sqrt(B) 2^-24 on
    sum |terms|, far below the bound) -- bound 2e-5 * max|g| of the tensor + 1e-9."""
    from oracle import grad as ograd
    M = nqs.made_create(params)
    e32 = np.stack([eloc_c64.real, eloc_c64.imag], axis=1).astype(np.float32)
    g, b = nqs.energy_grad(M, _dev_u64(samples), torch.from_numpy(counts).to(DEV) if counts is not None else None,
                           torch.from_numpy(e32).to(DEV), minibatch=minibatch)
    g = g.cpu().numpy().astype(np.float64)
    cnt = counts if counts is not None else np.ones(len(samples))
    ref, bref = ograd.energy_gradient(params, samples, cnt, e32[:, 0].astype(np.float64) + 1j * e32[:, 1].astype(np.float64))
    assert g.shape == ref.shape == (M.num_params(),)
    assert abs(b - bref) <= 1e-12 * max(1.0, abs(bref))
    worst = 0.0
    for t, sl in enumerate(_grad_tensor_slices(params)):
        scale = np.abs(ref[sl]).max()
        err = np.abs(g[sl] - ref[sl]).max()
        worst = max(worst, err / (scale + 1e-30))
        assert err <= 2e-5 * scale + 1e-9, (tag, t, err, scale)
    # masked entries are exactly zero
    masks = omade.build_masks(params.n_qubits, params.deg_hidden)
    sls = _grad_tensor_slices(params)
    for k, mk in enumerate(masks):
        assert np.all(g[sls[2 * k]].reshape(mk.shape)[mk == 0] == 0.0)
    print(f"[parity] gradient {tag}: max rel err over tensors {worst:.2e}")
    return g


@pytest.mark.parametrize("cfg,B,mb", [(1, 256, 100), (2, 4096, 1500), (3, 3000, 0)])
def test_energy_gradient_all_samples(cfg, B, mb):
    """Every sample of cfg 1-2 (3,000 of cfg 3), all parameter tensors, E_loc from the library itself (AUTO path), with
    gradient-accumulation mini-batches that do not divide B."""
    w, (x, z, c), params, H, M = workload(cfg)
    samples, counts = wl.make_samples(w.n_spatial, w.n_alpha, w.n_beta, B, w.max_count, w.seed_samples, w.unique)
    e, _ = nqs.local_energy(H, M, _dev_u64(samples), torch.from_numpy(counts).to(DEV))
    e = e.cpu().numpy().astype(np.float64)
    _check_grad(params, samples, counts, e[:, 0] + 1j * e[:, 1], mb, f"cfg {cfg}")


def test_energy_gradient_cfg5_sampled_rows_and_complex_energies():
    """cfg 5 shape (76 qubits, h = 512): 700 samples with synthetic COMPLEX local energies (so that the phase-net
    tensors get a non-zero gradient), unit counts, two mini-batches."""
    w = wl.WORKLOADS[5]
    params = wl.make_made_params(w.n_qubits, w.hidden, w.seed_weights)
    samples, _ = wl.make_samples(w.n_spatial, w.n_alpha, w.n_beta, 700, w.max_count, w.seed_samples, w.unique)
    rng = np.random.default_rng(55)
    e = -300.0 + rng.standard_normal(700) + 1j * rng.standard_normal(700)
    g = _check_grad(params, samples, None, e, 512, "cfg 5 shape, complex E")
    sls = _grad_tensor_slices(params)
    assert np.abs(g[sls[-4]]).max() > 0 and np.abs(g[sls[-2]]).max() > 0      # P1, P2 gradients are exercised


@pytest.mark.parametrize("n,h,L,order", [(13, 48, 1, "random"), (65, 100, 2, "random"), (128, 64, 2, "reverse"), (3, 8, 1, "identity")])
def test_energy_gradient_shapes(n, h, L, order):
    """One hidden layer (the paper's own architecture), random degrees, widths that are not multiples of the tile."""
    p = wl.make_made_params(n, h, 200 + n, n_hidden_layers=L, order=order)
    rng = np.random.default_rng(n)
    p.deg_hidden = rng.integers(1, n, size=(L, h)).astype(np.int32)
    samples = wl.pack_bits(rng.integers(0, 2, size=(333, n)).astype(np.uint8))
    counts = rng.integers(1, 50, size=333).astype(np.int64)
    e = rng.standard_normal(333) + 1j * rng.standard_normal(333)
    _check_grad(p, samples, counts, e, 128, f"n={n} h={h} L={L}")
    # B = 0
    M = nqs.made_create(p)
    g0, _ = nqs.energy_grad(M, _dev_u64(samples[:0]), None, torch.zeros((0, 2), device=DEV))
    assert torch.all(g0 == 0)


def test_energy_gradient_global_stats_shards_sum_to_whole_batch():
    """nqs_energy_grad(global_stats_host = ...) on two shards: the SUM equals the gradient of the whole batch
    (the data-parallel exchange of PAPER.md:146, distributed.all_reduce_gradient)."""
    p = wl.make_made_params(20, 128, 5)
    rng = np.random.default_rng(12)
    samples = wl.pack_bits(rng.integers(0, 2, size=(500, 20)).astype(np.uint8))
    counts = rng.integers(1, 30, size=500).astype(np.int64)
    e = (rng.standard_normal((500, 2)) + np.array([-20.0, 0.0])).astype(np.float32)
    M = nqs.made_create(p)
    xs, cs, es = _dev_u64(samples), torch.from_numpy(counts).to(DEV), torch.from_numpy(e).to(DEV)
    g_all, b_all = nqs.energy_grad(M, xs, cs, es)
    cd = counts.astype(np.float64)
    gstats = np.array([cd.sum(), (cd * e[:, 0]).sum(), (cd * e[:, 1]).sum()])
    g0, b0 = nqs.energy_grad(M, xs[:180], cs[:180], es[:180], global_stats=gstats)
    g1, b1 = nqs.energy_grad(M, xs[180:], cs[180:], es[180:], global_stats=gstats, minibatch=100)
    assert abs(b0 - b_all) < 1e-12 and abs(b1 - b_all) < 1e-12
    d = (g0 + g1 - g_all).abs().max().item()
    assert d <= 2e-6 * g_all.abs().max().item() + 1e-10, d


# ---- batched autoregressive sampler ---------------------------------------------------
def _check_sampler(params, n_draws, seed, n_up, n_down, cap, tag):
    """CUDA sampler against oracle.sampler on the same Philox-keyed draws.  Integer work is bit-exact EXCEPT where
    floating point decides a bit: a draw whose uniform lies within EPS of a conditional may fall on the other side in
    the kernel's fp32 forward pass (measured |p_gpu - p_oracle| <~ 3e-6).  The oracle reports the margin |u - p| of
    every draw; with a of them below EPS, the two count tables may differ by at most 2a in L1 (each ambiguous draw can
    leave one entry and join another), and must be identical when a = 0 and no elimination tie is affected."""
    from oracle import sampler as osamp
    EPS = 2e-5
    M = nqs.made_create(params)
    s_gpu, c_gpu = nqs.made_sample(M, n_draws, seed, n_up, n_down, cap, device=DEV)
    s_gpu = s_gpu.cpu().numpy().view(np.uint64)
    c_gpu = c_gpu.cpu().numpy()
    s_ref, c_ref, margins = osamp.sample(params, n_draws, seed, n_up, n_down, cap)
    amb = int((margins < EPS).sum())
    # validity that holds whatever the rounding: unique rows, positive counts, total, cap, constraint
    assert len(set(map(tuple, s_gpu.tolist()))) == len(s_gpu)
    assert np.all(c_gpu > 0)
    assert (c_gpu.sum() == n_draws) if cap == 0 else (c_gpu.sum() <= n_draws and len(c_gpu) <= cap)
    n = params.n_qubits
    bits = wl.unpack_bits(s_gpu, n)
    assert not np.any(s_gpu[:, 1] >> np.uint64(max(n - 64, 0))) if n > 64 else np.all(s_gpu[:, 1] == 0)
    if n_up >= 0:
        assert np.all(bits[:, 0::2].sum(axis=1) == n_up) and np.all(bits[:, 1::2].sum(axis=1) == n_down)
    tab_g = {tuple(r): int(c) for r, c in zip(s_gpu.tolist(), c_gpu)}
    tab_r = {tuple(r): int(c) for r, c in zip(s_ref.tolist(), c_ref)}
    l1 = sum(abs(tab_g.get(k, 0) - tab_r.get(k, 0)) for k in set(tab_g) | set(tab_r))
    print(f"[parity] sampler {tag}: {len(c_gpu)} unique (oracle {len(c_ref)}), ambiguous draws {amb}, L1 count distance {l1}")
    if cap == 0:
        assert l1 <= 2 * amb, (l1, amb)
        if amb == 0:
            assert np.array_equal(s_gpu, s_ref) and np.array_equal(c_gpu, c_ref)      # same rows, same buffer order
    else:
        # elimination decides by counter rank: an ambiguous draw can swap which of two tied entries survives
        assert l1 <= 2 * amb * max(1, int(c_ref.max())) + 2 * amb, (l1, amb)
        if amb == 0:
            assert np.array_equal(s_gpu, s_ref) and np.array_equal(c_gpu, c_ref)


@pytest.mark.parametrize("n,h,L,order,nu,nd,N,cap", [
    (8, 32, 2, "reverse", 2, 2, 4000, 0),            # cfg 1 model shape: the whole 36-state sector gets populated
    (8, 32, 2, "reverse", -1, -1, 4000, 0),          # unconstrained
    (20, 128, 2, "reverse", 5, 5, 20000, 0),         # cfg 2 shape
    (20, 128, 2, "random", 5, 5, 20000, 300),        # elimination of the lowest counters
    (30, 64, 1, "random", 7, 7, 5000, 1000),         # one hidden layer, cap below the draws
    (76, 128, 2, "reverse", 15, 15, 3000, 0),        # 76 qubits: two mask words, 15 + 15 electrons
    (11, 16, 2, "identity", 3, 2, 2000, 0),          # odd n: 6 up positions, 5 down
])
def test_sampler_replays_the_oracle_draws(n, h, L, order, nu, nd, N, cap):
    p = wl.make_made_params(n, h, 700 + n + cap, n_hidden_layers=L, order=order)
    _check_sampler(p, N, 4242 + n, nu, nd, cap, f"n={n} h={h} L={L} {order} ({nu},{nd}) N={N} cap={cap}")


def test_sampler_feeds_the_local_energy_path():
    """sample -> E_loc -> gradient through the ABI only: the sampler's output is what nqs_local_energy consumes."""
    w, (x, z, c), params, H, M = workload(2)
    s, cnt = nqs.made_sample(M, 50000, 7, w.n_alpha, w.n_beta, 2048, device=DEV)
    assert 0 < s.shape[0] <= 2048 and cnt.sum().item() <= 50000
    e, st = nqs.local_energy(H, M, s, cnt)
    assert np.isfinite(st).all() and st[0] == cnt.sum().item()
    g, b = nqs.energy_grad(M, s, cnt, e)
    assert torch.isfinite(g).all() and abs(b.real - st[1] / st[0]) < 1e-9 * abs(b.real)
    # edge cases: zero draws, bad constraint
    s0, c0 = nqs.made_sample(M, 0, 1, device=DEV)
    assert s0.shape[0] == 0
    with pytest.raises(nqs.NqsError):
        nqs.made_sample(M, 10, 1, 3, -1, device=DEV)


# ---- second workload: symmetry-sparse Hamiltonian + the paper's one-hidden-layer architecture ------
@pytest.mark.parametrize("N,n_irreps,h", [(10, 2, 512), (13, 4, 384)])
def test_symmetric_workload_one_hidden_layer_on_tensor_cores(N, n_irreps, h):
    """Integrals with point-group selection rules (the sparsity of Table 1's molecules), the paper's own
    modulus net with ONE hidden layer, Hamiltonian handed over as TEXT; E_loc on the tensor-core path
    against the oracle at the north_star bound, all rows against the fp32 CUDA-core path."""
    n = 2 * N
    hh, gg = wl.make_integrals_symmetric(N, 991 + N, n_irreps)
    x, z, c = wl.jw_pauli_terms(hh, gg)
    codes = wl.masks_to_codes(x, z, n)
    text = "\n".join(f"{repr(float(cc))} [" + " ".join("IXYZ"[v] + str(j) for j, v in enumerate(row) if v) + "]" for row, cc in zip(codes, c))
    H = nqs.ham_compile_text(n, text)
    H2 = nqs.ham_compile_packed(n, x, z, c)
    assert (H.K, H.G) == (H2.K, H2.G) and H.export()["coef"].tobytes() == H2.export()["coef"].tobytes()
    p = wl.make_made_params(n, h, 55 + N, n_hidden_layers=1)
    M = nqs.made_create(p)
    assert M.resolved_path(nqs.PATH_AUTO) == nqs.PATH_TC
    samples, counts = wl.make_samples(N, N // 2, N // 2, 700, 64, 5, True)
    e_tc, st = nqs.local_energy(H, M, _dev_u64(samples), torch.from_numpy(counts).to(DEV))
    e_si, _ = nqs.local_energy(H, M, _dev_u64(samples), None, path=nqs.PATH_SIMT)
    tol = 1e-5 * H.sum_abs_coeff
    pick = _spread_rows(700, 12, N)
    ref = oeloc.local_energy(codes, c, p, samples[pick], memo=True)
    et = e_tc.cpu().numpy().astype(np.float64)
    err = np.abs(et[pick, 0] + 1j * et[pick, 1] - ref).max()
    d = (e_tc - e_si).cpu().numpy().astype(np.float64)
    print(f"[parity] symmetric workload n={n} ({n_irreps} irreps) K={H.K} G={H.G}, 1 hidden layer h={h}, TC: max|dE_loc|/tol = {err / tol:.4f}; "
          f"max|TC - SIMT|/tol = {np.hypot(d[:, 0], d[:, 1]).max() / tol:.4f}")
    assert err <= tol
    assert np.hypot(d[:, 0], d[:, 1]).max() <= 2 * tol


# ---- constrained model: nqs_made_set_constraint (Eq. 14, readings A12 / A13) ---------------------
@pytest.mark.parametrize("n,h,L,order,nu,nd", [(8, 32, 2, "reverse", 2, 2), (20, 128, 2, "random", 5, 5), (76, 512, 2, "reverse", 15, 15),
                                                (30, 128, 1, "identity", 7, 6)])
def test_constrained_logpsi_both_paths(n, h, L, order, nu, nd):
    """log|psi| of the constrained model on valid strings (clamped conditionals skipped) and -inf on strings that
    violate Eq. 12, on the CUDA-core and the tensor-core path."""
    from oracle import sampler as osamp
    p = wl.make_made_params(n, h, 900 + n, n_hidden_layers=L, order=order)
    N = n // 2
    valid_s, _ = wl.make_samples(N, nu, nd, 200, 4, 3, False)
    rng = np.random.default_rng(n)
    rand_s = wl.pack_bits(rng.integers(0, 2, size=(133, n)).astype(np.uint8))
    cfgs = np.concatenate([valid_s, rand_s])
    ref = osamp.constrained_logpsi(p, cfgs, nu, nd)
    M = nqs.made_create(p)
    M.set_constraint(nu, nd)
    for path in _paths(M, min_hidden_tc=0):
        out = nqs.made_logpsi(M, _dev_u64(cfgs), path=path).cpu().numpy().astype(np.float64)
        fin = np.isfinite(ref.real)
        assert fin[:200].all()
        assert np.array_equal(np.isneginf(out[:, 0]), ~fin), path
        tol = 2e-4 if path == nqs.PATH_SIMT else TC_LOGPSI_TOL
        assert np.abs(out[fin, 0] - ref.real[fin]).max() < tol
        assert np.abs(out[:, 1] - ref.imag).max() < tol
    M.set_constraint(-1, -1)                                    # off again: the raw model
    out = nqs.made_logpsi(M, _dev_u64(cfgs), path=nqs.PATH_SIMT).cpu().numpy().astype(np.float64)
    assert np.abs(out[:, 0] - omade.logpsi(p, cfgs).real).max() < 2e-4


def test_constrained_local_energy_and_gradient_cfg2():
    """cfg 2 with the constrained wavefunction (5 up + 5 down): E_loc against the oracle's term-by-term sum with the
    constrained log f (the JW Hamiltonian conserves both spin populations, so every connected string is valid), and the
    gradient of Eq. 7 of the constrained model."""
    from oracle import sampler as osamp
    from oracle import grad as ograd
    w, (x, z, c), params, H, _ = workload(2)
    M = nqs.made_create(params)
    M.set_constraint(w.n_alpha, w.n_beta)
    samples, counts = wl.make_samples(w.n_spatial, w.n_alpha, w.n_beta, 400, w.max_count, w.seed_samples, True)
    codes = wl.masks_to_codes(x, z, w.n_qubits)
    pick = np.arange(0, 400, 25)
    ref = oeloc.local_energy_generic(codes, c, samples[pick], lambda cf: osamp.constrained_logpsi(params, cf, w.n_alpha, w.n_beta))
    tol = 1e-5 * H.sum_abs_coeff
    for path, fac in ((nqs.PATH_SIMT, 1.0), (nqs.PATH_TC, TC_NARROW_FACTOR)):
        e, st = nqs.local_energy(H, M, _dev_u64(samples), torch.from_numpy(counts).to(DEV), path=path)
        en = e.cpu().numpy().astype(np.float64)
        err = np.abs(en[pick, 0] + 1j * en[pick, 1] - ref).max()
        print(f"[parity] cfg 2 constrained model, path {path}: max|dE_loc|/tol = {err / tol:.4f}")
        assert err <= fac * tol
        if path == nqs.PATH_SIMT:
            g, b = nqs.energy_grad(M, _dev_u64(samples), torch.from_numpy(counts).to(DEV), e)
            e64 = en[:, 0] + 1j * en[:, 1]
            gref, _ = ograd.energy_gradient(params, samples, counts, e64, w.n_alpha, w.n_beta)
            g = g.cpu().numpy().astype(np.float64)
            for sl in _grad_tensor_slices(params):
                assert np.abs(g[sl] - gref[sl]).max() <= 2e-5 * np.abs(gref[sl]).max() + 1e-9
            # and it differs from the unconstrained gradient (the flag is really in effect)
            gun, _ = ograd.energy_gradient(params, samples, counts, e64)
            assert np.abs(gun - gref).max() > 1e-4 * np.abs(gref).max()


def test_sampler_takes_the_constraint_of_the_handle():
    """A handle with a constraint samples that constraint: (-1, -1) means the handle's pair, the same pair explicitly gives
    the same buffer, a different pair is refused (include/nqs.h) — samples, log psi, E_loc and gradient share one pi_hat."""
    p = wl.make_made_params(12, 32, 55)
    M = nqs.made_create(p)
    M.set_constraint(3, 2)
    s0, c0 = nqs.made_sample(M, 3000, 11, device=DEV)
    s1, c1 = nqs.made_sample(M, 3000, 11, 3, 2, device=DEV)
    assert torch.equal(s0, s1) and torch.equal(c0, c1)
    bits = wl.unpack_bits(s0.cpu().numpy().view(np.uint64), 12)
    assert np.all(bits[:, 0::2].sum(axis=1) == 3) and np.all(bits[:, 1::2].sum(axis=1) == 2)
    with pytest.raises(nqs.NqsError) as ei:
        nqs.made_sample(M, 3000, 11, 2, 3, device=DEV)
    assert ei.value.status == -1
    M.set_constraint(-1, -1)                                   # no constraint on the handle: the pair clamps the sampler alone
    s2, _ = nqs.made_sample(M, 3000, 11, 2, 3, device=DEV)
    bits = wl.unpack_bits(s2.cpu().numpy().view(np.uint64), 12)
    assert np.all(bits[:, 0::2].sum(axis=1) == 2) and np.all(bits[:, 1::2].sum(axis=1) == 3)


@pytest.mark.parametrize("cfg,B,mb", [(1, 256, 0), (3, 1101, 0), (3, 1101, 512), (4, 300, 0)])
def test_tc_eloc_is_bit_reproducible(cfg, B, mb):
    """The tensor-core path adds each row's per-CTA partial sums in a fixed order (no float atomics): the same call gives
    the same bytes, whatever the order the CTAs ran in.  cfg 1 puts 25 clusters on one sample block (50 slots per row),
    cfg 3 / 4 have clusters that straddle sample blocks; the mini-batch variant reuses the partial buffer at another size."""
    w, (x, z, c), params, H, M = workload(cfg)
    samples, counts = wl.make_samples(w.n_spatial, w.n_alpha, w.n_beta, B, w.max_count, w.seed_samples, w.unique)
    xs = _dev_u64(samples)
    e0, s0 = nqs.local_energy(H, M, xs, None, minibatch=mb, path=nqs.PATH_TC)
    e0 = e0.clone()
    junk, _ = nqs.local_energy(H, M, xs[: B // 3].contiguous(), None, path=nqs.PATH_TC)      # another shape in between
    e1, s1 = nqs.local_energy(H, M, xs, None, minibatch=mb, path=nqs.PATH_TC)
    assert torch.equal(e0, e1) and np.array_equal(s0, s1)
    e_si, _ = nqs.local_energy(H, M, xs, None, path=nqs.PATH_SIMT)
    d = (e0 - e_si).cpu().numpy().astype(np.float64)
    assert np.hypot(d[:, 0], d[:, 1]).max() <= 1e-5 * H.sum_abs_coeff
