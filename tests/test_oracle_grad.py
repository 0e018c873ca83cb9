"""Pins for oracle/grad.py (CPU only): Eq. 7.

  * d log f by central finite differences of oracle.made.logpsi (every parameter tensor, masked entries included);
  * the same derivatives through torch autograd (fp64) of an independently written network;
  * the ESTIMATOR on tiny systems by exact enumeration: with every configuration as a sample and |psi|^2 as its
    weight, Eq. 7 is the exact gradient of L = 1/2 <f|H|f> (Eq. 5; the MADE state is normalised for every
    theta, :86-88), which is checked against finite differences of 1/2 psi^H H psi with a dense Kronecker-product H
    carrying odd-Y strings (so a missing conjugate / a swapped Re, Im fails);
  * the baseline b does not change the exact gradient (E[conj sigma] = 0 for a normalised state), but it does change
    the finite-sample estimator: checked against the formula written out sample by sample.
"""
import copy

import numpy as np
import pytest
import torch

from oracle import grad as ograd
from oracle import made as omade
from oracle import eloc as oeloc
from oracle.pauli import pack_mask
from paper_2208_05637_b200 import workloads as wl
from tests import bruteforce as bf


def _params(n, h, L, seed, order="random", random_deg=True):
    p = wl.make_made_params(n, h, seed, n_hidden_layers=L, order=order)
    if random_deg:
        rng = np.random.default_rng(seed + 5)
        p.deg_hidden = rng.integers(1, n, size=(L, h)).astype(np.int32)
    # fp64 copies so that finite differences are clean
    p.weights = [w.astype(np.float64) for w in p.weights]
    p.biases = [b.astype(np.float64) for b in p.biases]
    p.phase_weights = [w.astype(np.float64) for w in p.phase_weights]
    p.phase_biases = [b.astype(np.float64) for b in p.phase_biases]
    return p


def _tensors(p):
    """The parameter tensors in the flat order of oracle.grad (views into p)."""
    out = []
    for W, b in zip(p.weights, p.biases):
        out += [W, b]
    return out + [p.phase_weights[0], p.phase_biases[0], p.phase_weights[1], p.phase_biases[1]]


@pytest.mark.parametrize("n,h,L", [(5, 6, 1), (7, 12, 2), (4, 9, 2)])
def test_dlogpsi_by_central_differences(n, h, L):
    p = _params(n, h, L, 40 + n)
    rng = np.random.default_rng(n)
    bits = rng.integers(0, 2, size=(3, n)).astype(np.uint8)
    cfgs = pack_mask(bits)
    for i in range(3):
        one = np.zeros(3); one[i] = 1.0
        g_mod = ograd.dlogpsi_weighted(p, cfgs, one, np.zeros(3))
        g_ph = ograd.dlogpsi_weighted(p, cfgs, np.zeros(3), one)
        tens = _tensors(p)
        for t, (T, gm, gp) in enumerate(zip(tens, g_mod, g_ph)):
            assert gm.shape == T.shape and gp.shape == T.shape
            flat = T.reshape(-1)
            for k in rng.choice(flat.size, size=min(flat.size, 12), replace=False):
                old = flat[k]
                eps = 1e-6
                flat[k] = old + eps; lp = omade.logpsi(p, cfgs[i:i + 1])[0]
                flat[k] = old - eps; lm = omade.logpsi(p, cfgs[i:i + 1])[0]
                flat[k] = old
                fd = (lp - lm) / (2 * eps)
                assert abs(fd.real - gm.reshape(-1)[k]) < 1e-8, (t, k, fd, gm.reshape(-1)[k])
                assert abs(fd.imag - gp.reshape(-1)[k]) < 1e-8, (t, k, fd, gp.reshape(-1)[k])


def test_dlogpsi_against_torch_autograd():
    n, h, L = 8, 16, 2
    p = _params(n, h, L, 77)
    masks = omade.build_masks(n, p.deg_hidden)
    rng = np.random.default_rng(5)
    bits = rng.integers(0, 2, size=(20, n)).astype(np.uint8)
    w_mod, w_ph = rng.standard_normal(20), rng.standard_normal(20)
    Ws = [torch.tensor(W, requires_grad=True) for W in p.weights]
    bs = [torch.tensor(b, requires_grad=True) for b in p.biases]
    P1, P2 = (torch.tensor(W, requires_grad=True) for W in p.phase_weights)
    c1, c2 = (torch.tensor(b, requires_grad=True) for b in p.phase_biases)
    z = torch.tensor(bits[:, p.order].astype(np.float64))
    a = 2 * z - 1
    for k in range(L + 1):
        a = torch.nn.functional.linear(a, Ws[k] * torch.tensor(masks[k]), bs[k])
        if k < L:
            a = torch.relu(a)
    prob = torch.sigmoid(a)
    logmod = 0.5 * (z * torch.log(prob) + (1 - z) * torch.log(1 - prob)).sum(dim=1)
    o = torch.nn.functional.linear(torch.relu(torch.nn.functional.linear(2 * z[:, : n - 2] - 1, P1, c1)), P2, c2)
    phi = torch.gather(o, 1, (2 * z[:, n - 2] + z[:, n - 1]).long()[:, None])[:, 0]
    loss = (torch.tensor(w_mod) * logmod).sum() + (torch.tensor(w_ph) * phi).sum()
    loss.backward()
    ref = []
    for W, b in zip(Ws, bs):
        ref += [W.grad.numpy(), b.grad.numpy()]
    ref += [P1.grad.numpy(), c1.grad.numpy(), P2.grad.numpy(), c2.grad.numpy()]
    got = ograd.dlogpsi_weighted(p, pack_mask(bits), w_mod, w_ph)
    for r, g in zip(ref, got):
        np.testing.assert_allclose(g, r, rtol=0, atol=1e-12)
    # masked entries receive exactly zero
    for k in range(L + 1):
        assert np.all(got[2 * k][masks[k] == 0] == 0.0)


def _random_pauli_list(n, K, seed):
    rng = np.random.default_rng(seed)
    codes = rng.integers(0, 4, size=(K, n)).astype(np.uint8)
    codes[0] = 0
    codes[1] = 2                                            # all Y
    return codes, rng.standard_normal(K)


@pytest.mark.parametrize("n,h,L", [(5, 8, 2), (6, 10, 1)])
def test_estimator_is_exact_gradient_under_full_enumeration(n, h, L):
    """Every x with weight |psi(x)|^2: Eq. 7 == grad of 1/2 <psi|H|psi> (finite differences, dense H with odd-Y)."""
    p = _params(n, h, L, 11 * n)
    codes, coeffs = _random_pauli_list(n, 40, n)
    H = bf.dense_pauli_sum(codes, coeffs)
    xs = bf.all_configs(n)

    def loss():
        psi = np.exp(omade.logpsi(p, xs))
        assert abs(np.vdot(psi, psi).real - 1.0) < 1e-12    # normalised for every theta
        return 0.5 * np.vdot(psi, H @ psi).real             # PAPER.md:62 Eq. 5

    lp = omade.logpsi(p, xs)
    weights = np.exp(2 * lp.real)
    e = oeloc.local_energy(codes, coeffs, p, xs)
    g, b = ograd.energy_gradient(p, xs, weights, e)
    assert abs(0.5 * b.real - loss()) < 1e-12               # Eq. 6: L = 1/2 E[l]
    rng = np.random.default_rng(3)
    tens = _tensors(p)
    sizes = [T.size for T in tens]
    offs = np.concatenate([[0], np.cumsum(sizes)])
    assert g.size == offs[-1]
    for t, T in enumerate(tens):
        flat = T.reshape(-1)
        for k in rng.choice(flat.size, size=min(flat.size, 6), replace=False):
            old = flat[k]
            eps = 1e-6
            flat[k] = old + eps; lplus = loss()
            flat[k] = old - eps; lminus = loss()
            flat[k] = old
            fd = (lplus - lminus) / (2 * eps)
            assert abs(fd - g[offs[t] + k]) < 2e-8, (t, k, fd, g[offs[t] + k])
    # the phase-net gradient is not identically zero here (Im E_loc != 0 because of the odd-Y strings)
    assert np.abs(g[offs[2 * (L + 1)]:]).max() > 1e-4


def test_estimator_formula_sample_by_sample_and_baseline():
    """Finite sample set with integer multiplicities: Eq. 7 written out one sample at a time, b = weighted mean."""
    n, h, L = 6, 8, 2
    p = _params(n, h, L, 9)
    rng = np.random.default_rng(8)
    bits = rng.integers(0, 2, size=(7, n)).astype(np.uint8)
    cfgs = pack_mask(bits)
    counts = rng.integers(1, 9, size=7)
    e = rng.standard_normal(7) + 1j * rng.standard_normal(7)
    g, b = ograd.energy_gradient(p, cfgs, counts, e)
    assert abs(b - (counts * e).sum() / counts.sum()) < 1e-14
    acc = 0.0
    for i in range(7):
        one = np.zeros(7); one[i] = 1.0
        s_mod = ograd.flatten(ograd.dlogpsi_weighted(p, cfgs, one, np.zeros(7)))
        s_ph = ograd.flatten(ograd.dlogpsi_weighted(p, cfgs, np.zeros(7), one))
        sigma = s_mod + 1j * s_ph                            # grad log f = grad log|psi| + i grad phi
        acc = acc + counts[i] * ((e[i] - b) * np.conj(sigma)).real
    np.testing.assert_allclose(g, acc / counts.sum(), rtol=0, atol=1e-13)
    # expanding multiplicities into repeated rows gives the same estimator
    rep = np.repeat(np.arange(7), counts)
    g2, b2 = ograd.energy_gradient(p, cfgs[rep], np.ones(len(rep)), e[rep])
    np.testing.assert_allclose(g2, g, rtol=0, atol=1e-13)
