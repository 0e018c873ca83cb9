"""Pins for oracle/made.py (CPU only): normalisation over 2^n ("Normalization follows
automatically"), autoregressive property, closed forms, an independent library evaluation."""
import numpy as np
import pytest
import torch

from oracle import made as omade
from oracle.pauli import pack_mask
from paper_2208_05637_b200 import workloads as wl
from tests import bruteforce as bf


def _params(n, h, L, seed, order="reverse", random_deg=False):
    p = wl.make_made_params(n, h, seed, n_hidden_layers=L, order=order)
    if random_deg:
        rng = np.random.default_rng(seed + 5)
        p.deg_hidden = rng.integers(1, n, size=(L, h)).astype(np.int32)   # any assignment in 1..n-1 is legal
    return p


@pytest.mark.parametrize("n,h,L,order,rd", [(3, 8, 2, "reverse", False), (6, 16, 2, "reverse", False),
                                            (7, 16, 1, "identity", False), (8, 32, 2, "random", True),
                                            (10, 32, 2, "reverse", True), (5, 4, 2, "random", False)])
def test_normalisation_over_all_configs(n, h, L, order, rd):
    """sum_x |f(x)|^2 = sum_x pi(x) = 1 — fails for any mask / ordering / log-sigmoid error."""
    p = _params(n, h, L, 11 + n, order, rd)
    lp = omade.logpsi(p, bf.all_configs(n))
    assert abs(np.exp(2 * lp.real).sum() - 1.0) < 1e-12


def test_autoregressive_property():
    """Flipping the input at position d changes only the logits at positions > d."""
    n, h = 9, 24
    p = _params(n, h, 2, 3, "random", True)
    rng = np.random.default_rng(0)
    z = rng.integers(0, 2, size=(1, n)).astype(np.uint8)
    a0 = omade.conditionals_logits(p, z)
    for d in range(n):
        z2 = z.copy(); z2[0, d] ^= 1
        a1 = omade.conditionals_logits(p, z2)
        assert np.array_equal(a0[0, : d + 1], a1[0, : d + 1])
    # and with the default (sorted) rule every later logit really does depend on earlier inputs
    p = _params(n, 64, 2, 4)
    a0 = omade.conditionals_logits(p, z)
    z2 = z.copy(); z2[0, 0] ^= 1
    assert np.all(omade.conditionals_logits(p, z2)[0, 1:] != a0[0, 1:])


def test_zero_weights_closed_form():
    """All weights zero: pi_d = sigmoid(b_out[d]) independent of x; log|psi| has a closed form."""
    n, h = 6, 8
    p = _params(n, h, 2, 5, "identity")
    p.weights = [np.zeros_like(w) for w in p.weights]
    b = np.asarray(p.biases[-1], dtype=np.float64)
    xs = bf.all_configs(n)
    lp = omade.logpsi(p, xs)
    bits = ((xs[:, 0:1] >> np.arange(n, dtype=np.uint64)) & np.uint64(1)).astype(np.float64)
    sig = 1.0 / (1.0 + np.exp(-b))
    expect = 0.5 * (bits * np.log(sig) + (1 - bits) * np.log(1 - sig)).sum(axis=1)
    np.testing.assert_allclose(lp.real, expect, rtol=0, atol=1e-13)


def test_order_is_a_relabelling():
    """logpsi with order=perm on x equals logpsi with identity order on the permuted bits."""
    n, h = 8, 16
    rng = np.random.default_rng(9)
    p = _params(n, h, 2, 6, "random")
    q = _params(n, h, 2, 6, "random")
    q.order = np.arange(n, dtype=np.int32)
    bits = rng.integers(0, 2, size=(20, n)).astype(np.uint8)
    lp = omade.logpsi(p, pack_mask(bits))
    lq = omade.logpsi(q, pack_mask(bits[:, p.order]))
    np.testing.assert_allclose(lp, lq, atol=1e-14)


def test_against_torch_dense_mlp():
    """Same network through a different library (torch.nn.functional, fp64) with W*M pre-multiplied and
    the sigmoid/log written the textbook way."""
    n, h = 10, 32
    p = _params(n, h, 2, 7)
    masks = omade.build_masks(n, p.deg_hidden)
    rng = np.random.default_rng(1)
    bits = rng.integers(0, 2, size=(50, n)).astype(np.uint8)
    z = torch.tensor(bits[:, p.order].astype(np.float64))
    a = 2 * z - 1
    for k, (W, b) in enumerate(zip(p.weights, p.biases)):
        a = torch.nn.functional.linear(a, torch.tensor(W.astype(np.float64) * masks[k]), torch.tensor(b.astype(np.float64)))
        if k < len(p.weights) - 1:
            a = torch.relu(a)
    prob = torch.sigmoid(a)
    logpi = (z * torch.log(prob) + (1 - z) * torch.log(1 - prob)).sum(dim=1)
    lp = omade.logpsi(p, pack_mask(bits))
    np.testing.assert_allclose(lp.real, 0.5 * logpi.numpy(), atol=1e-12)
    # phase net (reading A11) through the same independent library: dense n-2 -> h -> 4 on the
    # first n-2 POSITIONS, output picked by torch.gather with the last two positions' bits
    u = 2 * z[:, : n - 2] - 1
    hid = torch.relu(torch.nn.functional.linear(u, torch.tensor(p.phase_weights[0].astype(np.float64)),
                                                torch.tensor(p.phase_biases[0].astype(np.float64))))
    o = torch.nn.functional.linear(hid, torch.tensor(p.phase_weights[1].astype(np.float64)),
                                   torch.tensor(p.phase_biases[1].astype(np.float64)))
    sel = (2 * z[:, n - 2] + z[:, n - 1]).long()
    phi = torch.gather(o, 1, sel[:, None])[:, 0]
    np.testing.assert_allclose(lp.imag, phi.numpy(), atol=1e-12)


def test_log_sigmoid_vs_long_double_and_symmetry():
    t = np.linspace(-30, 30, 2001)
    ref = np.log(1.0 / (1.0 + np.exp(-t.astype(np.longdouble)))).astype(np.float64)
    np.testing.assert_allclose(omade.log_sigmoid(t), ref, rtol=0, atol=2e-15)
    np.testing.assert_allclose(omade.log_sigmoid(t) - omade.log_sigmoid(-t), t, rtol=0, atol=1e-14)
    assert np.isfinite(omade.log_sigmoid(np.array([-800.0, 800.0]))).all()


def test_phase_selector_and_input_independence():
    """phi depends on the last two positions only through the selector 2*z[n-2] + z[n-1] (reading A11)."""
    n, h = 7, 16
    p = _params(n, h, 2, 8, "identity")
    rng = np.random.default_rng(2)
    base = rng.integers(0, 2, size=n).astype(np.uint8)
    z = np.tile(base, (4, 1))
    for k in range(4):
        z[k, n - 2], z[k, n - 1] = k >> 1, k & 1
    phis = omade.phase(p, z)
    u = 2.0 * base[: n - 2] - 1.0
    hid = np.maximum(p.phase_weights[0].astype(np.float64) @ u + p.phase_biases[0], 0)
    o = p.phase_weights[1].astype(np.float64) @ hid + p.phase_biases[1]
    np.testing.assert_allclose(phis, o, atol=1e-14)
    lp = omade.logpsi(p, pack_mask(z))
    np.testing.assert_allclose(lp.imag, o, atol=1e-14)


def test_phase_reads_positions_not_qubits():
    """The phase net's n-2 inputs and its 2-bit selector are taken in autoregressive POSITION order
    (z_d = x[order[d]], reading A10/A11), not in qubit order: with a non-trivial order (i) flipping the QUBITS
    order[n-2], order[n-1] moves phi only among the four outputs of the same hidden state, while flipping
    qubits n-2, n-1 (which sit at other positions) changes the hidden state; (ii) phi equals a hand evaluation
    that gathers inputs through `order`, and differs from the one that ignores `order`."""
    n, h = 9, 16
    p = _params(n, h, 2, 21, "reverse")                      # position d reads qubit n-1-d
    rng = np.random.default_rng(4)
    bits = rng.integers(0, 2, size=(16, n)).astype(np.uint8)  # by qubit
    P1, P2 = p.phase_weights[0].astype(np.float64), p.phase_weights[1].astype(np.float64)
    c1, c2 = p.phase_biases[0].astype(np.float64), p.phase_biases[1].astype(np.float64)

    def by_hand(zrow):                                        # zrow: bits already in the order the net reads them
        hid = np.maximum(P1 @ (2.0 * zrow[: n - 2] - 1.0) + c1, 0.0)
        return (P2 @ hid + c2)[2 * int(zrow[n - 2]) + int(zrow[n - 1])]

    lp = omade.logpsi(p, pack_mask(bits))
    pos = np.array([by_hand(bits[b][p.order].astype(np.float64)) for b in range(16)])
    qub = np.array([by_hand(bits[b].astype(np.float64)) for b in range(16)])
    np.testing.assert_allclose(lp.imag, pos, atol=1e-13)
    assert np.abs(lp.imag - qub).max() > 1e-3
    # (i) selector qubits are order[n-2], order[n-1] = qubits 1, 0 under the reverse order
    q_hi, q_lo = int(p.order[n - 2]), int(p.order[n - 1])
    assert (q_hi, q_lo) == (1, 0)
    b0 = bits[:1].copy()
    outs = []
    for k in range(4):
        b = b0.copy(); b[0, q_hi], b[0, q_lo] = k >> 1, k & 1
        outs.append(omade.logpsi(p, pack_mask(b)).imag[0])
    hid = np.maximum(P1 @ (2.0 * b0[0][p.order][: n - 2] - 1.0) + c1, 0.0)
    np.testing.assert_allclose(outs, P2 @ hid + c2, atol=1e-13)
