"""Pins for oracle/sampler.py (CPU only): PAPER.md:105-107 (buffer / counter sampler), :109-120, :136-142 (Eq. 11-14).

  * Philox4x32-10 against the known-answer vectors published with the generator (Salmon et al., SC'11, Random123);
  * the constrained conditionals: sum over all 2^n strings of pi_hat(x) = 1, pi_hat(x) = 0 exactly for the strings that
    violate Eq. 12 and > 0 for the C(n/2, n_up) C(n/2, n_down) that satisfy it, several orders;
  * without constraints pi_hat is |psi|^2 of oracle.made;
  * the buffer bookkeeping against a draw-by-draw replay written independently (dict of prefixes, python loops), with
    and without pruning; total count conserved without pruning;
  * the distribution: counts / N within 5 sigma of pi_hat(x) for every string at n = 6.
"""
from math import comb

import numpy as np
import pytest

from oracle import made as omade
from oracle import sampler as osamp
from oracle.pauli import unpack_mask
from paper_2208_05637_b200 import workloads as wl
from tests import bruteforce as bf


def test_philox_known_answers():
    kat = [((0, 0, 0, 0), (0, 0), (0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8)),
           ((0xffffffff,) * 4, (0xffffffff,) * 2, (0x408f276d, 0x41c83b0e, 0xa20bc7c6, 0x6d5451fd)),
           ((0x243f6a88, 0x85a308d3, 0x13198a2e, 0x03707344), (0xa4093822, 0x299f31d0), (0xd16cfe09, 0x94fdcceb, 0x5001e420, 0x24126ea1))]
    ctr = np.array([k[0] for k in kat], dtype=np.uint32)
    key = np.array([k[1] for k in kat], dtype=np.uint32)
    out = osamp.philox4x32_10(ctr, key)
    assert out.tolist() == [list(k[2]) for k in kat]


def test_uniforms_are_in_the_open_interval_and_keyed_by_slot_and_position():
    u = osamp.draw_uniform(7, np.arange(100000), 3)
    assert u.min() > 0 and u.max() < 1 and abs(u.mean() - 0.5) < 5e-3
    assert np.array_equal(u[:10], osamp.draw_uniform(7, np.arange(10), 3))
    assert not np.array_equal(u[:10], osamp.draw_uniform(7, np.arange(10), 4))
    assert not np.array_equal(u[:10], osamp.draw_uniform(8, np.arange(10), 3))
    big = np.array([2 ** 32 + 5], dtype=np.uint64)                 # the high counter word is used
    assert osamp.draw_uniform(7, big, 3)[0] != osamp.draw_uniform(7, np.array([5]), 3)[0]


@pytest.mark.parametrize("n,nu,nd,order", [(8, 2, 2, "reverse"), (8, 1, 3, "random"), (8, 0, 4, "identity"), (6, 3, 0, "random"),
                                            (10, 2, 3, "reverse")])
def test_constrained_conditionals_normalise_and_vanish_on_invalid_strings(n, nu, nd, order):
    p = wl.make_made_params(n, 16, 31 + n + nu, order=order)
    xs = bf.all_configs(n)
    lp = osamp.constrained_logprob(p, xs, nu, nd)
    prob = np.exp(lp)
    bits = unpack_mask(xs, n)
    valid = (bits[:, 0::2].sum(axis=1) == nu) & (bits[:, 1::2].sum(axis=1) == nd)      # Eq. 12: even = up, odd = down
    assert valid.sum() == comb(n // 2, nu) * comb(n // 2, nd)
    assert np.all(prob[~valid] == 0.0)
    assert np.all(prob[valid] > 0.0)
    assert abs(prob.sum() - 1.0) < 1e-12


def test_unconstrained_is_the_made_distribution():
    p = wl.make_made_params(7, 12, 3, order="random")
    xs = bf.all_configs(7)
    np.testing.assert_allclose(osamp.constrained_logprob(p, xs, -1, -1), 2 * omade.logpsi(p, xs).real, atol=1e-12)


def _replay(p, n_draws, seed, nu, nd, max_unique):
    """Independent draw-by-draw bookkeeping: an ordered list of prefixes (tuples in position order), one python loop per
    draw; the doubled buffer lists the children of entry i at 2i, 2i+1."""
    n = p.n_qubits
    buf = [()]
    members = [list(range(n_draws))]
    for d in range(n):
        children, cm = [], []
        for pre, mem in zip(buf, members):
            z = np.zeros((1, n), dtype=np.int64)
            z[0, :d] = pre
            p1 = osamp.conditional_p1(p, z, d, nu, nd)[0]
            m0, m1 = [], []
            for s in mem:
                (m1 if osamp.draw_uniform(seed, np.array([s]), d)[0] < p1 else m0).append(s)
            children += [pre + (0,), pre + (1,)]
            cm += [m0, m1]
        idx = [i for i in range(len(children)) if cm[i]]
        if max_unique and len(idx) > max_unique:
            idx = sorted(sorted(idx, key=lambda i: (-len(cm[i]), i))[:max_unique])
        buf, members = [children[i] for i in idx], [cm[i] for i in idx]
    return buf, [len(m) for m in members]


@pytest.mark.parametrize("nu,nd,cap", [(-1, -1, 0), (2, 1, 0), (2, 2, 5), (-1, -1, 7)])
def test_buffer_bookkeeping_equals_draw_by_draw_replay(nu, nd, cap):
    n = 6
    p = wl.make_made_params(n, 10, 90 + cap, order="random")
    samples, counts, _ = osamp.sample(p, 300, 1234, nu, nd, cap)
    buf, cnt = _replay(p, 300, 1234, nu, nd, cap)
    z = unpack_mask(samples, n)[:, p.order]
    assert [tuple(int(v) for v in row) for row in z] == buf
    assert counts.tolist() == cnt
    assert len(set(map(tuple, samples.tolist()))) == len(samples)
    if cap == 0:
        assert counts.sum() == 300                                  # every draw ends in exactly one entry
    else:
        assert len(counts) <= cap and counts.sum() <= 300


@pytest.mark.parametrize("nu,nd", [(-1, -1), (2, 1)])
def test_sampled_frequencies_follow_pi_hat(nu, nd):
    n, N = 6, 200000
    p = wl.make_made_params(n, 12, 17, order="reverse")
    samples, counts, _ = osamp.sample(p, N, 99, nu, nd, 0)
    assert counts.sum() == N
    xs = bf.all_configs(n)
    prob = np.exp(osamp.constrained_logprob(p, xs, nu, nd))
    freq = np.zeros(2 ** n)
    freq[samples[:, 0].astype(np.int64)] = counts / N
    sigma = np.sqrt(prob * (1 - prob) / N)
    assert np.all(np.abs(freq - prob) <= 5 * sigma + 1e-12)
    assert np.all(freq[prob == 0] == 0)


def test_constrained_logpsi_forced_positions_and_its_gradient():
    """forced_positions restates Eq. 14's clamps: skipping them in the plain MADE sum reproduces constrained_logprob;
    the gradient of the constrained log f (oracle.grad with n_up, n_down) equals central differences of it."""
    from oracle import grad as ograd
    n, nu, nd = 8, 2, 3
    p = wl.make_made_params(n, 12, 5, order="random")
    p.weights = [w.astype(np.float64) for w in p.weights]; p.biases = [b.astype(np.float64) for b in p.biases]
    p.phase_weights = [w.astype(np.float64) for w in p.phase_weights]; p.phase_biases = [b.astype(np.float64) for b in p.phase_biases]
    xs = bf.all_configs(n)
    z = unpack_mask(xs, n)[:, p.order].astype(np.int64)
    forced, valid = osamp.forced_positions(p, z, nu, nd)
    lp = osamp.constrained_logpsi(p, xs, nu, nd)
    assert np.array_equal(valid, np.isfinite(lp.real))
    a = omade.conditionals_logits(p, z)
    terms = np.where(z == 1, omade.log_sigmoid(a), omade.log_sigmoid(-a))
    np.testing.assert_allclose(0.5 * np.where(forced, 0.0, terms).sum(axis=1)[valid], lp.real[valid], atol=1e-13)
    np.testing.assert_allclose(lp.imag, omade.logpsi(p, xs).imag, atol=1e-14)
    # gradient by central differences on three valid strings
    vi = np.flatnonzero(valid)[[0, 7, 20]]
    cf = xs[vi]
    rng = np.random.default_rng(0)
    for i in range(3):
        one = np.zeros(3); one[i] = 1
        g = ograd.dlogpsi_weighted(p, cf, one, np.zeros(3), nu, nd)
        for T, gt in zip([p.weights[0], p.weights[1], p.weights[2], p.biases[2]], [g[0], g[2], g[4], g[5]]):
            flat = T.reshape(-1)
            for k in rng.choice(flat.size, size=8, replace=False):
                old = flat[k]
                flat[k] = old + 1e-6; lpl = osamp.constrained_logpsi(p, cf[i:i + 1], nu, nd)[0].real
                flat[k] = old - 1e-6; lmi = osamp.constrained_logpsi(p, cf[i:i + 1], nu, nd)[0].real
                flat[k] = old
                assert abs((lpl - lmi) / 2e-6 - gt.reshape(-1)[k]) < 1e-8
