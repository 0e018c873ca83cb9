"""Gradient of the energy objective (oracle; test infrastructure) — PAPER.md:71 Eq. 7:

    grad L(theta) = Re E[ (l_theta(x) - b) * conj(sigma_theta(x)) ],   sigma_theta = grad_theta f / f = grad_theta log f,

with b = E[l_theta(x)] and the expectation over the unique samples weighted by their multiplicities
(PAPER.md:105 counter, :200 Eq. 17).  L = 1/2 <f|H|f> (Eq. 5), so for the normalised autoregressive
state this IS the exact gradient of 1/2 <H> when the samples are all 2^n configurations weighted by |psi|^2
(pinned that way in tests/test_oracle_grad.py).

log f = log|psi| + i phi (Eq. 10) with both parts real-valued networks, so
    Re[(E - b) conj(d log f)] = Re(E - b) * d log|psi|  +  Im(E - b) * d phi:
the MADE parameters receive Re(E - b) through log|psi| only, the phase-net parameters Im(E - b) through phi only.

Everything is written out layer by layer in fp64 (manual backward pass, no autograd): obviously slow, checkable by eye.
Parameter order of the flat gradient (the C ABI's, include/nqs.h): for k = 0..L: W_k [out][in] then b_k; then
P1 [h][n-2], c1 [h], P2 [4][h], c2 [4]; all in autoregressive POSITION order as in `params`.  Gradients are with respect
to the UNMASKED weights the ABI takes, i.e. masked entries receive exactly 0.
"""
import numpy as np

from .pauli import unpack_mask
from . import made as _made


def _sigmoid(t):
    return 0.5 * (1.0 + np.tanh(0.5 * t))


def dlogpsi_weighted(params, configs, w_mod, w_phase, n_up=-1, n_down=-1):
    """sum_i [ w_mod[i] * grad log|psi|(x_i) + w_phase[i] * grad phi(x_i) ] as a list of arrays shaped like the
    parameters: [dW_0, db_0, ..., dW_L, db_L, dP1, dc1, dP2, dc2].  Manual backward pass through Eq. 8-10.
    With n_up, n_down >= 0 the model is the constrained one: a conditional that Eq. 14 clamps to 0 / 1
    is a constant, so its logit receives no gradient (strings that violate Eq. 12 have psi = 0 and must not be passed)."""
    n = params.n_qubits
    bits = unpack_mask(np.asarray(configs, dtype=np.uint64), n)
    z = bits[:, np.asarray(params.order, dtype=np.int64)].astype(np.float64)      # [B, n] by position
    u = 2.0 * z - 1.0                                                              # reading A9
    w_mod = np.asarray(w_mod, dtype=np.float64)
    w_phase = np.asarray(w_phase, dtype=np.float64)
    masks = _made.build_masks(n, params.deg_hidden)
    nl = len(params.weights)
    Wm = [np.asarray(params.weights[k], dtype=np.float64) * masks[k] for k in range(nl)]
    bs = [np.asarray(params.biases[k], dtype=np.float64) for k in range(nl)]
    # ---- modulus net forward: keep every layer's input and pre-activation ----
    acts = [u]
    pre = []
    for k in range(nl):
        a = acts[-1] @ Wm[k].T + bs[k]
        pre.append(a)
        acts.append(np.maximum(a, 0.0) if k < nl - 1 else a)
    a_out = pre[-1]                                                                # logits [B, n]
    # log|psi| = 1/2 sum_d log sigmoid(s_d a_d), s_d = +1 if z_d = 1 else -1;  d/da log sigmoid(s a) = s sigmoid(-s a)
    s = u
    g = w_mod[:, None] * 0.5 * s * _sigmoid(-s * a_out)                            # d loss / d logits
    if n_up >= 0:
        from .sampler import forced_positions
        forced, valid = forced_positions(params, z.astype(np.int64), n_up, n_down)
        if not valid.all():
            raise ValueError("a sample violates the Hamming-weight constraint: psi = 0 there")
        g = np.where(forced, 0.0, g)
    grads = [None] * (2 * nl)
    for k in range(nl - 1, -1, -1):
        grads[2 * k] = (g.T @ acts[k]) * masks[k]                                  # dW_k (masked entries: exactly 0)
        grads[2 * k + 1] = g.sum(axis=0)                                           # db_k
        if k > 0:
            g = (g @ Wm[k]) * (pre[k - 1] > 0.0)                                   # through ReLU of layer k-1
    # ---- phase net (reading A11) ----
    P1 = np.asarray(params.phase_weights[0], dtype=np.float64)
    P2 = np.asarray(params.phase_weights[1], dtype=np.float64)
    c1 = np.asarray(params.phase_biases[0], dtype=np.float64)
    up = u[:, : n - 2]
    hp = up @ P1.T + c1
    hid = np.maximum(hp, 0.0)
    sel = (2 * z[:, n - 2] + z[:, n - 1]).astype(np.int64)
    go = np.zeros((z.shape[0], 4))
    go[np.arange(z.shape[0]), sel] = w_phase                                       # d loss / d o (only the selected output)
    dP2 = go.T @ hid
    dc2 = go.sum(axis=0)
    gh = (go @ P2) * (hp > 0.0)
    dP1 = gh.T @ up
    dc1 = gh.sum(axis=0)
    return grads + [dP1, dc1, dP2, dc2]


def flatten(grads):
    return np.concatenate([np.asarray(g, dtype=np.float64).reshape(-1) for g in grads])


def energy_gradient(params, samples, counts, eloc, n_up=-1, n_down=-1):
    """Eq. 7 with b = weighted mean of E_loc: returns (flat gradient fp64, b complex).

    samples uint64 [B,2], counts [B] (multiplicities; any non-negative weights), eloc complex [B]."""
    c = np.asarray(counts, dtype=np.float64)
    e = np.asarray(eloc, dtype=np.complex128)
    tot = c.sum()
    b = (c * e).sum() / tot
    w_mod = c * (e.real - b.real) / tot
    w_phase = c * (e.imag - b.imag) / tot
    return flatten(dlogpsi_weighted(params, samples, w_mod, w_phase, n_up, n_down)), b
