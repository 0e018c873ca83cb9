"""Naive fp64 MADE modulus net + phase MLP (oracle; test infrastructure).

PAPER.md:84 (architecture: MaskedFC -> ReLU -> MaskedFC -> Sigmoid; phase net [B,n-2] -> h -> 4),
:88 Eq. 8 (pi(x) = prod_i pi_i(x_i | x_<i)), :93-96 Eq. 9-10 (log f = i phi + 1/2 sum_i log pi_i).
Readings: A7 n_hidden_layers in {1, 2}; A8 masks from degrees; A9 input u = 2z - 1;
A10 `order`; A11 dense phase net selected by the last two bits in autoregressive order; A12 raw
(unconstrained) sigmoid conditionals.

`params` is any object with fields n_qubits, hidden, n_hidden_layers, order[n], deg_hidden[L][h],
weights (L+1 unmasked [out][in] matrices), biases, phase_weights ([h][n-2], [4][h]), phase_biases.
"""
import numpy as np

from .pauli import unpack_mask


def build_masks(n: int, deg_hidden: np.ndarray):
    """MADE masks from degrees (Germain et al. rule; reading A8).

    m_in[d] = d + 1 for autoregressive position d (0-based).  Hidden degrees in 1..n-1.
      M1[j][d]  = (m_hid1[j] >= m_in[d])
      Mk[j'][j] = (m_hid_k[j'] >= m_hid_{k-1}[j])          (hidden -> hidden)
      Mout[d][j] = (m_in[d] > m_hid_L[j])                   (strict: output d sees inputs < d only)
    """
    deg_hidden = np.asarray(deg_hidden, dtype=np.int64)
    m_in = np.arange(1, n + 1, dtype=np.int64)
    masks = [(deg_hidden[0][:, None] >= m_in[None, :])]
    for k in range(1, deg_hidden.shape[0]):
        masks.append(deg_hidden[k][:, None] >= deg_hidden[k - 1][None, :])
    masks.append(m_in[:, None] > deg_hidden[-1][None, :])
    return [m.astype(np.float64) for m in masks]


def log_sigmoid(t: np.ndarray) -> np.ndarray:
    """log(1/(1+e^-t)) = min(t, 0) - log1p(exp(-|t|)), stable for all t."""
    return np.minimum(t, 0.0) - np.log1p(np.exp(-np.abs(t)))


def conditionals_logits(params, z: np.ndarray) -> np.ndarray:
    """Logits a[b, d] of pi_d(z_d = 1 | z_<d); z [B, n] in autoregressive order (0/1)."""
    n = params.n_qubits
    masks = build_masks(n, params.deg_hidden)
    a = 2.0 * z.astype(np.float64) - 1.0                       # u = 2z - 1 (reading A9)
    nl = len(params.weights)
    for k in range(nl):
        Wm = np.asarray(params.weights[k], dtype=np.float64) * masks[k]
        a = a @ Wm.T + np.asarray(params.biases[k], dtype=np.float64)
        if k < nl - 1:
            a = np.maximum(a, 0.0)                             # ReLU
    return a


def phase(params, z: np.ndarray) -> np.ndarray:
    """phi(x): two-layer dense MLP on the first n-2 inputs, 4 outputs, picked by the last two bits."""
    n = params.n_qubits
    u = 2.0 * z[:, : n - 2].astype(np.float64) - 1.0
    P1 = np.asarray(params.phase_weights[0], dtype=np.float64)
    P2 = np.asarray(params.phase_weights[1], dtype=np.float64)
    hid = np.maximum(u @ P1.T + np.asarray(params.phase_biases[0], dtype=np.float64), 0.0)
    o = hid @ P2.T + np.asarray(params.phase_biases[1], dtype=np.float64)          # [B, 4]
    sel = 2 * z[:, n - 2].astype(np.int64) + z[:, n - 1].astype(np.int64)
    return o[np.arange(z.shape[0]), sel]


def logpsi(params, configs: np.ndarray) -> np.ndarray:
    """log f(x) = i phi(x) + 1/2 sum_d log pi_d(x_d | x_<d)  (Eq. 10), complex128 [B].

    configs: uint64 [B, 2] bit-packed, bit j = qubit j.  Position d of the autoregressive order reads
    qubit order[d].
    """
    n = params.n_qubits
    bits = unpack_mask(np.asarray(configs, dtype=np.uint64), n)                    # [B, n] by qubit
    z = bits[:, np.asarray(params.order, dtype=np.int64)]                          # by position
    a = conditionals_logits(params, z)
    zf = z.astype(np.float64)
    logpi = (zf * log_sigmoid(a) + (1.0 - zf) * log_sigmoid(-a)).sum(axis=1)       # Eq. 8 in log form
    return 0.5 * logpi + 1j * phase(params, z)
