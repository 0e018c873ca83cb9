"""Seeded random MADE + phase-MLP parameters (BASELINE.json configs; readings A7-A14 in DESIGN.md).

Shapes only (PAPER.md:84 architecture diagram); no forward arithmetic here.  Weights are
UNMASKED fp32, row-major [out][in]; the masks are applied by whoever evaluates the model
from `order` and `deg_hidden`.
"""
from dataclasses import dataclass, field
from typing import List

import numpy as np


@dataclass
class MadeParams:
    n_qubits: int
    hidden: int
    n_hidden_layers: int
    order: np.ndarray            # int32 [n]; autoregressive position d reads qubit order[d]
    deg_hidden: np.ndarray       # int32 [layers, h]; degrees in 1..n-1
    weights: List[np.ndarray] = field(default_factory=list)   # L+1 matrices: [h,n], ([h,h]), [n,h]
    biases: List[np.ndarray] = field(default_factory=list)    # [h], ([h]), [n]
    phase_weights: List[np.ndarray] = field(default_factory=list)  # [h,n-2], [4,h]
    phase_biases: List[np.ndarray] = field(default_factory=list)   # [h], [4]


def default_degrees(n_qubits: int, hidden: int, n_hidden_layers: int) -> np.ndarray:
    """Sorted rule m_hid[j] = 1 + floor(j*(n-1)/h) for every hidden layer (reading A8)."""
    j = np.arange(hidden, dtype=np.int64)
    d = 1 + (j * (n_qubits - 1)) // hidden
    return np.tile(d.astype(np.int32), (n_hidden_layers, 1))


def make_made_params(n_qubits: int, hidden: int, seed: int, n_hidden_layers: int = 2,
                     order: str = "reverse", bias_std: float = 0.1) -> MadeParams:
    n, h, L = int(n_qubits), int(hidden), int(n_hidden_layers)
    rng = np.random.default_rng(seed)
    if order == "reverse":          # sample "in a reversed order beginning with the nth qubit"
        perm = np.arange(n - 1, -1, -1, dtype=np.int32)
    elif order == "identity":
        perm = np.arange(n, dtype=np.int32)
    elif order == "random":
        perm = rng.permutation(n).astype(np.int32)
    else:
        raise ValueError(order)

    def mat(o, i):
        return (rng.standard_normal((o, i)) / np.sqrt(i)).astype(np.float32)   # variance 1/fan_in

    def vec(o):
        return (bias_std * rng.standard_normal(o)).astype(np.float32)

    dims = [n] + [h] * L + [n]
    weights = [mat(dims[i + 1], dims[i]) for i in range(L + 1)]
    biases = [vec(dims[i + 1]) for i in range(L + 1)]
    phase_weights = [mat(h, n - 2), mat(4, h)]
    phase_biases = [vec(h), vec(4)]
    return MadeParams(n, h, L, perm, default_degrees(n, h, L), weights, biases, phase_weights, phase_biases)
