"""Batched autoregressive sampler (oracle; test infrastructure) — PAPER.md:105-107 (sampling), :109-120 and :136-142
(Hamming-weight constraints, Eq. 11-14).

The paper's scheme: "keep track of a sample buffer ... associated with a counter storing the number of
occurrences for each sample in the buffer.  We start with a buffer containing only one ... sample.  At each of the n
iterations, we first double the size of the buffer by alternating +-1 value for existing samples at a fixed entry.
Then, we update the counter for all samples in the buffer through Bernoulli sampling with probabilities computed by
forward pass.  Finally, we eliminate the samples in the batch that have the lowest numbers of occurrences".

Readings adopted where the paper is silent or garbled (A13 / A25):
  * positions are visited in the autoregressive order of the model, d = 0..n-1, position d = qubit order[d] (the paper's
    default order is reversed, :107, and is a property of `params.order`);
  * the "Bernoulli sampling" of a counter holding c occurrences is c independent Bernoulli(p) trials, one per DRAW:
    draw s (0 <= s < n_draws) at position d uses the uniform u = (w + 1/2) 2^-32 with w the first word of
    Philox4x32-10(key = seed, counter = (s, d)); it takes bit 1 iff u < p.  The split of a counter is therefore
    Binomial(c, p) exactly, and the draws do not depend on how the buffer is ordered — both implementations of this
    repository (this one and the CUDA one) replay the same draws;
  * entries whose counter falls to zero leave the buffer; if more than `max_unique` remain, the `max_unique` entries
    with the largest counters are kept (ties: the entry that comes first in buffer order; children of entry i sit at
    2i, 2i+1) and the draws of the dropped entries are discarded (the total count shrinks);
  * Eq. 13-14 are garbled in the source (the fourth case repeats x_{2i-1} with n_down; the sums run to ceil(k/2), which
    would include x_k itself).  Reading: at position d, whose qubit has spin sigma (even qubit = up, odd = down,
    Eq. 12), with c = number of spin-sigma bits already set at positions < d and m = number of spin-sigma positions
    >= d:  pi_hat(1) = 0 if c = n_sigma;  pi_hat(1) = 1 if n_sigma - c = m;  pi otherwise.  Every completed string
    then satisfies Eq. 12 and the modified conditionals still normalise (:142).
"""
import numpy as np

from . import made as _made
from .pauli import unpack_mask, pack_mask

_M0, _M1 = np.uint64(0xD2511F53), np.uint64(0xCD9E8D57)
_W0, _W1 = np.uint32(0x9E3779B9), np.uint32(0xBB67AE85)
_MASK32 = np.uint64(0xFFFFFFFF)


def philox4x32_10(counter, key):
    """Philox4x32 with 10 rounds (Salmon et al., SC'11), vectorised: counter uint32 [..., 4], key uint32 [..., 2] ->
    uint32 [..., 4]."""
    c = [np.asarray(counter[..., i], dtype=np.uint32).copy() for i in range(4)]
    k0 = np.asarray(key[..., 0], dtype=np.uint32).copy()
    k1 = np.asarray(key[..., 1], dtype=np.uint32).copy()
    with np.errstate(over="ignore"):
        for _ in range(10):
            p0 = _M0 * c[0].astype(np.uint64)
            p1 = _M1 * c[2].astype(np.uint64)
            hi0, lo0 = (p0 >> np.uint64(32)).astype(np.uint32), (p0 & _MASK32).astype(np.uint32)
            hi1, lo1 = (p1 >> np.uint64(32)).astype(np.uint32), (p1 & _MASK32).astype(np.uint32)
            c = [hi1 ^ c[1] ^ k0, lo1, hi0 ^ c[3] ^ k1, lo0]
            k0 = (k0 + _W0).astype(np.uint32)
            k1 = (k1 + _W1).astype(np.uint32)
    return np.stack(c, axis=-1)


def draw_uniform(seed: int, slots: np.ndarray, position: int) -> np.ndarray:
    """u in (0, 1) of draw `slots` at autoregressive position `position` (fp64, exactly representable)."""
    slots = np.asarray(slots, dtype=np.uint64)
    ctr = np.zeros(slots.shape + (4,), dtype=np.uint32)
    ctr[..., 0] = (slots & _MASK32).astype(np.uint32)
    ctr[..., 1] = (slots >> np.uint64(32)).astype(np.uint32)
    ctr[..., 2] = np.uint32(position)
    key = np.zeros(slots.shape + (2,), dtype=np.uint32)
    key[..., 0] = np.uint32(seed & 0xFFFFFFFF)
    key[..., 1] = np.uint32((seed >> 32) & 0xFFFFFFFF)
    w = philox4x32_10(ctr, key)[..., 0]
    return (w.astype(np.float64) + 0.5) * 2.0 ** -32


def _spin_of_positions(params):
    """spin[d] = 0 (up, even qubit) or 1 (down, odd qubit) of autoregressive position d (Eq. 12)."""
    return (np.asarray(params.order, dtype=np.int64) & 1).astype(np.int64)


def clamp_conditional(params, z_prefix: np.ndarray, d: int, p1: np.ndarray, n_up: int, n_down: int) -> np.ndarray:
    """Eq. 14 under the reading in the module docstring: z_prefix [E, n] (positions >= d ignored), p1 [E]."""
    if n_up < 0:
        return p1
    spin = _spin_of_positions(params)
    sig = spin[d]
    target = n_up if sig == 0 else n_down
    same_before = (spin[:d] == sig)
    c = z_prefix[:, :d][:, same_before].sum(axis=1)
    m = int((spin[d:] == sig).sum())                               # spin-sigma positions not yet decided, this one included
    out = p1.copy()
    out[c >= target] = 0.0
    out[(target - c) >= m] = 1.0
    return out


def conditional_p1(params, z_prefix: np.ndarray, d: int, n_up: int = -1, n_down: int = -1) -> np.ndarray:
    """pi_hat(z_d = 1 | z_<d) for every buffer entry; z_prefix [E, n] in POSITION order, entries >= d arbitrary
    (the autoregressive masks make logit d independent of them — pinned in tests/test_oracle_made.py)."""
    a = _made.conditionals_logits(params, z_prefix)[:, d]
    p1 = 1.0 / (1.0 + np.exp(-a))
    return clamp_conditional(params, z_prefix, d, p1, n_up, n_down)


def constrained_logprob(params, configs: np.ndarray, n_up: int, n_down: int) -> np.ndarray:
    """log pi_hat(x) = sum_d log pi_hat(x_d | x_<d): -inf for strings that violate Eq. 12."""
    n = params.n_qubits
    bits = unpack_mask(np.asarray(configs, dtype=np.uint64), n)
    z = bits[:, np.asarray(params.order, dtype=np.int64)].astype(np.int64)
    out = np.zeros(z.shape[0])
    with np.errstate(divide="ignore"):
        for d in range(n):
            p1 = conditional_p1(params, z, d, n_up, n_down)
            out += np.where(z[:, d] == 1, np.log(p1), np.log1p(-p1))
    return out


def forced_positions(params, z: np.ndarray, n_up: int, n_down: int):
    """(forced [B, n] bool, valid [B] bool): positions whose conditional Eq. 14 clamps to 0 or 1 given the bits before
    them, and whether the string respects every clamp (i.e. satisfies Eq. 12).  z [B, n] in POSITION order."""
    B, n = z.shape
    forced = np.zeros((B, n), dtype=bool)
    valid = np.ones(B, dtype=bool)
    if n_up < 0:
        return forced, valid
    spin = _spin_of_positions(params)
    for d in range(n):
        sig = spin[d]
        target = n_up if sig == 0 else n_down
        c = z[:, :d][:, spin[:d] == sig].sum(axis=1)
        m = int((spin[d:] == sig).sum())
        f0, f1 = c >= target, (target - c) >= m
        forced[:, d] = f0 | f1
        valid &= ~(f0 & (z[:, d] == 1)) & ~(f1 & (z[:, d] == 0))
    return forced, valid


def constrained_logpsi(params, configs: np.ndarray, n_up: int, n_down: int) -> np.ndarray:
    """log f of the CONSTRAINED model (PAPER.md:138-142 with :96 Eq. 10): log|psi| = 1/2 sum_d log pi_hat_d, phase
    unchanged.  -inf + i phi for strings that violate Eq. 12 (psi = 0 there)."""
    n = params.n_qubits
    bits = unpack_mask(np.asarray(configs, dtype=np.uint64), n)
    z = bits[:, np.asarray(params.order, dtype=np.int64)]
    return 0.5 * constrained_logprob(params, configs, n_up, n_down) + 1j * _made.phase(params, z)


def sample(params, n_draws: int, seed: int, n_up: int = -1, n_down: int = -1, max_unique: int = 0):
    """The buffer / counter sampler.  Returns (samples uint64 [U, 2] in qubit order, counts int64 [U]) in buffer order,
    and the list of |u - p| margins of every draw taken (for the parity test's ambiguity budget)."""
    n = params.n_qubits
    order = np.asarray(params.order, dtype=np.int64)
    z = np.zeros((1, n), dtype=np.int64)                            # the buffer, POSITION order; undecided entries 0
    counts = np.array([n_draws], dtype=np.int64)
    entry = np.zeros(n_draws, dtype=np.int64)                       # buffer entry of every live draw
    slots = np.arange(n_draws, dtype=np.uint64)                     # identity of every live draw
    margins = []
    for d in range(n):
        p1 = conditional_p1(params, z, d, n_up, n_down)             # forward pass on the buffer
        u = draw_uniform(seed, slots, d)
        bit = (u < p1[entry]).astype(np.int64)                      # Bernoulli trial of every draw
        margins.append(np.abs(u - p1[entry]))
        child = 2 * entry + bit                                     # doubled buffer: children of entry i at 2i, 2i+1
        ccount = np.bincount(child, minlength=2 * len(counts)).astype(np.int64)
        keep = ccount > 0
        if max_unique and keep.sum() > max_unique:                  # eliminate the lowest counters
            idx = np.flatnonzero(keep)
            rank = np.lexsort((idx, -ccount[idx]))                  # largest count first, ties by buffer order
            keep[:] = False
            keep[idx[rank[:max_unique]]] = True
        newidx = np.cumsum(keep) - 1                                # stable compaction
        kept = np.flatnonzero(keep)
        znew = z[kept // 2].copy()
        znew[:, d] = kept & 1
        z, counts = znew, ccount[kept]
        alive = keep[child]
        entry, slots = newidx[child[alive]], slots[alive]
    bits = np.zeros((z.shape[0], n), dtype=np.uint8)
    bits[:, order] = z.astype(np.uint8)                             # position d -> qubit order[d]
    return pack_mask(bits), counts, np.concatenate(margins) if margins else np.zeros(0)
