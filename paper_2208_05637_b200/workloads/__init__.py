"""Seeded synthetic input generators shared by the oracle tests and the CUDA path.

Holds NONE of the method's arithmetic (no matrix elements, no MADE forward, no E_loc):
only the recipes that produce integrals, the Jordan-Wigner Pauli list, random model
parameters and samples.  See DESIGN.md "Input recipe".
"""
from .configs import WORKLOADS, Workload
from .integrals import make_integrals, make_integrals_symmetric
from .jw import jw_pauli_terms, masks_to_codes, codes_to_strings, build_jwgen
from .made_params import MadeParams, make_made_params, default_degrees
from .samples import make_samples, pack_bits, unpack_bits


def make_workload(cfg: int, batch: int = None):
    """Everything one config needs: (workload, (x, z, coeffs), MadeParams, samples, counts)."""
    w = WORKLOADS[cfg]
    h, g = make_integrals(w.n_spatial, w.seed_integrals)
    x, z, c = jw_pauli_terms(h, g)
    params = make_made_params(w.n_qubits, w.hidden, w.seed_weights)
    samples, counts = make_samples(w.n_spatial, w.n_alpha, w.n_beta, batch or w.batch,
                                   w.max_count, w.seed_samples, w.unique)
    return w, (x, z, c), params, samples, counts
