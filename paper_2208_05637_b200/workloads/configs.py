"""The five synthetic workloads of BASELINE.json (`configs[0..4]`, called cfg 1..5 here).

These stand in for the paper's molecule set (Table 1: n = 4..76 qubits,
K = 15..1,625,991 Pauli terms), whose Hamiltonians need OpenFermion-Psi4/PubChem and are
not available offline.  Only shapes/recipes live here; no method arithmetic.
"""
from dataclasses import dataclass

SEED_BASE = 220805637 * 10  # seed = 220805637*10 + cfg (+100 weights, +200 samples)


@dataclass(frozen=True)
class Workload:
    cfg: int            # 1..5
    n_spatial: int      # N spatial orbitals; n_qubits = 2N
    n_alpha: int
    n_beta: int
    hidden: int         # MADE hidden width h (= phase-MLP width)
    batch: int          # number of (unique) samples B
    minibatch: int      # gradient-accumulation mini-batch
    max_count: int      # multiplicities uniform in [1, max_count]
    unique: bool        # reject duplicate samples (cfg 1 cannot: sector has 36 states, A16)

    @property
    def n_qubits(self) -> int:
        return 2 * self.n_spatial

    @property
    def seed_integrals(self) -> int:
        return SEED_BASE + self.cfg

    @property
    def seed_weights(self) -> int:
        return SEED_BASE + self.cfg + 100

    @property
    def seed_samples(self) -> int:
        return SEED_BASE + self.cfg + 200


WORKLOADS = {
    1: Workload(1, 4, 2, 2, 32, 256, 256, 16, False),
    2: Workload(2, 10, 5, 5, 128, 4096, 4096, 64, True),
    3: Workload(3, 15, 7, 7, 256, 16384, 16384, 256, True),
    4: Workload(4, 26, 10, 10, 512, 32768, 8192, 512, True),
    5: Workload(5, 38, 15, 15, 512, 65536, 8192, 1024, True),
}
